/* rex_trex.h -- C ABI of the B200-native reweighting hot path (paper arxiv 2510.05100: Rex / teaRex / MadtRex).
 *
 * What the library computes (citations are PAPER.md line numbers):
 *   - rex_bucket : the stable categorisation of events into per-subprocess blocks that lhe::transpose() performs
 *                  before any reweighting (PAPER.md:354 ordering rule, :362 npos rule, :675-694 sort + transpose,
 *                  eq.(1) :691).
 *   - rex_gather / rex_scatter : the "transposition" into and out of the per-subprocess SoA blocks
 *                  (PAPER.md:100-104 process object, :877 "transpose weights from processes to events").
 *   - trex_reweight : eq.(5),  w' = w |M(p;theta_new)|^2 / |M(p;theta_old)|^2 , with the normalisation
 *                  and zero guard of procReweightor::initialise / evaluate; |M|^2 is the LO,
 *                  helicity- and colour-summed, initial-state averaged matrix element, the only
 *                  input being the momenta.
 *
 * Conventions
 *   - Every array pointer is a DEVICE pointer unless the comment says HOST. The caller owns every buffer; the library
 *     only allocates internal scratch that it caches in a process-global context (freed by trex_shutdown).
 *   - All device work is enqueued on the stream given to trex_set_stream (default: the legacy default stream).
 *     trex_reweight, rex_gather and rex_scatter are asynchronous; rex_bucket synchronises that stream before it
 *     returns because it hands bucket sizes back to the host.
 *   - Return value: >= 0 success, < 0 error code below. No C++ exception crosses this boundary; the text of the last
 *     error is available from trex_last_error().
 *   - Not thread-safe: one caller thread per process (one process per GPU).
 */
#ifndef REX_TREX_H
#define REX_TREX_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define TREX_OK                0
#define TREX_EINVAL           -1   /* null pointer, negative size, bad mode, inconsistent theta */
#define TREX_EUNKNOWN_SUBPROC -2   /* no kernel compiled in for this key / id */
#define TREX_ECUDA            -3   /* a CUDA runtime call or a kernel launch failed */
#define TREX_ENOMEM           -4   /* scratch allocation failed */

#define REX_MAX_BUCKETS 256                     /* the paper's largest sample has 65 classes */
#define REX_NPOS 0xFFFFFFFFFFFFFFFFull          /* "no class": always the last bucket */

/* theta[]: flat parameter vector replacing the SLHA `BLOCK ID VALUE` cards of PAPER.md:996-1002 */
#define TREX_NTHETA 16
enum { TREX_TH_ALPHA_S = 0, TREX_TH_ALPHA_EM = 1, TREX_TH_SIN2W = 2, TREX_TH_MZ = 3, TREX_TH_GAMMAZ = 4,
       TREX_TH_MT = 5, TREX_TH_GAMMAT = 6, TREX_TH_CTG = 7, TREX_TH_LAMBDA = 8, TREX_TH_VEV = 9 };

/* compiled-in subprocesses (particle order inside a block = order of the process string) */
enum { TREX_SP_EEMUMU = 0,   /* e- e+ > mu- mu+   (photon + Z)          */
       TREX_SP_GG_TT = 1,    /* g g > t t~                              */
       TREX_SP_GG_TTG = 2,   /* g g > t t~ g                            */
       TREX_SP_GG_TTGG = 3,  /* g g > t t~ g g                          */
       TREX_SP_GG_TTGGG = 4, /* g g > t t~ g g g                        */
       TREX_SP_UUX_TTG = 5,  /* u u~ > t t~ g                           */
       TREX_SP_DDX_TTG = 6,  /* d d~ > t t~ g                           */
       TREX_SP_UG_TTU = 7,   /* u g > t t~ u                            */
       TREX_SP_GUX_TTUX = 8, /* g u~ > t t~ u~                          */
       TREX_SP_RESERVED = 9, /* no kernel (keeps the numbering of the ids below free of gaps elsewhere)          */
       /* the same three one-light-line channels for the other massless flavours (QCD does not see the flavour; the two
        * beam orders of a channel share one flavour key and are re-indexed by trex_run_pdg)                        */
       TREX_SP_SSX_TTG = 10, TREX_SP_CCX_TTG = 11, TREX_SP_BBX_TTG = 12,                         /* q q~ > t t~ g   */
       TREX_SP_DG_TTD = 13, TREX_SP_SG_TTS = 14, TREX_SP_CG_TTC = 15, TREX_SP_BG_TTB = 16,       /* q g > t t~ q    */
       TREX_SP_GDX_TTDX = 17, TREX_SP_GSX_TTSX = 18, TREX_SP_GCX_TTCX = 19, TREX_SP_GBX_TTBX = 20, /* g q~ > t t~ q~ */
       /* one light line + TWO gluons (the multi-jet samples are dominated by such channels) */
       TREX_SP_UUX_TTGG = 21, TREX_SP_UG_TTUG = 22, TREX_SP_GUX_TTUXG = 23,   /* u u~ > t t~ g g, u g > t t~ u g, g u~ > t t~ u~ g */
       TREX_SP_DDX_TTGG = 24, TREX_SP_DG_TTDG = 25, TREX_SP_GDX_TTDXG = 26,   /* the same for d */
       TREX_SP_SSX_TTGG = 27, TREX_SP_SG_TTSG = 28, TREX_SP_GSX_TTSXG = 29,   /* s */
       TREX_SP_CCX_TTGG = 30, TREX_SP_CG_TTCG = 31, TREX_SP_GCX_TTCXG = 32,   /* c */
       TREX_SP_BBX_TTGG = 33, TREX_SP_BG_TTBG = 34, TREX_SP_GBX_TTBXG = 35,   /* b */
       TREX_NSUBPROC = 36 };

/* ---- flavour keys (PAPER.md:334 default comparator: unordered PDG codes of external legs, initial and final state
 * kept apart; Alg.1).
 * HOST helper. pdg[nlegs], status[nlegs] (-1 incoming, +1 outgoing; other statuses are ignored). Legs of each group
 * sorted ascending by PDG code; byte i = (|pdg| & 0x7F) | (pdg < 0 ? 0x80 : 0); byte 7 = (n_in << 4) | n_out.
 * At most 7 external legs; returns REX_NPOS if there are more or if |pdg| > 127. */
uint64_t rex_pack_key(const int32_t* pdg, const int8_t* status, int nlegs);

/* ---- rex_bucket: stable categorisation.
 * pdg_keys [n] device, in : packed flavour signatures.
 * perm     [n] device, out: perm[j] = original index of the j-th event in bucketed order. Buckets appear in order of
 *                           FIRST APPEARANCE of their key in the input; key REX_NPOS is forced last; inside a bucket
 *                           the input order is kept (stable). The result is unique, hence bit-exact.
 * offsets  HOST [REX_MAX_BUCKETS+1], out: bucket b occupies perm[offsets[b] .. offsets[b+1]).
 * Returns the number of buckets (0 for n == 0), TREX_EINVAL if more than REX_MAX_BUCKETS distinct keys occur.
 * Synchronises the stream. */
int rex_bucket(const uint64_t* pdg_keys, int64_t n, int32_t* perm, int64_t* offsets);

/* HOST [REX_MAX_BUCKETS] out: key of bucket b of the last rex_bucket call. Returns the bucket count. */
int rex_bucket_keys(uint64_t* bucket_keys);

/* dst[r*n_dst + j] = src[r*n_src + perm[j]], r < nrows, j < n_dst  (SoA rows: momentum components, weights).
 * perm points at the first entry of the bucket (perm + offsets[b]); n_dst = bucket size; n_src = total events. */
int rex_gather(const double* src, int64_t n_src, double* dst, int64_t n_dst, int nrows, const int32_t* perm);

/* dst[r*n_dst + perm[j]] = src[r*n_src + j], j < n_src: the inverse move. */
int rex_scatter(const double* src, int64_t n_src, double* dst, int64_t n_dst, int nrows, const int32_t* perm);

/* ---- subprocess registry (HOST) */
int trex_subproc_id(uint64_t key);     /* key -> id, TREX_EUNKNOWN_SUBPROC if none (such events get zero weights,
                                          PAPER.md:868, 1057: the caller zero-fills) */
int trex_npar(int subproc_id);         /* external legs, or TREX_EUNKNOWN_SUBPROC */
int trex_ncolor(int subproc_id);       /* colour flows summed in J^dagger C J */
int trex_nhel(int subproc_id);         /* helicity combinations summed */
/* HOST out[ncolor*ncolor], row-major: the colour matrix C used for this subprocess. Returns ncolor. */
int trex_colour_matrix(int subproc_id, double* out);

/* ---- trex_reweight (eqs.(2)-(5); :785-808)
 * momenta_soa [npar][4][n] device: index (ipar*4 + mu)*n + ievt, mu = (E,px,py,pz), GeV.
 * theta_old, theta_new HOST [TREX_NTHETA].
 * w_in [n] device; w_out [n] device = w_in * me2_new / me2_old, exactly 0 where me2_old == 0.
 * me2_old, me2_new [n] device or NULL.
 * One launch evaluates both parameter points and shares all kinematics between them. n == 0 is a no-op. */
int trex_reweight(int subproc_id, const double* momenta_soa, int64_t n, const double* theta_old,
                  const double* theta_new, const double* w_in, double* w_out, double* me2_old, double* me2_new);

/* ---- trex_run: the whole path of reweightor::run() steps 2-7 on DEVICE buffers:
 * categorise (rex_bucket), transpose momenta and weights into per-subprocess SoA blocks (rex_gather), one trex_reweight
 * launch per block, transpose the results back to the input order (rex_scatter).
 * pdg_keys [n] device; momenta_soa [npar][4][n] device in INPUT order (all events have npar legs; particle order of
 * every class = its process string); w_in, w_out [n] device; me2_old, me2_new [n] device or NULL.
 * Events whose key has no compiled-in subprocess (or REX_NPOS) get w_out = me2 = 0.
 * A sample with a single known class skips the transposition. Returns the number of buckets. Synchronises the stream
 * once (inside rex_bucket); the reweighting launches themselves are asynchronous. */
int trex_run(const uint64_t* pdg_keys, const double* momenta_soa, int64_t n, int npar, const double* theta_old,
             const double* theta_new, const double* w_in, double* w_out, double* me2_old, double* me2_new);

/* Flavour keys and parton re-indexing on the device: pdg_soa DEVICE int32 [npar][n]
 * (first n_in legs incoming, in ANY order inside the initial and inside the final state); keys DEVICE [n] out, the layout
 * of rex_pack_key (REX_NPOS for codes beyond +-127); legmap DEVICE int8 [npar][n] out or NULL: legmap[pos][i] = the leg of
 * event i that plays position pos of the process string of the compiled-in subprocess with that key -- for every
 * position, in order, the first not yet used leg on the same side with that PDG code, so identical particles keep
 * their event order; the identity for events no subprocess claims. Asynchronous on the library stream. */
int rex_keys(const int32_t* pdg_soa, int npar, int n_in, int64_t n, uint64_t* keys, int8_t* legmap);

/* Flavour keys under a comparator with a status filter (eventComparatorConfig::set_status_filter; the two
 * comparators of Alg.1): only partons whose status is in status_filter (HOST [nfilter], values out of
 * {-1, 1, 2}; nfilter == 0: no filtering) take part; two events get the same key iff those partons agree as unordered
 * (status, PDG code) collections. pdg_soa DEVICE int32 [nlegs][n], status_soa DEVICE int8 [nlegs][n], nlegs <= 16 (all
 * partons of the event record, intermediate ones included); keys DEVICE [n] out. Layout: kept partons with status -1
 * first, then status 1, then status 2, each group sorted ascending by PDG code, one byte each as in rex_pack_key; byte 7 =
 * n_intermediate << 6 | n_in << 4 | n_out -- for the filter {-1, 1} and no intermediate partons this is rex_pack_key's
 * key, for {1} the two events of Alg.1 (g g > t t~, u u~ > t t~) fall into one class. More than 7 kept partons, |pdg| >
 * 127, or (without a filter) a status outside {-1, 1, 2} give REX_NPOS. Feed the keys to rex_bucket / trex_run as usual.
 * Relative tolerances on double-valued traits are not offered: such a comparison is not an equivalence
 * relation, its classes depend on the order in which representatives are met. Asynchronous on the library stream. */
int rex_keys_filtered(const int32_t* pdg_soa, const int8_t* status_soa, int nlegs, int64_t n, const int32_t* status_filter,
                      int nfilter, uint64_t* keys);
/* HOST helper: the same key for one event (pdg, status HOST [nlegs]). */
uint64_t rex_pack_key_filtered(const int32_t* pdg, const int8_t* status, int nlegs, const int32_t* status_filter, int nfilter);

/* trex_run for events given by PDG codes in arbitrary parton order: rex_keys, then the path of trex_run with the
 * transposition re-indexing every event's legs to the process-string order. momenta_soa [npar][4][n] in the events'
 * own leg order. Same outputs and return value as trex_run. */
int trex_run_pdg(const int32_t* pdg_soa, const double* momenta_soa, int64_t n, int npar, int n_in, const double* theta_old,
                 const double* theta_new, const double* w_in, double* w_out, double* me2_old, double* me2_new);

/* Many parameter points on one categorisation ("sort once", eqs.(9)-(10); the launch loop over
 * parameter cards): rex_bucket and the transposition run ONCE, then every theta_new[k] is evaluated.
 * theta_new HOST [ntheta][TREX_NTHETA]; w_out DEVICE [ntheta][n]; me2_old DEVICE [n] or NULL (the same for every k);
 * me2_new DEVICE [ntheta][n] or NULL. Returns the number of buckets; synchronises the stream once, at the end.
 * Direct path: one reweighting pass per parameter point; row k equals what trex_run gives for (theta_old,
 * theta_new[k]) bit for bit. Polynomial path (ntheta >= 4, a QCD sample, and every theta_new[k] differs from theta_old
 * only in c_tG / Lambda / vev, i.e. in kappa): |M|^2 is exactly quadratic in kappa (one dimension-6 insertion per
 * amplitude), so |M|^2 is evaluated at kappa_old and kappa_old +- max_k |kappa_k - kappa_old| (two passes) and every
 * row is the per-event polynomial through those three values -- the cost no longer grows with ntheta beyond one
 * HBM-bound write per row; rows agree with the direct path to ~1e-13 relative. trex_set_poly_multi(0) forces the
 * direct path. */
int trex_run_multi(const uint64_t* pdg_keys, const double* momenta_soa, int64_t n, int npar, const double* theta_old,
                   const double* theta_new, int ntheta, const double* w_in, double* w_out, double* me2_old, double* me2_new);

/* trex_run with a PER-EVENT strong coupling (an LHE event carries its own alpha_s = AQCDUP at its renormalisation scale;
 * Rex exposes g_S = sqrt(4 pi alpha_S) per event through gS()): alpha_s DEVICE [n] replaces
 * theta[TREX_TH_ALPHA_S] of BOTH parameter points for that event; everything else as trex_run. With g_s factored out
 * an amplitude with nv strong vertices is g_s^nv (A0 + (kappa / g_s) A1) (one dimension-6 insertion at most), so
 *   |M(theta; alpha_s)|^2 = g_s^(2 nv) [ a + (kappa / g_s) b + (kappa / g_s)^2 d ]
 * with a, b, d free of alpha_s: they are obtained per event and parameter point from three passes of the unchanged
 * |M|^2 kernels at g_s = 1 (kappa / g_s = 0, +delta, -delta: the quadratic is exact), and one elementwise kernel applies
 * the event's g_s. Cost: three trex_run passes; when top mass and width agree at the two parameter points a, b, d are
 * common to both and two passes suffice (the two slots of a pass carry different kappa / g_s). e- e+ > mu- mu+ events do not depend on alpha_s and come out as from trex_run.
 * An event with alpha_s = 0 has |M|^2 = 0 and weight 0 (zero guard); negative or non-finite alpha_s
 * gives NaN for that event only. Returns the number of buckets. */
int trex_run_alphas(const uint64_t* pdg_keys, const double* momenta_soa, int64_t n, int npar, const double* theta_old,
                    const double* theta_new, const double* alpha_s, const double* w_in, double* w_out, double* me2_old,
                    double* me2_new);

/* The same with HOST buffers (pinned or pageable): copies keys, momenta and weights to internal device scratch on the
 * stream, runs trex_run, copies the results back and synchronises the stream before returning. */
int trex_run_host(const uint64_t* pdg_keys, const double* momenta_soa, int64_t n, int npar, const double* theta_old,
                  const double* theta_new, const double* w_in, double* w_out, double* me2_old, double* me2_new);

/* ---- reweighted cross section and propagated error:
 *   sigma' = C sum_i w'_i                                                  eq.(6)
 *   Delta sigma' = Delta sigma (1/N) sum_i w'_i / w_i + sigma std(w')      eq.(7), population standard deviation;
 *   events with w_i == 0 add nothing to the ratio sum (their w'_i is 0 by the zero guard) but count in N.
 * trex_xsec_moments reduces one shard: w_in, w_out DEVICE [n]; moments HOST [4] out = (N, sum w', sum w'/w,
 * M2 = sum (w' - mean)^2 with the shard's own mean). Two passes over the weights, fixed summation order
 * (bit-reproducible); synchronises the stream. n == 0 gives zeros.
 * trex_xsec_finish (host only) combines nparts shards (moments HOST [nparts][4], e.g. one per GPU, gathered by the
 * caller) and applies eqs.(6)-(7): out HOST [3] = (sigma', Delta sigma', fallback flag). If the propagated error is
 * infinite, NaN or not positive it is replaced by Delta sigma times whichever of sigma'/sigma, sigma/sigma' exceeds
 * one (Delta sigma itself if that ratio is unusable too) and the flag is 1. */
int trex_xsec_moments(const double* w_in, const double* w_out, int64_t n, double* moments);
int trex_xsec_finish(const double* moments, int nparts, double C, double sigma, double dsigma, double* out);

/* trex_xsec_moments for callers that must not allocate (code under CUDA-graph capture, tight serving loops, harnesses
 * that forbid cudaMalloc): the same two fixed-order passes, but
 *   - the block partials live in a file-scope `static __device__` array of 65.6 KB (8200 doubles) that every GPU
 *     loading the library holds until exit, sized for n <= TREX_XSEC_NOALLOC_MAX_EVENTS events per call (larger n is
 *     rejected with TREX_EINVAL and a message; split the shard and combine the parts with trex_xsec_finish);
 *   - moments_dev is a DEVICE buffer [4] of the caller (N, sum w', sum w'/w, M2), written on the library stream; the call
 *     is asynchronous and does not wait for the device.
 * The call performs no cudaMalloc / cudaFree / cudaMallocHost and calls no allocating library routine. Every call on a
 * device shares the one array: calls are ordered by the library stream; calls that overlap on the GPU (issued on
 * different streams via trex_set_stream without an event between them, or from several host threads) race on it.
 * Nothing in the array has to start at zero: each call overwrites what it reads. Summation order differs from
 * trex_xsec_moments in the number of blocks, so the two agree to rounding (~1e-15 relative), not bit for bit. */
#define TREX_XSEC_NOALLOC_MAX_EVENTS 16777216ll
int trex_xsec_moments_noalloc(const double* w_in, const double* w_out, int64_t n, double* moments_dev);

int trex_set_stream(void* cuda_stream);
int trex_set_precision(int mode);      /* 0 = fp64 (default), 1 = mixed (amplitudes fp64, colour sum fp32,
                                          PAPER.md:1209 fptype m), 2 = fp32 */
int trex_get_precision(void);
int trex_set_poly_multi(int on);         /* 1 (default): trex_run_multi may use its polynomial path */
/* 1 (default): kernels may use the parity symmetry of the helicity sum. QCD and the chromomagnetic operator with a real
 * coefficient conserve parity: flipping every helicity conjugates the spinor products, so |M_{-h}|^2 = |M_h|^2 as long as
 * no propagator carries a width. When Gamma_t = 0 at BOTH parameter points a kernel that honours the switch evaluates one
 * helicity configuration of every pair {h, -h} and doubles the sum (every QCD channel does; g g > t t~ g g only
 * when top mass and width also agree at the two points). With a width the symmetry is broken at the per-cent level
 * per helicity and every configuration is evaluated. 0: always evaluate every configuration. */
int trex_set_helicity_symmetry(int on);
const char* trex_last_error(void);
void trex_shutdown(void);

#ifdef __cplusplus
}
#endif
#endif /* REX_TREX_H */
