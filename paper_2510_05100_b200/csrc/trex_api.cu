// trex_api.cu -- reweighting kernels and the C ABI of include/rex_trex.h.
#include <algorithm>
#include <cstdlib>
#include <cstring>
#include <vector>

#include "trex_colour.h"
#include "trex_ctx.h"
#include "trex_host.h"
#include "trex_kernels.cuh"

namespace trex {

Context& ctx() { static Context c; return c; }

namespace {

#ifndef TREX_QQ_MINB
#define TREX_QQ_MINB 1
#endif

// One light-quark line + t t~ + gluon (q q~ -> t t~ g and crossings; trex_proc.cuh). A block is 32 consecutive events x
// 8 warps. Helicity selection on the massless light line: in the chiral basis a massless spinor has one non-zero
// 2-block (u(+), v(-): lower; u(-), v(+): upper; the bar swaps them) and gamma^mu couples upper to lower, so the
// light-line currents vanish EXACTLY unless row and column sit in different blocks: 2 light-line combinations c, hence
// 8 of the 16 helicity units (c, lambda_g, lambda_t), one per warp.
//   phase A : the 10 external wavefunctions of the event (row / column spinor of the light line for c = 0, 1; gluon
//             polarisation -/+; ubar(t) -/+; v(t~) -/+), one per warp (warps 0, 1 take two), parked in shared memory
//   phase A2: the 10 light-line currents (Jq[c]; Jq3[c][lambda_g], Jq4[c][lambda_g]: the line after radiating the gluon at
//             its row / column end), one per warp
//   phase B : warp = unit: top line (qq_close) with operands read back (lane = event: conflict-free)
// per class: legs of the light line and 1 / N_avg (0 for ids that are not quark channels)
__constant__ QLineLegs c_qlegs[TREX_NSUBPROC];
__constant__ double c_qinvnavg[TREX_NSUBPROC];

// DBG: the instantiation trex_debug_helicity_me2 launches -- the same code with the per-helicity dump compiled in
// HS (helicity symmetry, R-21; Gamma_t = 0): only the light-line combination c = 0 is evaluated (and doubled):
// four units, eight wavefunctions and five currents per event, so the block takes TWO groups of 32 events, four warps each
// (dynamic shared memory: the arrays below once per group)
constexpr int QQ_SMEM_GROUP = (20 + 80 + 80) * 32 * (int)sizeof(double);
template <class R, class RC, bool DBG = false, bool HS = false>
__global__ void __launch_bounds__(WARPS * 32, TREX_QQ_MINB) k_qq(const ReweightArgs a) {
  static_assert(WARPS == 8, "one allowed helicity unit per warp");
  constexpr int NG = HS ? 2 : 1, NWG = WARPS / NG, EPB = 32 * NG;       // groups, warps per group, events per block
  extern __shared__ __align__(16) unsigned char qq_raw[];
  const int grp = HS ? (int)(threadIdx.x >> 7) : 0;
  double (*pm)[32] = reinterpret_cast<double (*)[32]>(qq_raw + (size_t)grp * QQ_SMEM_GROUP);
  double (*wf)[8][32] = reinterpret_cast<double (*)[8][32]>(pm + 20);
  double (*cur)[8][32] = wf + 10;
  // which class this block belongs to: given by the call (trex_reweight), or found in the device plan when one launch
  // serves every quark-channel class of a run (blocks are dealt to the classes in id order, 32 events each)
  int sid = a.sid;
  long blk = blockIdx.x;
  if (a.plan && a.qfamily) {
    sid = -1;
    for (int s = 0; s < TREX_NSUBPROC; ++s) {
      if (c_qinvnavg[s] == 0.0) continue;
      const long nb = (a.plan->cnt[s] + EPB - 1) / EPB;
      if (blk < nb) { sid = s; break; }
      blk -= nb;
    }
    if (sid < 0) return;
  }
  const EvIO io = resolve_io(a, sid);
  if (blk * EPB >= io.n) return;
  const int lane = threadIdx.x & 31, warp = (int)(threadIdx.x >> 5) - grp * NWG;       // warp within its group
  const long e = blk * EPB + grp * 32 + lane;
  const long ev = e < io.n ? e : io.n - 1;
  for (int r = warp; r < 20; r += NWG) pm[r][lane] = io.mom[(long)r * io.ld + ev];
  __syncthreads();
  const QLineLegs L = c_qlegs[sid];
  const bool row_in = L.lrow < 2, col_in = L.lcol < 2, g_in = L.lg < 2;
  auto leg = [&](int l, double p[4]) {
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) p[mu] = pm[l * 4 + mu][lane];
  };
  auto put4 = [&](double (*dst)[32], const cx<double>* c4) {
#pragma unroll
    for (int i = 0; i < 4; ++i) { dst[2 * i][lane] = c4[i].re; dst[2 * i + 1][lane] = c4[i].im; }
  };
  auto get_spinor = [&](double (*src)[32]) {
    spinor<R> o;
#pragma unroll
    for (int i = 0; i < 4; ++i) o.c[i] = cx<R>(R(src[2 * i][lane]), R(src[2 * i + 1][lane]));
    return o;
  };
  auto get_vec = [&](double (*src)[32]) {
    vec4<R> o;
#pragma unroll
    for (int i = 0; i < 4; ++i) o.c[i] = cx<R>(R(src[2 * i][lane]), R(src[2 * i + 1][lane]));
    return o;
  };
  // ---- phase A (HS: the items of c = 0 only: 0, 2, 4 .. 9)
  for (int it = warp; it < (HS ? 8 : 10); it += NWG) {
    const int item = HS ? (it < 2 ? 2 * it : it + 2) : it;
    double p[4];
    if (item < 4) {
      const int c = item & 1;                               // row spinor sits in the upper block for c = 1
      const bool row_upper = c != 0, col_upper = !row_upper;
      if (item < 2) {
        leg(L.lrow, p);
        const int lam = (row_in ? !row_upper : row_upper) ? 1 : -1;     // vbar(+): lower, ubar(+): upper
        const spinor<double> w = row_in ? bar(spinor_v<double>(p, lam, true)) : bar(spinor_u<double>(p, lam, true));
        put4(wf[item], w.c);
      } else {
        leg(L.lcol, p);
        const int lam = (col_in ? !col_upper : col_upper) ? 1 : -1;     // u(+): lower, v(+): upper
        const spinor<double> x = col_in ? spinor_u<double>(p, lam, true) : spinor_v<double>(p, lam, true);
        put4(wf[item], x.c);
      }
    } else if (item < 6) {
      leg(L.lg, p);
      const vec4<double> eg = polvec<double>(p, (item & 1) ? 1 : -1, !g_in);
      put4(wf[item], eg.c);
    } else {
      leg(item < 8 ? 2 : 3, p);
      const int lam = (item & 1) ? 1 : -1;
      const spinor<double> sp = item < 8 ? bar(spinor_u<double>(p, lam, false)) : spinor_v<double>(p, lam, false);
      put4(wf[item], sp.c);
    }
  }
  __syncthreads();
  rvec4<double> Kr, Kc, Kg, Kq, Ptot, pt;
#pragma unroll
  for (int mu = 0; mu < 4; ++mu) {
    const double pr = pm[L.lrow * 4 + mu][lane], pc = pm[L.lcol * 4 + mu][lane], pg = pm[L.lg * 4 + mu][lane];
    Kr.c[mu] = row_in ? pr : -pr; Kc.c[mu] = col_in ? pc : -pc; Kg.c[mu] = g_in ? pg : -pg;
    Kq.c[mu] = Kr.c[mu] + Kc.c[mu];
    pt.c[mu] = pm[8 + mu][lane];
  }
  Ptot = radd(Kq, Kg);
  // ---- phase A2 (HS: Jq[0], Jq3[0][-/+], Jq4[0][-/+] = items 0, 2, 3, 6, 7)
  for (int it = warp; it < (HS ? 5 : 10); it += NWG) {
    const int item = HS ? (it == 0 ? 0 : (it < 3 ? it + 1 : it + 3)) : it;
    vec4<R> J;
    if (item < 2) {
      // quark-pair current  Jq = (w gamma^mu x) / Kq^2        [ (i g_s) * (-i / Kq^2) at g_s = 1 ]
      J = bilinear(get_spinor(wf[item]), get_spinor(wf[2 + item]));
      const R sc = R(1.0 / rdot(Kq, Kq));
#pragma unroll
      for (int i = 0; i < 4; ++i) J.c[i] = J.c[i] * sc;
    } else {
      const int k = item - 2, c = (k >> 1) & 1, lg = k & 1, col_end = k >> 2;
      const spinor<R> w = get_spinor(wf[c]), x = get_spinor(wf[2 + c]);
      const vec4<R> eg = get_vec(wf[4 + lg]);
      const double iP2 = 1.0 / rdot(Ptot, Ptot);
      if (!col_end) {
        // W = w (i eslash)(i qslash)/q^2, q = -(Kr + Kg)
        rvec4<double> q;
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) q.c[mu] = -(Kr.c[mu] + Kg.c[mu]);
        const spinor<R> W = row_slash(row_slash(w, eg), cast<R>(q));
        const R sc = R(-iP2 / rdot(q, q));
        J = bilinear(W, x);
#pragma unroll
        for (int i = 0; i < 4; ++i) J.c[i] = J.c[i] * sc;
      } else {
        // X = (i qslash)(i eslash) x / q^2, q = Kc + Kg
        const rvec4<double> q = radd(Kc, Kg);
        const spinor<R> X = slash_col(cast<R>(q), slash_col(eg, x));
        const R sc = R(-iP2 / rdot(q, q));
        J = bilinear(w, X);
#pragma unroll
        for (int i = 0; i < 4; ++i) J.c[i] = J.c[i] * sc;
      }
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) { cur[item][2 * i][lane] = (double)J.c[i].re; cur[item][2 * i + 1][lane] = (double)J.c[i].im; }
  }
  __syncthreads();
  // ---- phase B: unit = (lambda_g, lambda_t, light-line combination)
  const int lg = warp & 1, lt = (warp >> 1) & 1, c = HS ? 0 : (warp >> 2) & 1;
  RC acc[2];
  {
    const vec4<R> eg = get_vec(wf[4 + lg]), Jq = get_vec(cur[c]), Jq3 = get_vec(cur[2 + c * 2 + lg]), Jq4 = get_vec(cur[6 + c * 2 + lg]);
    const spinor<R> ubar_t = get_spinor(wf[6 + lt]);
    const spinor<R> vtb[2] = {get_spinor(wf[8]), get_spinor(wf[9])};
    qq_close<R, RC>(eg, Kg, Jq, Kq, Jq3, Jq4, Ptot, ubar_t, vtb, pt, a.T, acc, (DBG && !HS && a.dbg && e == 0) ? a.dbg + warp * 4 : nullptr);
  }
  // fixed-order reduction over the 8 units (the light row spinors of phase A are dead: their slots carry the partial sums)
  double (*red)[8][32] = reinterpret_cast<double (*)[8][32]>(&wf[0][0][0]);
  red[0][warp][lane] = (double)acc[0]; red[1][warp][lane] = (double)acc[1];
  __syncthreads();
  if (warp == 0 && e < io.n) {
    double s0 = 0.0, s1 = 0.0;
#pragma unroll
    for (int w = 0; w < NWG; ++w) { s0 += red[0][w][lane]; s1 += red[1][w][lane]; }
    const double hs = HS ? 2.0 : 1.0;
    const double mo = s0 * (a.T.gs2nv[0] * c_qinvnavg[sid] * hs), mn = s1 * (a.T.gs2nv[1] * c_qinvnavg[sid] * hs);
    const double norm = (mo == 0.0) ? 0.0 : 1.0 / mo;          // procReweightor::initialise
    io.w_out[e] = io.w_in[e] * norm * mn;                      // evaluate + append_wgts
    if (io.me2_old) io.me2_old[e] = mo;
    if (io.me2_new) io.me2_new[e] = mn;
  }
}

template <class R>
__global__ void __launch_bounds__(128) k_eemumu(const ReweightArgs a) {
  const EvIO io = resolve_io(a);
  const long e = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= io.n) return;
  R out[2];
  eemumu_event<R>(io.mom, io.ld, e, a.T, out);
  const double mo = (double)out[0] * a.T.pref[0], mn = (double)out[1] * a.T.pref[1];
  const double norm = (mo == 0.0) ? 0.0 : 1.0 / mo;
  io.w_out[e] = io.w_in[e] * norm * mn;
  if (io.me2_old) io.me2_old[e] = mo;
  if (io.me2_new) io.me2_new[e] = mn;
}

// Polynomial parameter points (R-4: |M|^2 is EXACTLY quadratic in kappa): from |M|^2 at kappa0 and kappa0 +- delta,
//   m(kappa0 + u delta) = m0 + u b + u^2 d,   b = (m+ - m-)/2,   d = (m+ + m-)/2 - m0,
// every further parameter point costs one fused multiply-add pair and 8-16 B of HBM traffic per event.
__global__ void __launch_bounds__(256) k_poly_weights(const double* __restrict__ w_in, const double* __restrict__ m0, const double* __restrict__ mp,
                                                      const double* __restrict__ mm, long n, int K, const double* __restrict__ u,
                                                      double* __restrict__ w_out, double* __restrict__ me2_new) {
  const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const double a = m0[i], p = mp[i], q = mm[i];
  const double b = 0.5 * (p - q), d = 0.5 * (p + q) - a;
  const double wn = (a == 0.0) ? 0.0 : w_in[i] * (1.0 / a);           // zero guard
  for (int k = 0; k < K; ++k) {
    const double uk = u[k];
    const double m = a + uk * (b + uk * d);
    w_out[(long)k * n + i] = wn * m;
    if (me2_new) me2_new[(long)k * n + i] = m;
  }
}

// diagnostic: colour-flow amplitudes of one event, one thread per full helicity index h (bit `leg` of h = helicity
// of that leg in process order)
template <int N> struct DebugSink {
  double* out; spinor<double> v; double gsN, gsN1;
  __device__ void operator()(int leaf, const spinor<double>* b0, const spinor<double>* b1) {
    cx<double> a0 = row_col(b0[0], v), a1 = row_col(b1[0], v);
    out[4 * leaf + 0] = a0.re * gsN; out[4 * leaf + 1] = a0.im * gsN;
    out[4 * leaf + 2] = a1.re * gsN1; out[4 * leaf + 3] = a1.im * gsN1;
  }
};
template <int N> __global__ void k_debug_flows(const double* mom, double mt, double mGt, double gs, double* out) {
  const int h = blockIdx.x * blockDim.x + threadIdx.x;
  if (h >= (1 << (N + 2))) return;
  DebugSink<N> sink;
  constexpr int NC = factorial(N);
  sink.out = out + (long)h * NC * 4;
  sink.gsN = pow(gs, (double)N); sink.gsN1 = pow(gs, (double)(N - 1));
  TTNG<double, N, 1, DebugSink<N>> t;
  for (int g = 0; g < N; ++g) {
    const int leg = g < 2 ? g : g + 2;
    double p[4]; load_leg<double>(mom, 1, 0, leg, p);
    const bool incoming = g < 2;
    t.eps[g] = polvec<double>(p, ((h >> leg) & 1) ? 1 : -1, !incoming);
    for (int mu = 0; mu < 4; ++mu) t.K[g].c[mu] = incoming ? p[mu] : -p[mu];
  }
  double p[4]; load_leg<double>(mom, 1, 0, 2, p);
  for (int mu = 0; mu < 4; ++mu) t.pt.c[mu] = p[mu];
  t.ubar_t = bar(spinor_u<double>(p, ((h >> 2) & 1) ? 1 : -1, false));
  double q[4]; load_leg<double>(mom, 1, 0, 3, q);
  sink.v = spinor_v<double>(q, ((h >> 3) & 1) ? 1 : -1, false);
  t.line[0].mt = mt; t.line[0].mGt = mGt;
  t.run(&sink);
}

const TtngLaunchFn kLaunch[4][3] = {
    {trex_tu_launch_n2_m0, trex_tu_launch_n2_m1, trex_tu_launch_n2_m2}, {trex_tu_launch_n3_m0, trex_tu_launch_n3_m1, trex_tu_launch_n3_m2},
    {trex_tu_launch_n4_m0, trex_tu_launch_n4_m1, trex_tu_launch_n4_m2}, {trex_tu_launch_n5_m0, trex_tu_launch_n5_m1, trex_tu_launch_n5_m2}};
const TtngUploadFn kUpload[4][3] = {
    {trex_tu_upload_n2_m0, trex_tu_upload_n2_m1, trex_tu_upload_n2_m2}, {trex_tu_upload_n3_m0, trex_tu_upload_n3_m1, trex_tu_upload_n3_m2},
    {trex_tu_upload_n4_m0, trex_tu_upload_n4_m1, trex_tu_upload_n4_m2}, {trex_tu_upload_n5_m0, trex_tu_upload_n5_m1, trex_tu_upload_n5_m2}};

#define TREX_TAB_ROW(stem) {{stem##3_m0, stem##3_m1, stem##3_m2}, {stem##4_m0, stem##4_m1, stem##4_m2}, {stem##5_m0, stem##5_m1, stem##5_m2}}
const TableLaunchFn kTableLaunch[3][3] = TREX_TAB_ROW(trex_tu_table_launch_n);
const TableMetaFn kTableMeta[3][3] = TREX_TAB_ROW(trex_tu_table_meta_n);
const TableFoldFn kTableFold[3][3] = TREX_TAB_ROW(trex_tu_table_fold_n);
const TableGeomFn kTableGeom[3][3] = TREX_TAB_ROW(trex_tu_table_geom_n);
#undef TREX_TAB_ROW

int ensure_colour() {
  Context& c = ctx();
  if (c.colour_ready) return 0;
  int dev = 0;
  TREX_CUDA_CHECK(cudaGetDevice(&dev));
  TREX_CUDA_CHECK(cudaDeviceGetAttribute(&c.nsm, cudaDevAttrMultiProcessorCount, dev));
  for (int N = 2; N <= 5; ++N) {
    std::vector<double> C = trex_colour::ttng_colour_matrix(N);
    if (N >= 3) {
      for (int m = 0; m < 3; ++m) {                     // the layout depends on the colour-sum variant of the mode
        std::vector<double> f((size_t)kTableFold[N - 3][m](C.data(), nullptr));
        kTableFold[N - 3][m](C.data(), f.data());
        TREX_CUDA_CHECK(cudaMalloc((void**)&c.Cfold[N - 3][m], sizeof(double) * f.size()));
        TREX_CUDA_CHECK(cudaMemcpy(c.Cfold[N - 3][m], f.data(), sizeof(double) * f.size(), cudaMemcpyHostToDevice));
      }
      std::vector<int> meta((size_t)kTableMeta[N - 3][0](nullptr));
      kTableMeta[N - 3][0](meta.data());
      TREX_CUDA_CHECK(cudaMalloc((void**)&c.table_meta[N - 3], sizeof(int) * meta.size()));
      TREX_CUDA_CHECK(cudaMemcpy(c.table_meta[N - 3], meta.data(), sizeof(int) * meta.size(), cudaMemcpyHostToDevice));
    }
    for (int m = 0; m < 3; ++m)
      if (kUpload[N - 2][m](C.data(), (int)C.size()) != 0) return fail(TREX_ECUDA, "colour matrix upload failed (N=%d)", N);
    if (N == 5) {
      TREX_CUDA_CHECK(cudaMalloc((void**)&c.C120, sizeof(double) * C.size()));
      TREX_CUDA_CHECK(cudaMemcpy(c.C120, C.data(), sizeof(double) * C.size(), cudaMemcpyHostToDevice));
    }
  }
  QLineLegs ql[TREX_NSUBPROC];
  double qi[TREX_NSUBPROC], qi2[TREX_NSUBPROC];
  for (int sid = 0; sid < TREX_NSUBPROC; ++sid) {
    const SubprocInfo* sp = subproc_info(sid);
    ql[sid] = sp ? sp->qlegs : QLineLegs{0, 0, 0, 0};
    qi[sid] = (sp && is_quark_channel(sid) && !is_two_gluon_quark_channel(sid)) ? 1.0 / sp->navg : 0.0;
    qi2[sid] = (sp && is_two_gluon_quark_channel(sid)) ? 1.0 / sp->navg : 0.0;
  }
  TREX_CUDA_CHECK(cudaMemcpyToSymbol(c_qlegs, ql, sizeof ql));
  TREX_CUDA_CHECK(cudaMemcpyToSymbol(c_qinvnavg, qi, sizeof qi));
  if (trex_tu_qq2_setup(ql, qi2, trex_colour::qq2_colour_matrix().data()) != 0)
    return fail(TREX_ECUDA, "upload of the two-gluon quark-channel tables failed: %s", cudaGetErrorString(cudaGetLastError()));
  c.colour_ready = true;
  return 0;
}

}  // namespace
}  // namespace trex

using namespace trex;

extern "C" int trex_subproc_id(uint64_t key) {
  for (int sid = 0; sid < TREX_NSUBPROC; ++sid) {
    const SubprocInfo* sp = subproc_info(sid);
    if (!sp) continue;
    int8_t status[7];
    for (int i = 0; i < sp->npar; ++i) status[i] = i < 2 ? -1 : 1;
    if (rex_pack_key(sp->pdg, status, sp->npar) == key) return sid;
  }
  return TREX_EUNKNOWN_SUBPROC;
}
extern "C" int trex_npar(int sid) { const SubprocInfo* sp = subproc_info(sid); return sp ? sp->npar : TREX_EUNKNOWN_SUBPROC; }
extern "C" int trex_ncolor(int sid) { const SubprocInfo* sp = subproc_info(sid); return sp ? sp->ncolor : TREX_EUNKNOWN_SUBPROC; }
extern "C" int trex_nhel(int sid) { const SubprocInfo* sp = subproc_info(sid); return sp ? sp->nhel : TREX_EUNKNOWN_SUBPROC; }

extern "C" int trex_colour_matrix(int sid, double* out) {
  const SubprocInfo* sp = subproc_info(sid);
  if (!sp) return fail(TREX_EUNKNOWN_SUBPROC, "trex_colour_matrix: unknown subprocess %d", sid);
  if (!out) return fail(TREX_EINVAL, "trex_colour_matrix: null pointer");
  if (sid == TREX_SP_EEMUMU) { out[0] = 1.0; return 1; }
  if (sid >= TREX_SP_GG_TT && sid <= TREX_SP_GG_TTGGG) {
    std::vector<double> C = trex_colour::ttng_colour_matrix(sp->npar - 2);
    std::memcpy(out, C.data(), C.size() * sizeof(double));
    return sp->ncolor;
  }
  if (is_two_gluon_quark_channel(sid)) {
    std::vector<double> C = trex_colour::qq2_colour_matrix();
    std::memcpy(out, C.data(), C.size() * sizeof(double));
    return sp->ncolor;
  }
  static const double CQ[16] = {12, 0, 4, 4, 0, 12, 4, 4, 4, 4, 12, 0, 4, 4, 0, 12};
  std::memcpy(out, CQ, sizeof CQ);
  return 4;
}

static int ensure_scratch(void** p, size_t* have, size_t need) {
  if (*have >= need) return 0;
  ctx().exec_valid = false;                           // a captured trex_run graph holds the old address
  if (*p) cudaFree(*p);
  *p = nullptr; *have = 0;
  TREX_CUDA_CHECK(cudaMalloc(p, need));
  *have = need;
  return 0;
}

// one launch: |M|^2 at theta_old and theta_new + epilogue. `a` carries the event arrays (a.io: caller's block; a.alt +
// a.plan: trex_run's bucketed scratch, ranges resolved on the device); nmax bounds the number of events of the launch
static int launch_reweight(int sid, ReweightArgs& a, long nmax, const ThetaPair& T) {
  Context& c = ctx();
  const SubprocInfo* sp = subproc_info(sid);
  if (int rc = ensure_colour()) return rc;
  a.T = T; a.sid = sid; a.q = sp->qlegs; a.C120 = c.C120; a.dbg = c.dbg_out;
  if (!a.plan || !is_quark_channel(sid)) a.qfamily = 0;
  // parity: |M_{-h}|^2 = |M_h|^2 when no propagator carries a width (R-21); the diagnostics dump every helicity
  a.hsym = (c.hel_sym && !c.dbg_out && sid != TREX_SP_EEMUMU && T.mGt[0] == 0.0 && T.mGt[1] == 0.0) ? 1 : 0;
  const unsigned grid32 = (unsigned)((nmax + 31) / 32);
  const int mode = c.precision;
  cudaEvent_t kt[2] = {nullptr, nullptr};
  if (c.ktiming) {
    for (int i = 0; i < 2; ++i) {
      if (!c.kev_pool.empty()) { kt[i] = c.kev_pool.back(); c.kev_pool.pop_back(); }
      else TREX_CUDA_CHECK(cudaEventCreate(&kt[i]));
    }
    TREX_CUDA_CHECK(cudaEventRecord(kt[0], c.stream));
  }
  if (sid == TREX_SP_EEMUMU) {
    const unsigned grid = (unsigned)((nmax + 127) / 128);
    if (mode == 2) k_eemumu<float><<<grid, 128, 0, c.stream>>>(a);
    else k_eemumu<double><<<grid, 128, 0, c.stream>>>(a);
  } else if (sid <= TREX_SP_GG_TTGGG) {
    const int N = sp->npar - 2;
    const int npass = (T.mt[0] != T.mt[1] || T.mGt[0] != T.mGt[1]) ? 2 : 1;
    if (N >= 3 && N >= c.table_min_n) {
      if (kTableLaunch[N - 3][mode](a, npass, nmax, c.table_meta[N - 3], c.Cfold[N - 3][mode], c.nsm, c.stream) != 0)
        return fail(TREX_ECUDA, "kernel launch failed: %s", cudaGetErrorString(cudaGetLastError()));
    } else if (kLaunch[N - 2][mode](a, npass, grid32, c.stream) != 0) {
      return fail(TREX_ECUDA, "kernel launch failed: %s", cudaGetErrorString(cudaGetLastError()));
    }
  } else if (is_two_gluon_quark_channel(sid)) {
    const unsigned gq = a.qfamily ? grid32 + (unsigned)TREX_NSUBPROC : grid32;
    if (trex_tu_qq2_launch(a, mode, gq, c.stream) != 0)
      return fail(TREX_ECUDA, "kernel launch failed: %s", cudaGetErrorString(cudaGetLastError()));
  } else {
    // a family launch (trex_run) serves every quark-channel class: each class rounds its events up to whole blocks
    const unsigned gq = a.qfamily ? grid32 + (unsigned)TREX_NSUBPROC : grid32;
    static bool qq_ready = false;
    if (!qq_ready) {
      TREX_CUDA_CHECK(cudaFuncSetAttribute(k_qq<double, double, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * QQ_SMEM_GROUP));
      TREX_CUDA_CHECK(cudaFuncSetAttribute(k_qq<double, float, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * QQ_SMEM_GROUP));
      TREX_CUDA_CHECK(cudaFuncSetAttribute(k_qq<float, float, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * QQ_SMEM_GROUP));
      qq_ready = true;
    }
    if (a.hsym && !a.dbg) {                                // two groups of 32 events per block
      const unsigned gh = (a.qfamily ? (grid32 + 1) / 2 + (unsigned)TREX_NSUBPROC : (grid32 + 1) / 2);
      if (mode == 0) k_qq<double, double, false, true><<<gh, WARPS * 32, 2 * QQ_SMEM_GROUP, c.stream>>>(a);
      else if (mode == 1) k_qq<double, float, false, true><<<gh, WARPS * 32, 2 * QQ_SMEM_GROUP, c.stream>>>(a);
      else k_qq<float, float, false, true><<<gh, WARPS * 32, 2 * QQ_SMEM_GROUP, c.stream>>>(a);
    } else if (mode == 0 && a.dbg) k_qq<double, double, true><<<gq, WARPS * 32, QQ_SMEM_GROUP, c.stream>>>(a);
    else if (mode == 0) k_qq<double, double><<<gq, WARPS * 32, QQ_SMEM_GROUP, c.stream>>>(a);
    else if (mode == 1) k_qq<double, float><<<gq, WARPS * 32, QQ_SMEM_GROUP, c.stream>>>(a);
    else k_qq<float, float><<<gq, WARPS * 32, QQ_SMEM_GROUP, c.stream>>>(a);
  }
  c.launches += 1;
  TREX_CUDA_CHECK(cudaGetLastError());
  if (c.ktiming) {
    TREX_CUDA_CHECK(cudaEventRecord(kt[1], c.stream));
    c.kev.push_back(kt[0]); c.kev.push_back(kt[1]);
  }
  return 0;
}

extern "C" int trex_reweight(int sid, const double* momenta_soa, int64_t n, const double* theta_old, const double* theta_new,
                             const double* w_in, double* w_out, double* me2_old, double* me2_new) {
  const SubprocInfo* sp = subproc_info(sid);
  if (!sp) return fail(TREX_EUNKNOWN_SUBPROC, "trex_reweight: unknown subprocess %d", sid);
  if (n < 0 || !theta_old || !theta_new) return fail(TREX_EINVAL, "trex_reweight: negative n or null theta");
  if (n == 0) return 0;
  if (!momenta_soa || !w_in || !w_out) return fail(TREX_EINVAL, "trex_reweight: null device pointer");
  ThetaPair T;
  if (!make_theta_pair(sid, theta_old, theta_new, T)) return fail(TREX_EINVAL, "trex_reweight: theta outside its domain");
  ReweightArgs a;
  a.io = EvIO{momenta_soa, (long)n, (long)n, w_in, w_out, me2_old, me2_new};
  a.alt = a.io; a.plan = nullptr; a.qfamily = 0;
  return launch_reweight(sid, a, n, T);
}

// key, leg count and process string of every compiled-in subprocess, for the device-side plan and rex_keys
int trex::ensure_plan() {
  Context& c = ctx();
  if (c.plan) return 0;
  unsigned long long sub[2 * TREX_NSUBPROC + 8 * TREX_NSUBPROC] = {0};
  for (int sid = 0; sid < TREX_NSUBPROC; ++sid) {
    const SubprocInfo* sp = subproc_info(sid);
    if (!sp) { sub[2 * sid] = REX_NPOS; sub[2 * sid + 1] = 0; continue; }
    int8_t status[7];
    for (int i = 0; i < sp->npar; ++i) status[i] = i < 2 ? -1 : 1;
    sub[2 * sid] = rex_pack_key(sp->pdg, status, sp->npar);
    sub[2 * sid + 1] = (unsigned long long)sp->npar;
    for (int i = 0; i < sp->npar; ++i) sub[2 * TREX_NSUBPROC + 8 * sid + i] = (unsigned long long)(long long)sp->pdg[i];
  }
  TREX_CUDA_CHECK(cudaMalloc(&c.plan_keys, sizeof sub));
  TREX_CUDA_CHECK(cudaMemcpy(c.plan_keys, sub, sizeof sub, cudaMemcpyHostToDevice));
  TREX_CUDA_CHECK(cudaMalloc((void**)&c.plan, sizeof(DevPlan)));
  return 0;
}

// The whole path on device buffers: categorise, transpose into per-subprocess blocks, reweight every block, transpose
// back. Everything is enqueued without waiting for the device: the bucket sizes stay on the device (DevPlan), every
// compiled-in subprocess with the right number of legs gets one launch sized for the whole sample whose blocks beyond its
// bucket exit at once, and a single-class sample is reweighted in place (gather / scatter return immediately). The
// host waits once, at the end, to read the number of buckets it has to return.
static int run_core(const uint64_t* pdg_keys, const double* momenta_soa, int64_t n, int64_t ld, int npar, const double* theta_old,
                    const double* theta_new, const double* w_in, double* w_out, double* me2_old, double* me2_new);

extern "C" int trex_run(const uint64_t* pdg_keys, const double* momenta_soa, int64_t n, int npar, const double* theta_old,
                        const double* theta_new, const double* w_in, double* w_out, double* me2_old, double* me2_new) {
  return run_core(pdg_keys, momenta_soa, n, n, npar, theta_old, theta_new, w_in, w_out, me2_old, me2_new);
}

// ld: row stride of momenta_soa (== n for a caller's block; trex_run_host hands in column ranges of a larger block)
static int run_core(const uint64_t* pdg_keys, const double* momenta_soa, int64_t n, int64_t ld, int npar, const double* theta_old,
                    const double* theta_new, const double* w_in, double* w_out, double* me2_old, double* me2_new) {
  Context& c = ctx();
  if (n < 0 || npar < 1 || npar > 7 || !theta_old || !theta_new) return fail(TREX_EINVAL, "trex_run: bad size or null theta");
  if (n == 0) return 0;
  if (!pdg_keys || !momenta_soa || !w_in || !w_out) return fail(TREX_EINVAL, "trex_run: null device pointer");
  if (n >= (int64_t(1) << 31)) return fail(TREX_EINVAL, "trex_run: n must be < 2^31");
  // parameter points first: nothing is enqueued if theta is unusable
  ThetaPair T[TREX_NSUBPROC];
  for (int sid = 0; sid < TREX_NSUBPROC; ++sid)
    if (npar_of_sid(sid) == npar && !make_theta_pair(sid, theta_old, theta_new, T[sid]))
      return fail(TREX_EINVAL, "trex_run: theta outside its domain");
  if (c.unit_gs)                                      // a pass of trex_run_alphas: g_s = 1, prescribed kappa / g_s per slot
    for (int sid = 0; sid < TREX_NSUBPROC; ++sid) {
      const SubprocInfo* sp = subproc_info(sid);
      if (!sp || sp->npar != npar || sid == TREX_SP_EEMUMU) continue;
      for (int k = 0; k < 2; ++k) { T[sid].kq[k] = c.unit_gs_kq[k]; T[sid].gs2nv[k] = 1.0; T[sid].pref[k] = 1.0 / sp->navg; }
    }
  if (int rc = ensure_plan()) return rc;
  if (int rc = ensure_colour()) return rc;
  const int nrows = 4 * npar;
  if (int rc = ensure_scratch(&c.run_perm, &c.run_perm_bytes, 2 * sizeof(int32_t) * (size_t)n)) return rc;
  if (int rc = ensure_scratch(&c.run_blocks, &c.run_blocks_bytes, sizeof(double) * (size_t)n * (nrows + 1 + 3))) return rc;
  if (int rc = bucket_reserve(n)) return rc;
  c.last_nbuckets = 0;

  // enqueue of the whole chain on c.stream
  auto enqueue = [&]() -> int {
    double* blk = (double*)c.run_blocks;              // [4 npar][n] momenta, [1][n] w_in  -- in bucketed order
    double* res = blk + (size_t)(nrows + 1) * n;      // [3][n]: w_out, me2_old, me2_new   -- in bucketed order
    if (int rc = bucket_enqueue(pdg_keys, n, (int32_t*)c.run_perm, npar, (int32_t*)c.run_perm + n)) return rc;
    if (int rc = run_gather(momenta_soa, ld, w_in, n, nrows, (const int32_t*)c.run_perm + n, blk, res)) return rc;
    bool quark_done = false;                          // ONE launch serves all quark-channel classes (k_qq finds the class in the plan)
    for (int sid = 0; sid < TREX_NSUBPROC; ++sid) {
      if (npar_of_sid(sid) != npar) continue;
      if (is_quark_channel(sid)) { if (quark_done) continue; quark_done = true; }
      ReweightArgs a;
      a.io = EvIO{momenta_soa, (long)n, (long)ld, w_in, w_out, me2_old, me2_new};
      a.alt = EvIO{blk, (long)n, (long)n, blk + (size_t)nrows * n, res, res + n, res + 2 * (size_t)n};
      a.plan = c.plan; a.qfamily = is_quark_channel(sid) ? 1 : 0;
      if (int rc = launch_reweight(sid, a, n, T[sid])) return rc;
    }
    return run_scatter(res, n, (const int32_t*)c.run_perm, w_out, me2_old, me2_new);
  };

  // the chain is a dozen short launches: a repeated call (same buffers, sizes, parameter points -- e.g. the next batch
  // of a streamed sample) replays it as one CUDA graph
  Context::RunKey key{};
  key.ptr[0] = pdg_keys; key.ptr[1] = momenta_soa; key.ptr[2] = w_in; key.ptr[3] = w_out; key.ptr[4] = me2_old; key.ptr[5] = me2_new;
  key.n = n; key.ld = ld; key.npar = npar; key.precision = c.precision; key.table_min_n = c.table_min_n; key.hel_sym = c.hel_sym ? 1 : 0;
  std::memcpy(key.th, theta_old, sizeof(double) * TREX_NTHETA);
  std::memcpy(key.th + TREX_NTHETA, theta_new, sizeof(double) * TREX_NTHETA);
  int64_t offsets[REX_MAX_BUCKETS + 1];
  // (not below trex_run_host: there the launches are issued while the input copies are still in flight, which hides them)
  const bool may_replay = !c.in_host_run && !c.ktiming;
  if (may_replay && c.exec_valid && std::memcmp(&key, &c.exec_key, sizeof key) == 0) {
    TREX_CUDA_CHECK(cudaGraphLaunch(c.run_exec, c.stream));
    c.launches += c.exec_launches; c.graph_replays += 1;
    return bucket_finish(offsets);
  }
  if (c.graphs_ok && std::getenv("TREX_NO_GRAPH")) c.graphs_ok = false;
  if (may_replay && c.graphs_ok && c.last_key_valid && std::memcmp(&key, &c.last_key, sizeof key) == 0) {
    if (!c.cap_stream) TREX_CUDA_CHECK(cudaStreamCreateWithFlags(&c.cap_stream, cudaStreamNonBlocking));
    cudaStream_t user = c.stream;
    const int64_t l0 = c.launches;
    cudaGraph_t graph = nullptr;
    c.stream = c.cap_stream;
    cudaError_t e1 = cudaStreamBeginCapture(c.cap_stream, cudaStreamCaptureModeThreadLocal);
    const int rc = e1 == cudaSuccess ? enqueue() : 0;
    cudaError_t e2 = e1 == cudaSuccess ? cudaStreamEndCapture(c.cap_stream, &graph) : e1;
    c.stream = user;
    const int64_t nl = c.launches - l0;
    c.launches = l0;
    cudaGraphExec_t exec = nullptr;
    if (rc == 0 && e2 == cudaSuccess && graph && cudaGraphInstantiate(&exec, graph, 0) == cudaSuccess) {
      if (c.run_exec) cudaGraphExecDestroy(c.run_exec);
      c.run_exec = exec; c.exec_key = key; c.exec_valid = true; c.exec_launches = nl;
      cudaGraphDestroy(graph);
      TREX_CUDA_CHECK(cudaGraphLaunch(c.run_exec, c.stream));
      c.launches += nl; c.graph_replays += 1;
      return bucket_finish(offsets);
    }
    if (graph) cudaGraphDestroy(graph);
    cudaGetLastError();
    c.graphs_ok = false;                              // capture not possible here: plain launches from now on
  }
  c.last_key = key; c.last_key_valid = true;
  if (int rc = enqueue()) return rc;
  return bucket_finish(offsets);
}

// |M|^2 = g_s^(2 nv) [a + x b + x^2 d], x = kappa / g_s, from its values m0, mp, mm at x = 0, +delta, -delta and g_s = 1
__global__ void __launch_bounds__(256) k_alphas_weights(const unsigned long long* __restrict__ keys, unsigned long long eemumu_key, int nv,
                                                        const double* __restrict__ alpha_s, const double* __restrict__ m /* [2][3][n] */,
                                                        int shared, long n, double xo, double xn, const double* __restrict__ w_in,
                                                        double* __restrict__ w_out, double* __restrict__ me2_old, double* __restrict__ me2_new) {
  const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  double res[2];
  const bool qcd = keys[i] != eemumu_key;
  const double gs = sqrt(4.0 * 3.14159265358979323846 * alpha_s[i]);
#pragma unroll
  for (int p = 0; p < 2; ++p) {
    // shared: top mass and width agree at the two points, so a, b, d do; rows 0, 1, 2 = x = 0 (theta_old slot), +delta
    // (theta_new slot), -delta. For e- e+ > mu- mu+ the two slots of the first pass are the two answers.
    const int r0 = shared ? 0 : 3 * p;
    const double m0 = m[(size_t)r0 * n + i], mp = m[(size_t)(r0 + 1) * n + i], mm = m[(size_t)(r0 + 2) * n + i];
    if (!qcd) { res[p] = shared ? (p == 0 ? m0 : mp) : m0; continue; }
    const double b = 0.5 * (mp - mm), d = 0.5 * (mp + mm) - m0;
    const double u = (p == 0 ? xo : xn) / gs;                 // (kappa / g_s) / delta
    double g2 = 1.0;
    for (int k = 0; k < nv; ++k) g2 *= gs * gs;
    res[p] = gs == 0.0 ? 0.0 : g2 * (m0 + u * (b + u * d));
  }
  const double norm = (res[0] == 0.0) ? 0.0 : 1.0 / res[0];   // zero guard
  w_out[i] = w_in[i] * norm * res[1];
  if (me2_old) me2_old[i] = res[0];
  if (me2_new) me2_new[i] = res[1];
}

extern "C" int trex_run_alphas(const uint64_t* pdg_keys, const double* momenta_soa, int64_t n, int npar, const double* theta_old,
                               const double* theta_new, const double* alpha_s, const double* w_in, double* w_out, double* me2_old,
                               double* me2_new) {
  Context& c = ctx();
  if (n < 0 || npar < 1 || npar > 7 || !theta_old || !theta_new) return fail(TREX_EINVAL, "trex_run_alphas: bad size or null theta");
  if (n == 0) return 0;
  if (!alpha_s || !pdg_keys || !momenta_soa || !w_in || !w_out) return fail(TREX_EINVAL, "trex_run_alphas: null device pointer");
  const auto kappa_of = [](const double* th) { return th[TREX_TH_CTG] * th[TREX_TH_VEV] / (std::sqrt(2.0) * th[TREX_TH_LAMBDA] * th[TREX_TH_LAMBDA]); };
  if (!(theta_old[TREX_TH_LAMBDA] > 0.0) || !(theta_new[TREX_TH_LAMBDA] > 0.0)) return fail(TREX_EINVAL, "trex_run_alphas: theta outside its domain");
  const double ko = kappa_of(theta_old), kn = kappa_of(theta_new);
  if (!std::isfinite(ko) || !std::isfinite(kn)) return fail(TREX_EINVAL, "trex_run_alphas: non-finite kappa");
  // support points of the quadratic in x = kappa / g_s: of the size x takes for g_s of order one
  double delta = std::fmax(std::fabs(ko), std::fabs(kn));
  if (delta == 0.0) delta = 1.0;
  if (int rc = ensure_scratch(&c.poly_tmp, &c.poly_tmp_bytes, sizeof(double) * 6 * (size_t)n)) return rc;
  double* m = (double*)c.poly_tmp;                    // [old, new][x = 0, +delta, -delta][n]
  // the passes read theta for everything but the strong coupling; alpha_s of theta must only be usable
  double tho[TREX_NTHETA], thn[TREX_NTHETA];
  std::memcpy(tho, theta_old, sizeof tho); std::memcpy(thn, theta_new, sizeof thn);
  tho[TREX_TH_ALPHA_S] = thn[TREX_TH_ALPHA_S] = 1.0;
  int rc = 0, nb = 0;
  // top mass and width equal at the two points (the usual case: only couplings move): a, b, d are common to both, and the
  // two slots of a pass can carry different x -- two passes (x = 0 | +delta, then -delta) instead of three
  const bool shared = theta_old[TREX_TH_MT] == theta_new[TREX_TH_MT] && theta_old[TREX_TH_GAMMAT] == theta_new[TREX_TH_GAMMAT];
  c.unit_gs = true; c.in_host_run = true;             // no graph replay: the key does not know about unit_gs_kq
  if (shared) {
    c.unit_gs_kq[0] = 0.0; c.unit_gs_kq[1] = delta;
    rc = run_core(pdg_keys, momenta_soa, n, n, npar, tho, thn, w_in, w_out, m, m + (size_t)n);
    if (rc >= 0) {
      nb = rc;
      c.unit_gs_kq[0] = c.unit_gs_kq[1] = -delta;
      rc = run_core(pdg_keys, momenta_soa, n, n, npar, tho, thn, w_in, w_out, m + 2 * (size_t)n, nullptr);
    }
  } else {
    for (int s = 0; s < 3 && rc >= 0; ++s) {
      c.unit_gs_kq[0] = c.unit_gs_kq[1] = s == 0 ? 0.0 : (s == 1 ? delta : -delta);
      rc = run_core(pdg_keys, momenta_soa, n, n, npar, tho, thn, w_in, w_out, m + (size_t)s * n, m + (size_t)(3 + s) * n);
      if (rc >= 0) nb = rc;
    }
  }
  c.unit_gs = false; c.in_host_run = false;
  if (rc < 0) return rc;
  const SubprocInfo* ee = subproc_info(TREX_SP_EEMUMU);
  int8_t status[4] = {-1, -1, 1, 1};
  const unsigned long long eekey = rex_pack_key(ee->pdg, status, 4);
  k_alphas_weights<<<(unsigned)((n + 255) / 256), 256, 0, c.stream>>>((const unsigned long long*)pdg_keys, eekey, npar - 2, alpha_s, m, shared ? 1 : 0, (long)n,
                                                                      ko / delta, kn / delta, w_in, w_out, me2_old, me2_new);
  c.launches += 1;
  TREX_CUDA_CHECK(cudaGetLastError());
  TREX_CUDA_CHECK(cudaStreamSynchronize(c.stream));
  return nb;
}

// The path for events that carry PDG codes in arbitrary parton order (an LHE file does not promise the order of the
// process string): flavour keys and per-event leg maps are formed on the device (rex_keys), the
// transposition re-indexes every event's legs to the representative's order on the fly.
extern "C" int trex_run_pdg(const int32_t* pdg_soa, const double* momenta_soa, int64_t n, int npar, int n_in, const double* theta_old,
                            const double* theta_new, const double* w_in, double* w_out, double* me2_old, double* me2_new) {
  Context& c = ctx();
  if (n < 0 || npar < 1 || npar > 7 || n_in < 0 || n_in > npar) return fail(TREX_EINVAL, "trex_run_pdg: bad size");
  if (n == 0) return 0;
  if (!pdg_soa) return fail(TREX_EINVAL, "trex_run_pdg: null device pointer");
  if (int rc = ensure_scratch(&c.pdg_tmp, &c.pdg_tmp_bytes, (size_t)n * (sizeof(uint64_t) + (size_t)npar))) return rc;
  uint64_t* keys = (uint64_t*)c.pdg_tmp;
  int8_t* legmap = (int8_t*)(keys + n);
  if (int rc = rex_keys(pdg_soa, npar, n_in, n, keys, legmap)) return rc;
  c.legmap = legmap; c.in_host_run = true;               // no graph replay: the chain depends on the leg maps
  const int rc = trex_run(keys, momenta_soa, n, npar, theta_old, theta_new, w_in, w_out, me2_old, me2_new);
  c.legmap = nullptr; c.in_host_run = false;
  return rc;
}

// Many parameter points on ONE categorisation (the paper's actual workload: "sort once", eqs.(9)-(10) PAPER.md:1306-1310;
// the iterator loop of PAPER.md:994-1002): bucketing and transposition run once, then every theta_new[k] gets its
// reweighting launches and its transposition back into w_out[k]. Nothing waits for the device until the end.
extern "C" int trex_run_multi(const uint64_t* pdg_keys, const double* momenta_soa, int64_t n, int npar, const double* theta_old,
                              const double* theta_new, int ntheta, const double* w_in, double* w_out, double* me2_old,
                              double* me2_new) {
  Context& c = ctx();
  if (n < 0 || npar < 1 || npar > 7 || ntheta < 0 || !theta_old || (ntheta > 0 && !theta_new))
    return fail(TREX_EINVAL, "trex_run_multi: bad size or null theta");
  if (n == 0 || ntheta == 0) return 0;
  if (!pdg_keys || !momenta_soa || !w_in || !w_out) return fail(TREX_EINVAL, "trex_run_multi: null device pointer");
  if (n >= (int64_t(1) << 31)) return fail(TREX_EINVAL, "trex_run_multi: n must be < 2^31");
  const int64_t ld = n;
  std::vector<ThetaPair> T((size_t)ntheta * TREX_NSUBPROC);
  for (int k = 0; k < ntheta; ++k)
    for (int sid = 0; sid < TREX_NSUBPROC; ++sid)
      if (npar_of_sid(sid) == npar &&
          !make_theta_pair(sid, theta_old, theta_new + (size_t)k * TREX_NTHETA, T[(size_t)k * TREX_NSUBPROC + sid]))
        return fail(TREX_EINVAL, "trex_run_multi: theta_new[%d] outside its domain", k);
  if (int rc = ensure_plan()) return rc;
  if (int rc = ensure_colour()) return rc;
  const int nrows = 4 * npar;
  if (int rc = ensure_scratch(&c.run_perm, &c.run_perm_bytes, 2 * sizeof(int32_t) * (size_t)n)) return rc;
  if (int rc = ensure_scratch(&c.run_blocks, &c.run_blocks_bytes, sizeof(double) * (size_t)n * (nrows + 1 + 3))) return rc;
  if (int rc = bucket_reserve(n)) return rc;
  c.last_nbuckets = 0;
  double* blk = (double*)c.run_blocks;
  double* res = blk + (size_t)(nrows + 1) * n;
  // Polynomial path: all parameter points differ from theta_old in kappa = c_tG v / (sqrt2 Lambda^2) only (same alpha_s,
  // top mass and width; a QCD process) -> three evaluations fix the exact quadratic, the rest is a polynomial per event.
  bool poly = ntheta >= 4 && npar >= 4 && c.poly_multi;
  const auto kappa_of = [](const double* th) { return th[TREX_TH_CTG] * th[TREX_TH_VEV] / (std::sqrt(2.0) * th[TREX_TH_LAMBDA] * th[TREX_TH_LAMBDA]); };
  const double k0 = kappa_of(theta_old);
  double delta = 0.0;
  for (int k = 0; k < ntheta && poly; ++k) {
    const double* th = theta_new + (size_t)k * TREX_NTHETA;
    for (int j = 0; j < TREX_NTHETA && poly; ++j)
      if (j != TREX_TH_CTG && j != TREX_TH_LAMBDA && j != TREX_TH_VEV && th[j] != theta_old[j]) poly = false;
    poly = poly && th[TREX_TH_LAMBDA] > 0.0;
    delta = std::fmax(delta, std::fabs(kappa_of(th) - k0));
  }
  if (poly && delta > 0.0) {
    if (int rc = ensure_scratch(&c.poly_tmp, &c.poly_tmp_bytes, sizeof(double) * (3 * (size_t)n + (size_t)ntheta))) return rc;
    double* tmp = (double*)c.poly_tmp;              // [3][n]: m(kappa0), m(kappa0 + delta), m(kappa0 - delta); then u[ntheta]
    double* du = tmp + 3 * (size_t)n;
    std::vector<double> u((size_t)ntheta);
    for (int k = 0; k < ntheta; ++k) u[k] = (kappa_of(theta_new + (size_t)k * TREX_NTHETA) - k0) / delta;
    TREX_CUDA_CHECK(cudaMemcpyAsync(du, u.data(), sizeof(double) * ntheta, cudaMemcpyHostToDevice, c.stream));
    // cudaMemcpyAsync from pageable memory returns after staging the source: u may go out of scope
    // support points kappa0 +- delta: kappa is carried into the kernel parameters directly (no round trip through c_tG,
    // which would divide by vev)
    const double gs0 = std::sqrt(4.0 * 3.14159265358979323846 * theta_old[TREX_TH_ALPHA_S]);
    if (!std::isfinite(k0) || !std::isfinite(delta)) return fail(TREX_EINVAL, "trex_run_multi: non-finite kappa");
    if (int rc = bucket_enqueue(pdg_keys, n, (int32_t*)c.run_perm, npar, (int32_t*)c.run_perm + n)) return rc;
    if (int rc = run_gather(momenta_soa, ld, w_in, n, nrows, (const int32_t*)c.run_perm + n, blk, res)) return rc;
    for (int s2 = 0; s2 < 2; ++s2) {
      double* mo_out = s2 == 0 ? tmp : nullptr;
      double* mn_out = tmp + (size_t)(1 + s2) * n;
      bool quark_done = false;
      for (int sid = 0; sid < TREX_NSUBPROC; ++sid) {
        if (npar_of_sid(sid) != npar) continue;
        if (is_quark_channel(sid)) { if (quark_done) continue; quark_done = true; }
        ThetaPair Tp;
        if (!make_theta_pair(sid, theta_old, theta_old, Tp)) return fail(TREX_EINVAL, "trex_run_multi: theta outside its domain");
        Tp.kq[1] = gs0 > 0.0 ? (k0 + (s2 == 0 ? delta : -delta)) / gs0 : 0.0;
        ReweightArgs a;
        a.io = EvIO{momenta_soa, (long)n, (long)n, w_in, w_out, mo_out, mn_out};      // w_out row 0 doubles as a dummy here
        a.alt = EvIO{blk, (long)n, (long)n, blk + (size_t)nrows * n, res, res + n, res + 2 * (size_t)n};
        a.plan = c.plan; a.qfamily = is_quark_channel(sid) ? 1 : 0;
        if (int rc = launch_reweight(sid, a, n, Tp)) return rc;
      }
      if (int rc = run_scatter(res, n, (const int32_t*)c.run_perm, w_out, mo_out, mn_out)) return rc;
    }
    k_poly_weights<<<(unsigned)((n + 255) / 256), 256, 0, c.stream>>>(w_in, tmp, tmp + n, tmp + 2 * (size_t)n, n, ntheta, du, w_out, me2_new);
    c.launches += 1;
    if (me2_old) TREX_CUDA_CHECK(cudaMemcpyAsync(me2_old, tmp, sizeof(double) * n, cudaMemcpyDeviceToDevice, c.stream));
    TREX_CUDA_CHECK(cudaGetLastError());
    int64_t offs[REX_MAX_BUCKETS + 1];
    return bucket_finish(offs);
  }
  if (int rc = bucket_enqueue(pdg_keys, n, (int32_t*)c.run_perm, npar, (int32_t*)c.run_perm + n)) return rc;
  if (int rc = run_gather(momenta_soa, ld, w_in, n, nrows, (const int32_t*)c.run_perm + n, blk, res)) return rc;
  for (int k = 0; k < ntheta; ++k) {
    double* wk = w_out + (size_t)k * n;
    double* mok = k == 0 ? me2_old : nullptr;                   // |M(theta_old)|^2 is the same for every k
    double* mnk = me2_new ? me2_new + (size_t)k * n : nullptr;
    bool quark_done = false;
    for (int sid = 0; sid < TREX_NSUBPROC; ++sid) {
      if (npar_of_sid(sid) != npar) continue;
      if (is_quark_channel(sid)) { if (quark_done) continue; quark_done = true; }
      ReweightArgs a;
      a.io = EvIO{momenta_soa, (long)n, (long)n, w_in, wk, mok, mnk};
      a.alt = EvIO{blk, (long)n, (long)n, blk + (size_t)nrows * n, res, res + n, res + 2 * (size_t)n};
      a.plan = c.plan; a.qfamily = is_quark_channel(sid) ? 1 : 0;
      if (int rc = launch_reweight(sid, a, n, T[(size_t)k * TREX_NSUBPROC + sid])) return rc;
    }
    if (int rc = run_scatter(res, n, (const int32_t*)c.run_perm, wk, mok, mnk)) return rc;
  }
  int64_t offsets[REX_MAX_BUCKETS + 1];
  return bucket_finish(offsets);
}

// the same with HOST buffers (bench.py's end-to-end figure). Events are independent, so the sample is cut into column
// ranges ("chunks") that go through the whole path one after the other on the library stream while a second stream
// copies the NEXT chunk in and the PREVIOUS chunk's weights out: the transfers hide behind the kernels. Per-event results
// do not depend on the cut; the number of buckets returned is that of the whole sample (union of the chunks' keys, in
// order of first appearance, REX_NPOS last).
extern "C" int trex_run_host(const uint64_t* pdg_keys, const double* momenta_soa, int64_t n, int npar, const double* theta_old,
                             const double* theta_new, const double* w_in, double* w_out, double* me2_old, double* me2_new) {
  Context& c = ctx();
  if (n < 0 || npar < 1 || npar > 7) return fail(TREX_EINVAL, "trex_run_host: bad size");
  if (n == 0) return 0;
  if (!pdg_keys || !momenta_soa || !w_in || !w_out) return fail(TREX_EINVAL, "trex_run_host: null pointer");
  const size_t nn = (size_t)n, rows = (size_t)4 * npar;
  if (int rc = ensure_scratch(&c.host_io, &c.host_io_bytes, 8 * nn * (1 + rows + 1 + 3))) return rc;
  if (!c.copy_stream) {
    TREX_CUDA_CHECK(cudaStreamCreateWithFlags(&c.copy_stream, cudaStreamNonBlocking));
    for (int i = 0; i < 2; ++i) TREX_CUDA_CHECK(cudaEventCreateWithFlags(&c.copy_ev[i], cudaEventDisableTiming));
  }
  uint64_t* d_keys = (uint64_t*)c.host_io;
  double* d_mom = (double*)c.host_io + nn;
  double* d_win = d_mom + rows * nn;
  double* d_out = d_win + nn;
  const int nchunk = (int)std::max<int64_t>(1, std::min<int64_t>(8, n / 65536));
  const auto lo_of = [&](int k) { return (size_t)(nn * (size_t)k / (size_t)nchunk); };
  const auto copy_in = [&](int k) -> int {
    const size_t lo = lo_of(k), w = lo_of(k + 1) - lo;
    TREX_CUDA_CHECK(cudaMemcpyAsync(d_keys + lo, pdg_keys + lo, 8 * w, cudaMemcpyHostToDevice, c.copy_stream));
    TREX_CUDA_CHECK(cudaMemcpy2DAsync(d_mom + lo, 8 * nn, momenta_soa + lo, 8 * nn, 8 * w, rows, cudaMemcpyHostToDevice, c.copy_stream));
    TREX_CUDA_CHECK(cudaMemcpyAsync(d_win + lo, w_in + lo, 8 * w, cudaMemcpyHostToDevice, c.copy_stream));
    TREX_CUDA_CHECK(cudaEventRecord(c.copy_ev[k & 1], c.copy_stream));
    return 0;
  };
  // the caller's earlier work on the library stream comes first
  TREX_CUDA_CHECK(cudaEventRecord(c.copy_ev[1], c.stream));
  TREX_CUDA_CHECK(cudaStreamWaitEvent(c.copy_stream, c.copy_ev[1], 0));
  if (int rc = copy_in(0)) return rc;
  uint64_t keys_seen[REX_MAX_BUCKETS + 1];
  int nseen = 0;
  bool npos_seen = false;
  c.in_host_run = true;
  int rc = 0;
  for (int k = 0; k < nchunk && rc >= 0; ++k) {
    const size_t lo = lo_of(k), w = lo_of(k + 1) - lo;
    if (k + 1 < nchunk) { if (int r2 = copy_in(k + 1)) { rc = r2; break; } }
    if (cudaStreamWaitEvent(c.stream, c.copy_ev[k & 1], 0) != cudaSuccess) { rc = fail(TREX_ECUDA, "trex_run_host: cudaStreamWaitEvent failed"); break; }
    // run_core returns after the chunk's kernels have finished (it reads the bucket sizes back)
    rc = run_core(d_keys + lo, d_mom + lo, (int64_t)w, n, npar, theta_old, theta_new, d_win + lo, d_out + lo,
                  me2_old ? d_out + nn + lo : nullptr, me2_new ? d_out + 2 * nn + lo : nullptr);
    if (rc < 0) break;
    for (int b = 0; b < c.last_nbuckets; ++b) {
      const uint64_t key = c.last_keys[b];
      if (key == REX_NPOS) { npos_seen = true; continue; }
      bool have = false;
      for (int j = 0; j < nseen && !have; ++j) have = keys_seen[j] == key;
      if (!have && nseen <= REX_MAX_BUCKETS) keys_seen[nseen++] = key;
    }
    cudaMemcpyAsync(w_out + lo, d_out + lo, 8 * w, cudaMemcpyDeviceToHost, c.copy_stream);
    if (me2_old) cudaMemcpyAsync(me2_old + lo, d_out + nn + lo, 8 * w, cudaMemcpyDeviceToHost, c.copy_stream);
    if (me2_new) cudaMemcpyAsync(me2_new + lo, d_out + 2 * nn + lo, 8 * w, cudaMemcpyDeviceToHost, c.copy_stream);
  }
  c.in_host_run = false;
  cudaError_t e1 = cudaStreamSynchronize(c.copy_stream), e2 = cudaStreamSynchronize(c.stream);
  if (rc < 0) return rc;
  TREX_CUDA_CHECK(e1); TREX_CUDA_CHECK(e2); TREX_CUDA_CHECK(cudaGetLastError());
  const int total = nseen + (npos_seen ? 1 : 0);
  if (total > REX_MAX_BUCKETS) return fail(TREX_EINVAL, "rex_bucket: more than %d distinct flavour keys", REX_MAX_BUCKETS);
  for (int j = 0; j < nseen; ++j) c.last_keys[j] = keys_seen[j];
  if (npos_seen) c.last_keys[nseen] = REX_NPOS;
  c.last_nbuckets = total;
  return total;
}

extern "C" int trex_debug_flow_amps(int sid, const double* momenta_one, const double* theta, double* out) {
  Context& c = ctx();
  const SubprocInfo* sp = subproc_info(sid);
  if (!sp || sid < TREX_SP_GG_TT || sid > TREX_SP_GG_TTGGG) return fail(TREX_EUNKNOWN_SUBPROC, "trex_debug_flow_amps: only g g > t t~ (+g..)");
  if (!momenta_one || !theta || !out) return fail(TREX_EINVAL, "trex_debug_flow_amps: null pointer");
  const int N = sp->npar - 2, nhel = sp->nhel;
  const size_t nout = (size_t)nhel * sp->ncolor * 4;
  double *d_mom = nullptr, *d_out = nullptr;
  TREX_CUDA_CHECK(cudaMalloc((void**)&d_mom, sizeof(double) * 4 * sp->npar));
  TREX_CUDA_CHECK(cudaMalloc((void**)&d_out, sizeof(double) * nout));
  TREX_CUDA_CHECK(cudaMemcpyAsync(d_mom, momenta_one, sizeof(double) * 4 * sp->npar, cudaMemcpyHostToDevice, c.stream));
  const double gs = std::sqrt(4.0 * 3.14159265358979323846 * theta[TREX_TH_ALPHA_S]);
  const double mt = theta[TREX_TH_MT], mGt = mt * theta[TREX_TH_GAMMAT];
  const unsigned grid = (unsigned)((nhel + 63) / 64);
  switch (N) {
    case 2: k_debug_flows<2><<<grid, 64, 0, c.stream>>>(d_mom, mt, mGt, gs, d_out); break;
    case 3: k_debug_flows<3><<<grid, 64, 0, c.stream>>>(d_mom, mt, mGt, gs, d_out); break;
    case 4: k_debug_flows<4><<<grid, 64, 0, c.stream>>>(d_mom, mt, mGt, gs, d_out); break;
    default: k_debug_flows<5><<<grid, 64, 0, c.stream>>>(d_mom, mt, mGt, gs, d_out); break;
  }
  c.launches += 1;
  cudaError_t e1 = cudaGetLastError();
  cudaError_t e2 = cudaMemcpyAsync(out, d_out, sizeof(double) * nout, cudaMemcpyDeviceToHost, c.stream);
  cudaError_t e3 = cudaStreamSynchronize(c.stream);
  cudaFree(d_mom); cudaFree(d_out);
  TREX_CUDA_CHECK(e1); TREX_CUDA_CHECK(e2); TREX_CUDA_CHECK(e3);
  return 0;
}

// Colour-flow amplitudes of ONE event as the PRODUCTION kernels form them (k_gg_tt, k_table<3>, k_table4w, k_table<5>):
// the kernel that trex_reweight launches copies its X tile (the operand of the colour sum) for event 0 to a scratch
// buffer; here the columns are sorted into the full helicity index h (bit `leg` of h = helicity of that leg, process
// order) and the couplings g_s^N are restored. out HOST [nhel][ncolor][2: theta_old, theta_new][re, im].
extern "C" int trex_debug_xtile(int sid, const double* momenta_one, const double* theta_old, const double* theta_new, double* out) {
  Context& c = ctx();
  const SubprocInfo* sp = subproc_info(sid);
  if (!sp || sid < TREX_SP_GG_TT || sid > TREX_SP_GG_TTGGG) return fail(TREX_EUNKNOWN_SUBPROC, "trex_debug_xtile: only g g > t t~ (+g..)");
  if (!momenta_one || !theta_old || !theta_new || !out) return fail(TREX_EINVAL, "trex_debug_xtile: null pointer");
  if (c.precision != 0) return fail(TREX_EINVAL, "trex_debug_xtile: fp64 mode only");
  ThetaPair T;
  if (!make_theta_pair(sid, theta_old, theta_new, T)) return fail(TREX_EINVAL, "trex_debug_xtile: theta outside its domain");
  const int N = sp->npar - 2, nhel = sp->nhel, nc = sp->ncolor;
  int geom[5] = {0, 1, 1, 2, 0};
  if (N >= 3) kTableGeom[N - 3][0](geom);
  const int NFIX = geom[0], NIT = geom[1], NLT = geom[2], NCOLT = geom[4];
  const size_t ndump = N == 2 ? (size_t)8 * 2 * 2 * 2 : (size_t)NIT * NLT * nc * NCOLT;
  double *d_mom = nullptr, *d_w = nullptr, *d_dbg = nullptr;
  TREX_CUDA_CHECK(cudaMalloc((void**)&d_mom, sizeof(double) * 4 * sp->npar));
  TREX_CUDA_CHECK(cudaMalloc((void**)&d_w, sizeof(double) * 4));
  TREX_CUDA_CHECK(cudaMalloc((void**)&d_dbg, sizeof(double) * 2 * ndump));
  const double one[4] = {1.0, 0.0, 0.0, 0.0};
  cudaMemcpyAsync(d_mom, momenta_one, sizeof(double) * 4 * sp->npar, cudaMemcpyHostToDevice, c.stream);
  cudaMemcpyAsync(d_w, one, sizeof one, cudaMemcpyHostToDevice, c.stream);
  cudaMemsetAsync(d_dbg, 0, sizeof(double) * 2 * ndump, c.stream);
  c.dbg_out = d_dbg;
  ReweightArgs a;
  a.io = EvIO{d_mom, 1, 1, d_w, d_w + 1, d_w + 2, d_w + 3};
  a.alt = a.io; a.plan = nullptr; a.qfamily = 0;
  const int rc = launch_reweight(sid, a, 1, T);
  c.dbg_out = nullptr;
  std::vector<double> dump(2 * ndump);
  cudaError_t e1 = cudaMemcpyAsync(dump.data(), d_dbg, sizeof(double) * 2 * ndump, cudaMemcpyDeviceToHost, c.stream);
  cudaError_t e2 = cudaStreamSynchronize(c.stream);
  cudaFree(d_mom); cudaFree(d_w); cudaFree(d_dbg);
  if (rc < 0) return rc;
  TREX_CUDA_CHECK(e1); TREX_CUDA_CHECK(e2);
  const double pi = 3.14159265358979323846;
  const double gsN[2] = {std::pow(std::sqrt(4.0 * pi * theta_old[TREX_TH_ALPHA_S]), N), std::pow(std::sqrt(4.0 * pi * theta_new[TREX_TH_ALPHA_S]), N)};
  for (int h = 0; h < nhel; ++h) {
    const int lt = (h >> 2) & 1, ltb = (h >> 3) & 1;
    unsigned gbits = 0;                                   // bit g = helicity of gluon g (legs 0, 1, 4, 5, ..)
    for (int g = 0; g < N; ++g) gbits |= (unsigned)((h >> (g < 2 ? g : g + 2)) & 1) << g;
    for (int s = 0; s < nc; ++s)
      for (int th = 0; th < 2; ++th) {
        size_t src;
        if (N == 2) src = (size_t)((((gbits * 2 + lt) * 2 + s) * 2 + ltb) * 2 + th);
        else {
          const unsigned itb = gbits & ((1u << NFIX) - 1u), hfree = gbits >> NFIX;
          const int lti = NLT == 2 ? lt : 0;
          const int col = NLT == 2 ? (int)((hfree * 2 + ltb) * 2 + th) : (int)(((hfree * 2 + lt) * 2 + ltb) * 2 + th);
          src = (((size_t)itb * NLT + lti) * nc + s) * NCOLT + col;
        }
        double* o = out + (((size_t)h * nc + s) * 2 + th) * 2;
        o[0] = dump[2 * src] * gsN[th]; o[1] = dump[2 * src + 1] * gsN[th];
      }
  }
  return 0;
}

// per-helicity |M_h|^2 of the quark-channel production kernels (k_qq, k_qq2): see include/rex_trex_diag.h
extern "C" int trex_debug_helicity_me2(int sid, const double* momenta_one, const double* theta_old, const double* theta_new, double* out) {
  Context& c = ctx();
  const SubprocInfo* sp = subproc_info(sid);
  if (!sp || !is_quark_channel(sid)) return fail(TREX_EUNKNOWN_SUBPROC, "trex_debug_helicity_me2: quark channels only");
  if (!momenta_one || !theta_old || !theta_new || !out) return fail(TREX_EINVAL, "trex_debug_helicity_me2: null pointer");
  if (c.precision != 0) return fail(TREX_EINVAL, "trex_debug_helicity_me2: fp64 mode only");
  ThetaPair T;
  if (!make_theta_pair(sid, theta_old, theta_new, T)) return fail(TREX_EINVAL, "trex_debug_helicity_me2: theta outside its domain");
  const bool two = is_two_gluon_quark_channel(sid);
  const size_t ndump = two ? 8 * 8 : 8 * 4;               // units x (lambda_t, lambda_tbar, theta) resp. (lambda_tbar, theta)
  double *d_mom = nullptr, *d_w = nullptr, *d_dbg = nullptr;
  TREX_CUDA_CHECK(cudaMalloc((void**)&d_mom, sizeof(double) * 4 * sp->npar));
  TREX_CUDA_CHECK(cudaMalloc((void**)&d_w, sizeof(double) * 4));
  TREX_CUDA_CHECK(cudaMalloc((void**)&d_dbg, sizeof(double) * ndump));
  const double one[4] = {1.0, 0.0, 0.0, 0.0};
  cudaMemcpyAsync(d_mom, momenta_one, sizeof(double) * 4 * sp->npar, cudaMemcpyHostToDevice, c.stream);
  cudaMemcpyAsync(d_w, one, sizeof one, cudaMemcpyHostToDevice, c.stream);
  cudaMemsetAsync(d_dbg, 0, sizeof(double) * ndump, c.stream);
  c.dbg_out = d_dbg;
  ReweightArgs a;
  a.io = EvIO{d_mom, 1, 1, d_w, d_w + 1, d_w + 2, d_w + 3};
  a.alt = a.io; a.plan = nullptr; a.qfamily = 0;
  const int rc = launch_reweight(sid, a, 1, T);
  c.dbg_out = nullptr;
  std::vector<double> dump(ndump);
  cudaError_t e1 = cudaMemcpyAsync(dump.data(), d_dbg, sizeof(double) * ndump, cudaMemcpyDeviceToHost, c.stream);
  cudaError_t e2 = cudaStreamSynchronize(c.stream);
  cudaFree(d_mom); cudaFree(d_w); cudaFree(d_dbg);
  if (rc < 0) return rc;
  TREX_CUDA_CHECK(e1); TREX_CUDA_CHECK(e2);
  for (int i = 0; i < 2 * sp->nhel; ++i) out[i] = 0.0;
  const QLineLegs L = sp->qlegs;
  const bool row_in = L.lrow < 2, col_in = L.lcol < 2;
  for (int u = 0; u < 8; ++u) {
    // unit -> helicities: the light-line combination c fixes both ends (see k_qq / qq2_unit)
    const int cc = two ? (u & 1) : ((u >> 2) & 1);
    const bool row_upper = cc != 0, col_upper = !row_upper;
    const int hrow = (row_in ? !row_upper : row_upper) ? 1 : 0, hcol = (col_in ? !col_upper : col_upper) ? 1 : 0;
    for (int lt = 0; lt < 2; ++lt) {
      if (!two && lt != ((u >> 1) & 1)) continue;
      for (int iv = 0; iv < 2; ++iv) {
        int h = (hrow << L.lrow) | (hcol << L.lcol) | (lt << 2) | (iv << 3);
        size_t src;
        if (two) { h |= (((u >> 1) & 1) << L.lg) | (((u >> 2) & 1) << L.lg2); src = (size_t)u * 8 + (lt * 2 + iv) * 2; }
        else { h |= ((u & 1) << L.lg); src = (size_t)u * 4 + iv * 2; }
        for (int th = 0; th < 2; ++th) out[2 * h + th] = dump[src + th] * T.gs2nv[th] / sp->navg;
      }
    }
  }
  return 0;
}

extern "C" int trex_set_stream(void* cuda_stream) { ctx().stream = (cudaStream_t)cuda_stream; return 0; }
extern "C" int trex_set_precision(int mode) {
  if (mode < 0 || mode > 2) return fail(TREX_EINVAL, "trex_set_precision: mode must be 0, 1 or 2");
  ctx().precision = mode; return 0;
}
extern "C" int trex_get_precision(void) { return ctx().precision; }
extern "C" int trex_set_poly_multi(int on) { ctx().poly_multi = on != 0; return 0; }
extern "C" int trex_set_helicity_symmetry(int on) { ctx().hel_sym = on != 0; return 0; }
extern "C" int trex_set_algorithm(int algo) {
  if (algo != 0 && (algo < 3 || algo > 5)) return fail(TREX_EINVAL, "trex_set_algorithm: algo must be 0, 3, 4 or 5");
  ctx().table_min_n = algo == 0 ? 99 : algo; return 0;
}
extern "C" int64_t trex_launch_count(void) { return ctx().launches; }
extern "C" int64_t trex_graph_replays(void) { return ctx().graph_replays; }
extern "C" int trex_kernel_timing(int on) { ctx().ktiming = on != 0; return 0; }
extern "C" int trex_kernel_time(double* total_ms, int64_t* launches) {
  Context& c = ctx();
  if (!total_ms || !launches) return fail(TREX_EINVAL, "trex_kernel_time: null pointer");
  TREX_CUDA_CHECK(cudaStreamSynchronize(c.stream));
  double sum = 0.0;
  for (size_t i = 0; i + 1 < c.kev.size(); i += 2) {
    float ms = 0.f;
    TREX_CUDA_CHECK(cudaEventElapsedTime(&ms, c.kev[i], c.kev[i + 1]));
    sum += ms;
  }
  *total_ms = sum; *launches = (int64_t)(c.kev.size() / 2);
  c.kev_pool.insert(c.kev_pool.end(), c.kev.begin(), c.kev.end());
  c.kev.clear();
  return 0;
}
extern "C" const char* trex_last_error(void) { return ctx().err; }
extern "C" void trex_shutdown(void) {
  Context& c = ctx();
  if (c.bucket_scratch) cudaFree(c.bucket_scratch);
  if (c.bucket_host) cudaFreeHost(c.bucket_host);
  if (c.C120) cudaFree(c.C120);
  for (int i = 0; i < 3; ++i) {
    for (int m = 0; m < 3; ++m) { if (c.Cfold[i][m]) cudaFree(c.Cfold[i][m]); c.Cfold[i][m] = nullptr; }
    if (c.table_meta[i]) cudaFree(c.table_meta[i]);
    c.table_meta[i] = nullptr;
  }
  if (c.run_perm) cudaFree(c.run_perm);
  if (c.run_blocks) cudaFree(c.run_blocks);
  if (c.host_io) cudaFree(c.host_io);
  if (c.probe_out) cudaFree(c.probe_out);
  if (c.pdg_tmp) cudaFree(c.pdg_tmp);
  c.pdg_tmp = nullptr; c.pdg_tmp_bytes = 0;
  if (c.poly_tmp) cudaFree(c.poly_tmp);
  c.poly_tmp = nullptr; c.poly_tmp_bytes = 0;
  if (c.xsec_scratch) cudaFree(c.xsec_scratch);
  if (c.xsec_host) cudaFreeHost(c.xsec_host);
  c.xsec_scratch = c.xsec_host = nullptr;
  for (cudaEvent_t e : c.kev) cudaEventDestroy(e);
  for (cudaEvent_t e : c.kev_pool) cudaEventDestroy(e);
  c.kev.clear(); c.kev_pool.clear();
  if (c.copy_stream) { cudaStreamDestroy(c.copy_stream); cudaEventDestroy(c.copy_ev[0]); cudaEventDestroy(c.copy_ev[1]); c.copy_stream = nullptr; }
  if (c.run_exec) cudaGraphExecDestroy(c.run_exec);
  if (c.cap_stream) cudaStreamDestroy(c.cap_stream);
  c.run_exec = nullptr; c.cap_stream = nullptr; c.exec_valid = false; c.last_key_valid = false;
  if (c.plan) cudaFree(c.plan);
  if (c.plan_keys) cudaFree(c.plan_keys);
  c.plan = nullptr; c.plan_keys = nullptr;
  c.probe_out = nullptr;
  c.run_perm = c.run_blocks = c.host_io = nullptr; c.run_perm_bytes = c.run_blocks_bytes = c.host_io_bytes = 0;
  c.bucket_scratch = nullptr; c.bucket_scratch_bytes = 0; c.bucket_host = nullptr; c.C120 = nullptr; c.colour_ready = false;
}
