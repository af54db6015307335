// rex_bucket.cu -- device-side stable categorisation of events by flavour signature and the SoA "transposition"
// (SURVEY.md 8(a) a2-a4, a10; PAPER.md:354 bucket order, :362 npos rule, :675-694 sort + transpose, :877 scatter back).
//
// rex_bucket in five small launches, all bound by HBM traffic (keys are read three times, perm written once):
//   discover : distinct keys + index of first appearance, per-block shared-memory hash table merged into a global one
//   rank     : bucket id = rank of the key's first appearance; REX_NPOS forced last
//   hist     : per (bucket, warp-chunk) counts; a warp owns a contiguous chunk of events
//   scan     : exclusive scan of the counts in (bucket-major, chunk-minor) order -> write positions, bucket offsets
//   scatter  : every warp walks its chunk in input order, 32 events at a time, ranks equal buckets inside the warp
//              with __match_any_sync and writes perm; running positions live in shared memory  => stable, bit-exact
#include "trex_ctx.h"

namespace trex {

namespace {

constexpr int TS = 1024;                       // hash slots (>= 4 x REX_MAX_BUCKETS)
constexpr uint64_t EMPTY = REX_NPOS;           // REX_NPOS never enters the table: it has its own bucket
constexpr int NBMAX = REX_MAX_BUCKETS;
constexpr int WARPS = 8;

struct BucketResult {                          // copied to pinned host memory at the end of the scan
  int64_t offsets[NBMAX + 1];
  uint64_t keys[NBMAX];
  int nb;
  int err;                                     // 1: more than REX_MAX_BUCKETS distinct keys
};

struct Table {
  unsigned long long* keys;   // [TS]
  unsigned* first;            // [TS] index of first appearance
  int* bid;                   // [TS] bucket id
  int* meta;                  // [0] ndistinct, [1] has_npos, [2] overflow, [3] nb, [4] single known class: chain finished by k_rank
  unsigned* npos_first;       // [1]
};

__device__ __forceinline__ unsigned hash_key(unsigned long long k) { return (unsigned)((k * 0x9E3779B97F4A7C15ull) >> 54); }

__global__ void k_init(Table t) {
  int i = threadIdx.x;
  t.keys[i] = EMPTY; t.first[i] = 0xFFFFFFFFu; t.bid[i] = -1;
  if (i < 8) t.meta[i] = 0;
  if (i == 0) *t.npos_first = 0xFFFFFFFFu;
}

__global__ void __launch_bounds__(256) k_discover(const unsigned long long* __restrict__ keys, long n, long per_block, Table t) {
  __shared__ unsigned long long sk[TS];
  __shared__ unsigned sf[TS];
  __shared__ unsigned s_npos;
  __shared__ int s_over;
  for (int i = threadIdx.x; i < TS; i += blockDim.x) { sk[i] = EMPTY; sf[i] = 0xFFFFFFFFu; }
  if (threadIdx.x == 0) { s_npos = 0xFFFFFFFFu; s_over = 0; }
  __syncthreads();
  const long lo = (long)blockIdx.x * per_block, hi = min(n, lo + per_block);
  for (long i = lo + threadIdx.x; i < hi; i += blockDim.x) {
    const unsigned long long k = keys[i];
    if (k == EMPTY) { if ((unsigned)i < s_npos) atomicMin(&s_npos, (unsigned)i); continue; }
    unsigned h = hash_key(k);
    int slot = -1;
    for (int probe = 0; probe < TS; ++probe) {
      const unsigned s = (h + probe) & (TS - 1);
      unsigned long long cur = sk[s];
      if (cur == EMPTY) cur = atomicCAS(&sk[s], EMPTY, k);
      if (cur == EMPTY || cur == k) { slot = (int)s; break; }
    }
    if (slot < 0) { s_over = 1; continue; }
    // indices seen by one thread only grow and sf only shrinks: a stale read can only cause a redundant atomic
    if ((unsigned)i < sf[slot]) atomicMin(&sf[slot], (unsigned)i);
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    if (s_npos != 0xFFFFFFFFu) { atomicMin(t.npos_first, s_npos); t.meta[1] = 1; }
    if (s_over) t.meta[2] = 1;
  }
  for (int i = threadIdx.x; i < TS; i += blockDim.x) {
    const unsigned long long k = sk[i];
    if (k == EMPTY) continue;
    unsigned h = hash_key(k);
    int slot = -1;
    for (int probe = 0; probe < TS; ++probe) {
      const unsigned s = (h + probe) & (TS - 1);
      unsigned long long cur = t.keys[s];
      if (cur == EMPTY) { cur = atomicCAS(&t.keys[s], EMPTY, k); if (cur == EMPTY) atomicAdd(&t.meta[0], 1); }
      if (cur == EMPTY || cur == k) { slot = (int)s; break; }
    }
    if (slot < 0) { t.meta[2] = 1; continue; }
    atomicMin(&t.first[slot], sf[i]);
  }
}

// (trex_run only, npar > 0) A sample of ONE class that a compiled-in subprocess claims is reweighted in place: no
// permutation is needed, so the plan is written here and histogram, scan and scatter return at once (meta[4]).
__global__ void __launch_bounds__(TS) k_rank(Table t, BucketResult* res, long n, const unsigned long long* __restrict__ sub, int npar,
                                             DevPlan* __restrict__ plan, int force_gather) {
  __shared__ unsigned sf[NBMAX + 1];
  __shared__ int s_cnt;
  const int s = threadIdx.x;
  if (s == 0) s_cnt = 0;
  __syncthreads();
  const unsigned long long k = t.keys[s];
  const unsigned f = t.first[s];
  // the occupied slots are few (one per class): compact their first-appearance indices, then rank among those
  if (k != EMPTY) { const int j = atomicAdd(&s_cnt, 1); if (j <= NBMAX) sf[j] = f; }
  __syncthreads();
  const int nd = t.meta[0], has_npos = t.meta[1];
  const int nb = nd + has_npos;
  const bool bad = (nb > NBMAX) || t.meta[2];
  if (k != EMPTY && !bad) {
    int rank = 0;
    for (int j = 0; j < nd; ++j) rank += (sf[j] < f) ? 1 : 0;
    t.bid[s] = rank;
    res->keys[rank] = k;
  }
  if (s == 0) {
    t.meta[3] = bad ? 0 : nb;
    res->nb = bad ? 0 : nb;
    res->err = bad ? 1 : 0;
    if (!bad && has_npos) res->keys[nd] = EMPTY;
  }
  if (npar <= 0 || bad || nd != 1 || has_npos || force_gather) return;       // uniform over the block
  __shared__ unsigned long long the_key;
  __shared__ int claimed;
  if (s == 0) claimed = 0;
  if (k != EMPTY) the_key = k;
  __syncthreads();
  if (s < TREX_NSUBPROC && (int)sub[2 * s + 1] == npar && sub[2 * s] == the_key) claimed = 1;
  __syncthreads();
  if (!claimed) return;
  if (s < TREX_NSUBPROC) {
    const bool mine = (int)sub[2 * s + 1] == npar && sub[2 * s] == the_key;
    plan->off[s] = 0; plan->cnt[s] = mine ? n : 0;
  }
  if (s == 0) { plan->single = 1; plan->nb = 1; res->offsets[0] = 0; res->offsets[1] = n; t.meta[4] = 1; }
}

// shared-memory copy of the key -> bucket table for the lookups of hist / scatter
struct SmemTable {
  unsigned long long k[TS];
  int b[TS];
  __device__ void load(const Table& t) {
    for (int i = threadIdx.x; i < TS; i += blockDim.x) { k[i] = t.keys[i]; b[i] = t.bid[i]; }
  }
  __device__ __forceinline__ int lookup(unsigned long long key, int npos_bid) const {
    if (key == EMPTY) return npos_bid;
    unsigned h = hash_key(key);
    for (int probe = 0; probe < TS; ++probe) {
      const unsigned s = (h + probe) & (TS - 1);
      if (k[s] == key) return b[s];
    }
    return npos_bid;   // unreachable: every key was inserted by k_discover
  }
};

__global__ void __launch_bounds__(WARPS * 32) k_hist(const unsigned long long* __restrict__ keys, long n, long wch, long nchunks,
                                                   Table t, unsigned* __restrict__ counts) {
  __shared__ SmemTable tab;
  __shared__ unsigned hist[WARPS][NBMAX];
  const int nb = t.meta[3];
  if (nb == 0 || t.meta[4]) return;
  tab.load(t);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  for (int i = lane; i < nb; i += 32) hist[warp][i] = 0;
  __syncthreads();
  const long chunk = (long)blockIdx.x * WARPS + warp;
  if (chunk >= nchunks) return;
  const long lo = chunk * wch, hi = min(n, lo + wch);
  for (long i = lo + lane; i < hi; i += 32) atomicAdd(&hist[warp][tab.lookup(keys[i], nb - 1)], 1u);
  __syncwarp();
  for (int b = lane; b < nb; b += 32) counts[(long)b * nchunks + chunk] = hist[warp][b];
}

__global__ void __launch_bounds__(1024) k_scan(unsigned* __restrict__ counts, long nchunks, long n, Table t, BucketResult* res,
                                               const unsigned long long* __restrict__ sub, int npar, DevPlan* __restrict__ plan, int force_gather) {
  __shared__ unsigned long long part[1024];
  if (t.meta[4]) return;
  const int nb = t.meta[3];
  const long total = (long)nb * nchunks;
  const long seg = (total + 1023) / 1024;
  const long lo = min(total, (long)threadIdx.x * seg), hi = min(total, lo + seg);
  unsigned long long s = 0;
  for (long i = lo; i < hi; ++i) s += counts[i];
  part[threadIdx.x] = s;
  __syncthreads();
  // inclusive Hillis-Steele scan over the 1024 partial sums
  for (int off = 1; off < 1024; off <<= 1) {
    unsigned long long v = threadIdx.x >= off ? part[threadIdx.x - off] : 0ull;
    __syncthreads();
    part[threadIdx.x] += v;
    __syncthreads();
  }
  unsigned long long run = part[threadIdx.x] - s;
  for (long i = lo; i < hi; ++i) {
    const unsigned c = counts[i];
    counts[i] = (unsigned)run;
    if (i % nchunks == 0) res->offsets[i / nchunks] = (int64_t)run;
    run += c;
  }
  if (threadIdx.x == 0) res->offsets[nb] = nb ? n : 0;
  if (npar <= 0) return;
  // device plan of trex_run: bucket of every compiled-in subprocess (key in sub[2 sid], leg count in sub[2 sid + 1])
  __threadfence_block();
  __syncthreads();
  const int sid = threadIdx.x;
  bool found = false;
  if (sid < TREX_NSUBPROC) {
    long long off = 0, cnt = 0;
    if ((int)sub[2 * sid + 1] == npar)
      for (int b = 0; b < nb; ++b)
        if (res->keys[b] == sub[2 * sid]) { off = res->offsets[b]; cnt = res->offsets[b + 1] - off; found = true; }
    plan->off[sid] = off; plan->cnt[sid] = cnt;
  }
  const int any = __syncthreads_or(found ? 1 : 0);
  if (sid == 0) { plan->single = (nb == 1 && any && !force_gather) ? 1 : 0; plan->nb = nb; }
}

__global__ void __launch_bounds__(WARPS * 32) k_scatter(const unsigned long long* __restrict__ keys, long n, long wch, long nchunks,
                                                      Table t, const unsigned* __restrict__ base, int* __restrict__ perm, int* __restrict__ inv) {
  __shared__ SmemTable tab;
  __shared__ unsigned pos[WARPS][NBMAX];
  const int nb = t.meta[3];
  if (nb == 0 || t.meta[4]) return;
  tab.load(t);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const long chunk = (long)blockIdx.x * WARPS + warp;
  if (chunk < nchunks)
    for (int b = lane; b < nb; b += 32) pos[warp][b] = base[(long)b * nchunks + chunk];
  __syncthreads();
  if (chunk >= nchunks) return;
  const long lo = chunk * wch, hi = min(n, lo + wch);
  for (long i0 = lo; i0 < hi; i0 += 32) {
    const long i = i0 + lane;
    const bool live = i < hi;
    const unsigned active = __ballot_sync(0xFFFFFFFFu, live);
    if (live) {
      const int b = tab.lookup(keys[i], nb - 1);
      const unsigned peers = __match_any_sync(active, b);
      const unsigned rank = __popc(peers & ((1u << lane) - 1u));
      const unsigned dst = pos[warp][b] + rank;
      perm[dst] = (int)i;
      if (inv) inv[i] = (int)dst;                            // inverse permutation: coalesced, for the transposition
      __syncwarp(active);
      if (rank == 0) pos[warp][b] += __popc(peers);
    }
    __syncwarp();
  }
}

__global__ void k_gather(const double* __restrict__ src, long n_src, double* __restrict__ dst, long n_dst, int nrows,
                         const int* __restrict__ perm) {
  const long j = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= n_dst) return;
  const long p = perm[j];
  for (int r = 0; r < nrows; ++r) dst[(long)r * n_dst + j] = src[(long)r * n_src + p];
}

__global__ void k_scatter_rows(const double* __restrict__ src, long n_src, double* __restrict__ dst, long n_dst, int nrows,
                               const int* __restrict__ perm) {
  const long j = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= n_src) return;
  const long p = perm[j];
  for (int r = 0; r < nrows; ++r) dst[(long)r * n_dst + p] = src[(long)r * n_src + j];
}

// ---------------------------------------------------------------- small samples: the whole chain in ONE block
// For n <= SMALL_N the six launches above are latency, not bandwidth: one block of 1024 threads does discover -> rank ->
// per-warp histogram -> scan -> stable scatter (+ the device plan of trex_run) with block barriers in between. Same
// definitions, same result bit for bit: bucket id = rank of the key's first appearance, REX_NPOS last, a warp owns a
// contiguous chunk and ranks equal buckets with __match_any_sync.
constexpr long SMALL_N = 8192;      // beyond this one SM's load latency loses against six launches (16-bit counts: n <= 65536)
constexpr int SB_WARPS = 32;

__global__ void __launch_bounds__(1024) k_bucket_small(const unsigned long long* __restrict__ keys, long n, int* __restrict__ perm,
                                                       int* __restrict__ inv, BucketResult* __restrict__ res, const unsigned long long* __restrict__ sub,
                                                       int npar, DevPlan* __restrict__ plan, int force_gather) {
  __shared__ unsigned long long sk[TS];
  __shared__ unsigned sf[TS];
  __shared__ int sb[TS];
  __shared__ unsigned short cnt[SB_WARPS][NBMAX + 1];     // per (warp, bucket) counts, then write cursors relative to the bucket
  __shared__ unsigned s_npos;
  __shared__ int s_over, s_nd;
  __shared__ int slots[NBMAX + 1];
  __shared__ long long boff[NBMAX + 2];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  sk[tid] = EMPTY; sf[tid] = 0xFFFFFFFFu; sb[tid] = -1;
  if (tid == 0) { s_npos = 0xFFFFFFFFu; s_over = 0; s_nd = 0; }
  __syncthreads();
  // discover
  for (long i = tid; i < n; i += 1024) {
    const unsigned long long k = keys[i];
    if (k == EMPTY) { if ((unsigned)i < s_npos) atomicMin(&s_npos, (unsigned)i); continue; }
    const unsigned h = hash_key(k);
    int slot = -1;
    for (int probe = 0; probe < TS; ++probe) {
      const unsigned s = (h + probe) & (TS - 1);
      unsigned long long cur = sk[s];
      if (cur == EMPTY) cur = atomicCAS(&sk[s], EMPTY, k);
      if (cur == EMPTY || cur == k) { slot = (int)s; break; }
    }
    if (slot < 0) { s_over = 1; continue; }
    if ((unsigned)i < sf[slot]) atomicMin(&sf[slot], (unsigned)i);
  }
  __syncthreads();
  // rank: compact the occupied slots, rank them by first appearance
  if (sk[tid] != EMPTY) { const int j = atomicAdd(&s_nd, 1); if (j <= NBMAX) slots[j] = tid; }
  __syncthreads();
  const int nd = s_nd, has_npos = s_npos != 0xFFFFFFFFu ? 1 : 0;
  const int nbr = nd + has_npos;
  const bool bad = nbr > NBMAX || s_over;
  const int nb = bad ? 0 : nbr;
  if (!bad && tid < nd) {
    const int s = slots[tid];
    int rank = 0;
    for (int j = 0; j < nd; ++j) rank += sf[slots[j]] < sf[s] ? 1 : 0;
    sb[s] = rank;
    res->keys[rank] = sk[s];
  }
  if (tid == 0) { res->nb = nb; res->err = bad ? 1 : 0; if (!bad && has_npos) res->keys[nd] = EMPTY; }
  // trex_run on a sample of ONE known class: nothing has to move (no permutation is read when plan->single is set)
  if (npar > 0 && !bad && nd == 1 && !has_npos && !force_gather) {              // uniform over the block
    const unsigned long long the_key = sk[slots[0]];
    const bool mine = tid < TREX_NSUBPROC && (int)sub[2 * tid + 1] == npar && sub[2 * tid] == the_key;
    if (__syncthreads_or(mine ? 1 : 0)) {
      if (tid < TREX_NSUBPROC) { plan->off[tid] = 0; plan->cnt[tid] = mine ? n : 0; }
      if (tid == 0) { plan->single = 1; plan->nb = 1; res->offsets[0] = 0; res->offsets[1] = n; }
      return;
    }
  }
  for (int i = lane; i <= NBMAX; i += 32) cnt[warp][i] = 0;
  __syncthreads();
  auto lookup = [&](unsigned long long key) -> int {
    if (key == EMPTY) return nb - 1;
    const unsigned h = hash_key(key);
    for (int probe = 0; probe < TS; ++probe) { const unsigned s = (h + probe) & (TS - 1); if (sk[s] == key) return sb[s]; }
    return nb - 1;
  };
  // histogram: warp w owns events [w * wch, (w + 1) * wch)
  const long wch = (n + SB_WARPS - 1) / SB_WARPS;
  const long lo = min(n, warp * wch), hi = min(n, lo + wch);
  if (nb) {
    for (long i0 = lo; i0 < hi; i0 += 32) {
      const long i = i0 + lane;
      const bool live = i < hi;
      const unsigned active = __ballot_sync(0xFFFFFFFFu, live);
      if (live) {
        const int b = lookup(keys[i]);
        const unsigned peers = __match_any_sync(active, b);
        if (lane == __ffs(peers) - 1) cnt[warp][b] += (unsigned short)__popc(peers);
      }
      __syncwarp();
    }
  }
  __syncthreads();
  // scan: bucket totals (thread b), bucket offsets (thread 0), per-warp write cursors (thread b)
  if (tid < nb) {
    unsigned run = 0;
    for (int w = 0; w < SB_WARPS; ++w) { const unsigned c = cnt[w][tid]; cnt[w][tid] = (unsigned short)run; run += c; }
    boff[tid + 1] = run;
  }
  __syncthreads();
  if (tid == 0) {
    long long run = 0;
    boff[0] = 0;
    for (int b = 0; b < nb; ++b) { const long long c = boff[b + 1]; boff[b] = run; run += c; }
    boff[nb] = nb ? n : 0;
  }
  __syncthreads();
  if (tid <= nb) res->offsets[tid] = boff[tid];
  // stable scatter
  if (nb) {
    for (long i0 = lo; i0 < hi; i0 += 32) {
      const long i = i0 + lane;
      const bool live = i < hi;
      const unsigned active = __ballot_sync(0xFFFFFFFFu, live);
      if (live) {
        const int b = lookup(keys[i]);
        const unsigned peers = __match_any_sync(active, b);
        const unsigned rank = __popc(peers & ((1u << lane) - 1u));
        const long dst = boff[b] + cnt[warp][b] + rank;
        perm[dst] = (int)i;
        if (inv) inv[i] = (int)dst;
        __syncwarp(active);
        if (rank == 0) cnt[warp][b] += (unsigned short)__popc(peers);
      }
      __syncwarp();
    }
  }
  // device plan of trex_run
  if (npar > 0) {
    bool found = false;
    if (tid < TREX_NSUBPROC) {
      long long off = 0, c = 0;
      if ((int)sub[2 * tid + 1] == npar)
        for (int b = 0; b < nd && !bad; ++b)
          if (sk[slots[b]] == sub[2 * tid]) { const int r = sb[slots[b]]; off = boff[r]; c = boff[r + 1] - off; found = true; }
      plan->off[tid] = off; plan->cnt[tid] = c;
    }
    const int any = __syncthreads_or(found ? 1 : 0);
    if (tid == 0) { plan->single = (nb == 1 && any && !force_gather) ? 1 : 0; plan->nb = nb; }
  }
}

// flavour key and leg map of every event from its PDG codes (SoA [npar][n], first n_in legs incoming). Key: rex_pack_key's
// layout. Leg map: for every position of the process string of the subprocess with that key, in order, the first not yet
// used leg on the same side with that PDG code (identical particles keep their event order); identity if nobody claims
// the event. sub: registry uploaded by ensure_plan (keys, leg counts, process strings).
__global__ void __launch_bounds__(256) k_keys(const int* __restrict__ pdg, int npar, int n_in, long n, const unsigned long long* __restrict__ sub,
                                              unsigned long long* __restrict__ keys, signed char* __restrict__ legmap) {
  const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  int ev[7], srt[7];
  bool bad = false;
  for (int l = 0; l < npar; ++l) { ev[l] = pdg[(long)l * n + i]; srt[l] = ev[l]; bad = bad || ev[l] > 127 || ev[l] < -127; }
  for (int side = 0; side < 2; ++side) {                     // insertion sort inside the initial and the final state
    const int lo = side ? n_in : 0, hi = side ? npar : n_in;
    for (int a = lo + 1; a < hi; ++a) { const int x = srt[a]; int b = a - 1; while (b >= lo && srt[b] > x) { srt[b + 1] = srt[b]; --b; } srt[b + 1] = x; }
  }
  unsigned long long key = 0;
  for (int l = 0; l < npar; ++l) { const int q = srt[l]; key |= (unsigned long long)(((q < 0 ? -q : q) & 0x7F) | (q < 0 ? 0x80 : 0)) << (8 * l); }
  key |= (unsigned long long)((n_in << 4) | (npar - n_in)) << 56;
  if (bad) key = EMPTY;
  keys[i] = key;
  if (!legmap) return;
  int sid = -1;
  for (int s = 0; s < TREX_NSUBPROC; ++s) if (sub[2 * s] == key && (int)sub[2 * s + 1] == npar) sid = s;
  unsigned used = 0;
  for (int pos = 0; pos < npar; ++pos) {
    int pick = pos;
    if (sid >= 0) {
      const int want = (int)(long long)sub[2 * TREX_NSUBPROC + 8 * sid + pos];
      const int lo = pos < n_in ? 0 : n_in, hi = pos < n_in ? n_in : npar;
      for (int l = hi - 1; l >= lo; --l) if (!((used >> l) & 1u) && ev[l] == want) pick = l;
      used |= 1u << pick;
    }
    legmap[(long)pos * n + i] = (signed char)pick;
  }
}

// flavour key under a comparator with a status filter (Alg.1 :419-444): the partons whose status the
// filter keeps -- incoming (-1) first, then final (1), then intermediate (2), each group sorted ascending by PDG code --
// one byte per parton as in rex_pack_key; byte 7 = n_other << 6 | n_in << 4 | n_out. fmask: bit 0 keeps status -1,
// bit 1 status 1, bit 2 status 2, bit 3 = no filtering at all (then any other status makes the event "no class").
__host__ __device__ inline unsigned long long filtered_key(const int* pdg, const signed char* status, int nlegs, long stride, unsigned fmask) {
  int grp[3][8];
  int cnt[3] = {0, 0, 0};
  bool bad = false;
  for (int l = 0; l < nlegs; ++l) {
    const int st = status[(long)l * stride], q = pdg[(long)l * stride];
    const int g = st == -1 ? 0 : (st == 1 ? 1 : (st == 2 ? 2 : -1));
    if (g < 0) { bad = bad || (fmask & 8u); continue; }
    if (!(fmask & 8u) && !((fmask >> g) & 1u)) continue;
    if (cnt[g] >= 7 || q > 127 || q < -127) { bad = true; continue; }
    int b = cnt[g]++;
    while (b > 0 && grp[g][b - 1] > q) { grp[g][b] = grp[g][b - 1]; --b; }      // insertion sort inside the group
    grp[g][b] = q;
  }
  if (bad || cnt[0] + cnt[1] + cnt[2] > 7 || cnt[0] > 3 || cnt[2] > 3) return REX_NPOS;
  unsigned long long key = 0;
  int pos = 0;
  for (int g = 0; g < 3; ++g)
    for (int i = 0; i < cnt[g]; ++i) {
      const int q = grp[g][i];
      key |= (unsigned long long)(((q < 0 ? -q : q) & 0x7F) | (q < 0 ? 0x80 : 0)) << (8 * pos++);
    }
  return key | (unsigned long long)((cnt[2] << 6) | (cnt[0] << 4) | cnt[1]) << 56;
}

__global__ void __launch_bounds__(256) k_keys_filtered(const int* __restrict__ pdg, const signed char* __restrict__ status, int nlegs, long n,
                                                       unsigned fmask, unsigned long long* __restrict__ keys) {
  const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  keys[i] = filtered_key(pdg + i, status + i, nlegs, n, fmask);
}

// momenta rows + weights into bucketed order; result rows cleared (classes nobody claims keep zero weights).
// A thread owns one event of the INPUT order and sends it to position inv[i]: the reads are fully coalesced and the
// 8-byte writes of neighbouring events of a class land in the same 32-byte sectors while those are still in L2, so the
// transposition moves its algorithmic bytes (reading at perm[j] instead fetched a whole sector per 8 bytes).
__global__ void k_run_gather(const DevPlan* __restrict__ plan, const double* __restrict__ mom, long ld, const double* __restrict__ w_in, long n,
                             int nrows, const int* __restrict__ inv, double* __restrict__ blk, double* __restrict__ res,
                             const signed char* __restrict__ legmap) {
  if (plan->single || plan->nb == 0) return;         // nb == 0: categorisation failed, perm was never written
  const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const long j = inv[i];
  if (legmap) {
    // parton re-indexing: position `leg` of the process string is played by leg legmap[leg] of the event
    for (int leg = 0; leg < nrows / 4; ++leg) {
      const int src = legmap[(long)leg * n + i];
      for (int mu = 0; mu < 4; ++mu) blk[(long)(leg * 4 + mu) * n + j] = mom[(long)(src * 4 + mu) * ld + i];
    }
  } else
  for (int r = 0; r < nrows; ++r) blk[(long)r * n + j] = mom[(long)r * ld + i];
  blk[(long)nrows * n + j] = w_in[i];
  res[i] = 0.0; res[n + i] = 0.0; res[2 * n + i] = 0.0;
}

__global__ void k_run_scatter(const DevPlan* __restrict__ plan, const double* __restrict__ res, long n, const int* __restrict__ perm,
                              double* __restrict__ w_out, double* __restrict__ me2_old, double* __restrict__ me2_new) {
  if (plan->single || plan->nb == 0) return;         // nb == 0: categorisation failed, perm was never written
  const long j = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= n) return;
  const long p = perm[j];
  w_out[p] = res[j];
  if (me2_old) me2_old[p] = res[n + j];
  if (me2_new) me2_new[p] = res[2 * n + j];
}

size_t align_up(size_t x) { return (x + 255) & ~size_t(255); }

}  // namespace

}  // namespace trex

using namespace trex;

namespace {
struct BucketLayout {
  long wch, nchunks;
  size_t off_keys, off_first, off_bid, off_meta, off_npos, off_res, off_counts, total;
};
BucketLayout bucket_layout(int64_t n) {
  BucketLayout L;
  // a warp owns `wch` consecutive events; at most 4096 chunks so that the single-block scan stays short
  // (small samples: short chunks, so that the launches still cover the machine)
  L.wch = 64;
  while (L.wch < 1024 && (n + L.wch - 1) / L.wch > 2368) L.wch *= 2;
  while ((n + L.wch - 1) / L.wch > 4096) L.wch *= 2;
  L.nchunks = (n + L.wch - 1) / L.wch;
  L.off_keys = 0; L.off_first = align_up(L.off_keys + TS * 8); L.off_bid = align_up(L.off_first + TS * 4);
  L.off_meta = align_up(L.off_bid + TS * 4); L.off_npos = align_up(L.off_meta + 32); L.off_res = align_up(L.off_npos + 4);
  L.off_counts = align_up(L.off_res + sizeof(BucketResult));
  L.total = align_up(L.off_counts + (size_t)NBMAX * L.nchunks * 4);
  return L;
}
}  // namespace

int trex::bucket_reserve(int64_t n) {
  Context& c = ctx();
  const BucketLayout L = bucket_layout(n);
  if (c.bucket_scratch_bytes < L.total) {
    c.exec_valid = false;                             // a captured trex_run graph holds the old address
    if (c.bucket_scratch) cudaFree(c.bucket_scratch);
    c.bucket_scratch = nullptr; c.bucket_scratch_bytes = 0;
    TREX_CUDA_CHECK(cudaMalloc(&c.bucket_scratch, L.total));
    c.bucket_scratch_bytes = L.total;
  }
  if (!c.bucket_host) TREX_CUDA_CHECK(cudaMallocHost(&c.bucket_host, sizeof(BucketResult)));
  return 0;
}

int trex::bucket_enqueue(const uint64_t* pdg_keys, int64_t n, int32_t* perm, int npar, int32_t* inv) {
  Context& c = ctx();
  const BucketLayout L = bucket_layout(n);
  const long wch = L.wch, nchunks = L.nchunks;
  char* base = (char*)c.bucket_scratch;
  Table t{(unsigned long long*)(base + L.off_keys), (unsigned*)(base + L.off_first), (int*)(base + L.off_bid),
          (int*)(base + L.off_meta), (unsigned*)(base + L.off_npos)};
  BucketResult* res = (BucketResult*)(base + L.off_res);
  unsigned* counts = (unsigned*)(base + L.off_counts);
  const unsigned long long* keys = (const unsigned long long*)pdg_keys;

  if (n <= SMALL_N) {
    k_bucket_small<<<1, 1024, 0, c.stream>>>(keys, n, perm, inv, res, (const unsigned long long*)c.plan_keys, npar, c.plan, c.legmap ? 1 : 0);
    c.launches += 1;
    TREX_CUDA_CHECK(cudaGetLastError());
    TREX_CUDA_CHECK(cudaMemcpyAsync(c.bucket_host, res, sizeof(BucketResult), cudaMemcpyDeviceToHost, c.stream));
    return 0;
  }
  k_init<<<1, TS, 0, c.stream>>>(t);
  long per_block = 512;
  while (per_block < 8192 && (n + per_block - 1) / per_block > 592) per_block *= 2;
  const unsigned nblk = (unsigned)((n + per_block - 1) / per_block);
  k_discover<<<nblk, 256, 0, c.stream>>>(keys, n, per_block, t);
  k_rank<<<1, TS, 0, c.stream>>>(t, res, (long)n, (const unsigned long long*)c.plan_keys, npar, c.plan, c.legmap ? 1 : 0);
  const unsigned cblk = (unsigned)((nchunks + WARPS - 1) / WARPS);
  k_hist<<<cblk, WARPS * 32, 0, c.stream>>>(keys, n, wch, nchunks, t, counts);
  k_scan<<<1, 1024, 0, c.stream>>>(counts, nchunks, n, t, res, (const unsigned long long*)c.plan_keys, npar, c.plan, c.legmap ? 1 : 0);
  k_scatter<<<cblk, WARPS * 32, 0, c.stream>>>(keys, n, wch, nchunks, t, counts, perm, inv);
  c.launches += 6;
  TREX_CUDA_CHECK(cudaGetLastError());
  TREX_CUDA_CHECK(cudaMemcpyAsync(c.bucket_host, res, sizeof(BucketResult), cudaMemcpyDeviceToHost, c.stream));
  return 0;
}

int trex::bucket_finish(int64_t* offsets) {
  Context& c = ctx();
  TREX_CUDA_CHECK(cudaStreamSynchronize(c.stream));
  const BucketResult* h = (const BucketResult*)c.bucket_host;
  if (h->err) return fail(TREX_EINVAL, "rex_bucket: more than %d distinct flavour keys", REX_MAX_BUCKETS);
  for (int b = 0; b <= h->nb; ++b) offsets[b] = h->offsets[b];
  for (int b = 0; b < h->nb; ++b) c.last_keys[b] = h->keys[b];
  c.last_nbuckets = h->nb;
  return h->nb;
}

extern "C" int rex_bucket(const uint64_t* pdg_keys, int64_t n, int32_t* perm, int64_t* offsets) {
  Context& c = ctx();
  if (n < 0 || !offsets || (n > 0 && (!pdg_keys || !perm))) return fail(TREX_EINVAL, "rex_bucket: null pointer or negative n");
  if (n >= (int64_t(1) << 31)) return fail(TREX_EINVAL, "rex_bucket: n must be < 2^31 (perm is int32)");
  c.last_nbuckets = 0;
  if (n == 0) { offsets[0] = 0; return 0; }
  if (int rc = bucket_reserve(n)) return rc;
  if (int rc = bucket_enqueue(pdg_keys, n, perm, 0, nullptr)) return rc;
  return bucket_finish(offsets);
}

int trex::run_gather(const double* mom, int64_t ld, const double* w_in, int64_t n, int nrows, const int32_t* inv, double* blk, double* res) {
  Context& c = ctx();
  k_run_gather<<<(unsigned)((n + 255) / 256), 256, 0, c.stream>>>(c.plan, mom, ld, w_in, n, nrows, inv, blk, res, (const signed char*)c.legmap);
  c.launches += 1;
  TREX_CUDA_CHECK(cudaGetLastError());
  return 0;
}

int trex::run_scatter(const double* res, int64_t n, const int32_t* perm, double* w_out, double* me2_old, double* me2_new) {
  Context& c = ctx();
  k_run_scatter<<<(unsigned)((n + 255) / 256), 256, 0, c.stream>>>(c.plan, res, n, perm, w_out, me2_old, me2_new);
  c.launches += 1;
  TREX_CUDA_CHECK(cudaGetLastError());
  return 0;
}

extern "C" int rex_keys(const int32_t* pdg_soa, int npar, int n_in, int64_t n, uint64_t* keys, int8_t* legmap) {
  Context& c = ctx();
  if (n < 0 || npar < 1 || npar > 7 || n_in < 0 || n_in > npar) return fail(TREX_EINVAL, "rex_keys: bad size");
  if (n == 0) return 0;
  if (!pdg_soa || !keys) return fail(TREX_EINVAL, "rex_keys: null device pointer");
  if (int rc = ensure_plan()) return rc;
  k_keys<<<(unsigned)((n + 255) / 256), 256, 0, c.stream>>>(pdg_soa, npar, n_in, n, (const unsigned long long*)c.plan_keys,
                                                           (unsigned long long*)keys, (signed char*)legmap);
  c.launches += 1;
  TREX_CUDA_CHECK(cudaGetLastError());
  return 0;
}

static bool filter_mask(const int32_t* status_filter, int nfilter, unsigned& fmask) {
  if (nfilter < 0 || (nfilter > 0 && !status_filter)) return false;
  fmask = nfilter == 0 ? 8u : 0u;
  for (int k = 0; k < nfilter; ++k) {
    const int st = status_filter[k];
    if (st == -1) fmask |= 1u; else if (st == 1) fmask |= 2u; else if (st == 2) fmask |= 4u; else return false;
  }
  return true;
}

extern "C" uint64_t rex_pack_key_filtered(const int32_t* pdg, const int8_t* status, int nlegs, const int32_t* status_filter, int nfilter) {
  unsigned fmask = 0;
  if (!pdg || !status || nlegs < 0 || nlegs > 16 || !filter_mask(status_filter, nfilter, fmask)) return REX_NPOS;
  return filtered_key(pdg, (const signed char*)status, nlegs, 1, fmask);
}

extern "C" int rex_keys_filtered(const int32_t* pdg_soa, const int8_t* status_soa, int nlegs, int64_t n, const int32_t* status_filter,
                                 int nfilter, uint64_t* keys) {
  Context& c = ctx();
  unsigned fmask = 0;
  if (n < 0 || nlegs < 1 || nlegs > 16) return fail(TREX_EINVAL, "rex_keys_filtered: bad size (1 <= nlegs <= 16)");
  if (!filter_mask(status_filter, nfilter, fmask)) return fail(TREX_EINVAL, "rex_keys_filtered: the filter may hold the statuses -1, 1, 2");
  if (n == 0) return 0;
  if (!pdg_soa || !status_soa || !keys) return fail(TREX_EINVAL, "rex_keys_filtered: null device pointer");
  k_keys_filtered<<<(unsigned)((n + 255) / 256), 256, 0, c.stream>>>(pdg_soa, (const signed char*)status_soa, nlegs, n, fmask, (unsigned long long*)keys);
  c.launches += 1;
  TREX_CUDA_CHECK(cudaGetLastError());
  return 0;
}

extern "C" int rex_bucket_keys(uint64_t* bucket_keys) {
  Context& c = ctx();
  if (!bucket_keys) return fail(TREX_EINVAL, "rex_bucket_keys: null pointer");
  for (int b = 0; b < c.last_nbuckets; ++b) bucket_keys[b] = c.last_keys[b];
  return c.last_nbuckets;
}

extern "C" int rex_gather(const double* src, int64_t n_src, double* dst, int64_t n_dst, int nrows, const int32_t* perm) {
  Context& c = ctx();
  if (n_src < 0 || n_dst < 0 || nrows < 0) return fail(TREX_EINVAL, "rex_gather: negative size");
  if (n_dst == 0 || nrows == 0) return 0;
  if (!src || !dst || !perm) return fail(TREX_EINVAL, "rex_gather: null pointer");
  k_gather<<<(unsigned)((n_dst + 255) / 256), 256, 0, c.stream>>>(src, n_src, dst, n_dst, nrows, perm);
  c.launches += 1;
  TREX_CUDA_CHECK(cudaGetLastError());
  return 0;
}

extern "C" int rex_scatter(const double* src, int64_t n_src, double* dst, int64_t n_dst, int nrows, const int32_t* perm) {
  Context& c = ctx();
  if (n_src < 0 || n_dst < 0 || nrows < 0) return fail(TREX_EINVAL, "rex_scatter: negative size");
  if (n_src == 0 || nrows == 0) return 0;
  if (!src || !dst || !perm) return fail(TREX_EINVAL, "rex_scatter: null pointer");
  k_scatter_rows<<<(unsigned)((n_src + 255) / 256), 256, 0, c.stream>>>(src, n_src, dst, n_dst, nrows, perm);
  c.launches += 1;
  TREX_CUDA_CHECK(cudaGetLastError());
  return 0;
}

extern "C" uint64_t rex_pack_key(const int32_t* pdg, const int8_t* status, int nlegs) {
  if (!pdg || !status || nlegs < 0) return REX_NPOS;
  int ini[8], fin[8], ni = 0, nf = 0;
  for (int i = 0; i < nlegs; ++i) {
    if (status[i] != -1 && status[i] != 1) continue;
    const int a = pdg[i] < 0 ? -pdg[i] : pdg[i];
    if (a > 127 || ni + nf >= 7) return REX_NPOS;
    (status[i] == -1 ? ini[ni++] : fin[nf++]) = pdg[i];
  }
  auto sort_small = [](int* v, int m) { for (int i = 1; i < m; ++i) { int x = v[i], j = i - 1; while (j >= 0 && v[j] > x) { v[j + 1] = v[j]; --j; } v[j + 1] = x; } };
  sort_small(ini, ni); sort_small(fin, nf);
  uint64_t key = 0;
  int pos = 0;
  auto put = [&](int p) { const uint64_t b = (uint64_t)((p < 0 ? -p : p) & 0x7F) | (p < 0 ? 0x80u : 0u); key |= b << (8 * pos++); };
  for (int i = 0; i < ni; ++i) put(ini[i]);
  for (int i = 0; i < nf; ++i) put(fin[i]);
  key |= (uint64_t)((ni << 4) | nf) << 56;
  return key;
}
