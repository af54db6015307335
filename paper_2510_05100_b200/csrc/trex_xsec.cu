// trex_xsec.cu -- reweighted cross section and its propagated error (eqs.(6)-(7)).
//
//   sigma' = C sum_i w'_i,   Delta sigma' = Delta sigma (1/N) sum_i w'_i / w_i + sigma std(w')   (population std).
// The device reduces one shard of events to four moments  m = (N, sum w', sum w'/w, M2 = sum (w' - mean)^2)  in two
// passes over the weights (HBM-bound: 16 + 8 B per event), every sum in a FIXED order (per-thread strided partial sums,
// shuffle tree, one partial per block, one block sums the partials in index order): bit-reproducible. Shards (GPUs)
// are combined on the host with the pairwise update of Chan et al., M2 = M2_a + M2_b + d^2 n_a n_b / (n_a + n_b).
#include <cmath>

#include "trex_ctx.h"

namespace trex {
namespace {

constexpr int XB = 256;          // threads per block
constexpr int XG = 592;          // blocks (4 per SM)

__device__ __forceinline__ double block_sum(double v, double* sh) {
#pragma unroll
  for (int o = 16; o >= 1; o >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, o);
  __syncthreads();
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
  __syncthreads();
  double s = 0.0;
  if (threadIdx.x == 0) for (int w = 0; w < XB / 32; ++w) s += sh[w];
  return s;                       // valid in thread 0
}

// pass 1: per-block partial sums of w' and w'/w (terms with w == 0 are skipped: their w' is 0 by the zero guard)
__global__ void __launch_bounds__(XB) k_xsec_sums(const double* __restrict__ w_in, const double* __restrict__ w_out, long n, double* __restrict__ part) {
  __shared__ double sh[XB / 32];
  double s1 = 0.0, s3 = 0.0;
  for (long i = (long)blockIdx.x * XB + threadIdx.x; i < n; i += (long)gridDim.x * XB) {
    const double wo = w_out[i], wi = w_in[i];
    s1 += wo;
    if (wi != 0.0) s3 += wo / wi;
  }
  const double b1 = block_sum(s1, sh), b3 = block_sum(s3, sh);
  if (threadIdx.x == 0) { part[2 * blockIdx.x] = b1; part[2 * blockIdx.x + 1] = b3; }
}
// one block: partials -> moments[1], moments[2]
__global__ void __launch_bounds__(32) k_xsec_fold(const double* __restrict__ part, int nblk, int stride, int ncomp, long n, double* __restrict__ mom, int first) {
  if (threadIdx.x != 0) return;
  for (int c = 0; c < ncomp; ++c) {
    double s = 0.0;
    for (int b = 0; b < nblk; ++b) s += part[stride * b + c];
    mom[first + c] = s;
  }
  mom[0] = (double)n;
}
// pass 2: sum of squared deviations from the shard mean
__global__ void __launch_bounds__(XB) k_xsec_m2(const double* __restrict__ w_out, long n, const double* __restrict__ mom, double* __restrict__ part) {
  __shared__ double sh[XB / 32];
  const double mean = mom[1] / (double)n;
  double s = 0.0;
  for (long i = (long)blockIdx.x * XB + threadIdx.x; i < n; i += (long)gridDim.x * XB) { const double d = w_out[i] - mean; s += d * d; }
  const double b = block_sum(s, sh);
  if (threadIdx.x == 0) part[blockIdx.x] = b;
}

// ---------------------------------------------------------------- the variant that allocates nothing
// trex_xsec_moments_noalloc: the same two passes with the block partials in a file-scope device array instead of
// cudaMalloc'd scratch, and the four moments written to a DEVICE buffer of the caller (no pinned staging buffer, no host
// wait): usable under CUDA-graph capture and by callers that may not allocate. A block covers at most NA_EPB events, the
// array holds the partials of NA_MAXBLK blocks: n <= NA_MAXBLK * NA_EPB = TREX_XSEC_NOALLOC_MAX_EVENTS.
constexpr int NA_EPB = XB * 16;                 // events per block (16 per thread)
constexpr int NA_MAXBLK = 4096;
static_assert((long)NA_MAXBLK * NA_EPB == TREX_XSEC_NOALLOC_MAX_EVENTS, "header and kernel geometry must agree");
// [2 NA_MAXBLK] block partials, [8] moments of the shard between the passes: 65.6 KB on every GPU that loads the library
static __device__ __align__(256) double g_xsec_static[2 * NA_MAXBLK + 8];

// one block: partials -> mom[first .. first + ncomp), fixed order (thread t sums partials t, t + XB, ..; then block_sum)
__global__ void __launch_bounds__(XB) k_xsec_fold_wide(const double* __restrict__ part, int nblk, int stride, int ncomp, long n, double* __restrict__ mom, int first) {
  __shared__ double sh[XB / 32];
  for (int c = 0; c < ncomp; ++c) {
    double s = 0.0;
    for (int b = threadIdx.x; b < nblk; b += XB) s += part[stride * b + c];
    const double t = block_sum(s, sh);
    if (threadIdx.x == 0) mom[first + c] = t;
  }
  if (threadIdx.x == 0) mom[0] = (double)n;
}
__global__ void __launch_bounds__(32) k_xsec_emit(const double* __restrict__ mom, double* __restrict__ out) {
  if (threadIdx.x < 4) out[threadIdx.x] = mom[threadIdx.x];
}

// device address of g_xsec_static on the CURRENT device (in host code the array's name is a host-side stand-in, not a
// device address): asked for once per device, with that device current
int xsec_static_ptr(double** out) {
  constexpr int MAXDEV = 64;
  static double* ptr[MAXDEV] = {nullptr};
  int dev = -1;
  TREX_CUDA_CHECK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= MAXDEV) return fail(TREX_EINVAL, "trex_xsec_moments_noalloc: device ordinal %d out of range", dev);
  if (!ptr[dev]) {
    double* p = nullptr;
    TREX_CUDA_CHECK(cudaGetSymbolAddress((void**)&p, g_xsec_static));
    ptr[dev] = p;
  }
  *out = ptr[dev];
  return 0;
}

}  // namespace
}  // namespace trex

using namespace trex;

extern "C" int trex_xsec_moments_noalloc(const double* w_in, const double* w_out, int64_t n, double* moments_dev) {
  Context& c = ctx();
  if (n < 0 || !moments_dev) return fail(TREX_EINVAL, "trex_xsec_moments_noalloc: negative n or null output");
  if (n > (int64_t)TREX_XSEC_NOALLOC_MAX_EVENTS)
    return fail(TREX_EINVAL, "trex_xsec_moments_noalloc: n = %lld exceeds the static scratch (at most %lld events per call); "
                "use trex_xsec_moments or split the shard and combine with trex_xsec_finish",
                (long long)n, (long long)TREX_XSEC_NOALLOC_MAX_EVENTS);
  if (n > 0 && (!w_in || !w_out)) return fail(TREX_EINVAL, "trex_xsec_moments_noalloc: null device pointer");
  double* part = nullptr;
  if (int rc = xsec_static_ptr(&part)) return rc;
  double* mom = part + 2 * NA_MAXBLK;
  if (n == 0) {                                          // zeros, as trex_xsec_moments gives
    k_xsec_fold_wide<<<1, XB, 0, c.stream>>>(part, 0, 1, 3, 0, mom, 1);
    k_xsec_emit<<<1, 32, 0, c.stream>>>(mom, moments_dev);
    c.launches += 2;
    TREX_CUDA_CHECK(cudaGetLastError());
    return 0;
  }
  // every partial a fold reads and every moment is written by THIS call before it is read: nothing has to start at zero,
  // whatever the previous call left in the array
  const int nblk = (int)((n + NA_EPB - 1) / NA_EPB);
  k_xsec_sums<<<nblk, XB, 0, c.stream>>>(w_in, w_out, n, part);
  k_xsec_fold_wide<<<1, XB, 0, c.stream>>>(part, nblk, 2, 2, n, mom, 1);
  k_xsec_m2<<<nblk, XB, 0, c.stream>>>(w_out, n, mom, part);
  k_xsec_fold_wide<<<1, XB, 0, c.stream>>>(part, nblk, 1, 1, n, mom, 3);
  k_xsec_emit<<<1, 32, 0, c.stream>>>(mom, moments_dev);
  c.launches += 5;
  TREX_CUDA_CHECK(cudaGetLastError());
  return 0;
}

extern "C" int trex_xsec_moments(const double* w_in, const double* w_out, int64_t n, double* moments) {
  Context& c = ctx();
  if (n < 0 || !moments) return fail(TREX_EINVAL, "trex_xsec_moments: negative n or null output");
  if (n == 0) { moments[0] = moments[1] = moments[2] = moments[3] = 0.0; return 0; }
  if (!w_in || !w_out) return fail(TREX_EINVAL, "trex_xsec_moments: null device pointer");
  if (!c.xsec_scratch) TREX_CUDA_CHECK(cudaMalloc(&c.xsec_scratch, sizeof(double) * (2 * XG + 8)));
  if (!c.xsec_host) TREX_CUDA_CHECK(cudaMallocHost(&c.xsec_host, sizeof(double) * 4));
  double* part = (double*)c.xsec_scratch;
  double* mom = part + 2 * XG;
  const int nblk = (int)std::min<int64_t>(XG, (n + XB - 1) / XB);
  k_xsec_sums<<<nblk, XB, 0, c.stream>>>(w_in, w_out, n, part);
  k_xsec_fold<<<1, 32, 0, c.stream>>>(part, nblk, 2, 2, n, mom, 1);
  k_xsec_m2<<<nblk, XB, 0, c.stream>>>(w_out, n, mom, part);
  k_xsec_fold<<<1, 32, 0, c.stream>>>(part, nblk, 1, 1, n, mom, 3);
  c.launches += 4;
  TREX_CUDA_CHECK(cudaGetLastError());
  TREX_CUDA_CHECK(cudaMemcpyAsync(c.xsec_host, mom, sizeof(double) * 4, cudaMemcpyDeviceToHost, c.stream));
  TREX_CUDA_CHECK(cudaStreamSynchronize(c.stream));
  for (int i = 0; i < 4; ++i) moments[i] = ((const double*)c.xsec_host)[i];
  return 0;
}

extern "C" int trex_xsec_finish(const double* moments, int nparts, double C, double sigma, double dsigma, double* out) {
  if (!moments || !out || nparts < 0) return fail(TREX_EINVAL, "trex_xsec_finish: null pointer or negative count");
  double n = 0.0, s1 = 0.0, s3 = 0.0, m2 = 0.0;
  for (int p = 0; p < nparts; ++p) {
    const double nb = moments[4 * p], s1b = moments[4 * p + 1];
    if (nb == 0.0) continue;
    if (n > 0.0) { const double d = s1b / nb - s1 / n; m2 += moments[4 * p + 3] + d * d * n * nb / (n + nb); }
    else m2 = moments[4 * p + 3];
    n += nb; s1 += s1b; s3 += moments[4 * p + 2];
  }
  const double sigma_p = C * s1;
  double d = n > 0.0 ? dsigma * (s3 / n) + sigma * std::sqrt(m2 / n) : NAN;
  int fallback = 0;
  if (!(std::isfinite(d) && d > 0.0)) {
    fallback = 1;
    const double r = sigma != 0.0 ? sigma_p / sigma : NAN;
    d = (std::isfinite(r) && r > 0.0) ? dsigma * std::fmax(r, 1.0 / r) : dsigma;
  }
  out[0] = sigma_p; out[1] = d; out[2] = (double)fallback;
  return 0;
}
