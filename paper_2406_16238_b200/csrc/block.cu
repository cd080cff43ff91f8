// block.cu - what sits between walker steps in a block ("population control,
// and estimator calculation"; local population control on one GPU, PAPER.md:489;
// estimator sums of Code Snippet 9):
//
//   comb_kernel       population control by the comb (reading S21): one uniform xi per
//                     call; new walker k copies the old walker whose cumulative-weight interval
//                     holds the tooth (k + xi) W / Nw; all new weights W / Nw.
//   gather kernels    walkers / overlaps permuted by the comb's map (HBM streaming, 16-byte lanes)
//   estimator_kernel  (ENumer, EDenom, E1Body, E2Body) = sum w (Re E0, 1, Re E1, Re E2)
//
// Floating point decides integers in the comb, so its arithmetic is fixed to the last bit:
// sequential left-to-right running sum, one division, one add + one multiply per tooth with no
// FMA contraction (__dadd_rn / __dmul_rn), comparison c_j <= tooth.
#include "internal.h"

namespace afq {

namespace {

// One CTA.  cum[nw] is scratch in global memory.
__global__ void __launch_bounds__(256) comb_kernel(double* weights, const double* xi_p, double* cum, int* map,
                                                   int nw) {
  __shared__ int s_last;
  __shared__ int s_ok;
  __shared__ double s_spacing;
  if (threadIdx.x == 0) {
    double s = 0.0;
    for (int i = 0; i < nw; ++i) {
      s = __dadd_rn(s, weights[i]);
      cum[i] = s;
    }
    const double total = s;
    const int ok = isfinite(total) && total > 0.0;
    int last = 0;
    if (ok)
      while (cum[last] != total) ++last;
    s_ok = ok;
    s_last = last;
    s_spacing = __ddiv_rn(total, (double)nw);
  }
  __syncthreads();
  if (!s_ok) {                       // nothing to resample: identity, weights untouched
    for (int k = threadIdx.x; k < nw; k += blockDim.x) map[k] = k;
    return;
  }
  // xi is the caller's uniform in [0, 1); a device-resident value cannot be rejected by the host-side check,
  // so it is clamped here (NaN -> 0): a tooth can then never leave its own interval of the comb
  double xi = *xi_p;
  xi = xi >= 0.0 ? (xi < 1.0 ? xi : 0x1.fffffffffffffp-1) : 0.0;
  const double spacing = s_spacing;
  const int last = s_last;
  for (int k = threadIdx.x; k < nw; k += blockDim.x) {
    const double tooth = __dmul_rn(__dadd_rn((double)k, xi), spacing);
    // #{j : cum[j] <= tooth}, cum non-decreasing: upper bound by bisection
    int lo = 0, hi = nw;
    while (lo < hi) {
      const int mid = (lo + hi) >> 1;
      if (cum[mid] <= tooth) lo = mid + 1; else hi = mid;
    }
    map[k] = lo < last ? lo : last;
    weights[k] = spacing;            // cum[] holds what the weights were
  }
}

// dst[k][:] = src[map[k]][:], rows of n16 16-byte words; grid (chunks, nw)
__global__ void __launch_bounds__(256) gather_rows_kernel(uint4* dst, const uint4* src, const int* map, long n16) {
  const int k = blockIdx.y;
  const uint4* s = src + (size_t)map[k] * n16;
  uint4* d = dst + (size_t)k * n16;
  for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < n16; i += (long)gridDim.x * blockDim.x) d[i] = s[i];
}

// rows that moved are copied back; rows with map[k] == k never left
__global__ void __launch_bounds__(256) scatter_moved_kernel(uint4* dst, const uint4* src, const int* map, long n16) {
  const int k = blockIdx.y;
  if (map[k] == k) return;
  const uint4* s = src + (size_t)k * n16;
  uint4* d = dst + (size_t)k * n16;
  for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < n16; i += (long)gridDim.x * blockDim.x) d[i] = s[i];
}

__global__ void estimator_kernel(const double* weights, const double* E, double* out4, int nw) {
  __shared__ double red[8 * 4];
  double v[4] = {0.0, 0.0, 0.0, 0.0};
  for (int w = threadIdx.x; w < nw; w += blockDim.x) {
    const double wt = weights[w];
    v[0] += wt * E[6 * w + 0];
    v[1] += wt;
    v[2] += wt * E[6 * w + 2];
    v[3] += wt * E[6 * w + 4];
  }
#pragma unroll
  for (int k = 0; k < 4; ++k)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v[k] += __shfl_down_sync(0xffffffffu, v[k], o);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (lane == 0)
    for (int k = 0; k < 4; ++k) red[warp * 4 + k] = v[k];
  __syncthreads();
  if (threadIdx.x < 4) {
    double s = 0.0;
    for (int w = 0; w < (int)(blockDim.x >> 5); ++w) s += red[w * 4 + threadIdx.x];
    out4[threadIdx.x] = s;
  }
}

}  // namespace

int run_comb(double* weights, const double* xi, double* cum, int* map, int nw, cudaStream_t st) {
  comb_kernel<<<1, 256, 0, st>>>(weights, xi, cum, map, nw);
  return 1;
}

// walkers (row_bytes per walker, multiple of 16) permuted in place through `tmp`
int run_permute_rows(void* rows, void* tmp, const int* map, long row_bytes, int nw, cudaStream_t st) {
  const long n16 = row_bytes / 16;
  int chunks = (int)((n16 + 256 * 8 - 1) / (256 * 8));
  if (chunks < 1) chunks = 1;
  if (chunks > 64) chunks = 64;
  gather_rows_kernel<<<dim3(chunks, nw), 256, 0, st>>>((uint4*)tmp, (const uint4*)rows, map, n16);
  scatter_moved_kernel<<<dim3(chunks, nw), 256, 0, st>>>((uint4*)rows, (const uint4*)tmp, map, n16);
  return 2;
}

int run_estimators(const double* weights, const double* E, double* out4, int nw, cudaStream_t st) {
  estimator_kernel<<<1, 256, 0, st>>>(weights, E, out4, nw);
  return 1;
}

}  // namespace afq
