// setup.cu - streaming kernels of afqmc_create (Eqs. 4-6, PAPER.md:63-69;
// mean-field shift PAPER.md:108).  All of them are HBM-bound passes over L.
#include "internal.h"

namespace afq {

namespace {

// m_g = sum_pq L[g][p][q] P[p][q]; one CTA per g
__global__ void __launch_bounds__(256) mean_field_kernel(const double* L, const double* P, double* m, long MM) {
  __shared__ double red[8];
  const double* Lg = L + (size_t)blockIdx.x * MM;
  double s = 0.0;
  for (long i = threadIdx.x; i < MM; i += blockDim.x) s = fma(Lg[i], P[i], s);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x == 0) {
    double tot = 0.0;
    for (int k = 0; k < 8; ++k) tot += red[k];
    m[blockIdx.x] = tot;
  }
}

// out[pq] = sum_g m[g] L[g][pq]; one thread per pq, g ascending (deterministic)
__global__ void sum_mL_kernel(const double* L, const double* m, double* out, long MM, int n_chol) {
  const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= MM) return;
  double s = 0.0;
  for (int g = 0; g < n_chol; ++g) s = fma(m[g], L[(size_t)g * MM + i], s);
  out[i] = s;
}

__global__ void hmod_kernel(const double* h1, const double* part, int nsplit, const double* mL, double* hmod, long MM) {
  const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= MM) return;
  double s = 0.0;
  for (int k = 0; k < nsplit; ++k) s += part[(size_t)k * MM + i];
  hmod[i] = h1[i] - 0.5 * s + mL[i];
}

__global__ void axpby_identity_kernel(double* P, double a, double idval, int M) {
  const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= (long)M * M) return;
  const int r = (int)(i / M), c = (int)(i % M);
  P[i] = a * P[i] + (r == c ? idval : 0.0);
}

__global__ void scale_copy_kernel(double* dst, const double* src, double a, long n) {
  const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) dst[i] = a * src[i];
}

}  // namespace

int run_mean_field(const double* L, const double* P, double* m, int M, int n_chol, cudaStream_t st) {
  mean_field_kernel<<<n_chol, 256, 0, st>>>(L, P, m, (long)M * M);
  return 1;
}
int run_sum_mL(const double* L, const double* m, double* out, int M, int n_chol, cudaStream_t st) {
  const long MM = (long)M * M;
  sum_mL_kernel<<<(unsigned)((MM + 127) / 128), 128, 0, st>>>(L, m, out, MM, n_chol);
  return 1;
}
int run_hmod(const double* h1, const double* part, int nsplit, const double* mL, double* hmod, int M, cudaStream_t st) {
  const long MM = (long)M * M;
  hmod_kernel<<<(unsigned)((MM + 255) / 256), 256, 0, st>>>(h1, part, nsplit, mL, hmod, MM);
  return 1;
}
int run_axpby_identity(double* P, double a, double idval, int M, cudaStream_t st) {
  const long MM = (long)M * M;
  axpby_identity_kernel<<<(unsigned)((MM + 255) / 256), 256, 0, st>>>(P, a, idval, M);
  return 1;
}
int run_scale_copy(double* dst, const double* src, double a, long n, cudaStream_t st) {
  scale_copy_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(dst, src, a, n);
  return 1;
}

}  // namespace afq
