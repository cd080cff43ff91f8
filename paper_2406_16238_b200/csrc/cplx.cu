// cplx.cu - complex Cholesky vectors ("Support of complex Cholesky vectors"; SURVEY 8f
// NEXT-4).  With L_g = A_g + i B_g (A, B Hermitian) the symmetric tensor is (ps|qr) = sum_g (A_ps A_qr +
// B_ps B_qr), so the walker step is the one of the real case with the 2n Hermitian matrices K = (A_1..A_n,
// B_1..B_n) in place of the n real symmetric L_g - "twice as many auxiliary fields" (derivation and pins:
// oracle/complex_chol_oracle.py, tests/test_oracle_complex_pins.py).
//
// The handle keeps K as REAL planes  Ks = [Re K_1 .. Re K_2n | Im K_1 .. Im K_2n]  ([4n][M][M], Re symmetric,
// Im antisymmetric) and runs the REAL kernels over these 4n pseudo-vectors; the kernels here put the complex
// numbers back together:
//   hermitian_planes_kernel   L (complex, interleaved) -> Ks
//   field_shift_cplx_kernel   X_g = Xs_g + i Xs_{2n+g};  xbar, xs, c_fb, c_mf;  V_HS coefficients of all 4n planes
//   energy_cplx_kernel        E_C = 1/2 sum X^2;  E_X = -1/2 sum tr(T T) with T = T_r + i T_i:
//                             tr(T T) = tr(T_r T_r) - tr(T_i T_i) + i [tr((T_r + T_i)^2) - tr(T_r T_r) - tr(T_i T_i)]
//                             (three runs of the exchange kernel: Lrot_r, Lrot_i and Lrot_r + Lrot_i)
//   add_antisym_kernel        sign fix of the antisymmetric part of V_HS computed by the symmetric-half kernel
//   deinterleave / caxpby_identity   helpers of the complex expm(-dt/2 h_mod) (api.cu: build_E1_complex)
#include "internal.h"

namespace afq {

namespace {

// Ks[g] = Re A_g, Ks[n + g] = Re B_g, Ks[2n + g] = Im A_g, Ks[3n + g] = Im B_g;  grid (chunks, n)
__global__ void __launch_bounds__(256) hermitian_planes_kernel(const double2* __restrict__ L, double* __restrict__ Ks,
                                                               int M, int n) {
  const int g = blockIdx.y;
  const size_t MM = (size_t)M * M;
  const double2* Lg = L + (size_t)g * MM;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < MM; i += (size_t)gridDim.x * blockDim.x) {
    const int p = (int)(i / M), q = (int)(i % M);
    const double2 a = Lg[i], b = Lg[(size_t)q * M + p];       // L_pq, L_qp
    // A = (L + L^+)/2: A_pq = (L_pq + conj(L_qp))/2;   B = (L - L^+)/(2i): B_pq = (L_pq - conj(L_qp))/(2i)
    Ks[(size_t)g * MM + i] = 0.5 * (a.x + b.x);
    Ks[(size_t)(2 * n + g) * MM + i] = 0.5 * (a.y - b.y);
    Ks[(size_t)(n + g) * MM + i] = 0.5 * (a.y + b.y);
    Ks[(size_t)(3 * n + g) * MM + i] = -0.5 * (a.x - b.x);
  }
}

__global__ void axpy_kernel(double* dst, const double* a, const double* b, long n) {
  const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) dst[i] = a[i] + b[i];
}

__global__ void axpy_scaled_kernel(double* dst, const double* a, const double* b, double sb, long n) {
  const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) dst[i] = a[i] + sb * b[i];
}

__global__ void add_antisym_kernel(double* A, const double* B, long MM, int M, long total) {
  const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= total) return;
  const long e = i % MM;
  const int p = (int)(e / M), q = (int)(e % M);
  if (q > p) A[i] += B[i];
  else if (q < p) A[i] -= B[i];
}

// planar [2][M][M] <- interleaved [M][2M]
__global__ void deinterleave_kernel(double* planar, const double* inter, long MM) {
  const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= MM) return;
  planar[i] = inter[2 * i];
  planar[MM + i] = inter[2 * i + 1];
}
// interleaved complex M x M: P = a P + idval 1
__global__ void caxpby_identity_kernel(double* P, double a, double idval, int M) {
  const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= (long)M * M) return;
  const int r = (int)(i / M), c = (int)(i % M);
  P[2 * i] = a * P[2 * i] + (r == c ? idval : 0.0);
  P[2 * i + 1] = a * P[2 * i + 1];
}

template <int NV>
__device__ __forceinline__ void block_sum256(double (&v)[NV], double* scratch /* 8 * NV */) {
#pragma unroll
  for (int k = 0; k < NV; ++k)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v[k] += __shfl_down_sync(0xffffffffu, v[k], o);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  __syncthreads();
  if (lane == 0)
#pragma unroll
    for (int k = 0; k < NV; ++k) scratch[warp * NV + k] = v[k];
  __syncthreads();
  if (threadIdx.x == 0)
#pragma unroll
    for (int k = 0; k < NV; ++k) {
      double s = 0.0;
      for (int w = 0; w < 8; ++w) s += scratch[w * NV + k];
      v[k] = s;
    }
}

// one CTA per walker; nf = 2n fields, nv = 2 nf pseudo-vectors
__global__ void __launch_bounds__(256) field_shift_cplx_kernel(CShiftArgs a) {
  __shared__ double red[8 * 4];
  const int w = blockIdx.x, nf = a.nf, nv = 2 * a.nf;
  const double sq = a.sqrt_dt;
  double v[4] = {0.0, 0.0, 0.0, 0.0};
  for (int g = threadIdx.x; g < nf; g += blockDim.x) {
    double rr = 0.0, ri = 0.0, ir = 0.0, ii = 0.0;      // (Lrot_r . Theta) re/im, (Lrot_i . Theta) re/im
    for (int s = 0; s < a.nsplit; ++s) {
      const double* xr = a.Xp + (size_t)s * a.sXp + (size_t)(2 * w) * nv;
      const double* xi = xr + nv;
      rr += xr[g]; ri += xi[g]; ir += xr[nf + g]; ii += xi[nf + g];
    }
    // X = sf [ (rr + i ri) + i (ir + i ii) ]
    const double Xr = a.spin_factor * (rr - ii), Xi = a.spin_factor * (ri + ir);
    a.X[(size_t)(2 * w) * nf + g] = Xr;
    a.X[(size_t)(2 * w + 1) * nf + g] = Xi;
    const double mg = a.m[g], x = a.x[(size_t)w * nf + g];
    double br = -sq * Xi, bi = sq * (Xr - mg);           // xbar = i sqrt(dt) (X - m)
    if (a.xbar_bound > 0.0) {                            // reading S8b: cap the modulus, keep the phase
      const double mag = hypot(br, bi);
      if (mag > a.xbar_bound) { const double sc = a.xbar_bound / mag; br *= sc; bi *= sc; }
    }
    const double sr = x - br, si = -bi;                  // xs = x - xbar
    v[0] += x * br - 0.5 * (br * br - bi * bi);
    v[1] += x * bi - br * bi;
    v[2] += sr * mg;
    v[3] += si * mg;
    // A = sum_g c_g (Kr_g + i Ki_g), c = -i sqrt(dt) xs = sqrt(dt) (si - i sr):
    //   planes of Kr_g: (Re c, Im c) = sqrt(dt) (si, -sr);  planes of Ki_g: i c = sqrt(dt) (sr, si)
    a.Cf[(size_t)(2 * w) * nv + g] = sq * si;
    a.Cf[(size_t)(2 * w + 1) * nv + g] = -sq * sr;
    a.Cf[(size_t)(2 * w) * nv + nf + g] = sq * sr;
    a.Cf[(size_t)(2 * w + 1) * nv + nf + g] = sq * si;
  }
  block_sum256<4>(v, red);
  if (threadIdx.x == 0) {
    a.cfb[2 * w] = v[0];
    a.cfb[2 * w + 1] = v[1];
    a.cmf[2 * w] = -sq * v[3];                           // c_mf = i sqrt(dt) sum xs m
    a.cmf[2 * w + 1] = sq * v[2];
  }
}

// one CTA per walker: E_out[w] = (E, E1b, E2)
__global__ void __launch_bounds__(256) energy_cplx_kernel(CEnergyArgs a) {
  __shared__ double red[8 * 8];
  const int w = blockIdx.x, nf = a.nf, nw = a.nw;
  double v[8] = {0, 0, 0, 0, 0, 0, 0, 0};   // sum X^2 (re, im); sums of tr(TT) for the sets r, i, s (re, im each)
  for (int g = threadIdx.x; g < nf; g += blockDim.x) {
    const double* xr = a.Xr + ((size_t)g * nw + w) * 2;   // tr(T_r) of this field (complex)
    double Xre = a.spin_factor * xr[0], Xim = a.spin_factor * xr[1];
    if (!a.pair) {
      const double* xi = a.Xi + ((size_t)g * nw + w) * 2;
      Xre = a.spin_factor * (xr[0] - xi[1]); Xim = a.spin_factor * (xr[1] + xi[0]);
    }
    v[0] += Xre * Xre - Xim * Xim;
    v[1] += 2.0 * Xre * Xim;
  }
  for (int k = 0; k < (a.pair ? 1 : 3); ++k)
    for (int b = 0; b < a.nblk; ++b)
      for (int q = threadIdx.x; q < a.ngroups[b]; q += blockDim.x) {
        const double* e = a.expart[k][b] + ((size_t)q * nw + w) * 2;
        v[2 + 2 * k] += e[0];
        v[3 + 2 * k] += e[1];
      }
  block_sum256<8>(v, red);
  if (threadIdx.x == 0) {
    double e1r = 0.0, e1i = 0.0;
    for (int b = 0; b < a.nblk; ++b) {
      const double* er = a.e1r + ((size_t)w * a.nblk + b) * 2;   // sum Re(h)rot . Theta
      const double* ei = a.e1i + ((size_t)w * a.nblk + b) * 2;   // sum Im(h)rot . Theta
      e1r += er[0] - ei[1];
      e1i += er[1] + ei[0];
    }
    e1r *= a.spin_factor;
    e1i *= a.spin_factor;
    // tr(TT) = t_r - t_i + i (t_s - t_r - t_i), each t complex
    const double tr_re = a.pair ? v[2] : v[2] - v[4] - (v[7] - v[3] - v[5]);
    const double tr_im = a.pair ? v[3] : v[3] - v[5] + (v[6] - v[2] - v[4]);
    const double e2r = 0.5 * v[0] - 0.5 * a.spin_factor * tr_re;
    const double e2i = 0.5 * v[1] - 0.5 * a.spin_factor * tr_im;
    double* o = a.E_out + (size_t)w * 6;
    o[0] = e1r + e2r; o[1] = e1i + e2i;
    o[2] = e1r;       o[3] = e1i;
    o[4] = e2r;       o[5] = e2i;
  }
}

}  // namespace

int run_hermitian_planes(const double* L_cplx, double* Ks, int M, int n, cudaStream_t st) {
  hermitian_planes_kernel<<<dim3(64, n), 256, 0, st>>>(reinterpret_cast<const double2*>(L_cplx), Ks, M, n);
  return 1;
}
int run_add(double* dst, const double* a, const double* b, long n, cudaStream_t st) {
  axpy_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(dst, a, b, n);
  return 1;
}
int run_add_scaled(double* dst, const double* a, const double* b, double sb, long n, cudaStream_t st) {
  axpy_scaled_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(dst, a, b, sb, n);
  return 1;
}
int run_add_antisym(double* A, const double* B, int rows, int M, cudaStream_t st) {
  const long MM = (long)M * M, total = MM * rows;
  add_antisym_kernel<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(A, B, MM, M, total);
  return 1;
}
int run_deinterleave(double* planar, const double* inter, int M, cudaStream_t st) {
  const long MM = (long)M * M;
  deinterleave_kernel<<<(unsigned)((MM + 255) / 256), 256, 0, st>>>(planar, inter, MM);
  return 1;
}
int run_caxpby_identity(double* P, double a, double idval, int M, cudaStream_t st) {
  const long MM = (long)M * M;
  caxpby_identity_kernel<<<(unsigned)((MM + 255) / 256), 256, 0, st>>>(P, a, idval, M);
  return 1;
}
int run_field_shift_cplx(const CShiftArgs& a, int nw, cudaStream_t st) {
  field_shift_cplx_kernel<<<nw, 256, 0, st>>>(a);
  return 1;
}
int run_energy_cplx(const CEnergyArgs& a, cudaStream_t st) {
  energy_cplx_kernel<<<a.nw, 256, 0, st>>>(a);
  return 1;
}

}  // namespace afq
