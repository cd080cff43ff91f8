// small.cu - the small-matrix and element-wise stages of the walker step (plain FP64 ALU).
//
//   a1/a2  overlap O = psi^T phi, Gauss-Jordan inverse with row pivoting, det, Theta = phi O^-1
//
//   a4     force bias -> shifted fields, c_fb, c_mf           (Eqs. 12, 14, 16)
//   a9     phaseless weight update                            (Eqs. 13, 15-18)
//   a10    re-orthonormalisation by two Cholesky-QR passes
//
// One CTA per (spin block, walker); these stages are <= 1 % of the flops of a step.
#include <cstring>

#include "internal.h"

namespace afq {

namespace {

constexpr int kRows = 32;  // walker rows staged per chunk

__device__ __forceinline__ double2 cmul(double2 a, double2 b) {
  return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
__device__ __forceinline__ double2 cinv(double2 a) {
  double d = a.x * a.x + a.y * a.y;
  return make_double2(a.x / d, -a.y / d);
}

// block-wide sum of NV doubles per thread; result valid in thread 0
template <int NV>
__device__ __forceinline__ void block_sum(double (&v)[NV], double* scratch /* >= 8*NV */) {
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
  if (threadIdx.x == 0) {
    const int nwarp = blockDim.x >> 5;
#pragma unroll
    for (int k = 0; k < NV; ++k) {
      double s = 0.0;
      for (int w = 0; w < nwarp; ++w) s += scratch[w * NV + k];
      v[k] = s;
    }
  }
}

// ------------------------------------------------------------------------------ a1 / a2
__global__ void __launch_bounds__(256) overlap_theta_kernel(OTArgs a) {
  extern __shared__ __align__(16) unsigned char smraw[];
  const int blk = blockIdx.x, w = blockIdx.y;
  const int ns = a.ns[blk], off = a.off[blk], M = a.M, Nt = a.Nt;
  const int tid = threadIdx.x;
  const int ld2 = 2 * ns;      // augmented row length
  const int ldp = ns | 1;      // odd row stride (double2 units) of the staged walker rows

  double2* Aug = reinterpret_cast<double2*>(smraw);             // [ns][2 ns]
  double2* sphi = Aug + (size_t)ns * ld2;                       // [kRows][ldp]
  double2* fcol = sphi + (size_t)kRows * ldp;                   // [ns]
  double* spsi = reinterpret_cast<double*>(fcol + ns);          // [kRows][ns]
  double* red = spsi + (size_t)kRows * ns;                      // [32] reduction scratch
  double* spsi_i = red + 32;                                    // [kRows][ns], complex trial only
  __shared__ int s_piv;
  __shared__ double2 s_det;

  const double2* Wc = reinterpret_cast<const double2*>(a.W) + (size_t)w * M * Nt;

  // ---- O = psi^+ phi (psi^T for a real trial) ------------------------------------------
  const int nout = ns * ns;
  double2 acc[16];
#pragma unroll
  for (int k = 0; k < 16; ++k) acc[k] = make_double2(0.0, 0.0);
  for (int p0 = 0; p0 < M; p0 += kRows) {
    const int pr = min(kRows, M - p0);
    __syncthreads();
    for (int c = tid; c < pr * ns; c += blockDim.x) {
      int pl = c / ns, j = c % ns;
      sphi[pl * ldp + j] = Wc[(size_t)(p0 + pl) * Nt + off + j];
      spsi[pl * ns + j] = a.trial[(size_t)(p0 + pl) * Nt + off + j];
      if (a.trial_im) spsi_i[pl * ns + j] = a.trial_im[(size_t)(p0 + pl) * Nt + off + j];
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < 16; ++k) {
      const int idx = tid + k * 256;
      if (idx < nout) {
        const int i = idx / ns, j = idx % ns;
        double2 s = acc[k];
        for (int pl = 0; pl < pr; ++pl) {
          const double ps = spsi[pl * ns + i];
          const double2 z = sphi[pl * ldp + j];
          s.x = fma(ps, z.x, s.x);
          s.y = fma(ps, z.y, s.y);
        }
        if (a.trial_im)                       // conj(psi) z = (pr - i pi)(zr + i zi)
          for (int pl = 0; pl < pr; ++pl) {
            const double pi = spsi_i[pl * ns + i];
            const double2 z = sphi[pl * ldp + j];
            s.x = fma(pi, z.y, s.x);
            s.y = fma(-pi, z.x, s.y);
          }
        acc[k] = s;
      }
    }
  }
  __syncthreads();
#pragma unroll
  for (int k = 0; k < 16; ++k) {
    const int idx = tid + k * 256;
    if (idx < nout) {
      const int i = idx / ns, j = idx % ns;
      Aug[i * ld2 + j] = acc[k];
      Aug[i * ld2 + ns + j] = make_double2(i == j ? 1.0 : 0.0, 0.0);
    }
  }
  if (tid == 0) s_det = make_double2(1.0, 0.0);
  __syncthreads();

  // ---- Gauss-Jordan with row pivoting on [O | I] -------------------------------------
  for (int c = 0; c < ns; ++c) {
    if (tid < 32) {
      double best = -1.0;
      int bi = c;
      for (int r = c + tid; r < ns; r += 32) {
        double2 v = Aug[r * ld2 + c];
        double m = v.x * v.x + v.y * v.y;
        if (!(m <= best)) { best = m; bi = r; }   // NaN counts as a candidate so it propagates
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        double ob = __shfl_down_sync(0xffffffffu, best, o);
        int oi = __shfl_down_sync(0xffffffffu, bi, o);
        if (ob > best || (ob == best && oi < bi)) { best = ob; bi = oi; }
      }
      if (tid == 0) s_piv = bi;
    }
    __syncthreads();
    const int piv = s_piv;
    if (piv != c) {
      for (int j = tid; j < ld2; j += blockDim.x) {
        double2 u = Aug[c * ld2 + j];
        Aug[c * ld2 + j] = Aug[piv * ld2 + j];
        Aug[piv * ld2 + j] = u;
      }
      if (tid == 0) s_det = make_double2(-s_det.x, -s_det.y);
    }
    __syncthreads();
    const double2 pv = Aug[c * ld2 + c];
    __syncthreads();
    const double2 ipv = cinv(pv);
    if (tid == 0) s_det = cmul(s_det, pv);
    for (int j = tid; j < ld2; j += blockDim.x) Aug[c * ld2 + j] = cmul(Aug[c * ld2 + j], ipv);
    for (int r = tid; r < ns; r += blockDim.x)
      if (r != c) fcol[r] = Aug[r * ld2 + c];
    __syncthreads();
    for (int idx = tid; idx < ns * ld2; idx += blockDim.x) {
      const int r = idx / ld2, j = idx % ld2;
      if (r != c) {
        const double2 f = fcol[r], pc = Aug[c * ld2 + j];
        double2 v = Aug[idx];
        v.x -= f.x * pc.x - f.y * pc.y;
        v.y -= f.x * pc.y + f.y * pc.x;
        Aug[idx] = v;
      }
    }
    __syncthreads();
  }
  if (tid == 0) reinterpret_cast<double2*>(a.det)[(size_t)w * a.nblk + blk] = s_det;
  if (!a.want_theta) return;

  // ---- Theta = phi O^-1, written transposed and planar; E1b partial ------------------
  double e1[2] = {0.0, 0.0};
  const int ql = tid & 31, i0 = tid >> 5;
  double* th_re = a.ThT + ((size_t)(w * 2 + 0) * Nt + off) * M;
  double* th_im = a.ThT + ((size_t)(w * 2 + 1) * Nt + off) * M;
  for (int q0 = 0; q0 < M; q0 += kRows) {
    const int qr = min(kRows, M - q0);
    __syncthreads();
    for (int c = tid; c < qr * ns; c += blockDim.x) {
      int pl = c / ns, j = c % ns;
      sphi[pl * ldp + j] = Wc[(size_t)(q0 + pl) * Nt + off + j];
    }
    __syncthreads();
    if (ql < qr) {
      for (int i = i0; i < ns; i += 8) {
        double2 s = make_double2(0.0, 0.0);
        for (int j = 0; j < ns; ++j) {
          const double2 z = sphi[ql * ldp + j];
          const double2 o = Aug[j * ld2 + ns + i];
          s.x += z.x * o.x - z.y * o.y;
          s.y += z.x * o.y + z.y * o.x;
        }
        th_re[(size_t)i * M + q0 + ql] = s.x;
        th_im[(size_t)i * M + q0 + ql] = s.y;
        if (a.want_e1) {
          const double hr = a.hrot[(size_t)(off + i) * M + q0 + ql];
          e1[0] = fma(hr, s.x, e1[0]);
          e1[1] = fma(hr, s.y, e1[1]);
        }
      }
    }
  }
  if (a.want_e1) {
    block_sum<2>(e1, red);
    if (tid == 0) reinterpret_cast<double2*>(a.e1)[(size_t)w * a.nblk + blk] = make_double2(e1[0], e1[1]);
  }
}

// ------------------------------------------------------------------------------ a1 / a2 on DMMA
// The same stage as overlap_theta_kernel with its two contractions on the tensor cores:
//   O = psi^T phi          batched KN GEMM (gemm_ws.cu), all blocks at once: Obuf[w][Nt][2 Nt]
//   gj_kernel              per (block, walker): Gauss-Jordan inverse + det of the diagonal block, and the
//                          inverse written as the real (2 Nt) x (2 Nt) operand
//                              Aop[(plane, i)][(j, plane')] = [[Re Oinv^T, -Im Oinv^T], [Im Oinv^T, Re Oinv^T]]
//   Theta^T = Aop W^T      batched NK GEMM: ThT[w][(plane, i)][q] = sum_k Aop[(plane, i)][k] W[q][k]
//   e1_kernel              one-body energy sum hrot . Theta
__global__ void __launch_bounds__(256) gj_kernel(OTArgs a) {
  extern __shared__ __align__(16) unsigned char smraw[];
  const int blk = blockIdx.x, w = blockIdx.y;
  const int ns = a.ns[blk], off = a.off[blk], Nt = a.Nt;
  const int tid = threadIdx.x, tx = tid & 31, ty = tid >> 5;
  const int ld2 = 2 * ns;
  double2* Aug = reinterpret_cast<double2*>(smraw);             // [ns][2 ns]
  double2* fcol = Aug + (size_t)ns * ld2;                       // [ns]
  __shared__ int s_piv;
  __shared__ double2 s_det;
  const double2* O = reinterpret_cast<const double2*>(a.Obuf) + (size_t)w * Nt * Nt;
  for (int i = ty; i < ns; i += 8)
    for (int j = tx; j < ns; j += 32) {
      Aug[i * ld2 + j] = O[(size_t)(off + i) * Nt + off + j];
      Aug[i * ld2 + ns + j] = make_double2(i == j ? 1.0 : 0.0, 0.0);
    }
  if (tid == 0) s_det = make_double2(1.0, 0.0);
  __syncthreads();
  // Gauss-Jordan with row pivoting on [O | I]: four barriers per column (pivot found / column c and the pivot
  // read / rows swapped and scaled / rows eliminated); thread (ty, tx) owns rows ty, ty + 8, ... and columns
  // tx, tx + 32, ... of the elimination, so no index arithmetic with divisions is needed.
  for (int c = 0; c < ns; ++c) {
    if (ty == 0) {
      double best = -1.0;
      int bi = c;
      for (int r = c + tx; r < ns; r += 32) {
        const double2 v = Aug[r * ld2 + c];
        const double m = v.x * v.x + v.y * v.y;
        if (!(m <= best)) { best = m; bi = r; }   // NaN counts as a candidate so it propagates
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        const double ob = __shfl_down_sync(0xffffffffu, best, o);
        const int oi = __shfl_down_sync(0xffffffffu, bi, o);
        if (ob > best || (ob == best && oi < bi)) { best = ob; bi = oi; }
      }
      if (tx == 0) s_piv = bi;
    }
    __syncthreads();
    const int piv = s_piv;
    const double2 pv = Aug[piv * ld2 + c];         // read by everyone before anyone writes (barrier below)
    // the eliminated rows need their column-c entries as they are now (row piv will sit in row c after the swap)
    for (int r = tid; r < ns; r += blockDim.x)
      if (r != c) fcol[r] = r == piv ? Aug[c * ld2 + c] : Aug[r * ld2 + c];
    __syncthreads();
    const double2 ipv = cinv(pv);
    if (tid == 0) {
      double2 d = cmul(s_det, pv);
      s_det = piv != c ? make_double2(-d.x, -d.y) : d;
    }
    // swap rows c and piv and scale the new row c by 1 / pivot, one column per thread
    for (int j = tid; j < ld2; j += blockDim.x) {
      const double2 top = Aug[piv * ld2 + j];
      if (piv != c) Aug[piv * ld2 + j] = Aug[c * ld2 + j];
      Aug[c * ld2 + j] = cmul(top, ipv);
    }
    __syncthreads();
    for (int r = ty; r < ns; r += 8) {
      if (r == c) continue;
      const double2 f = fcol[r];
      for (int j = tx; j < ld2; j += 32) {
        const double2 pc = Aug[c * ld2 + j];
        double2 v = Aug[r * ld2 + j];
        v.x -= f.x * pc.x - f.y * pc.y;
        v.y -= f.x * pc.y + f.y * pc.x;
        Aug[r * ld2 + j] = v;
      }
    }
    __syncthreads();
  }
  if (tid == 0) reinterpret_cast<double2*>(a.det)[(size_t)w * a.nblk + blk] = s_det;
  if (!a.want_theta) return;
  // rows (plane, off + i) of Aop, all 2 Nt columns (zero outside this spin block)
  const int K2 = 2 * Nt;
  double* Aop = a.Aop + (size_t)w * K2 * K2;
  for (int idx = tid; idx < ns * Nt; idx += blockDim.x) {
    const int i = idx / Nt, jc = idx % Nt;           // jc: column of the walker, all blocks
    double2 o = make_double2(0.0, 0.0);
    if (jc >= off && jc < off + ns) o = Aug[(jc - off) * ld2 + ns + i];   // Oinv[j][i]
    double* r0 = Aop + (size_t)(off + i) * K2 + 2 * jc;               // plane re
    double* r1 = Aop + (size_t)(Nt + off + i) * K2 + 2 * jc;          // plane im
    r0[0] = o.x; r0[1] = -o.y;
    r1[0] = o.y; r1[1] = o.x;
  }
}

// e1[w][blk] = sum_{i in block, q} hrot[off + i][q] * Theta^T[w][.][off + i][q]; grid (nblk, nw)
__global__ void __launch_bounds__(1024) e1_kernel(OTArgs a) {
  __shared__ double red[32 * 2];
  const int blk = blockIdx.x, w = blockIdx.y;
  const int ns = a.ns[blk], off = a.off[blk], M = a.M, Nt = a.Nt;
  const double* tr = a.ThT + ((size_t)(w * 2 + 0) * Nt + off) * M;
  const double* ti = a.ThT + ((size_t)(w * 2 + 1) * Nt + off) * M;
  const double* hr = a.hrot + (size_t)off * M;
  double e1[2] = {0.0, 0.0};
  for (long idx = threadIdx.x; idx < (long)ns * M; idx += blockDim.x) {
    const double h = hr[idx];
    e1[0] = fma(h, tr[idx], e1[0]);
    e1[1] = fma(h, ti[idx], e1[1]);
  }
  block_sum<2>(e1, red);
  if (threadIdx.x == 0) reinterpret_cast<double2*>(a.e1)[(size_t)w * a.nblk + blk] = make_double2(e1[0], e1[1]);
}

// ------------------------------------------------------------------------------ a4
__global__ void __launch_bounds__(256) field_shift_kernel(ShiftArgs a) {
  __shared__ double red[8 * 4];
  const int w = blockIdx.x, nc = a.n_chol;
  const double sq = a.sqrt_dt;
  double v[4] = {0.0, 0.0, 0.0, 0.0};  // cfb.re, cfb.im, sum xs_re m, sum xs_im m
  for (int g = threadIdx.x; g < nc; g += blockDim.x) {
    double xr = 0.0, xi = 0.0;
    for (int s = 0; s < a.nsplit; ++s) {
      xr += a.Xp[(size_t)s * a.sXp + (size_t)(2 * w) * nc + g];
      xi += a.Xp[(size_t)s * a.sXp + (size_t)(2 * w + 1) * nc + g];
    }
    xr *= a.spin_factor;
    xi *= a.spin_factor;
    a.X[(size_t)(2 * w) * nc + g] = xr;
    a.X[(size_t)(2 * w + 1) * nc + g] = xi;
    const double mg = a.m[g], x = a.x[(size_t)w * nc + g];
    // xbar = i sqrt(dt) (X - m)
    double br = -sq * xi, bi = sq * (xr - mg);
    if (a.xbar_bound > 0.0) {                           // reading S8b: cap the modulus, keep the phase
      const double mag = hypot(br, bi);
      if (mag > a.xbar_bound) { const double sc = a.xbar_bound / mag; br *= sc; bi *= sc; }
    }
    const double sr = x - br, si = -bi;                 // xs = x - xbar
    // c_fb = sum x xbar - 1/2 sum xbar^2 (bilinear)
    v[0] += x * br - 0.5 * (br * br - bi * bi);
    v[1] += x * bi - br * bi;
    v[2] += sr * mg;
    v[3] += si * mg;
    // A = -i sqrt(dt) sum xs L : Re A = sqrt(dt) sum Im(xs) L, Im A = -sqrt(dt) sum Re(xs) L
    a.Cf[(size_t)(2 * w) * nc + g] = sq * si;
    a.Cf[(size_t)(2 * w + 1) * nc + g] = -sq * sr;
  }
  block_sum<4>(v, red);
  if (threadIdx.x == 0) {
    a.cfb[2 * w] = v[0];
    a.cfb[2 * w + 1] = v[1];
    // c_mf = i sqrt(dt) sum xs m
    a.cmf[2 * w] = -sq * v[3];
    a.cmf[2 * w + 1] = sq * v[2];
  }
}

// ------------------------------------------------------------------------------ a9
__device__ __forceinline__ double2 block_prod(const double* det, int w, int nblk, int rhf) {
  double2 o = make_double2(1.0, 0.0);
  for (int b = 0; b < nblk; ++b) {
    double2 d = reinterpret_cast<const double2*>(det)[(size_t)w * nblk + b];
    o = cmul(o, d);
    if (rhf) o = cmul(o, d);
  }
  return o;
}

__global__ void weight_update_kernel(WeightArgs a, int nw) {
  const int w = blockIdx.x * blockDim.x + threadIdx.x;
  if (w >= nw) return;
  const double2 oo = block_prod(a.det_old, w, a.nblk, a.rhf);
  const double2 on = block_prod(a.det_new, w, a.nblk, a.rhf);
  reinterpret_cast<double2*>(a.ovlp)[w] = on;
  // r = on / oo
  const double d = oo.x * oo.x + oo.y * oo.y;
  const double2 r = make_double2((on.x * oo.x + on.y * oo.y) / d, (on.y * oo.x - on.x * oo.y) / d);
  const double cmr = a.cmf[2 * w], cmi = a.cmf[2 * w + 1];
  const double em = exp(cmr);
  double sn, cs;
  sincos(cmi, &sn, &cs);
  const double2 S = cmul(r, make_double2(em * cs, em * sn));        // Eq. (17)
  const double absS = hypot(S.x, S.y);
  double absI = absS * exp(a.cfb[2 * w]) * exp(a.expo);              // |I|, Eq. (16) + reading S7
  const bool finI = isfinite(absI);                                  // judged BEFORE the bound: an overflowed |I| kills
  if (a.ehyb_bound > 0.0 && absI > 0.0) {                            // reading S8b: clip D = -log|I| / dt
    const double D = -log(absI) / a.dt;
    if (fabs(D) > a.ehyb_bound) absI = exp(-a.dt * copysign(a.ehyb_bound, D));
  }
  const bool ok = isfinite(S.x) && isfinite(S.y) && finI && absS > 0.0 &&
                  (oo.x != 0.0 || oo.y != 0.0) && isfinite(on.x) && isfinite(on.y) &&
                  isfinite(a.cfb[2 * w + 1]);
  double wt = a.weights[w];
  if (!ok) {
    wt = 0.0;
  } else {
    const double c = S.x / absS;                                     // cos(arg S), Eq. (18)
    wt = wt * absI * (c > 0.0 ? c : 0.0);                            // Eqs. (13), (15)
  }
  a.weights[w] = wt;
}

// ------------------------------------------------------------------------------ a10
// Thin QR with R_ii > 0 by repeated Cholesky-QR passes inside ONE kernel (a CTA owns its walker-block):
//     G = phi^H phi = R^H R,  phi <- phi R^-1,  detR *= prod R_ii
// until the Gram matrix found at the start of a pass is within 0.05 of the identity: that pass then leaves
// ||Q^H Q - 1|| = O(eps).  Well-conditioned walkers take the two passes of Cholesky-QR2.  When the Cholesky
// factorisation breaks down (a pivot <= 1e-11 of its diagonal entry, or not finite: cond(phi)^2 reached 1/eps) the
// pass is redone on G + s 1 with s = 11 (M n + n (n + 1)) eps tr(G) - shifted Cholesky-QR (Fukaya et al., SIAM J. Sci.
// Comput. 42 (2020)): it brings cond(phi) ~ 1e12 down to ~1e7, which the next two passes finish.  R is the product
// of the passes' triangles, so its diagonal stays real positive: the unique thin QR, as the oracle's (S9).
// A walker that is not finite stays not finite (its weight is already 0, S10).  shifted[0] counts shifted passes.
__global__ void __launch_bounds__(256) cholqr_kernel(QRArgs a) {
  extern __shared__ __align__(16) unsigned char smraw[];
  const int blk = blockIdx.x, w = blockIdx.y;
  const int ns = a.ns[blk], off = a.off[blk], M = a.M, Nt = a.Nt;
  const int tid = threadIdx.x;
  const int ldp = ns | 1;
  double2* G = reinterpret_cast<double2*>(smraw);     // [ns][ns]
  double2* Ri = G + (size_t)ns * ns;                  // [ns][ns] inverse of R (backup of G during the Cholesky)
  double2* sphi = Ri + (size_t)ns * ns;               // [kRows][ldp]
  double2* Wc = reinterpret_cast<double2*>(a.W) + (size_t)w * M * Nt;
  __shared__ double s_red[8];
  __shared__ double s_diag0[kMaxOcc];
  __shared__ int s_bad;
  const int nout = ns * ns;
  double detR = 1.0;

  for (int pass = 0; pass < 8; ++pass) {
    double2 acc[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) acc[k] = make_double2(0.0, 0.0);
    for (int p0 = 0; p0 < M; p0 += kRows) {
      const int pr = min(kRows, M - p0);
      __syncthreads();
      for (int c = tid; c < pr * ns; c += blockDim.x) {
        int pl = c / ns, j = c % ns;
        sphi[pl * ldp + j] = Wc[(size_t)(p0 + pl) * Nt + off + j];
      }
      __syncthreads();
#pragma unroll
      for (int k = 0; k < 16; ++k) {
        const int idx = tid + k * 256;
        if (idx < nout) {
          const int i = idx / ns, j = idx % ns;
          double2 s = acc[k];
          for (int pl = 0; pl < pr; ++pl) {
            const double2 u = sphi[pl * ldp + i], z = sphi[pl * ldp + j];
            s.x += u.x * z.x + u.y * z.y;               // conj(u) z
            s.y += u.x * z.y - u.y * z.x;
          }
          acc[k] = s;
        }
      }
    }
    __syncthreads();
    // G, its backup, and max |G - 1| (NaN counts as far from the identity)
    double dev = 0.0;
#pragma unroll
    for (int k = 0; k < 16; ++k) {
      const int idx = tid + k * 256;
      if (idx < nout) {
        G[idx] = acc[k];
        Ri[idx] = acc[k];
        const int i = idx / ns, j = idx % ns;
        const double e = fmax(fabs(acc[k].x - (i == j ? 1.0 : 0.0)), fabs(acc[k].y));
        dev = (e > dev || !(e == e)) ? (e == e ? e : 1e300) : dev;
        if (i == j) s_diag0[i] = acc[k].x;
      }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) dev = fmax(dev, __shfl_down_sync(0xffffffffu, dev, o));
    if ((tid & 31) == 0) s_red[tid >> 5] = dev;
    if (tid == 0) s_bad = 0;
    __syncthreads();
    dev = 0.0;
    for (int k = 0; k < 8; ++k) dev = fmax(dev, s_red[k]);
    const bool last = dev <= 0.05;

    // Cholesky G = R^H R, R upper, in place; one retry on the shifted matrix
    for (int attempt = 0; attempt < 2; ++attempt) {
      bool bad = false;
      for (int k = 0; k < ns; ++k) {
        const double d2 = G[k * ns + k].x;
        if (attempt == 0 && !(d2 > 1e-11 * s_diag0[k])) { bad = true; break; }     // uniform: every thread reads the same
        const double d = sqrt(d2);
        __syncthreads();
        for (int j = k + tid; j < ns; j += blockDim.x) {
          double2 v = G[k * ns + j];
          G[k * ns + j] = (j == k) ? make_double2(d, 0.0) : make_double2(v.x / d, v.y / d);
        }
        __syncthreads();
        const int rem = ns - k - 1;
        for (int idx = tid; idx < rem * rem; idx += blockDim.x) {
          const int i = k + 1 + idx / rem, j = k + 1 + idx % rem;
          if (j >= i) {
            const double2 u = G[k * ns + i], z = G[k * ns + j];
            double2 v = G[i * ns + j];
            v.x -= u.x * z.x + u.y * z.y;
            v.y -= u.x * z.y - u.y * z.x;
            G[i * ns + j] = v;
          }
        }
        __syncthreads();
      }
      if (!bad) break;
      // breakdown: restore G from the backup with the shift on the diagonal
      __syncthreads();
      double tr = 0.0;
      for (int k = 0; k < ns; ++k) tr += s_diag0[k];
      const double shift = 11.0 * ((double)M * ns + (double)ns * (ns + 1)) * 1.1102230246251565e-16 * tr;
      for (int idx = tid; idx < nout; idx += blockDim.x) {
        double2 v = Ri[idx];
        if (idx / ns == idx % ns) v.x += shift;
        G[idx] = v;
      }
      if (tid == 0) { s_bad = 1; if (a.shifted) atomicAdd(a.shifted, 1); }
      __syncthreads();
    }
    for (int idx = tid; idx < nout; idx += blockDim.x) Ri[idx] = make_double2(0.0, 0.0);
    __syncthreads();
    // R^-1 by back substitution, one column per thread
    if (tid < ns) {
      const int c = tid;
      for (int i = c; i >= 0; --i) {
        double2 s = make_double2(i == c ? 1.0 : 0.0, 0.0);
        for (int k = i + 1; k <= c; ++k) {
          const double2 r = G[i * ns + k], x = Ri[k * ns + c];
          s.x -= r.x * x.x - r.y * x.y;
          s.y -= r.x * x.y + r.y * x.x;
        }
        const double rii = G[i * ns + i].x;
        Ri[i * ns + c] = make_double2(s.x / rii, s.y / rii);
      }
    }
    for (int k = 0; k < ns; ++k) detR *= G[k * ns + k].x;
    __syncthreads();
    // phi <- phi R^-1, rows are independent
    const int lane = tid & 31, rw = tid >> 5;
    for (int q0 = 0; q0 < M; q0 += kRows) {
      const int qr = min(kRows, M - q0);
      __syncthreads();
      for (int c = tid; c < qr * ns; c += blockDim.x) {
        int pl = c / ns, j = c % ns;
        sphi[pl * ldp + j] = Wc[(size_t)(q0 + pl) * Nt + off + j];
      }
      __syncthreads();
      for (int pl = rw; pl < qr; pl += 8)
        for (int i = lane; i < ns; i += 32) {
          double2 s = make_double2(0.0, 0.0);
          for (int j = 0; j <= i; ++j) {
            const double2 z = sphi[pl * ldp + j], o = Ri[j * ns + i];
            s.x += z.x * o.x - z.y * o.y;
            s.y += z.x * o.y + z.y * o.x;
          }
          Wc[(size_t)(q0 + pl) * Nt + off + i] = s;
        }
    }
    __syncthreads();
    // stop after the pass that started within 0.05 of orthonormal, or when the walker is not finite
    if (last || !(detR == detR) || !(fabs(detR) < 1e308)) break;
  }
  if (tid == 0) a.detR[(size_t)w * a.nblk + blk] *= detR;
}

__global__ void ovlp_div_detR_kernel(double* ovlp, const double* detR, int nblk, int rhf, int nw) {
  const int w = blockIdx.x * blockDim.x + threadIdx.x;
  if (w >= nw) return;
  double d = 1.0;
  for (int b = 0; b < nblk; ++b) d *= rhf ? detR[w * nblk + b] * detR[w * nblk + b] : detR[w * nblk + b];
  ovlp[2 * w] /= d;
  ovlp[2 * w + 1] /= d;
}

__global__ void fill_kernel(double* p, double v, long n) {
  long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) p[i] = v;
}

}  // namespace

static size_t ot_smem(int ns) {
  const int ldp = ns | 1;
  return (size_t)ns * 2 * ns * 16 + (size_t)kRows * ldp * 16 + (size_t)ns * 16 + (size_t)2 * kRows * ns * 8 + 32 * 8 + 64;
}

// the DMMA route; returns launches or -1 if a GEMM cannot be served (caller falls back to the one-kernel route)
static int run_overlap_theta_gemm(const OTArgs& a, int nw, cudaStream_t st) {
  const int M = a.M, Nt = a.Nt, K2 = 2 * Nt;
  int launches = 0;
  // O[w] = trial^T (Nt x M, shared) * W[w] (M x 2 Nt); complex trial: conj(trial)^T as the planar pair
  // (Re psi^T, -Im psi^T) of the planar-complex GEMM
  int r = run_gemm_ws_kn(a.trialT, M, a.trial_im ? (long)Nt * M : 0, 0, a.trial_im != nullptr, a.W, K2, (long)M * K2, a.Obuf,
                         nullptr, K2, (long)Nt * K2, Nt, K2, M, nw, 1.0, 0, st);
  if (r < 0) return -1;
  launches += r;
  int nsmax = a.ns[0];
  if (a.nblk > 1 && a.ns[1] > nsmax) nsmax = a.ns[1];
  const size_t sm = (size_t)nsmax * 2 * nsmax * 16 + (size_t)nsmax * 16 + 64;
  static size_t cur[64] = {0};
  if (auto grow_ = grow_on_device(cur, sm)) cudaFuncSetAttribute(gj_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
  gj_kernel<<<dim3(a.nblk, nw), 256, sm, st>>>(a);
  ++launches;
  if (!a.want_theta) return launches;
  // ThT[w] (2 Nt x M) = Aop[w] (2 Nt x 2 Nt, k contiguous) * W[w]^T (W: M x 2 Nt, k contiguous)
  GemmArgs g;
  memset(&g, 0, sizeof(g));
  g.A = a.Aop; g.lda = K2; g.sA = (long)K2 * K2;
  g.B = a.W; g.ldb = K2; g.sB = (long)M * K2;
  g.C = a.ThT; g.ldc = M; g.sC = (long)K2 * M;
  g.M = K2; g.N = M; g.K = K2; g.batch = nw; g.splitK = 1; g.alpha = 1.0;
  launches += run_gemm(GEMM_NK, g, st);
  if (a.want_e1) {
    e1_kernel<<<dim3(a.nblk, nw), 1024, 0, st>>>(a);
    ++launches;
  }
  return launches;
}

int run_e1(const OTArgs& a, int nw, cudaStream_t st) {
  e1_kernel<<<dim3(a.nblk, nw), 1024, 0, st>>>(a);
  return 1;
}

int run_overlap_theta(const OTArgs& a, int nw, cudaStream_t st) {
  if (a.Obuf && a.Aop && a.trialT) {
    const int r = run_overlap_theta_gemm(a, nw, st);
    if (r > 0) return r;
  }
  int nsmax = a.ns[0];
  if (a.nblk > 1 && a.ns[1] > nsmax) nsmax = a.ns[1];
  const size_t sm = ot_smem(nsmax);
  static size_t cur[64] = {0};
  if (auto grow_ = grow_on_device(cur, sm)) {
    cudaFuncSetAttribute(overlap_theta_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
  }
  overlap_theta_kernel<<<dim3(a.nblk, nw), 256, sm, st>>>(a);
  return 1;
}

int run_field_shift(const ShiftArgs& a, int nw, cudaStream_t st) {
  field_shift_kernel<<<nw, 256, 0, st>>>(a);
  return 1;
}

int run_weight_update(const WeightArgs& a, int nw, cudaStream_t st) {
  weight_update_kernel<<<(nw + 127) / 128, 128, 0, st>>>(a, nw);
  return 1;
}

int run_cholqr_pass(const QRArgs& a, int nw, cudaStream_t st) {
  int nsmax = a.ns[0];
  if (a.nblk > 1 && a.ns[1] > nsmax) nsmax = a.ns[1];
  const size_t sm = (size_t)2 * nsmax * nsmax * 16 + (size_t)kRows * (nsmax | 1) * 16 + 64;
  static size_t cur[64] = {0};
  if (auto grow_ = grow_on_device(cur, sm)) {
    cudaFuncSetAttribute(cholqr_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
  }
  cholqr_kernel<<<dim3(a.nblk, nw), 256, sm, st>>>(a);
  return 1;
}

int run_ovlp_div_detR(double* ovlp, const double* detR, int nblk, int rhf, int nw, cudaStream_t st) {
  ovlp_div_detR_kernel<<<(nw + 127) / 128, 128, 0, st>>>(ovlp, detR, nblk, rhf, nw);
  return 1;
}

int run_fill(double* p, double v, long n, cudaStream_t st) {
  fill_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(p, v, n);
  return 1;
}

}  // namespace afq
