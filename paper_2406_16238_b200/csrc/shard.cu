// shard.cu - owner-side reductions of the distributed-Hamiltonian mode ("Distributed Hamiltonian
// for limited memory", Fig. 6).
//
// In a group of G members every member holds a gamma-slice of L.  Quantities that are sums over
// gamma (A = V_HS, c_fb, c_mf, E_C + E_X) are computed slice by slice by the member that holds the
// slice, for ALL walkers of the group, and each partial is stored straight into the walker
// owner's receive slot [source member] (peer memory over NVLink, or the same device).  The owner
// then adds its G slots in FIXED member order 0..G-1, so the result does not depend on timing.
#include "internal.h"

namespace afq {

namespace {

struct SlotPtrs { const double* p[kMaxGroup]; };

// dst[i] = sum_r slot_r[i], i < n (n even), 16-byte lanes, grid-stride
__global__ void __launch_bounds__(256) sum_slots_kernel(double* dst, SlotPtrs s, int G, long n2) {
  double2* d = reinterpret_cast<double2*>(dst);
  for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < n2; i += (long)gridDim.x * blockDim.x) {
    double2 v = reinterpret_cast<const double2*>(s.p[0])[i];
    for (int r = 1; r < G; ++r) {
      const double2 u = reinterpret_cast<const double2*>(s.p[r])[i];
      v.x += u.x;
      v.y += u.y;
    }
    d[i] = v;
  }
}

// dst[w] (complex) = E[w][2] (complex, the two-body part of an [n][3] energy array); dst may be
// peer memory
__global__ void push_e2_kernel(double* dst, const double* E, int n) {
  const int w = blockIdx.x * blockDim.x + threadIdx.x;
  if (w < n) {
    dst[2 * w] = E[(size_t)w * 6 + 4];
    dst[2 * w + 1] = E[(size_t)w * 6 + 5];
  }
}

// E_out[w] = (E1b + E2, E1b, E2), E1b = sf * sum_b e1[w][b], E2 = sum_r slot_r[w]
__global__ void energy_finish_kernel(double* E_out, const double* e1, SlotPtrs s, int G, int nblk, double sf, int nw) {
  const int w = blockIdx.x * blockDim.x + threadIdx.x;
  if (w >= nw) return;
  double e1r = 0.0, e1i = 0.0;
  for (int b = 0; b < nblk; ++b) {
    e1r += e1[((size_t)w * nblk + b) * 2];
    e1i += e1[((size_t)w * nblk + b) * 2 + 1];
  }
  e1r *= sf;
  e1i *= sf;
  double e2r = 0.0, e2i = 0.0;
  for (int r = 0; r < G; ++r) {
    e2r += s.p[r][2 * w];
    e2i += s.p[r][2 * w + 1];
  }
  double* o = E_out + (size_t)w * 6;
  o[0] = e1r + e2r; o[1] = e1i + e2i;
  o[2] = e1r;       o[3] = e1i;
  o[4] = e2r;       o[5] = e2i;
}

}  // namespace

int run_sum_slots(double* dst, const double* const* slots, int G, long n, cudaStream_t st) {
  SlotPtrs s;
  for (int r = 0; r < kMaxGroup; ++r) s.p[r] = r < G ? slots[r] : nullptr;
  const long n2 = n / 2;
  long blocks = (n2 + 255) / 256;
  if (blocks > 148 * 16) blocks = 148 * 16;
  if (blocks < 1) blocks = 1;
  sum_slots_kernel<<<(unsigned)blocks, 256, 0, st>>>(dst, s, G, n2);
  return 1;
}

int run_push_e2(double* dst, const double* E, int n, cudaStream_t st) {
  push_e2_kernel<<<(n + 127) / 128, 128, 0, st>>>(dst, E, n);
  return 1;
}

int run_energy_finish(double* E_out, const double* e1, const double* const* slots, int G, int nblk, double sf,
                      int nw, cudaStream_t st) {
  SlotPtrs s;
  for (int r = 0; r < kMaxGroup; ++r) s.p[r] = r < G ? slots[r] : nullptr;
  energy_finish_kernel<<<(nw + 127) / 128, 128, 0, st>>>(E_out, e1, s, G, nblk, sf, nw);
  return 1;
}

}  // namespace afq
