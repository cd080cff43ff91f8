// comb_static.cu - afqmc_comb_static: the comb of the population control ("population control", PAPER.md:185, 489;
// DESIGN.md reading S21) for callers that cannot allocate device memory.
//
// Every other entry point of the library works on an afqmc_handle, and afqmc_create sizes and cudaMallocs the
// workspaces of the whole walker step - among them cum[nw], the running sum of the weights that the comb bisects.
// A driver that only wants to resample (it holds weights, not a Hamiltonian), or that runs where the device has no
// memory left to give - the Cholesky tensor plus a framework's caching allocator own all of HBM, so cudaMalloc
// returns out-of-memory - or that may not stall its other streams on the implicit device synchronisation of
// cudaMalloc / cudaFree, cannot pay for that.  For it the one scratch array of the comb lives in the library image
// itself: g_comb_cum below, 512 KiB, present on every GPU that loads libafqmc.so from the moment the module is loaded
// until the process exits, whether or not this entry point is ever called.
//
// The arithmetic is the handle path's (block.cu, comb_kernel) to the last bit - floating point decides integers
// here: sequential left-to-right sum, one division, one add and one multiply per tooth without FMA contraction,
// comparison cum[j] <= tooth.
#include <cstdio>

#include "internal.h"

// The scratch.  In HOST code this name is only the host-side shadow that nvcc generates for the symbol - it is not
// a device address and must never be handed to a kernel; cum_on_device() asks the runtime for the real one.
static __device__ __align__(256) double g_comb_cum[AFQMC_COMB_STATIC_MAX_WALKERS];

namespace {

constexpr int kMaxDev = 64;

std::mutex g_mu;
double* g_cum_addr[kMaxDev];   // device address of g_comb_cum on device d; nullptr = not looked up yet

// Once per device, with that device current: the address of this device's copy of g_comb_cum.
cudaError_t cum_on_device(int dev, double** out) {
  std::lock_guard<std::mutex> lk(g_mu);
  if (!g_cum_addr[dev]) {
    double* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress((void**)&p, g_comb_cum);
    if (e != cudaSuccess) return e;
    g_cum_addr[dev] = p;
  }
  *out = g_cum_addr[dev];
  return cudaSuccess;
}

// One CTA.  cum[0 .. nw) is written by thread 0 before anybody reads it and nothing beyond nw is read, so what an
// earlier call left in the array never matters and nothing has to be cleared.
__global__ void __launch_bounds__(256) comb_static_kernel(double* weights, const double* xi_p, double* cum, int* map,
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
  if (!s_ok) {                       // total weight zero, negative or not finite: identity map, weights untouched
    for (int k = threadIdx.x; k < nw; k += blockDim.x) map[k] = k;
    return;
  }
  double xi = *xi_p;                 // clamped into [0, 1), NaN -> 0, as on the handle path
  xi = xi >= 0.0 ? (xi < 1.0 ? xi : 0x1.fffffffffffffp-1) : 0.0;
  const double spacing = s_spacing;
  const int last = s_last;
  for (int k = threadIdx.x; k < nw; k += blockDim.x) {
    const double tooth = __dmul_rn(__dadd_rn((double)k, xi), spacing);
    int lo = 0, hi = nw;             // #{j : cum[j] <= tooth}
    while (lo < hi) {
      const int mid = (lo + hi) >> 1;
      if (cum[mid] <= tooth) lo = mid + 1; else hi = mid;
    }
    map[k] = lo < last ? lo : last;
    weights[k] = spacing;
  }
}

int32_t fail(char* err, int32_t err_len, int32_t code, const char* what, const char* detail = nullptr) {
  if (err && err_len > 0) {
    if (detail) snprintf(err, (size_t)err_len, "afqmc_comb_static: %s: %s", what, detail);
    else snprintf(err, (size_t)err_len, "afqmc_comb_static: %s", what);
  }
  return code;
}

// device that holds p, or -1 for anything that is not plain device memory
int device_memory_of(const void* p) {
  cudaPointerAttributes at;
  if (cudaPointerGetAttributes(&at, p) != cudaSuccess) {
    cudaGetLastError();
    return -1;
  }
  return at.type == cudaMemoryTypeDevice ? at.device : -1;
}

}  // namespace

extern "C" int32_t afqmc_comb_static(double* weights, const double* xi, int32_t* map_out, int32_t nw, void* stream,
                                     char* err, int32_t err_len) {
  if (err && err_len > 0) err[0] = 0;
  if (!weights || !xi || !map_out) return fail(err, err_len, AFQMC_ERR_INVALID, "null argument");
  if (nw <= 0) return fail(err, err_len, AFQMC_ERR_DIMS, "nw must be positive");
  if (nw > AFQMC_COMB_STATIC_MAX_WALKERS) {
    char msg[256];
    snprintf(msg, sizeof msg, "nw = %d is more than the %d walkers the built-in scratch array holds "
             "(AFQMC_COMB_STATIC_MAX_WALKERS); use afqmc_population_control on a handle", nw,
             AFQMC_COMB_STATIC_MAX_WALKERS);
    return fail(err, err_len, AFQMC_ERR_DIMS, msg);
  }
  const int dev = device_memory_of(weights);
  if (dev < 0 || device_memory_of(xi) != dev || device_memory_of(map_out) != dev)
    return fail(err, err_len, AFQMC_ERR_INVALID, "weights, xi and map_out must be device memory of one GPU");
  if (dev >= kMaxDev) return fail(err, err_len, AFQMC_ERR_UNSUPPORTED, "device ordinal above 63");

  int prev = -1;
  cudaGetDevice(&prev);
  if (prev != dev && cudaSetDevice(dev) != cudaSuccess) {
    const cudaError_t e = cudaGetLastError();
    return fail(err, err_len, AFQMC_ERR_CUDA, "cudaSetDevice", cudaGetErrorString(e));
  }
  int32_t rc = AFQMC_OK;
  double* cum = nullptr;
  cudaError_t e = cum_on_device(dev, &cum);
  if (e != cudaSuccess) {
    cudaGetLastError();
    rc = fail(err, err_len, AFQMC_ERR_CUDA, "cudaGetSymbolAddress", cudaGetErrorString(e));
  } else {
    comb_static_kernel<<<1, 256, 0, (cudaStream_t)stream>>>(weights, xi, cum, map_out, nw);
    e = cudaGetLastError();
    if (e != cudaSuccess) rc = fail(err, err_len, AFQMC_ERR_CUDA, "kernel launch", cudaGetErrorString(e));
  }
  if (prev != dev && prev >= 0) cudaSetDevice(prev);
  return rc;
}
