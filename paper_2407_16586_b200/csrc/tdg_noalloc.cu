// tdg_noalloc.cu — allocation-free entry point: Rys roots and weights (step a5) evaluated with ALL device
// workspace in a fixed file-scope device array, for callers that may not call cudaMalloc (code under CUDA graph capture, tight
// serving loops, harnesses that forbid allocation).  tdg_rys (tdg_api.cu) stages its arguments and results in three cudaMalloc'ed
// temporaries; tdg_rys_static stages them here instead and calls no cudaMalloc, cudaFree or allocating library routine.
//
// The array is held by every GPU that loads the library until the process exits (TDG_STATIC_SCRATCH_BYTES = 2 MiB + 256 B).
// ALL calls on a device share it and it keeps the last call's contents: the kernel reads and writes only the first `count`
// entries of each region, which the call has just uploaded or overwrites, and the one word that must start at zero (the
// invalid-argument counter) is cleared by every call.  Two calls that overlap on the GPU (different streams, different host
// threads, different contexts on one device) RACE on the array: callers serialise them.
//
// In host code the NAME of a __device__ array is a host-side stand-in, not a device address: a kernel handed `g_scratch` from the
// host would fault (or, where the GPU can reach host memory, silently use the wrong memory).  Host code therefore asks
// cudaGetSymbolAddress for the device address once per device, with that device current (scratch_address below); device code in
// this file names the array directly.
#include "tdg_common.cuh"
#include "tdg_internal.h"

#define TDG_STATIC_ITEM_DOUBLES (2 + 2 * RYS_NMAX)                      // T, rho, 2n <= 14 results per evaluation
#define TDG_STATIC_FLAG_DOUBLES 32                                      // one 256-byte line for the invalid-argument counter
#define TDG_STATIC_SCRATCH_DOUBLES (TDG_RYS_STATIC_MAX * TDG_STATIC_ITEM_DOUBLES + TDG_STATIC_FLAG_DOUBLES)
// regions: [0, MAX) T | [MAX, 2 MAX) rho | [2 MAX, 2 MAX + 14 MAX) results | 32 doubles: counter
#define TDG_STATIC_OFF_RHO TDG_RYS_STATIC_MAX
#define TDG_STATIC_OFF_OUT (2 * TDG_RYS_STATIC_MAX)
#define TDG_STATIC_OFF_FLAG (TDG_RYS_STATIC_MAX * TDG_STATIC_ITEM_DOUBLES)

static __device__ __align__(256) double g_scratch[TDG_STATIC_SCRATCH_DOUBLES];

// Same arithmetic as rys_test_kernel (tdg_aux.cu), operands and results in g_scratch (named directly: this is device code).
template <int N>
__global__ void rys_static_kernel(int count, double omega, const double* __restrict__ tab) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= count) return;
  const double T = g_scratch[i], rho = g_scratch[TDG_STATIC_OFF_RHO + i];
  double* out = g_scratch + TDG_STATIC_OFF_OUT + (size_t)i * 2 * N;
  if (!(T >= 0.0) || !(rho > 0.0) || isinf(T)) {   // also catches NaN
    atomicAdd(reinterpret_cast<unsigned long long*>(g_scratch + TDG_STATIC_OFF_FLAG), 1ULL);
    for (int r = 0; r < 2 * N; ++r) out[r] = 0.0;
    return;
  }
  double s2 = 1.0, ss = 1.0;
  if (omega > 0.0) { s2 = omega * omega / (omega * omega + rho); ss = sqrt(s2); }
  double x[N], w[N];
  rys_roots<N>(tab, s2 * T, x, w);
  for (int r = 0; r < N; ++r) { out[r] = x[r] * s2; out[N + r] = w[r] * ss; }
}

// Device address of g_scratch on `device` (which must be current): looked up once per device, then cached.
#define TDG_STATIC_MAX_DEVICES 64
static cudaError_t scratch_address(int device, double** ptr) {
  static double* cache[TDG_STATIC_MAX_DEVICES] = {};
  if (device < 0 || device >= TDG_STATIC_MAX_DEVICES) return cudaErrorInvalidDevice;
  double* p = cache[device];   // a racing first call on two host threads looks the same address up twice: harmless
  if (!p) {
    const cudaError_t e = cudaGetSymbolAddress((void**)&p, g_scratch);
    if (e != cudaSuccess) return e;
    cache[device] = p;
  }
  *ptr = p;
  return cudaSuccess;
}

int tdg_rys_static_max(void) { return TDG_RYS_STATIC_MAX; }

// Host T, rho -> g_scratch, kernel, g_scratch -> host out; *nbad = number of invalid (T, rho) arguments seen by the kernel.
// The device of `tab` must be current.  No allocation.
cudaError_t tdg_run_rys_static(int device, int n, int count, const double* T, const double* rho, double omega, const double* tab, double* out,
                               unsigned long long* nbad, cudaStream_t s) {
  if (n < 1 || n > RYS_NMAX || count < 1 || count > TDG_RYS_STATIC_MAX) return cudaErrorInvalidValue;
  double* scr = nullptr;
  cudaError_t e = scratch_address(device, &scr);
  if (e != cudaSuccess) return e;
  if ((e = cudaMemsetAsync(scr + TDG_STATIC_OFF_FLAG, 0, sizeof(double) * TDG_STATIC_FLAG_DOUBLES, s)) != cudaSuccess) return e;   // must start at zero
  if ((e = cudaMemcpyAsync(scr, T, sizeof(double) * count, cudaMemcpyHostToDevice, s)) != cudaSuccess) return e;
  if ((e = cudaMemcpyAsync(scr + TDG_STATIC_OFF_RHO, rho, sizeof(double) * count, cudaMemcpyHostToDevice, s)) != cudaSuccess) return e;
  const int nb = (count + 127) / 128;
  switch (n) {
    case 1: rys_static_kernel<1><<<nb, 128, 0, s>>>(count, omega, tab); break;
    case 2: rys_static_kernel<2><<<nb, 128, 0, s>>>(count, omega, tab); break;
    case 3: rys_static_kernel<3><<<nb, 128, 0, s>>>(count, omega, tab); break;
    case 4: rys_static_kernel<4><<<nb, 128, 0, s>>>(count, omega, tab); break;
    case 5: rys_static_kernel<5><<<nb, 128, 0, s>>>(count, omega, tab); break;
    case 6: rys_static_kernel<6><<<nb, 128, 0, s>>>(count, omega, tab); break;
    default: rys_static_kernel<7><<<nb, 128, 0, s>>>(count, omega, tab); break;
  }
  if ((e = cudaGetLastError()) != cudaSuccess) return e;
  if ((e = cudaMemcpyAsync(out, scr + TDG_STATIC_OFF_OUT, sizeof(double) * (size_t)count * 2 * n, cudaMemcpyDeviceToHost, s)) != cudaSuccess) return e;
  if ((e = cudaMemcpyAsync(nbad, scr + TDG_STATIC_OFF_FLAG, sizeof(unsigned long long), cudaMemcpyDeviceToHost, s)) != cudaSuccess) return e;
  return cudaStreamSynchronize(s);
}
