// nl_static.cu — mmf_apply_nonlinear_static: the Kerr operator of Eq. (1) for callers that must not
// allocate device memory.
//
// Who that is.  Everything else in this library is driven by a plan: mmf_plan_create cudaMallocs the plan's tables and
// the caller cudaMallocs (or lets torch allocate) a workspace.  Some hosts of this code can do neither.  A link
// simulator that has handed all of HBM to its own pool at start-up (several 15 GiB field copies do that quickly) gets
// "out of memory" from any later cudaMalloc; a framework with a caching allocator does not want a library to go behind
// the pool's back; and a caller inside a latency-critical loop or a driver callback cannot afford cudaMalloc /
// cudaFree at all, because both synchronise the whole device.  For those callers this file offers ONE entry point
// that takes the coupling matrix, the input field and the output field as device pointers the caller already owns and
// calls no cudaMalloc, no cudaFree and no library routine that allocates.
//
// What it runs.  The two-kernel form of the nonlinear step that the paper's Listing 1 and this library's row-sharded
// path use (nl_shard.cuh: k_shard_pow / k_shard_apply): first the mode powers P_b(t) = |U_bx(t)|^2 + |U_by(t)|^2 are
// written to global memory as a REAL [M][N] matrix ("calc_squareabs"), then every row takes
// S_a(t) = sum_b kappa_ab P_b(t) and OUT_{a,p}(t) = i h gamma S_a(t) U_{a,p}(t).  In the sharded
// path that power matrix is a buffer the caller allocates; here it lives in the file-scope device array below.
//
// The price of a static array, stated once:
//   * it has a fixed size, MMF_STATIC_SCRATCH_BYTES (4 MiB = 524 288 powers): M * N beyond that is refused with
//     MMF_ETOOBIG, nothing is launched;
//   * every GPU on which this library's code is loaded holds those 4 MiB until the process exits;
//   * all calls on a device share the one array.  A call overwrites the M * N entries it needs before it reads them, so
//     nothing has to be cleared and what the previous call left behind is never read; but two calls whose kernels can
//     be on the GPU at the same time (two streams, two host threads) race on it.  Keep calls on one device in one
//     stream, or order them yourself.
//   * the array's name means something different in host and in device code.  Kernels in this file could name it
//     directly; host code may not hand `g_static_powers` to a kernel as if it were a pointer (that is the address of a
//     host-side shadow object).  The device address is asked for with cudaGetSymbolAddress, once per device, on the
//     first call made with that device current, and remembered.  That first call may also make the CUDA runtime load
//     this module on the device, so make it once during set-up, before any stream capture is begun.
#include <cuda_runtime.h>

#include <cmath>
#include <mutex>

#include "../../include/mmf.h"

namespace {

constexpr long long kMaxPowers = (long long)(MMF_STATIC_SCRATCH_BYTES / sizeof(double));

// The scratch: P[b * N + t], b < M, t < N, for the call in flight.  256-byte aligned so that every row of a
// power-of-two N >= 32 starts on a full memory segment.
static __device__ __align__(256) double g_static_powers[kMaxPowers];

constexpr int kLanes = 32;   // consecutive time samples handled by one warp: 256-byte segments of P, 512-byte of U
constexpr int kWarps = 8;    // warps of a CTA stride over the modes

struct double2c { double re, im; };

// P[b][t] = |U_bx(t)|^2 + |U_by(t)|^2.  grid = ceil(N / 32), block = 256.
__global__ void __launch_bounds__(kLanes * kWarps) k_static_pow(const double2c* __restrict__ U, double* __restrict__ P,
                                                                 int M, long long N) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const long long t = (long long)blockIdx.x * kLanes + lane;
  if (t >= N) return;
  for (int b = warp; b < M; b += kWarps) {
    const double2c ux = U[(2LL * b) * N + t], uy = U[(2LL * b + 1) * N + t];
    P[(long long)b * N + t] = (ux.re * ux.re + ux.im * ux.im) + (uy.re * uy.re + uy.im * uy.im);
  }
}

// S_a(t) = sum_b kappa[a][b] P[b][t] (b ascending, one fused multiply-add per term: the order of nl_simt.cuh), then
// OUT_{a,p}(t) = i hg S_a(t) U_{a,p}(t).  U is read and OUT written by the same thread at the same index, so OUT may
// be U itself.  P is at most 4 MiB and stays in L2 between the two kernels and over the M passes of this loop.
__global__ void __launch_bounds__(kLanes * kWarps) k_static_apply(const double2c* U, double2c* OUT,
                                                                   const double* __restrict__ P,
                                                                   const double* __restrict__ kappa, double hg, int M,
                                                                   long long N) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const long long t = (long long)blockIdx.x * kLanes + lane;
  if (t >= N) return;
  for (int a = warp; a < M; a += kWarps) {
    const double* kr = kappa + (long long)a * M;
    double S = 0.0;
    for (int b = 0; b < M; ++b) S = fma(__ldg(kr + b), P[(long long)b * N + t], S);
    const double g = hg * S;
#pragma unroll
    for (int pol = 0; pol < 2; ++pol) {
      const long long i = (2LL * a + pol) * N + t;
      const double2c u = U[i];
      double2c k;
      k.re = -g * u.im;
      k.im = g * u.re;
      OUT[i] = k;
    }
  }
}

// Device address of g_static_powers, per device, filled on the first call made with that device current.
constexpr int kMaxDevices = 64;
std::mutex g_setup_mutex;
double* g_powers_addr[kMaxDevices] = {};

// Returns cudaSuccess and the address, or the error of the failing runtime call.
cudaError_t static_powers_address(double** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_setup_mutex);
  if (g_powers_addr[dev] == nullptr) {
    double* p = nullptr;
    e = cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_static_powers);   // NOT &g_static_powers: see the header comment
    if (e != cudaSuccess) return e;
    if (p == nullptr) return cudaErrorInvalidSymbol;
    g_powers_addr[dev] = p;
  }
  *out = g_powers_addr[dev];
  return cudaSuccess;
}

}  // namespace

namespace mmf {
int note_cuda_error(cudaError_t e);   // mmf_api.cu: records the text mmf_status_string(MMF_ECUDA) returns
}

extern "C" {

int mmf_apply_nonlinear_static(int M, long long N, double h, double gamma, const double* kappa_dev, const void* U_dev,
                               void* OUT_dev, void* cuda_stream) {
  if (M < 1 || N < 1 || kappa_dev == nullptr || U_dev == nullptr || OUT_dev == nullptr) return MMF_EINVAL;
  if (!std::isfinite(h) || !std::isfinite(gamma)) return MMF_EINVAL;
  if ((reinterpret_cast<size_t>(U_dev) & 15) || (reinterpret_cast<size_t>(OUT_dev) & 15) ||
      (reinterpret_cast<size_t>(kappa_dev) & 7))
    return MMF_EINVAL;
  if (N > kMaxPowers / M) return MMF_ETOOBIG;            // M * N powers would not fit the static array
  const long long tiles = (N + kLanes - 1) / kLanes;      // <= 16384
  double* P = nullptr;
  cudaError_t e = static_powers_address(&P);
  if (e != cudaSuccess) return mmf::note_cuda_error(e);
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  const double2c* U = static_cast<const double2c*>(U_dev);
  k_static_pow<<<(unsigned)tiles, kLanes * kWarps, 0, st>>>(U, P, M, N);
  k_static_apply<<<(unsigned)tiles, kLanes * kWarps, 0, st>>>(U, static_cast<double2c*>(OUT_dev), P, kappa_dev, h * gamma,
                                                              M, N);
  e = cudaGetLastError();
  return e == cudaSuccess ? MMF_OK : mmf::note_cuda_error(e);
}

}  // extern "C"
