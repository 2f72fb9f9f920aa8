// noise.cu — noise loading: mmf_add_noise (section 6: "White noise is added to the signals before the
// receiver, setting the optical signal-to-noise ratio (OSNR) to 20 dB"; reading R18 in DESIGN.md section 2).
//
// Two kernels on the caller's stream, no plan, no workspace:
//   k_mode_power   P_a = (1/N) sum_t (|A_ax(t)|^2 + |A_ay(t)|^2), one CTA per spatial mode (the two rows of a mode are
//                  2N contiguous complex samples), fixed summation tree: the result depends on N only, not on the
//                  launch, so repeated calls give the same noise level bit for bit;
//   k_add_noise    A_{a,p}(t) += sigma_a z(seed, 2a+p, t), sigma_a^2 = P_a / (nch 2 B_ref OSNR dt), z a unit complex
//                  normal sample from Philox-4x32-10 (counter = (t low, t high, row, 0), key = the seed's two words)
//                  and Box-Muller.  One read and one write of the field (2 F), everything else in registers; the
//                  generator is counter-based, so a sample depends on (seed, row, t) alone and not on the grid.
// Written from the generator's published definition (Salmon, Moraes, Dror, Shaw, SC'11), independently of the oracle.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdint>

#include "../../include/mmf.h"

namespace mmf {
int note_cuda_error(cudaError_t e);   // mmf_api.cu
}

namespace {

constexpr int kPowThreads = 1024;
constexpr int kPowUnroll = 8;
constexpr int kNoiseThreads = 256;

// grid = M, block = 1024.  Thread j sums the samples j, j + 1024, ... of the mode's 2N contiguous samples into
// kPowUnroll interleaved accumulators (independent loads in flight), then the CTA reduces: accumulators in index
// order, lanes by shuffle (xor 16 .. 1), warps in index order.
__global__ void __launch_bounds__(kPowThreads) k_mode_power(const double2* __restrict__ A, double* __restrict__ P,
                                                             long long N) {
  __shared__ double wsum[kPowThreads / 32];
  const double2* row = A + (size_t)blockIdx.x * 2 * (size_t)N;
  const long long n2 = 2 * N;
  double acc[kPowUnroll];
#pragma unroll
  for (int u = 0; u < kPowUnroll; ++u) acc[u] = 0.0;
  long long i = threadIdx.x;
  for (; i + (long long)(kPowUnroll - 1) * kPowThreads < n2; i += (long long)kPowUnroll * kPowThreads) {
    double2 v[kPowUnroll];
#pragma unroll
    for (int u = 0; u < kPowUnroll; ++u) v[u] = row[i + (long long)u * kPowThreads];
#pragma unroll
    for (int u = 0; u < kPowUnroll; ++u) acc[u] += v[u].x * v[u].x + v[u].y * v[u].y;
  }
  double tail = 0.0;
  for (; i < n2; i += kPowThreads) {
    const double2 v = row[i];
    tail += v.x * v.x + v.y * v.y;
  }
  double s = 0.0;
#pragma unroll
  for (int u = 0; u < kPowUnroll; ++u) s += acc[u];
  s += tail;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if ((threadIdx.x & 31) == 0) wsum[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0.0;
    for (int w = 0; w < kPowThreads / 32; ++w) t += wsum[w];
    P[blockIdx.x] = t / (double)N;
  }
}

// Philox-4x32, 10 rounds: round function (hi, lo of M0 c0 and M1 c2; xor with the neighbours and the key), key bumped
// by the two Weyl constants between rounds.
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1,
                                              uint32_t (&out)[4]) {
  constexpr uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t hi0 = __umulhi(M0, c0), lo0 = M0 * c0, hi1 = __umulhi(M1, c2), lo1 = M1 * c2;
    const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
    c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    k0 += W0;   // the bump after the last round is dead code
    k1 += W1;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// two words -> (k + 1/2) 2^-52 with k the top 52 bits of (hi : lo): the open unit interval, every value exact
__device__ __forceinline__ double unit_open(uint32_t hi, uint32_t lo) {
  const unsigned long long k = ((unsigned long long)hi << 20) | (unsigned long long)(lo >> 12);
  return ((double)k + 0.5) * 0x1p-52;
}

// grid = (ceil(N / 256) capped, 2M), block = 256: blockIdx.y is the row, the CTA strides over its samples.
__global__ void __launch_bounds__(kNoiseThreads) k_add_noise(double2* __restrict__ A, const double* __restrict__ P,
                                                              long long N, double dt, double osnr, double ref_bw, int nch,
                                                              uint32_t seed_lo, uint32_t seed_hi) {
  __shared__ double sigma_s;
  const uint32_t r = blockIdx.y;
  if (threadIdx.x == 0) sigma_s = sqrt(P[r >> 1] / (double)nch / (2.0 * ref_bw * osnr) / dt);
  __syncthreads();
  const double sigma = sigma_s;
  if (!(sigma > 0.0)) return;       // no signal in this mode, or an infinite OSNR: nothing is added
  double2* row = A + (size_t)r * (size_t)N;
  for (long long t = (long long)blockIdx.x * kNoiseThreads + threadIdx.x; t < N; t += (long long)gridDim.x * kNoiseThreads) {
    uint32_t w[4];
    philox4x32_10((uint32_t)t, (uint32_t)((unsigned long long)t >> 32), r, 0u, seed_lo, seed_hi, w);
    const double u1 = unit_open(w[0], w[1]), u2 = unit_open(w[2], w[3]);
    const double rad = sigma * sqrt(-log(u1));
    double sn, cs;
    sincospi(2.0 * u2, &sn, &cs);
    double2 v = row[t];
    v.x += rad * cs;
    v.y += rad * sn;
    row[t] = v;
  }
}

__global__ void k_noise_words(uint32_t* __restrict__ out, uint32_t seed_lo, uint32_t seed_hi, uint32_t row,
                              unsigned long long t0, long long count) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= count) return;
  const unsigned long long t = t0 + (unsigned long long)i;
  uint32_t w[4];
  philox4x32_10((uint32_t)t, (uint32_t)(t >> 32), row, 0u, seed_lo, seed_hi, w);
  reinterpret_cast<uint4*>(out)[i] = make_uint4(w[0], w[1], w[2], w[3]);
}

}  // namespace

extern "C" {

int mmf_add_noise(void* A_dev, int M, long long N, double dt, double osnr_db, double ref_bw, int nch,
                  unsigned long long seed, double* mode_power_dev, void* cuda_stream) {
  if (!A_dev || !mode_power_dev || M < 1 || M > 32767 || N < 1 || nch < 1) return MMF_EINVAL;
  if (!(dt > 0) || !std::isfinite(dt) || !(ref_bw > 0) || !std::isfinite(ref_bw) || std::isnan(osnr_db)) return MMF_EINVAL;
  if ((reinterpret_cast<size_t>(A_dev) & 15) || (reinterpret_cast<size_t>(mode_power_dev) & 7)) return MMF_EINVAL;
  const double osnr = std::pow(10.0, osnr_db / 10.0);   // +inf dB -> inf -> sigma = 0 -> nothing added
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  double2* A = static_cast<double2*>(A_dev);
  k_mode_power<<<(unsigned)M, kPowThreads, 0, st>>>(A, mode_power_dev, N);
  long long gx = (N + kNoiseThreads - 1) / kNoiseThreads;
  if (gx > 65536) gx = 65536;
  k_add_noise<<<dim3((unsigned)gx, (unsigned)(2 * M)), kNoiseThreads, 0, st>>>(A, mode_power_dev, N, dt, osnr, ref_bw, nch,
                                                                               (uint32_t)seed, (uint32_t)(seed >> 32));
  const cudaError_t e = cudaGetLastError();
  return e == cudaSuccess ? MMF_OK : mmf::note_cuda_error(e);
}

int mmf_debug_noise_words(unsigned long long seed, unsigned row, unsigned long long t0, long long count, void* words_dev,
                          void* cuda_stream) {
  if (!words_dev || count < 0 || (reinterpret_cast<size_t>(words_dev) & 15)) return MMF_EINVAL;
  if (count == 0) return MMF_OK;
  k_noise_words<<<(unsigned)((count + 255) / 256), 256, 0, reinterpret_cast<cudaStream_t>(cuda_stream)>>>(
      static_cast<uint32_t*>(words_dev), (uint32_t)seed, (uint32_t)(seed >> 32), row, t0, count);
  const cudaError_t e = cudaGetLastError();
  return e == cudaSuccess ? MMF_OK : mmf::note_cuda_error(e);
}

}  // extern "C"
