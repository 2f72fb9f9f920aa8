// nl_simt.cuh — the fused nonlinear kernel on the plain FP64 pipe (DFMA), used when M exceeds what the tensor-path
// kernel of nl_tma.cuh keeps in registers (M > 120).  Rows a4-a7 of the hot-path table.
#pragma once
#include "async_copy.cuh"
#include "fft_core.cuh"

namespace mmf {

// ------------------------------------------------------------------------------------------- fused nonlinear kernel
// Eq. (1) PAPER.md:36 and the stage combinations of Eq. (6b)-(6f) PAPER.md:78-88.  With
//   NL(u)_{a,p}(t) = i * hg * (sum_b kappa_ab (|u_bx(t)|^2 + |u_by(t)|^2)) * u_{a,p}(t),   hg = h * gamma:
//   NL_PLAIN       Y  <- NL(X)                                                   (first k1 bracket, Eq. 6b)
//   NL_STAGE2      Z  <- NL(X + Y/2)                                X = A_I, Y = k1   (Eq. 6c)
//   NL_STAGE3      k3 = NL(X + Z/2);  W <- X + k3;  Z <- X + Y/6 + Z/3 + k3/3          (Eq. 6d and the brackets of 6e, 6f)
//   NL_FINAL       X  <- Z + NL(W)/6                                W = u4, Z = exp(h/2 L)[...]   (Eq. 6e, 6f)
//   NL_FINAL_NEXT  as NL_FINAL, and Y <- NL(X_new)                  (the next step's Eq. 6b bracket, fused)
enum { NL_PLAIN = 0, NL_STAGE2 = 1, NL_STAGE3 = 2, NL_FINAL = 3, NL_FINAL_NEXT = 4 };

struct NlParams {
  cpx* X;
  cpx* Y;
  cpx* Z;
  cpx* W;
  const double* __restrict__ kappa;  // [M][M]
  double hg;
  double gain;  // NL_FINAL / NL_FINAL_NEXT: amplitude factor of a lumped amplifier applied to the new field (1 = none)
  int M;
  long long N;
};

#define MMF_NL_T 32
#define MMF_NL_WARPS 8

template <int MODE>
__device__ __forceinline__ cpx nl_arg(const NlParams& p, long long i) {
  if constexpr (MODE == NL_PLAIN) {
    return p.X[i];
  } else if constexpr (MODE == NL_STAGE2) {
    const cpx x = p.X[i], y = p.Y[i];
    return make_double2(fma(0.5, y.x, x.x), fma(0.5, y.y, x.y));
  } else if constexpr (MODE == NL_STAGE3) {
    const cpx x = p.X[i], z = p.Z[i];
    return make_double2(fma(0.5, z.x, x.x), fma(0.5, z.y, x.y));
  } else {
    return p.W[i];
  }
}

// grid = ceil(N / 32); block = 256 (8 warps); lane = time sample inside the tile, warps stride over modes.
// dynamic shared memory: 2 * M * 32 doubles.
template <int MODE>
__global__ void __launch_bounds__(MMF_NL_T* MMF_NL_WARPS) k_nl(NlParams p) {
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  double* P1 = reinterpret_cast<double*>(smem_raw);
  double* P2 = P1 + (size_t)p.M * MMF_NL_T;
  pdl_launch_dependents();
  pdl_wait();   // every thread reads the predecessor's output from global memory
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const long long tt = (long long)blockIdx.x * MMF_NL_T + lane;
  const bool live = tt < p.N;
  const int M = p.M;
  for (int a = warp; a < M; a += MMF_NL_WARPS) {
    double pw = 0.0;
    if (live) {
      const cpx ux = nl_arg<MODE>(p, (2LL * a) * p.N + tt), uy = nl_arg<MODE>(p, (2LL * a + 1) * p.N + tt);
      pw = (ux.x * ux.x + ux.y * ux.y) + (uy.x * uy.x + uy.y * uy.y);
    }
    P1[a * MMF_NL_T + lane] = pw;
  }
  __syncthreads();
  for (int a = warp; a < M; a += MMF_NL_WARPS) {
    double S = 0.0;
    const double* kr = p.kappa + (long long)a * M;
    for (int b = 0; b < M; ++b) S = fma(__ldg(kr + b), P1[b * MMF_NL_T + lane], S);
    const double g = p.hg * S;
    double pw2 = 0.0;
    if (live) {
#pragma unroll
      for (int pol = 0; pol < 2; ++pol) {
        const long long i = (2LL * a + pol) * p.N + tt;
        const cpx u = nl_arg<MODE>(p, i);
        const cpx k = make_double2(-g * u.y, g * u.x);
        if constexpr (MODE == NL_PLAIN) {
          p.Y[i] = k;
        } else if constexpr (MODE == NL_STAGE2) {
          p.Z[i] = k;
        } else if constexpr (MODE == NL_STAGE3) {
          const cpx x = p.X[i], y = p.Y[i], z = p.Z[i];
          p.W[i] = cadd(x, k);
          const double third = 1.0 / 3.0, sixth = 1.0 / 6.0;
          p.Z[i] = make_double2(x.x + sixth * y.x + third * z.x + third * k.x,
                                x.y + sixth * y.y + third * z.y + third * k.y);
        } else {
          const cpx z = p.Z[i];
          const double sixth = 1.0 / 6.0;
          const cpx an = make_double2(p.gain * fma(sixth, k.x, z.x), p.gain * fma(sixth, k.y, z.y));
          p.X[i] = an;
          pw2 += an.x * an.x + an.y * an.y;
        }
      }
    }
    if constexpr (MODE == NL_FINAL_NEXT) P2[a * MMF_NL_T + lane] = pw2;
  }
  if constexpr (MODE == NL_FINAL_NEXT) {
    __syncthreads();
    for (int a = warp; a < M; a += MMF_NL_WARPS) {
      double S = 0.0;
      const double* kr = p.kappa + (long long)a * M;
      for (int b = 0; b < M; ++b) S = fma(__ldg(kr + b), P2[b * MMF_NL_T + lane], S);
      const double g = p.hg * S;
      if (live) {
#pragma unroll
        for (int pol = 0; pol < 2; ++pol) {
          const long long i = (2LL * a + pol) * p.N + tt;
          const cpx u = p.X[i];  // written above by this same thread
          p.Y[i] = make_double2(-g * u.y, g * u.x);
        }
      }
    }
  }
}

}  // namespace mmf
