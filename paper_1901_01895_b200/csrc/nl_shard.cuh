// nl_shard.cuh — the nonlinear step of the ROW-SHARDED propagation (sections 4.1-4.3:
// "each process stores and modifies only a part of the signal matrix ... the squared absolute values have to be
// shared between the GPUs", Listing 1: calc_squareabs / all-gather / calc_nonlinear_own + others / apply_nonlinear_all).
//
// A rank owns M_local spatial modes (2 M_local rows) of a fibre with M_total modes, modes mode0 .. mode0 + M_local - 1.
// One evaluation of N = i h gamma (sum_b kappa_ab P_b) is two kernels with a collective between them:
//   k_shard_pow<STAGE>     P_all[mode0 + a][t] = |u_ax(t)|^2 + |u_ay(t)|^2   for the rank's own modes (real, PAPER.md:111:
//                          "stored real to halve the traffic"), u the argument of the stage's N;
//   (all-gather of the M_total x N real matrix P_all: torch.distributed / NCCL, driven by sharded.py)
//   k_shard_apply<STAGE>   S_a(t) = sum_{b < M_total} kappa_rows[a][b] P_all[b][t] for the own rows, then the stage sums
//                          of Eq. (6b)-(6f) in the four-buffer plan of nl_simt.cuh (one N evaluation per launch — an
//                          all-gather separates consecutive evaluations, so (6c)/(6d) cannot share a pass here).
// Stages: 0 PLAIN  Y <- NL(X);  1 STAGE2  Z <- NL(X + Y/2);  2 STAGE3  k3 = NL(X + Z/2), W <- X + k3,
//         Z <- X + Y/6 + Z/3 + k3/3;  3 FINAL  X <- gain (Z + NL(W)/6).
// Layout: lane = time sample (32 consecutive samples: 512-byte row segments of the fields, 256-byte segments of P),
// warps stride over the modes; the contraction runs on the plain fp64 pipe with P staged in shared memory.  The path is
// bound by the collective (M_total N 8 bytes per evaluation), not by these kernels.
#pragma once
#include "async_copy.cuh"
#include "fft_core.cuh"

namespace mmf {

enum { SH_PLAIN = 0, SH_STAGE2 = 1, SH_STAGE3 = 2, SH_FINAL = 3 };

struct ShardParams {
  cpx* X;
  cpx* Y;
  cpx* Z;
  cpx* W;
  const double* __restrict__ kappa_rows;  // [M_local][M_total]
  double* P_all;                          // [M_total][N]
  double hg, gain;
  int M_local, M_total, mode0;
  long long N;
};

#define MMF_SH_T 32
#define MMF_SH_WARPS 8

template <int STAGE>
__device__ __forceinline__ cpx shard_arg(const ShardParams& p, long long i) {
  if constexpr (STAGE == SH_PLAIN) {
    return p.X[i];
  } else if constexpr (STAGE == SH_STAGE2) {
    const cpx x = p.X[i], y = p.Y[i];
    return make_double2(fma(0.5, y.x, x.x), fma(0.5, y.y, x.y));
  } else if constexpr (STAGE == SH_STAGE3) {
    const cpx x = p.X[i], z = p.Z[i];
    return make_double2(fma(0.5, z.x, x.x), fma(0.5, z.y, x.y));
  } else {
    return p.W[i];
  }
}

// grid = ceil(N / 32), block = 256
template <int STAGE>
__global__ void __launch_bounds__(MMF_SH_T* MMF_SH_WARPS) k_shard_pow(ShardParams p) {
  pdl_launch_dependents();
  pdl_wait();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const long long tt = (long long)blockIdx.x * MMF_SH_T + lane;
  if (tt >= p.N) return;
  for (int a = warp; a < p.M_local; a += MMF_SH_WARPS) {
    const cpx ux = shard_arg<STAGE>(p, (2LL * a) * p.N + tt), uy = shard_arg<STAGE>(p, (2LL * a + 1) * p.N + tt);
    p.P_all[(long long)(p.mode0 + a) * p.N + tt] = (ux.x * ux.x + ux.y * ux.y) + (uy.x * uy.x + uy.y * uy.y);
  }
}

// grid = ceil(N / 32), block = 256, dynamic shared memory = M_total * 32 doubles
template <int STAGE>
__global__ void __launch_bounds__(MMF_SH_T* MMF_SH_WARPS) k_shard_apply(ShardParams p) {
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  double* P = reinterpret_cast<double*>(smem_raw);
  pdl_launch_dependents();
  pdl_wait();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const long long tt = (long long)blockIdx.x * MMF_SH_T + lane;
  const bool live = tt < p.N;
  for (int b = warp; b < p.M_total; b += MMF_SH_WARPS) P[b * MMF_SH_T + lane] = live ? p.P_all[(long long)b * p.N + tt] : 0.0;
  __syncthreads();
  const double third = 1.0 / 3.0, sixth = 1.0 / 6.0;
  for (int a = warp; a < p.M_local; a += MMF_SH_WARPS) {
    double S = 0.0;
    const double* kr = p.kappa_rows + (long long)a * p.M_total;
    for (int b = 0; b < p.M_total; ++b) S = fma(__ldg(kr + b), P[b * MMF_SH_T + lane], S);
    const double g = p.hg * S;
    if (!live) continue;
#pragma unroll
    for (int pol = 0; pol < 2; ++pol) {
      const long long i = (2LL * a + pol) * p.N + tt;
      const cpx u = shard_arg<STAGE>(p, i);
      const cpx k = make_double2(-g * u.y, g * u.x);
      if constexpr (STAGE == SH_PLAIN) {
        p.Y[i] = k;
      } else if constexpr (STAGE == SH_STAGE2) {
        p.Z[i] = k;
      } else if constexpr (STAGE == SH_STAGE3) {
        const cpx x = p.X[i], y = p.Y[i], z = p.Z[i];
        p.W[i] = cadd(x, k);
        p.Z[i] = make_double2(x.x + sixth * y.x + third * z.x + third * k.x, x.y + sixth * y.y + third * z.y + third * k.y);
      } else {
        const cpx z = p.Z[i];
        p.X[i] = make_double2(p.gain * fma(sixth, k.x, z.x), p.gain * fma(sixth, k.y, z.y));
      }
    }
  }
}

}  // namespace mmf
