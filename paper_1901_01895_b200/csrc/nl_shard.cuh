// nl_shard.cuh — the nonlinear step of the ROW-SHARDED propagation (sections 4.1-4.3:
// "each process stores and modifies only a part of the signal matrix ... the squared absolute values have to be
// shared between the GPUs", Listing 1: calc_squareabs / all-gather / calc_nonlinear_own + others / apply_nonlinear_all).
//
// A rank owns M_local spatial modes (2 M_local rows) of a fibre with M_total modes, modes mode0 .. mode0 + M_local - 1.
// One evaluation of N = i h gamma (sum_b kappa_ab P_b) is two kernels with a collective between them:
// Both kernels work on a TIME CHUNK [t_first, t_first + t_count) with its own contiguous [M_total][t_count] power block, so
// that the all-gather of one chunk overlaps the kernels of its neighbours (the B200 form of the paper's overlap of
// calc_nonlinear_own with the transfers; sharded.py pipelines them).
//   k_shard_pow<STAGE>     P_all[mode0 + a][t] = |u_ax(t)|^2 + |u_ay(t)|^2   for the rank's own modes (real, PAPER.md:111:
//                          "stored real to halve the traffic"), u the argument of the stage's N;
//   (all-gather of the M_total x N real matrix P_all: torch.distributed / NCCL, driven by sharded.py)
//   k_shard_apply<STAGE>   S_a(t) = sum_{b < M_total} kappa_rows[a][b] P_all[b][t] for the own rows, then the stage sums
//                          of Eq. (6b)-(6f) in the four-buffer plan of nl_simt.cuh (one N evaluation per launch — an
//                          all-gather separates consecutive evaluations, so (6c)/(6d) cannot share a pass here).
// Stages: 0 PLAIN  Y <- NL(X);  1 STAGE2  Z <- NL(X + Y/2);  2 STAGE3  k3 = NL(X + Z/2), W <- X + k3,
//         Z <- X + Y/6 + Z/3 + k3/3;  3 FINAL  X <- gain (Z + NL(W)/6).
// Layout: lane = time sample (32 consecutive samples: 512-byte row segments of the fields, 256-byte segments of P),
// warps stride over the modes; the contraction runs on the plain fp64 pipe with P and the kappa rows in shared memory.  The path is
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
  double* P_all;                          // [M_total][t_count]: the powers of samples t_first .. t_first + t_count - 1
  double hg, gain;
  int M_local, M_total, mode0;
  long long N;
  long long t_first, t_count;             // the time chunk this launch works on (the whole axis: 0, N)
};

#define MMF_SH_T 32
#define MMF_SH_WARPS 16

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

// grid = ceil(t_count / 32), block = 512
template <int STAGE>
__global__ void __launch_bounds__(MMF_SH_T* MMF_SH_WARPS) k_shard_pow(ShardParams p) {
  pdl_launch_dependents();
  pdl_wait();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const long long tc = (long long)blockIdx.x * MMF_SH_T + lane;   // sample inside the chunk
  if (tc >= p.t_count) return;
  const long long tt = p.t_first + tc;
  for (int a = warp; a < p.M_local; a += MMF_SH_WARPS) {
    const cpx ux = shard_arg<STAGE>(p, (2LL * a) * p.N + tt), uy = shard_arg<STAGE>(p, (2LL * a + 1) * p.N + tt);
    p.P_all[(long long)(p.mode0 + a) * p.t_count + tc] = (ux.x * ux.x + ux.y * ux.y) + (uy.x * uy.x + uy.y * uy.y);
  }
}

// Persistent: grid = a multiple of the SM count, every CTA walks the 32-sample tiles blockIdx.x, + gridDim.x, ...
// block = 512 (16 warps; lane = sample).  Dynamic shared memory: the rank's kappa rows TRANSPOSED and padded,
// ks[b][a] (a < MP = M_local rounded up to 4; loaded once per CTA), the power tile P[b][32] and the result S[a][32].
// Three phases per tile, so that the global loads of a phase are all in flight together (the kernel is bound by
// memory latency otherwise: it has few warps per SM):
//   1. P tile <- P_all (coalesced 256-byte rows);
//   2. S = kappa_rows * P from shared memory only; a warp computes FOUR modes at a time: per column b one read of
//      P[b][lane] and two broadcast 16-byte reads of ks[b][a..a+3] feed four FMAs;
//   3. the stage sums, four field rows per warp at a time: all loads of the four rows first, then the arithmetic.
__host__ __device__ inline size_t shard_apply_smem_bytes(int M_local, int M_total) {
  const int MP = (M_local + 3) & ~3;
  return sizeof(double) * ((size_t)M_total * MP + (size_t)M_total * MMF_SH_T + (size_t)MP * MMF_SH_T);
}
template <int STAGE>
__global__ void __launch_bounds__(MMF_SH_T* MMF_SH_WARPS) k_shard_apply(ShardParams p) {
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  const int MP = (p.M_local + 3) & ~3;
  double* ks = reinterpret_cast<double*>(smem_raw);          // [M_total][MP]
  double* P = ks + (size_t)p.M_total * MP;                    // [M_total][32]
  double* Ss = P + (size_t)p.M_total * MMF_SH_T;              // [MP][32]
  pdl_launch_dependents();
  for (int i = threadIdx.x; i < p.M_total * MP; i += blockDim.x) {
    const int b = i / MP, a = i - b * MP;
    ks[i] = a < p.M_local ? p.kappa_rows[(long long)a * p.M_total + b] : 0.0;   // kappa: a constant table
  }
  pdl_wait();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const double third = 1.0 / 3.0, sixth = 1.0 / 6.0;
  const int R = 2 * p.M_local;
  constexpr int U = 4;   // field rows per warp and batch in phase 3
  const long long ntile = (p.t_count + MMF_SH_T - 1) / MMF_SH_T;
  for (long long tile = blockIdx.x; tile < ntile; tile += gridDim.x) {
    const long long tc = tile * MMF_SH_T + lane;   // sample inside the chunk
    const long long tt = p.t_first + tc;
    const bool live = tc < p.t_count;
    __syncthreads();   // the previous tile's P and S are no longer read (and, first time round, ks is complete)
    for (int b = warp; b < p.M_total; b += MMF_SH_WARPS) P[b * MMF_SH_T + lane] = live ? p.P_all[(long long)b * p.t_count + tc] : 0.0;
    __syncthreads();
    for (int a0 = 4 * warp; a0 < p.M_local; a0 += 4 * MMF_SH_WARPS) {
      double S[4] = {0.0, 0.0, 0.0, 0.0};
      const double* kc = ks + a0;
#pragma unroll 4
      for (int b = 0; b < p.M_total; ++b) {
        const double pb = P[b * MMF_SH_T + lane];
        const double2 k01 = *reinterpret_cast<const double2*>(kc + (size_t)b * MP);
        const double2 k23 = *reinterpret_cast<const double2*>(kc + (size_t)b * MP + 2);
        S[0] = fma(k01.x, pb, S[0]);
        S[1] = fma(k01.y, pb, S[1]);
        S[2] = fma(k23.x, pb, S[2]);
        S[3] = fma(k23.y, pb, S[3]);
      }
#pragma unroll
      for (int da = 0; da < 4; ++da) Ss[(a0 + da) * MMF_SH_T + lane] = p.hg * S[da];
    }
    __syncthreads();
    if (!live) continue;
    for (int r0 = warp; r0 < R; r0 += MMF_SH_WARPS * U) {
      cpx x[U], y[U], z[U];   // stage 0: x = X; 1: x = X, y = Y; 2: x = X, y = Y, z = Z; 3: x = W, z = Z
#pragma unroll
      for (int j = 0; j < U; ++j) {
        const int r = r0 + MMF_SH_WARPS * j;
        if (r < R) {
          const long long i = (long long)r * p.N + tt;
          x[j] = (STAGE == SH_FINAL) ? p.W[i] : p.X[i];
          if constexpr (STAGE == SH_STAGE2 || STAGE == SH_STAGE3) y[j] = p.Y[i];
          if constexpr (STAGE == SH_STAGE3 || STAGE == SH_FINAL) z[j] = p.Z[i];
        }
      }
#pragma unroll
      for (int j = 0; j < U; ++j) {
        const int r = r0 + MMF_SH_WARPS * j;
        if (r < R) {
          const long long i = (long long)r * p.N + tt;
          const double g = Ss[(r >> 1) * MMF_SH_T + lane];
          cpx u = x[j];
          if constexpr (STAGE == SH_STAGE2) u = make_double2(fma(0.5, y[j].x, x[j].x), fma(0.5, y[j].y, x[j].y));
          if constexpr (STAGE == SH_STAGE3) u = make_double2(fma(0.5, z[j].x, x[j].x), fma(0.5, z[j].y, x[j].y));
          const cpx k = make_double2(-g * u.y, g * u.x);
          if constexpr (STAGE == SH_PLAIN) {
            p.Y[i] = k;
          } else if constexpr (STAGE == SH_STAGE2) {
            p.Z[i] = k;
          } else if constexpr (STAGE == SH_STAGE3) {
            p.W[i] = cadd(x[j], k);
            p.Z[i] = make_double2(x[j].x + sixth * y[j].x + third * z[j].x + third * k.x,
                                  x[j].y + sixth * y[j].y + third * z[j].y + third * k.y);
          } else {
            p.X[i] = make_double2(p.gain * fma(sixth, k.x, z[j].x), p.gain * fma(sixth, k.y, z[j].y));
          }
        }
      }
    }
  }
}

}  // namespace mmf
