// nl_mma.cuh — the fused nonlinear kernel of the RK4IP step (rows a4-a7 of the hot-path table), sm_100a, fp64.
//
// What it computes (Eq. 1 PAPER.md:36 and Eq. 6b-6f), for one tile of 8 time samples and ALL 2M rows:
//   NL(u)_{a,p}(t) = i * hg * S_a(t) * u_{a,p}(t),  S_a(t) = sum_b kappa_ab P_b(t),  P_b = |u_bx|^2 + |u_by|^2,  hg = h gamma
//   NLM_PLAIN   OUT <- NL(U)                                                    (the bracket of Eq. 6b; U, OUT any)
//   NLM_S23     X = A_I, Y = k1:  k2 = NL(X + Y/2),  k3 = NL(X + k2/2),
//               X <- X + k3  (the argument of Eq. 6e),  Y <- X + Y/6 + k2/3 + k3/3  (the bracket of Eq. 6f), IN PLACE.
//               Eq. (6c) and (6d) have no transform between them, so both are evaluated in one pass: 4 F of traffic
//               instead of the 8 F two kernels need.
//   NLM_FINAL   X = u4, Y = exp(h/2 L)[...]:  X <- Y + NL(X)/6                   (Eq. 6e + 6f; Y untouched)
//   NLM_FINAL_NEXT  as NLM_FINAL, then Y <- NL(X_new)                           (the next step's Eq. 6b bracket)
//
// Design.  The kappa contraction S = kappa * P is a (M x M) x (M x 8) fp64 matrix product per tile: it runs on the
// fp64 tensor path (mma.sync.m8n8k4.f64, SASS DMMA; tcgen05 has no fp64 kind).  Warp w of a tile group owns mode
// rows a = 8w .. 8w+7 and keeps its 8 x M slab of kappa in REGISTERS for the whole (persistent) kernel as A
// fragments (M/4 doubles per lane), so kappa is never re-read.  The C fragment a lane receives — S[a][t], S[a][t+1]
// for a = 8w + lane/4, t = 2 (lane%4) — is exactly the set of field elements that lane owns (both polarisations),
// so the products, the RK4 sums and P of the next round all happen in registers; only P (M x 8 doubles) crosses
// warps, through shared memory.  Input tiles are prefetched one tile ahead with cp.async into a double-buffered
// staging area (XOR-swizzled so the fragment-shaped reads are bank-conflict free); results go straight from
// registers to global memory (32 contiguous bytes per lane, 128 per quad).
#pragma once
#include "fft_core.cuh"

namespace mmf {

enum { NLM_PLAIN = 0, NLM_S23 = 1, NLM_FINAL = 2, NLM_FINAL_NEXT = 3 };

#define MMF_NLM_T 8           // time samples per tile
#define MMF_NLM_PSTRIDE 12    // doubles per P row in shared memory (8 + 4: conflict-free B-fragment reads)
#define MMF_NLM_MAXM 128      // kappa slab per warp: M/4 doubles per lane -> 16 warps x 8 rows

struct NlmParams {
  const cpx* U;    // NLM_PLAIN input (otherwise unused)
  cpx* X;          // in/out (see modes); NLM_PLAIN: output
  cpx* Y;
  const double* __restrict__ kappa;  // [M][M] row-major
  double hg;
  int M;
  int NW;          // warps per tile group = ceil(M / 8)
  int TG;          // tile groups per CTA
  long long N;
  long long ntiles;  // N / 8
};

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;\n" ::: "memory"); }

// bytes of dynamic shared memory one tile group needs
__host__ __device__ inline size_t nlm_group_smem(int M, int nk, int narr) {
  const size_t stage = (size_t)2 * narr * (2 * (size_t)M) * MMF_NLM_T * sizeof(cpx);      // double-buffered tiles
  const size_t pbuf = (size_t)2 * (4 * (size_t)nk) * MMF_NLM_PSTRIDE * sizeof(double);    // P of round 1 and 2
  return stage + pbuf;
}

template <int MODE>
__host__ __device__ constexpr int nlm_narr() { return MODE == NLM_PLAIN ? 1 : 2; }

// S = kappa_slab * P  for this warp's 8 rows and the tile's 8 samples
template <int NK>
__device__ __forceinline__ void nlm_contract(const double (&kf)[NK], const double* __restrict__ P, int g, int q,
                                             double& s0, double& s1) {
  double c0 = 0.0, c1 = 0.0, d0 = 0.0, d1 = 0.0;
  const double* pb = P + q * MMF_NLM_PSTRIDE + g;
#pragma unroll
  for (int ks = 0; ks < NK; ks += 2) {
    dmma884(c0, c1, kf[ks], pb[(4 * ks) * MMF_NLM_PSTRIDE]);
    if (ks + 1 < NK) dmma884(d0, d1, kf[ks + 1], pb[(4 * ks + 4) * MMF_NLM_PSTRIDE]);
  }
  s0 = c0 + d0;
  s1 = c1 + d1;
}

// NK = ceil(M / 4) k-steps of the contraction (compile-time: the kappa fragments are a register array).
// block = 32 * NW * TG threads; grid = persistent; dynamic smem = TG * nlm_group_smem(M, NK, narr).
// largest block the launcher can pick for NK k-steps (M <= 4 NK): NW = ceil(M/8) warps x floor(16/NW) tile groups
__host__ __device__ constexpr int nlm_max_threads(int nk) {
  const int nw = (4 * nk + 7) / 8;
  return 32 * nw * (16 / nw);
}

template <int NK, int MODE>
__global__ void __launch_bounds__(nlm_max_threads(NK), 1) k_nlm(NlmParams p) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  constexpr int NARR = nlm_narr<MODE>();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int grp = warp / p.NW, wg = warp - grp * p.NW;
  const int gthreads = 32 * p.NW, gtid = wg * 32 + lane;
  const int g = lane >> 2, q = lane & 3;
  const int M = p.M, R = 2 * M;
  const int a = wg * 8 + g;
  const bool valid = a < M;
  const long long N = p.N;

  // this warp's slab of kappa as A fragments: kf[ks] = kappa[a][4 ks + q]
  double kf[NK];
#pragma unroll
  for (int ks = 0; ks < NK; ++ks) {
    const int b = 4 * ks + q;
    kf[ks] = (valid && b < M) ? p.kappa[(long long)a * M + b] : 0.0;
  }

  unsigned char* gbase = smem_raw + (size_t)grp * nlm_group_smem(M, NK, NARR);
  const size_t tile_bytes = (size_t)R * MMF_NLM_T * sizeof(cpx);  // one array, one tile
  cpx* stage = reinterpret_cast<cpx*>(gbase);                     // [buf][arr][row][8 slots]
  double* Pb0 = reinterpret_cast<double*>(gbase + 2 * NARR * tile_bytes);
  double* Pb1 = Pb0 + 4 * NK * MMF_NLM_PSTRIDE;
  for (int i = gtid; i < 2 * 4 * NK * MMF_NLM_PSTRIDE; i += gthreads) Pb0[i] = 0.0;  // padding rows must stay 0

  const cpx* src0 = (MODE == NLM_PLAIN) ? p.U : p.X;
  const cpx* src1 = p.Y;
  const long long tstep = (long long)gridDim.x * p.TG;
  long long tile = (long long)blockIdx.x * p.TG + grp;

  auto prefetch = [&](long long tl, int buf) {
    cpx* dst = stage + (size_t)buf * NARR * R * MMF_NLM_T;
    const int per_arr = R * MMF_NLM_T;
    for (int idx = gtid; idx < NARR * per_arr; idx += gthreads) {
      const int arr = (NARR == 2 && idx >= per_arr) ? 1 : 0;
      const int rem = idx - arr * per_arr;
      const int row = rem >> 3, t = rem & 7;
      const cpx* s = (arr ? src1 : src0) + (long long)row * N + tl * MMF_NLM_T + t;
      cp_async16(dst + (size_t)arr * per_arr + row * MMF_NLM_T + (t ^ ((row >> 1) & 1)), s);
    }
  };

  int buf = 0;
  if (tile < p.ntiles) prefetch(tile, 0);
  cp_async_commit();
  const int sw = a & 1;  // staging swizzle of this lane's rows
  const double third = 1.0 / 3.0, sixth = 1.0 / 6.0;

  for (; tile < p.ntiles; tile += tstep, buf ^= 1) {
    cp_async_wait_all();
    group_barrier(grp, gthreads);  // tile `buf` visible to the group; everyone is done with buffer buf^1
    if (tile + tstep < p.ntiles) prefetch(tile + tstep, buf ^ 1);
    cp_async_commit();

    // this lane's elements: rows 2a (x) and 2a+1 (y), samples t = 2q, 2q+1
    cpx x[2][2], y[2][2];
    const cpx* st = stage + (size_t)buf * NARR * R * MMF_NLM_T;
#pragma unroll
    for (int pol = 0; pol < 2; ++pol)
#pragma unroll
      for (int i = 0; i < 2; ++i) {
        const int slot = (2 * q + i) ^ sw;
        x[pol][i] = valid ? st[(2 * a + pol) * MMF_NLM_T + slot] : make_double2(0.0, 0.0);
        if constexpr (NARR == 2)
          y[pol][i] = valid ? st[(size_t)R * MMF_NLM_T + (2 * a + pol) * MMF_NLM_T + slot] : make_double2(0.0, 0.0);
      }

    // ---- round 1 -------------------------------------------------------------------------------------------
    cpx u[2][2];
#pragma unroll
    for (int pol = 0; pol < 2; ++pol)
#pragma unroll
      for (int i = 0; i < 2; ++i) {
        if constexpr (MODE == NLM_S23)
          u[pol][i] = make_double2(fma(0.5, y[pol][i].x, x[pol][i].x), fma(0.5, y[pol][i].y, x[pol][i].y));
        else
          u[pol][i] = x[pol][i];
      }
    if (valid) {
      double2 pw;
      pw.x = (u[0][0].x * u[0][0].x + u[0][0].y * u[0][0].y) + (u[1][0].x * u[1][0].x + u[1][0].y * u[1][0].y);
      pw.y = (u[0][1].x * u[0][1].x + u[0][1].y * u[0][1].y) + (u[1][1].x * u[1][1].x + u[1][1].y * u[1][1].y);
      *reinterpret_cast<double2*>(Pb0 + a * MMF_NLM_PSTRIDE + 2 * q) = pw;
    }
    group_barrier(grp, gthreads);
    double s[2];
    nlm_contract<NK>(kf, Pb0, g, q, s[0], s[1]);
    const double g1[2] = {p.hg * s[0], p.hg * s[1]};
    const long long col = tile * MMF_NLM_T + 2 * q;

    if constexpr (MODE == NLM_PLAIN) {
      if (valid) {
#pragma unroll
        for (int pol = 0; pol < 2; ++pol)
#pragma unroll
          for (int i = 0; i < 2; ++i)
            p.X[(long long)(2 * a + pol) * N + col + i] = make_double2(-g1[i] * u[pol][i].y, g1[i] * u[pol][i].x);
      }
    } else if constexpr (MODE == NLM_FINAL) {
      if (valid) {
#pragma unroll
        for (int pol = 0; pol < 2; ++pol)
#pragma unroll
          for (int i = 0; i < 2; ++i) {
            const cpx k4 = make_double2(-g1[i] * u[pol][i].y, g1[i] * u[pol][i].x);
            p.X[(long long)(2 * a + pol) * N + col + i] =
                make_double2(fma(sixth, k4.x, y[pol][i].x), fma(sixth, k4.y, y[pol][i].y));
          }
      }
    } else {
      // ---- round 2 -----------------------------------------------------------------------------------------
      cpx v[2][2];  // S23: u3 = X + k2/2;  FINAL_NEXT: the new field A(z+h)
#pragma unroll
      for (int pol = 0; pol < 2; ++pol)
#pragma unroll
        for (int i = 0; i < 2; ++i) {
          const cpx k = make_double2(-g1[i] * u[pol][i].y, g1[i] * u[pol][i].x);  // k2 resp. k4
          if constexpr (MODE == NLM_S23)
            v[pol][i] = make_double2(fma(0.5, k.x, x[pol][i].x), fma(0.5, k.y, x[pol][i].y));
          else
            v[pol][i] = make_double2(fma(sixth, k.x, y[pol][i].x), fma(sixth, k.y, y[pol][i].y));
        }
      if (valid) {
        double2 pw;
        pw.x = (v[0][0].x * v[0][0].x + v[0][0].y * v[0][0].y) + (v[1][0].x * v[1][0].x + v[1][0].y * v[1][0].y);
        pw.y = (v[0][1].x * v[0][1].x + v[0][1].y * v[0][1].y) + (v[1][1].x * v[1][1].x + v[1][1].y * v[1][1].y);
        *reinterpret_cast<double2*>(Pb1 + a * MMF_NLM_PSTRIDE + 2 * q) = pw;
      }
      group_barrier(grp, gthreads);
      double s2[2];
      nlm_contract<NK>(kf, Pb1, g, q, s2[0], s2[1]);
      const double g2[2] = {p.hg * s2[0], p.hg * s2[1]};
      if (valid) {
#pragma unroll
        for (int pol = 0; pol < 2; ++pol)
#pragma unroll
          for (int i = 0; i < 2; ++i) {
            const long long o = (long long)(2 * a + pol) * N + col + i;
            const cpx kk = make_double2(-g2[i] * v[pol][i].y, g2[i] * v[pol][i].x);  // k3 resp. next bracket
            if constexpr (MODE == NLM_S23) {
              const cpx k2 = make_double2(-g1[i] * u[pol][i].y, g1[i] * u[pol][i].x);
              const cpx xx = x[pol][i], yy = y[pol][i];
              p.X[o] = cadd(xx, kk);
              p.Y[o] = make_double2(xx.x + sixth * yy.x + third * k2.x + third * kk.x,
                                    xx.y + sixth * yy.y + third * k2.y + third * kk.y);
            } else {
              p.X[o] = v[pol][i];
              p.Y[o] = kk;
            }
          }
      }
    }
  }
  cp_async_wait_all();
}

}  // namespace mmf
