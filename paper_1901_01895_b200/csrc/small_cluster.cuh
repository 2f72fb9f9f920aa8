// small_cluster.cuh — the WHOLE propagation of a small problem in one kernel: a thread-block cluster holds the field in
// distributed shared memory and alternates D and N with cluster barriers (hard part 6; "only
// a single CUDA kernel ... was launched" is the shape).  Rows a1-a8 of the hot-path table for N = 4096 and at most
// MMF_SMALL_MAXM spatial modes (config 0 of BASELINE.json: M = 2), where a step of the launch-by-launch plan is bound
// by launch latency and kernel prologues, not by any roofline.
//
// The cluster has T = 2 * 2M CTAs of 256 threads (one transform group each).  CTA c keeps ONE 4096-point tile in its
// shared memory for the whole propagation: row (c mod 2M) of buffer X (c < 2M) or of buffer Y (c >= 2M) — the two
// buffers of the RK4IP step driver (mmf_api.cu: X = A -> A_I -> A_I + k3 -> u4 -> A', Y = NL(A) -> k1 -> bracket -> ...).
//   D phase   every CTA applies exp(h/2 L) to its own tile in place: the 4096-point chains of tmem_exchange.cuh; the
//             thread's 16 exp(h/2 L) values and the stage tables are loaded ONCE per kernel (tensor memory / shared
//             memory), so a step reads nothing from global memory at all.
//   N phase   the time samples are dealt out over all T * 256 threads of the cluster; a thread reads the 2 * 2M values
//             of its sample from the owners' shared memory (ld.shared::cluster), evaluates the fused stage of
//             nl_tma.cuh (PLAIN, S23, FINAL, FINAL_NEXT — same formulas, plain loops over the M <= 4 modes) and writes
//             the results back to the owners (st.shared::cluster).
// barrier.cluster (arrive.release / wait.acquire) separates the phases: four per step.  The caller's field is read at
// the start and written at the end; nothing else touches global memory.
#pragma once
#include "async_copy.cuh"
#include "fft_core.cuh"
#include "fft_kernels.cuh"
#include "nl_tma.cuh"
#include "tmem_exchange.cuh"

namespace mmf {

#define MMF_SMALL_MAXM 4                     // 2 * 2M <= 16 CTAs: the largest (non-portable) cluster
#define MMF_SMALL_LOGN 12
#define MMF_SMALL_THREADS MMF_GROUP_THREADS  // one 256-thread transform group per CTA

struct SmallParams {
  cpx* A;                            // the caller's field [2M][4096], natural order (read at entry, written at exit)
  const cpx* __restrict__ E;         // exp(h/2 L) table [M][4096] in the slot order of k_etab
  const cpx* __restrict__ twtab;     // stage tables of the 4096-point transform
  const double* __restrict__ kappa;  // [M][M]
  double hg, gain;
  int M, nsteps, span;
};

__host__ __device__ constexpr size_t small_smem_bytes() {
  return sizeof(cpx) * ((size_t)(1 << MMF_SMALL_LOGN) + ((tw_total_entries(MMF_SMALL_LOGN, nstages(MMF_SMALL_LOGN)) + 7) & ~7)) +
         sizeof(double) * MMF_SMALL_MAXM * MMF_SMALL_MAXM + 64;
}

__device__ __forceinline__ uint32_t cluster_ctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;\n" : "=r"(r));
  return r;
}
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;\n" ::: "memory");
  asm volatile("barrier.cluster.wait.acquire.aligned;\n" ::: "memory");
}
// shared-memory address of the same variable in CTA `rank` of the cluster
__device__ __forceinline__ uint32_t cluster_map(uint32_t smem_addr, uint32_t rank) {
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;\n" : "=r"(r) : "r"(smem_addr), "r"(rank));
  return r;
}
__device__ __forceinline__ cpx ld_cluster(uint32_t addr) {
  cpx v;
  asm volatile("ld.shared::cluster.v2.f64 {%0, %1}, [%2];\n" : "=d"(v.x), "=d"(v.y) : "r"(addr) : "memory");
  return v;
}
__device__ __forceinline__ void st_cluster(uint32_t addr, cpx v) {
  asm volatile("st.shared::cluster.v2.f64 [%0], {%1, %2};\n" ::"r"(addr), "d"(v.x), "d"(v.y) : "memory");
}

enum { SM_PLAIN = 0, SM_S23 = 1, SM_FINAL = 2, SM_FINAL_NEXT = 3 };

// S_a = sum_b kappa_ab P_b for the M <= 4 modes of one sample.
// P, S are held in ROTATED positions: position a' is mode (a' + q) mod M (see small_nl_phase), and the sum runs over
// the positions in ascending order, i.e. over the modes in the order q, q + 1, ..., M - 1, 0, ..., q - 1 with q
// depending on CTA and warp.  That is NOT the oracle's b-ascending order: the result agrees with the oracle and with
// the kernel-per-stage plan to rounding (a few ulp of S), not bit for bit, and the rounding of a sample depends on the
// warp that owns it.  (include/mmf.h says so; test_small_cluster_kernel_matches_oracle_and_the_launch_by_launch_plan
// bounds the difference at 1e-13 relative L2 per field.)
template <int M>
__device__ __forceinline__ void small_contract(const double* __restrict__ kap, int q, const double (&P)[M], double (&S)[M]) {
#pragma unroll
  for (int a = 0; a < M; ++a) {
    const int am = a + q < M ? a + q : a + q - M;
    double s = 0.0;
#pragma unroll
    for (int b = 0; b < M; ++b) {
      const int bm = b + q < M ? b + q : b + q - M;
      s = fma(kap[am * M + bm], P[b], s);
    }
    S[a] = s;
  }
}

// One fused nonlinear stage on the samples n = first, first + stride, ... of all rows.  tile_addr: this CTA's tile
// (shared-memory address); the tile of row r of X lives in CTA r, that of Y in CTA 2M + r, at the same address.
// Every thread of the cluster needs every owner once per sample; if all of them walked the owners in the same order,
// one SM's shared memory would serve 2048 threads at a time while the others idle (measured: 4900 clk per phase at
// M = 2, the bandwidth of ONE SM).  So the walk is staggered per warp: position i of the register arrays holds row
// (i + 2 q) mod 2M with q = (CTA + warp) mod M, and every other warp group visits Y before X — the owners are busy
// together.  Two samples per trip (M <= 2): the remote loads of both are in flight before the first is worked on.
__device__ __forceinline__ int small_row(int i, int q, int R) { return i + 2 * q < R ? i + 2 * q : i + 2 * q - R; }
template <int MODE, int M>
__device__ __forceinline__ void small_nl_load(uint32_t off, int q, bool yfirst, cpx (&x)[2 * M], cpx (&y)[2 * M]) {
  constexpr int R = 2 * M;
  if (MODE == SM_PLAIN || !yfirst) {
#pragma unroll
    for (int i = 0; i < R; ++i) {
      const int r = small_row(i, q, R);
      x[i] = ld_cluster(cluster_map(off, (uint32_t)r));
      if constexpr (MODE != SM_PLAIN) y[i] = ld_cluster(cluster_map(off, (uint32_t)(R + r)));
    }
  } else {
#pragma unroll
    for (int i = 0; i < R; ++i) {
      const int r = small_row(i, q, R);
      y[i] = ld_cluster(cluster_map(off, (uint32_t)(R + r)));
      x[i] = ld_cluster(cluster_map(off, (uint32_t)r));
    }
  }
}
template <int MODE, int M>
__device__ __forceinline__ void small_nl_finish(uint32_t off, int q, const cpx (&x)[2 * M], const cpx (&y)[2 * M],
                                                const double* __restrict__ kap, double hg, double gain) {
  constexpr int R = 2 * M;
  const double third = 1.0 / 3.0, sixth = 1.0 / 6.0;
  double P[M], S[M];
  cpx u[R];
#pragma unroll
  for (int r = 0; r < R; ++r) u[r] = (MODE == SM_S23) ? axpy(0.5, y[r], x[r]) : x[r];
#pragma unroll
  for (int a = 0; a < M; ++a) P[a] = power2(u[2 * a], u[2 * a + 1]);
  small_contract<M>(kap, q, P, S);
  if constexpr (MODE == SM_PLAIN) {
#pragma unroll
    for (int r = 0; r < R; ++r) st_cluster(cluster_map(off, (uint32_t)(R + small_row(r, q, R))), times_ig(u[r], hg * S[r >> 1]));
  } else if constexpr (MODE == SM_FINAL) {
#pragma unroll
    for (int r = 0; r < R; ++r) {
      const cpx an = axpy(sixth, times_ig(u[r], hg * S[r >> 1]), y[r]);
      st_cluster(cluster_map(off, (uint32_t)small_row(r, q, R)), make_double2(gain * an.x, gain * an.y));
    }
  } else {
    cpx v[R];  // S23: u3 = X + k2/2;  FINAL_NEXT: the new field
#pragma unroll
    for (int r = 0; r < R; ++r) {
      const cpx k = times_ig(u[r], hg * S[r >> 1]);  // k2 resp. k4
      if constexpr (MODE == SM_S23) {
        v[r] = axpy(0.5, k, x[r]);
      } else {
        const cpx an = axpy(sixth, k, y[r]);
        v[r] = make_double2(gain * an.x, gain * an.y);
      }
    }
    double P2[M], S2[M];
#pragma unroll
    for (int a = 0; a < M; ++a) P2[a] = power2(v[2 * a], v[2 * a + 1]);
    small_contract<M>(kap, q, P2, S2);
#pragma unroll
    for (int r = 0; r < R; ++r) {
      const cpx kk = times_ig(v[r], hg * S2[r >> 1]);  // k3 resp. the next step's (6b) bracket
      if constexpr (MODE == SM_S23) {
        const cpx k2 = times_ig(u[r], hg * S[r >> 1]);
        st_cluster(cluster_map(off, (uint32_t)small_row(r, q, R)), cadd(x[r], kk));
        st_cluster(cluster_map(off, (uint32_t)(R + small_row(r, q, R))),
                   make_double2(x[r].x + sixth * y[r].x + third * k2.x + third * kk.x,
                                x[r].y + sixth * y[r].y + third * k2.y + third * kk.y));
      } else {
        st_cluster(cluster_map(off, (uint32_t)small_row(r, q, R)), v[r]);
        st_cluster(cluster_map(off, (uint32_t)(R + small_row(r, q, R))), kk);
      }
    }
  }
}
template <int MODE, int M>
__device__ __forceinline__ void small_nl_phase(uint32_t tile_addr, const double* __restrict__ kap, double hg, double gain,
                                               int first, int stride, int q, bool yfirst) {
  constexpr int NPT = 1 << MMF_SMALL_LOGN;
  if constexpr (M <= 2) {   // 4 resp. 2 samples per thread: two at a time
    for (int n = first; n < NPT; n += 2 * stride) {
      const int n2 = n + stride;
      const uint32_t off = tile_addr + (uint32_t)n * (uint32_t)sizeof(cpx), off2 = tile_addr + (uint32_t)n2 * (uint32_t)sizeof(cpx);
      cpx x[2 * M], y[2 * M], x2[2 * M], y2[2 * M];
      small_nl_load<MODE, M>(off, q, yfirst, x, y);
      if (n2 < NPT) small_nl_load<MODE, M>(off2, q, yfirst, x2, y2);
      small_nl_finish<MODE, M>(off, q, x, y, kap, hg, gain);
      if (n2 < NPT) small_nl_finish<MODE, M>(off2, q, x2, y2, kap, hg, gain);
    }
  } else {
    for (int n = first; n < NPT; n += stride) {
      const uint32_t off = tile_addr + (uint32_t)n * (uint32_t)sizeof(cpx);
      cpx x[2 * M], y[2 * M];
      small_nl_load<MODE, M>(off, q, yfirst, x, y);
      small_nl_finish<MODE, M>(off, q, x, y, kap, hg, gain);
    }
  }
}

// grid = cluster = 2 * 2M CTAs (launch attribute), block = 256, dynamic shared memory = small_smem_bytes()
template <int M>
__global__ void __launch_bounds__(MMF_SMALL_THREADS, 1) k_small(SmallParams p) {
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  constexpr int NPT = 1 << MMF_SMALL_LOGN;
  constexpr int TWN = tw_total_entries(MMF_SMALL_LOGN, nstages(MMF_SMALL_LOGN));
  cpx* tile = reinterpret_cast<cpx*>(smem_raw);
  cpx* tab = tile + NPT;
  double* kap = reinterpret_cast<double*>(tab + ((TWN + 7) & ~7));
  uint64_t* tabbar = reinterpret_cast<uint64_t*>(kap + MMF_SMALL_MAXM * MMF_SMALL_MAXM);
  uint32_t* tmem_word = reinterpret_cast<uint32_t*>(tabbar + 1);
  const int t = threadIdx.x;
  constexpr int R = 2 * M, T = 2 * R;
  const uint32_t c = cluster_ctarank();
  const int row = (int)c % R;
  const bool is_x = (int)c < R;

  if (t == 0) {
    mbar_init(tabbar, 1);
    mbar_init_fence();
    mbar_arrive_expect_tx(tabbar, TWN * (int)sizeof(cpx));
    bulk_load_1d(tab, p.twtab, TWN * (int)sizeof(cpx), tabbar);
  }
  if (t < 32) {
    __syncwarp();
    tmem_alloc(tmem_word, 256);   // per warp: 64 columns of E values + 64 of exchange buffer; two warps per lane quarter
  }
  tmem_fence_before_sync();
  if (t < M * M) kap[t] = p.kappa[t];
  __syncthreads();
  tmem_fence_after_sync();
  pdl_launch_dependents();   // after tcgen05.alloc, never before: see k_rows (a chain of these kernels allocates 256 columns each)
  pdl_wait();
  const uint32_t warp = (uint32_t)t >> 5;
  const uint32_t taddr = *tmem_word + (((warp & 3) * 32) << 16) + (warp >> 2) * 128;
  const Tm12 lay = tm12_layout(t);
  {  // the thread's 16 exp(h/2 L) values of this row's mode, for the whole propagation
    const cpx* e = p.E + ((size_t)(row >> 1) << MMF_SMALL_LOGN) + lay.tv;
#pragma unroll
    for (int cc = 0; cc < 8; ++cc) {
      const cpx pr[2] = {__ldg(e + ((2 * cc) << (MMF_SMALL_LOGN - 4))), __ldg(e + ((2 * cc + 1) << (MMF_SMALL_LOGN - 4)))};
      tmem_st_c2(taddr + 8 * cc, pr);
    }
    tmem_wait_st();
  }
  if (is_x) {  // the caller's row into the tile
    const cpx* g = p.A + ((size_t)row << MMF_SMALL_LOGN);
#pragma unroll
    for (int j = 0; j < 16; ++j) tile[t + 256 * j] = g[t + 256 * j];
  }
  mbar_wait(tabbar, 0);
  const uint32_t tile_addr = smem_u32(tile);
  const int first = (int)c * MMF_SMALL_THREADS + t, stride = T * MMF_SMALL_THREADS;
  const int qrot = ((int)c + (int)warp) % M;                       // staggered walk over the owners (small_nl_phase)
  const bool yfirst = ((((int)c + (int)warp) / M) & 1) != 0;

  auto apply_D = [&]() {   // exp(h/2 L) on the own tile, in place (fft_kernels.cuh: k_rows, one tile)
    cpx v[16];
    tile_lds_linear<8>(v, tile, lay.base1);
    fft12_dif_tm<+1>(v, tile, lay, tab, 1, taddr + 64);
#pragma unroll
    for (int hb = 0; hb < 2; ++hb) {
      int wa[4][8];
#pragma unroll
      for (int cc = 0; cc < 4; ++cc) tmem_ld_issue8(wa[cc], taddr + 32 * hb + 8 * cc);
#pragma unroll
      for (int cc = 0; cc < 4; ++cc) tmem_ld_wait8(wa[cc]);
#pragma unroll
      for (int cc = 0; cc < 4; ++cc) {
        cpx ev[2];
        tmem_words_to_c2(ev, wa[cc]);
        v[8 * hb + 2 * cc] = cmul(v[8 * hb + 2 * cc], ev[0]);
        v[8 * hb + 2 * cc + 1] = cmul(v[8 * hb + 2 * cc + 1], ev[1]);
      }
    }
    fft12_dit_tm<-1>(v, tile, lay, tab, 1, taddr + 64);
    __syncwarp();
    tile_sts_linear<8>(v, tile, lay.base1);
  };

  cluster_sync_all();                                                      // every X tile is in place
  small_nl_phase<SM_PLAIN, M>(tile_addr, kap, p.hg, 1.0, first, stride, qrot, yfirst);   // Y <- h N(A) A      (bracket of 6b)
  cluster_sync_all();
  for (int s = 0; s < p.nsteps; ++s) {
    apply_D();                                                             // (6a) A_I, (6b) k1
    cluster_sync_all();
    small_nl_phase<SM_S23, M>(tile_addr, kap, p.hg, 1.0, first, stride, qrot, yfirst);   // (6c), (6d), brackets of (6e) / (6f)
    cluster_sync_all();
    apply_D();                                                             // (6e) argument, (6f) first term
    cluster_sync_all();
    const double g = (p.span > 0 && (s + 1) % p.span == 0) ? p.gain : 1.0;
    if (s + 1 < p.nsteps) small_nl_phase<SM_FINAL_NEXT, M>(tile_addr, kap, p.hg, g, first, stride, qrot, yfirst);
    else small_nl_phase<SM_FINAL, M>(tile_addr, kap, p.hg, g, first, stride, qrot, yfirst);
    cluster_sync_all();
  }
  if (is_x) {
    cpx* g = p.A + ((size_t)row << MMF_SMALL_LOGN);
#pragma unroll
    for (int j = 0; j < 16; ++j) g[t + 256 * j] = tile[t + 256 * j];
  }
  tmem_fence_before_sync();
  __syncthreads();
  if (t < 32) tmem_dealloc(*tmem_word, 256);
}

}  // namespace mmf
