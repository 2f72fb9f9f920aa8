// nl_general.cuh — the nonlinear kernel for the GENERAL per-polarisation coupling matrix, sm_100a.
//
// What it computes (Fig. 2: "Storing all kappa values requires a matrix of 2M x 2M elements"): with
// R = 2M polarisation modes (rows), hg = h gamma,
//   NL(u)_r(t) = i * hg * S_r(t) * u_r(t),   S_r(t) = sum_{s < R} kappa2[r][s] |u_s(t)|^2
// — Eq. (1) PAPER.md:36 with one coefficient per PAIR OF ROWS; the Manakov kernel of nl_tma.cuh is the special case
// kappa2[2a+p][2b+q] = kappa_ab.  One evaluation per launch, with the stage sums of Eq. (6b)-(6f) folded in:
//   NLG_PLAIN    Y <- NL(X)                                                     (bracket of Eq. 6b)
//   NLG_STAGE2   Z <- NL(X + Y/2)                         X = A_I, Y = k1        (Eq. 6c)
//   NLG_STAGE3   k3 = NL(X + Z/2);  W <- X + k3;  Y <- X + Y/6 + Z/3 + k3/3      (Eq. 6d and the brackets of 6e, 6f)
//   NLG_FINAL    X <- Y + NL(W)/6                         W = u4, Y = exp(h/2 L)[...]   (Eq. 6e, 6f)
//
// Design.  The contraction is a (R x R) x (R x 8) fp64 product per 8-sample tile — 4 x the Manakov work, 0.48 TFLOP
// per evaluation at M = 120 (13 ms at the 37 TFLOP/s fp64 peak), so this kernel is bound by the fp64 tensor pipe
// (mma.sync.m8n8k4.f64, SASS DMMA), not by HBM.  kappa2 (460 KB at M = 120) fits no single SM, so the ROWS are split
// in two halves: CTA 2i + c (c = 0, 1) computes S for rows [cM, cM + M) of the tiles i, i + G/2, ... and keeps its
// M x 2M slab of kappa2 (230 KB) for the whole persistent kernel in TENSOR MEMORY (tcgen05.st once; the A fragments
// of every k-step stream back with tcgen05.ld, one load ahead of the DMMAs that consume it) — neither registers nor
// shared memory could hold it.  Warp w owns rows 8w..8w+7 of its half; the C fragment a lane receives is S of the
// row / samples whose field elements that lane holds.  Every CTA needs |u_s|^2 of ALL rows: it loads the full tile
// (its partner loads the same tile at the same time: one of the two reads is an L2 hit) and stores only its half,
// always into a buffer nobody reads in this launch (hence the four-buffer plan: no cross-CTA hazard, no cluster).
// Data movement: one producer thread, TMA through a two-slot ring, as in nl_tma.cuh.
#pragma once
#include "async_copy.cuh"
#include "fft_core.cuh"
#include "nl_tma.cuh"

namespace mmf {

enum { NLG_PLAIN = 0, NLG_STAGE2 = 1, NLG_STAGE3 = 2, NLG_FINAL = 3 };

#define MMF_NLG_SLOTS 2
#define MMF_NLG_MAXM 120   // 15 compute warps x 8 rows per half; 60 k-steps = 120 TMEM columns per warp

struct NlgParams {
  const double* __restrict__ kappa2;  // [2M][2M] row-major
  double hg;
  double gain;       // NLG_FINAL: amplitude factor of a lumped amplifier applied to the new field (1 = none)
  int M;             // rows per half (R = 2M)
  int NW;            // compute warps = ceil(M / 8); the producer is warp NW
  int nchunk;        // chunks of 4 k-steps (16 rows of P): ceil(2M / 16)
  long long ntiles;  // N / 8
};

template <int MODE>
__host__ __device__ constexpr int nlg_nfull() { return (MODE == NLG_STAGE2 || MODE == NLG_STAGE3) ? 2 : 1; }  // full-tile loads
template <int MODE>
__host__ __device__ constexpr bool nlg_half_in() { return MODE == NLG_STAGE3 || MODE == NLG_FINAL; }       // own-rows load

__host__ __device__ inline size_t nlg_slot_bytes(int M, int nfull, bool half) {
  return ((size_t)nfull * 2 * M + (half ? M : 0)) * MMF_NLM_T * sizeof(cpx);
}
__host__ __device__ inline size_t nlg_p_bytes(int nchunk) { return (size_t)16 * nchunk * MMF_NLM_PSTRIDE * sizeof(double); }
__host__ __device__ inline size_t nlg_smem_bytes(int M, int nchunk, int nfull, bool half) {
  return MMF_NLG_SLOTS * nlg_slot_bytes(M, nfull, half) + 2 * nlg_p_bytes(nchunk) + 128;
}

// four doubles (8 columns) of this thread's TMEM lane: issue the load / wait for it (the wait names the registers, so
// no use of them is scheduled ahead of it; DMMAs on OTHER registers issued in between overlap the load)
__device__ __forceinline__ void tmem_ld_issue(int (&r)[8], uint32_t taddr) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];\n"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
               : "r"(taddr));
}
__device__ __forceinline__ void tmem_ld_wait(int (&r)[8]) {
  asm volatile("tcgen05.wait::ld.sync.aligned;\n"
               : "+r"(r[0]), "+r"(r[1]), "+r"(r[2]), "+r"(r[3]), "+r"(r[4]), "+r"(r[5]), "+r"(r[6]), "+r"(r[7]));
}

// mapF0 / mapF1: full-tile loads (box = 16 doubles x 2M rows);  mapHin: own-rows load, mapHo0 / mapHo1: own-rows stores
// (box = 16 doubles x M rows at row cM).   PLAIN: F0 = X, Ho0 = Y.   STAGE2: F0 = X, F1 = Y, Ho0 = Z.
// STAGE3: F0 = X, F1 = Z, Hin = Y, Ho0 = W, Ho1 = Y.   FINAL: F0 = W, Hin = Y, Ho0 = X.
// block = 32 (NW + 1) threads; grid = an even number of persistent CTAs; dynamic smem = nlg_smem_bytes(...).
template <int MODE>
__global__ void __launch_bounds__(512, 1)
k_nlg(const __grid_constant__ CUtensorMap mapF0, const __grid_constant__ CUtensorMap mapF1,
      const __grid_constant__ CUtensorMap mapHin, const __grid_constant__ CUtensorMap mapHo0,
      const __grid_constant__ CUtensorMap mapHo1, NlgParams p) {
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  constexpr int NFULL = nlg_nfull<MODE>();
  constexpr bool HALF_IN = nlg_half_in<MODE>();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int M = p.M, R = 2 * M, NW = p.NW;
  const int half = blockIdx.x & 1;                             // which half of the rows this CTA computes S for
  const size_t full_bytes = (size_t)R * MMF_NLM_T * sizeof(cpx);
  const size_t half_bytes = (size_t)M * MMF_NLM_T * sizeof(cpx);
  const size_t slot_bytes = NFULL * full_bytes + (HALF_IN ? half_bytes : 0);
  const size_t pbytes = nlg_p_bytes(p.nchunk);
  double* Pb0 = reinterpret_cast<double*>(smem_raw + MMF_NLG_SLOTS * slot_bytes);
  double* Pb1 = reinterpret_cast<double*>(smem_raw + MMF_NLG_SLOTS * slot_bytes + pbytes);
  uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw + MMF_NLG_SLOTS * slot_bytes + 2 * pbytes);
  uint64_t* done = full + MMF_NLG_SLOTS;
  uint32_t* tmem_word = reinterpret_cast<uint32_t*>(done + MMF_NLG_SLOTS);

  if (threadIdx.x == 0) {
#pragma unroll
    for (int s = 0; s < MMF_NLG_SLOTS; ++s) {
      mbar_init(&full[s], 1);
      mbar_init(&done[s], NW);
    }
    mbar_init_fence();
  }
  if (warp == 0) {
    __syncwarp();
    tmem_alloc(tmem_word, 512);
  }
  tmem_fence_before_sync();
  pdl_launch_dependents();
  for (int i = threadIdx.x; i < (int)(2 * pbytes / sizeof(double)); i += blockDim.x) Pb0[i] = 0.0;  // padding rows stay 0
  __syncthreads();
  tmem_fence_after_sync();

  const long long npair = gridDim.x >> 1, first = blockIdx.x >> 1;

  if (warp == NW) {
    // ---------------------------------------------------------------------------------------------- producer warp
    if (lane == 0) {
      tma_prefetch_desc(&mapF0);
      tma_prefetch_desc(&mapF1);
      tma_prefetch_desc(&mapHin);
      tma_prefetch_desc(&mapHo0);
      tma_prefetch_desc(&mapHo1);
      pdl_wait();   // the fields are the predecessor's output (only this thread touches them in global memory)
      const int own_row = half * M;
      auto store_tile = [&](long long tl, int slot) {
        unsigned char* s = smem_raw + slot * slot_bytes;
        const int c0 = (int)(tl * 2 * MMF_NLM_T);
        if constexpr (MODE == NLG_FINAL) {
          tma_store_2d(&mapHo0, c0, own_row, s + NFULL * full_bytes);              // the new field (own rows)
        } else {
          tma_store_2d(&mapHo0, c0, own_row, s + (size_t)own_row * MMF_NLM_T * sizeof(cpx));  // own rows of array 0
          if constexpr (MODE == NLG_STAGE3) tma_store_2d(&mapHo1, c0, own_row, s + NFULL * full_bytes);
        }
        tma_store_commit();
      };
      long long tile = first;
      int j = 0;
      for (; tile < p.ntiles; tile += npair, ++j) {
        const int slot = j % MMF_NLG_SLOTS, use = j / MMF_NLG_SLOTS;
        unsigned char* s = smem_raw + slot * slot_bytes;
        if (use > 0) {  // the tile that occupied this slot: store it once computed, then wait until it has been read out
          mbar_wait(&done[slot], (use - 1) & 1);
          store_tile(tile - MMF_NLG_SLOTS * npair, slot);
          tma_store_wait_read();
        }
        mbar_arrive_expect_tx(&full[slot], (uint32_t)slot_bytes);
        const int c0 = (int)(tile * 2 * MMF_NLM_T);
        tma_load_2d(s, &mapF0, c0, 0, &full[slot]);
        if constexpr (NFULL == 2) tma_load_2d(s + full_bytes, &mapF1, c0, 0, &full[slot]);
        if constexpr (HALF_IN) tma_load_2d(s + NFULL * full_bytes, &mapHin, c0, own_row, &full[slot]);
      }
      for (int jj = (j > MMF_NLG_SLOTS ? j - MMF_NLG_SLOTS : 0); jj < j; ++jj) {  // drain
        const int slot = jj % MMF_NLG_SLOTS, use = jj / MMF_NLG_SLOTS;
        mbar_wait(&done[slot], use & 1);
        store_tile(first + jj * npair, slot);
      }
      tma_store_wait_all();
    }
  } else {
    // ---------------------------------------------------------------------------------------------- compute warps
    const int gthreads = 32 * NW;
    const int g = lane >> 2, q = lane & 3;
    const int lo = warp * 8 + g;                       // row inside the half
    const bool valid = lo < M;
    const int ro = half * M + lo, rt = (1 - half) * M + lo;   // own row, and the partner half's row this lane squares
    const int nchunk = p.nchunk;

    // this warp's slab of kappa2 as A fragments, parked in tensor memory: k-step ks holds kappa2[ro][4 ks + q]
    const uint32_t taddr = *tmem_word + (((uint32_t)(warp & 3) * 32) << 16) + (uint32_t)(warp >> 2) * 128;
    for (int kc = 0; kc < nchunk; ++kc) {
      double2 e[2];
      double v[4];
#pragma unroll
      for (int jk = 0; jk < 4; ++jk) {
        const int col = 4 * (4 * kc + jk) + q;
        v[jk] = (valid && col < R) ? p.kappa2[(long long)ro * R + col] : 0.0;
      }
      e[0] = make_double2(v[0], v[1]);
      e[1] = make_double2(v[2], v[3]);
      tmem_st_c2(taddr + 8 * kc, e);
    }
    tmem_wait_st();

    const double third = 1.0 / 3.0, sixth = 1.0 / 6.0;
    const int eo = ro * MMF_NLM_T + 2 * q, et = rt * MMF_NLM_T + 2 * q;   // this lane's elements in a full array
    const int eh = lo * MMF_NLM_T + 2 * q;                                 // ... in the own-rows array

    int j = 0;
    for (long long tile = first; tile < p.ntiles; tile += npair, ++j) {
      const int slot = j % MMF_NLG_SLOTS;
      cpx* f0 = reinterpret_cast<cpx*>(smem_raw + slot * slot_bytes);
      cpx* f1 = reinterpret_cast<cpx*>(smem_raw + slot * slot_bytes + full_bytes);
      cpx* hh = reinterpret_cast<cpx*>(smem_raw + slot * slot_bytes + NFULL * full_bytes);
      double* P = (j & 1) ? Pb1 : Pb0;
      mbar_wait(&full[slot], (j / MMF_NLG_SLOTS) & 1);

      cpx x[2], u[2], ut[2], w2[2];   // own row: first array, argument of N; partner row: argument; own second array
#pragma unroll
      for (int i = 0; i < 2; ++i) {
        x[i] = valid ? f0[eo + i] : make_double2(0.0, 0.0);
        const cpx xt = valid ? f0[et + i] : make_double2(0.0, 0.0);
        if constexpr (NFULL == 2) {
          w2[i] = valid ? f1[eo + i] : make_double2(0.0, 0.0);
          const cpx wt = valid ? f1[et + i] : make_double2(0.0, 0.0);
          u[i] = axpy(0.5, w2[i], x[i]);
          ut[i] = axpy(0.5, wt, xt);
        } else {
          u[i] = x[i];
          ut[i] = xt;
        }
      }
      if (valid) {
        *reinterpret_cast<double2*>(P + ro * MMF_NLM_PSTRIDE + 2 * q) =
            make_double2(u[0].x * u[0].x + u[0].y * u[0].y, u[1].x * u[1].x + u[1].y * u[1].y);
        *reinterpret_cast<double2*>(P + rt * MMF_NLM_PSTRIDE + 2 * q) =
            make_double2(ut[0].x * ut[0].x + ut[0].y * ut[0].y, ut[1].x * ut[1].x + ut[1].y * ut[1].y);
      }
      group_barrier(1, gthreads);

      // S = kappa2_slab * P: four independent accumulator chains, A fragments one TMEM load ahead of their DMMAs
      double c[4][2] = {{0.0, 0.0}, {0.0, 0.0}, {0.0, 0.0}, {0.0, 0.0}};
      const double* pb = P + q * MMF_NLM_PSTRIDE + g;
      int ka[8], kb[8];
      tmem_ld_issue(ka, taddr);
      tmem_ld_wait(ka);
      for (int kc = 0; kc < nchunk; ++kc) {
        if (kc + 1 < nchunk) tmem_ld_issue(kb, taddr + 8 * (kc + 1));
        const double* pr = pb + (size_t)(16 * kc) * MMF_NLM_PSTRIDE;
#pragma unroll
        for (int jk = 0; jk < 4; ++jk)
          dmma884(c[jk][0], c[jk][1], __hiloint2double(ka[2 * jk + 1], ka[2 * jk]), pr[(4 * jk) * MMF_NLM_PSTRIDE]);
        if (kc + 1 < nchunk) {
          tmem_ld_wait(kb);
#pragma unroll
          for (int i = 0; i < 8; ++i) ka[i] = kb[i];
        }
      }
      const double g1[2] = {p.hg * ((c[0][0] + c[1][0]) + (c[2][0] + c[3][0])),
                            p.hg * ((c[0][1] + c[1][1]) + (c[2][1] + c[3][1]))};
      if (valid) {
#pragma unroll
        for (int i = 0; i < 2; ++i) {
          const cpx k = times_ig(u[i], g1[i]);
          if constexpr (MODE == NLG_PLAIN || MODE == NLG_STAGE2) {
            f0[eo + i] = k;
          } else if constexpr (MODE == NLG_STAGE3) {
            const cpx y = hh[eh + i], z = w2[i], xx = x[i];
            f0[eo + i] = cadd(xx, k);
            hh[eh + i] = make_double2(xx.x + sixth * y.x + third * z.x + third * k.x,
                                      xx.y + sixth * y.y + third * z.y + third * k.y);
          } else {
            const cpx an = axpy(sixth, k, hh[eh + i]);
            hh[eh + i] = make_double2(p.gain * an.x, p.gain * an.y);
          }
        }
      }
      fence_proxy_async_smem();
      __syncwarp();
      if (lane == 0) mbar_arrive(&done[slot]);
    }
  }
  tmem_fence_before_sync();
  __syncthreads();
  if (warp == 0) tmem_dealloc(*tmem_word, 512);
}

}  // namespace mmf
