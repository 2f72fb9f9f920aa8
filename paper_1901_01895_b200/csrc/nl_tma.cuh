// nl_tma.cuh — the fused nonlinear kernel of the RK4IP step (rows a4-a7 of the hot-path table), sm_100a, fp64.
//
// What it computes (Eq. 1 PAPER.md:36 and Eq. 6b-6f), for one tile of 8 time samples and ALL 2M rows:
//   NL(u)_{a,p}(t) = i * hg * S_a(t) * u_{a,p}(t),  S_a(t) = sum_b kappa_ab P_b(t),  P_b = |u_bx|^2 + |u_by|^2,  hg = h gamma
//   NLM_PLAIN   OUT <- NL(U)                                                    (the bracket of Eq. 6b; U, OUT any)
//   NLM_S23     X = A_I, Y = k1:  k2 = NL(X + Y/2),  k3 = NL(X + k2/2),
//               X <- X + k3  (the argument of Eq. 6e),  Y <- X + Y/6 + k2/3 + k3/3  (the bracket of Eq. 6f), IN PLACE.
//               Eq. (6c) and (6d) have no transform between them, so both are evaluated in one pass: 4 F of traffic
//               instead of the 8 F two kernels need.
//   NLM_FINAL   X = u4, Y = exp(h/2 L)[...]:  X <- gain (Y + NL(X)/6)            (Eq. 6e + 6f; Y untouched; gain = 1
//               except at the end of a fibre span, where it is the lumped amplifier of PAPER.md:255)
//   NLM_FINAL_NEXT  as NLM_FINAL, then Y <- NL(X_new)                           (the next step's Eq. 6b bracket)
//   NLM_ENTER   first kernel of a propagation in the blocked order (fft_kernels.cuh): reads tile tn(t) of the caller's
//               field A (NATURAL order) and writes tile t of X <- A and of Y <- NL(A) (blocked order): the layout
//               conversion of the way in rides on the first nonlinear evaluation (3 F instead of 2 F + 2 F).
//   NLM_EXIT    last kernel: NLM_FINAL on the blocked X, Y with the result written to tile tn(t) of the caller's
//               field (natural order): no conversion pass on the way out.
//               A time tile is 8 consecutive samples in both orders; only its position differs.
//   NLM_RK4     X <- X + k1/6 + k2/3 + k3/3 + k4/6,  k1 = NL(X), k2 = NL(X + k1/2), k3 = NL(X + k2/2), k4 = NL(X + k3):
//               the nonlinear substep of the symmetric split step (Eq. 4, "SSFM-RK4"): classical RK4
//               over h of dA/dz = N(A) A, four contraction rounds per tile, the field read and written once (2 F).
//   NLM_AGR_S0 / NLM_AGR_IT1 / NLM_AGR_ITJ   the nonlinear part of the ITERATIVE symmetric split step ("SSFM-Agrawal",
//               Eq. 4; reading R14: trapezoidal rule with N(z+h) from the previous iterate):
//               S0:  T <- hg S(X)                      (|A|^2 "once at the position z"; T is a real [M][N] table)
//               IT1: Y <- exp(i T) X                   (first iteration, N(z+h) := N(z); X = exp(h/2 L) A(z))
//               ITJ: Y <- exp(i (T + hg S(Y)) / 2) X   (later iterations, |A|^2 "at the position z + h" from Y)
//
// Design.  The kappa contraction S = kappa * P is a (M x M) x (M x 8) fp64 matrix product per tile: it runs on the
// fp64 tensor path (mma.sync.m8n8k4.f64, SASS DMMA; tcgen05 has no fp64 kind).  Compute warp w owns mode rows
// a = 8w .. 8w+7 and keeps its 8 x M slab of kappa in REGISTERS for the whole (persistent) kernel as A fragments
// (M/4 doubles per lane), so kappa is never re-read.  The C fragment a lane receives — S[a][t], S[a][t+1] for
// a = 8w + lane/4, t = 2 (lane%4) — is exactly the set of field elements that lane owns (both polarisations), so the
// products, the RK4 sums and P of the next round all happen in registers; only P (M x 8 doubles) crosses warps,
// through shared memory.
// Data movement is entirely asynchronous: one PRODUCER thread moves tiles with TMA (cp.async.bulk.tensor, box =
// 8 samples x 2M rows per array) through a ring of three shared-memory slots — load (completes on a "full" mbarrier),
// compute in place, store from the same slot once the compute warps have arrived on its "done" mbarrier — so the
// compute warps issue no global memory instruction at all and loads run two tiles ahead of the arithmetic.
#pragma once
#include "async_copy.cuh"
#include "fft_core.cuh"

namespace mmf {

enum { NLM_PLAIN = 0, NLM_S23 = 1, NLM_FINAL = 2, NLM_FINAL_NEXT = 3, NLM_RK4 = 4, NLM_ENTER = 5, NLM_EXIT = 6,
       NLM_AGR_S0 = 7, NLM_AGR_IT1 = 8, NLM_AGR_ITJ = 9 };

#define MMF_NLM_T 8           // time samples per tile
#define MMF_NLM_PSTRIDE 12    // doubles per P row in shared memory (8 + 4: conflict-free B-fragment reads)
#define MMF_NLM_MAXM 120      // 15 compute warps x 8 modes + the producer warp = 512 threads; TMA box <= 256 rows
#define MMF_NLM_SLOTS 3       // ring depth

struct NltParams {
  const double* __restrict__ kappa;  // [M][M] row-major; GROUPED kernels: the G distinct rows, [G][M]
  const int* __restrict__ group_of;  // GROUPED kernels: [M], which distinct row mode a has
  int G;                             // GROUPED kernels: number of distinct rows; the first ceil(G / 8) warps contract
  double hg;
  double gain;       // FINAL / FINAL_NEXT / EXIT: amplitude factor of a lumped amplifier applied to the new field (1 = none)
  int M;
  int NW;            // compute warps = ceil(M / 8); the producer is warp NW
  int logn1, logn2, logwb;  // NLM_ENTER / NLM_EXIT: geometry of the blocked order (N = N1 N2, WB columns per block)
  long long ntiles;  // N / 8
};

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}

template <int MODE>
__host__ __device__ constexpr int nlm_narr() {  // field arrays per slot
  return (MODE == NLM_PLAIN || MODE == NLM_RK4 || MODE == NLM_AGR_S0 || MODE == NLM_AGR_IT1) ? 1 : 2;
}
template <int MODE>
__host__ __device__ constexpr bool nlm_has_table() {  // the slot also holds a tile of the real table T (M x 8 doubles)
  return MODE == NLM_AGR_S0 || MODE == NLM_AGR_IT1 || MODE == NLM_AGR_ITJ;
}

// bytes of dynamic shared memory: ring slots, two P buffers, mbarriers
__host__ __device__ inline size_t nlt_table_bytes(int M) { return ((size_t)M * MMF_NLM_T * sizeof(double) + 127) & ~(size_t)127; }
__host__ __device__ inline size_t nlt_slot_bytes(int M, int narr, bool table) {
  return (size_t)narr * 2 * M * MMF_NLM_T * sizeof(cpx) + (table ? nlt_table_bytes(M) : 0);
}
#define MMF_NLM_MAXG 32   // distinct kappa rows the grouped contraction handles (four warps of eight rows)
// G: distinct rows of the grouped contraction (0: dense kernel, no room for their S)
__host__ __device__ inline size_t nlt_sg_bytes(int G) { return (size_t)((G + 7) & ~7) * MMF_NLM_PSTRIDE * sizeof(double); }
__host__ __device__ inline size_t nlt_smem_bytes(int M, int nk, int narr, bool table, int G = 0) {
  return MMF_NLM_SLOTS * nlt_slot_bytes(M, narr, table) + (size_t)2 * (4 * nk) * MMF_NLM_PSTRIDE * sizeof(double) +
         nlt_sg_bytes(G) + 128;
}

// S = kappa_slab * P  for this warp's 8 rows and the tile's 8 samples (four independent accumulator chains)
template <int NK>
__device__ __forceinline__ void nlm_contract(const double (&kf)[NK], const double* __restrict__ P, int g, int q,
                                             double& s0, double& s1) {
  double c[4][2] = {{0.0, 0.0}, {0.0, 0.0}, {0.0, 0.0}, {0.0, 0.0}};
  const double* pb = P + q * MMF_NLM_PSTRIDE + g;
#pragma unroll
  for (int ks = 0; ks < NK; ++ks) dmma884(c[ks & 3][0], c[ks & 3][1], kf[ks], pb[(4 * ks) * MMF_NLM_PSTRIDE]);
  s0 = (c[0][0] + c[1][0]) + (c[2][0] + c[3][0]);
  s1 = (c[0][1] + c[1][1]) + (c[2][1] + c[3][1]);
}

__device__ __forceinline__ double power2(cpx a, cpx b) { return (a.x * a.x + a.y * a.y) + (b.x * b.x + b.y * b.y); }
__device__ __forceinline__ cpx times_ig(cpx u, double g) { return make_double2(-g * u.y, g * u.x); }  // (i g) u
__device__ __forceinline__ cpx axpy(double s, cpx a, cpx b) { return make_double2(fma(s, a.x, b.x), fma(s, a.y, b.y)); }

// GROUPED (mode groups, section 6: "The modes form strongly coupled groups of modes ... taken into account by
// choosing the appropriate nonlinear coupling coefficients kappa"): when kappa has only G << M DISTINCT
// rows (every mode of a group couples to the others alike), S has only G distinct rows too.  The first ceil(G / 8) warps
// contract the G distinct rows with P (the same DMMA chains, G M instead of M M products per sample), park the result
// in shared memory, and after one more barrier every lane picks the row of its mode's group.
// NK = ceil(M / 4) k-steps of the contraction (compile-time: the kappa fragments are a register array).
// mapA / mapB: 2-D tensor maps (inner = 2N doubles, outer = 2M rows, box = 16 doubles x 2M rows) of
//   PLAIN: U / OUT;  other modes: X / Y.  mapC: ENTER / EXIT the caller's field; AGR_*: the table T (inner = N doubles,
//   outer = M rows, box = 8 doubles x M rows).
// block = 32 (NW + 1) threads; grid = persistent; dynamic smem = nlt_smem_bytes(M, NK, narr).
template <int NK, int MODE, int GROUPED = 0>
__global__ void __launch_bounds__(512, 1)
k_nlt(const __grid_constant__ CUtensorMap mapA, const __grid_constant__ CUtensorMap mapB,
      const __grid_constant__ CUtensorMap mapC, NltParams p) {
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  constexpr int NARR = nlm_narr<MODE>();
  constexpr bool TWO_ROUNDS = (MODE == NLM_S23 || MODE == NLM_FINAL_NEXT);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int M = p.M, R = 2 * M, NW = p.NW;
  const size_t arr_elems = (size_t)R * MMF_NLM_T;            // cpx per array per slot
  constexpr bool TABLE = nlm_has_table<MODE>();
  const size_t tab_off = NARR * arr_elems * sizeof(cpx);      // the table tile sits behind the field arrays of a slot
  const size_t slot_bytes = tab_off + (TABLE ? nlt_table_bytes(M) : 0);
  double* Pb0 = reinterpret_cast<double*>(smem_raw + MMF_NLM_SLOTS * slot_bytes);
  double* Pb1 = Pb0 + 4 * NK * MMF_NLM_PSTRIDE;
  double* Sg = Pb1 + 4 * NK * MMF_NLM_PSTRIDE;   // GROUPED: S of the distinct rows, [G rounded up to 8][PSTRIDE]
  uint64_t* full = reinterpret_cast<uint64_t*>(Sg + (GROUPED ? ((p.G + 7) & ~7) * MMF_NLM_PSTRIDE : 0));
  uint64_t* done = full + MMF_NLM_SLOTS;

  if (threadIdx.x == 0) {
#pragma unroll
    for (int s = 0; s < MMF_NLM_SLOTS; ++s) {
      mbar_init(&full[s], 1);
      mbar_init(&done[s], NW);
    }
    mbar_init_fence();
  }
  pdl_launch_dependents();
  for (int i = threadIdx.x; i < 2 * 4 * NK * MMF_NLM_PSTRIDE; i += blockDim.x) Pb0[i] = 0.0;  // padding rows stay 0
  __syncthreads();

  const long long tstep = gridDim.x;

  // ------------------------------------------------------------------------------------------------ producer warp
  if (warp == NW) {
    if (lane != 0) return;
    tma_prefetch_desc(&mapA);
    tma_prefetch_desc(&mapB);
    tma_prefetch_desc(&mapC);
    pdl_wait();   // the fields are the predecessor's output (only this thread touches global memory)
    // natural-order tile that holds the samples of blocked tile t (ENTER reads it, EXIT writes it)
    auto natural_tile = [&](long long t) -> long long {
      const int u8 = p.logwb - 3;  // log2(tiles per unit of WB columns)
      const long long cbt = t & ((1LL << u8) - 1), unit = t >> u8;
      const long long n1 = unit & ((1LL << p.logn1) - 1), ctb = unit >> p.logn1;
      return (n1 << (p.logn2 - 3)) + (ctb << u8) + cbt;
    };
    auto store_tile = [&](long long tl, int slot) {
      unsigned char* s = smem_raw + slot * slot_bytes;
      const int c0 = (int)(tl * 2 * MMF_NLM_T);
      if constexpr (MODE == NLM_ENTER) {  // X <- A and Y <- NL(A), blocked order
        tma_store_2d(&mapB, c0, 0, s);
        tma_store_2d(&mapC, c0, 0, s + arr_elems * sizeof(cpx));
      } else if constexpr (MODE == NLM_EXIT) {  // the new field, natural order
        tma_store_2d(&mapC, (int)(natural_tile(tl) * 2 * MMF_NLM_T), 0, s);
      } else if constexpr (MODE == NLM_AGR_S0) {  // only the table leaves
        tma_store_2d(&mapC, (int)(tl * MMF_NLM_T), 0, s + tab_off);
      } else if constexpr (MODE == NLM_AGR_IT1) {
        tma_store_2d(&mapB, c0, 0, s);
      } else if constexpr (MODE == NLM_AGR_ITJ) {
        tma_store_2d(&mapB, c0, 0, s + arr_elems * sizeof(cpx));
      } else {
        tma_store_2d((MODE == NLM_PLAIN) ? &mapB : &mapA, c0, 0, s);
        if constexpr (MODE == NLM_S23 || MODE == NLM_FINAL_NEXT) tma_store_2d(&mapB, c0, 0, s + arr_elems * sizeof(cpx));
      }
      tma_store_commit();
    };
    constexpr uint32_t kLoadArrays = (MODE == NLM_ENTER) ? 1 : NARR;
    long long tile = blockIdx.x;
    int j = 0;
    for (; tile < p.ntiles; tile += tstep, ++j) {
      const int slot = j % MMF_NLM_SLOTS, use = j / MMF_NLM_SLOTS;
      unsigned char* s = smem_raw + slot * slot_bytes;
      if (use > 0) {  // the tile that occupied this slot: store it once computed, then wait until it has been read out
        mbar_wait(&done[slot], (use - 1) & 1);
        store_tile(tile - MMF_NLM_SLOTS * tstep, slot);
        tma_store_wait_read();
      }
      constexpr bool kLoadTable = MODE == NLM_AGR_IT1 || MODE == NLM_AGR_ITJ;
      mbar_arrive_expect_tx(&full[slot], (uint32_t)(kLoadArrays * arr_elems * sizeof(cpx) +
                                                    (kLoadTable ? (size_t)M * MMF_NLM_T * sizeof(double) : 0)));
      const long long tin = (MODE == NLM_ENTER) ? natural_tile(tile) : tile;
      tma_load_2d(s, &mapA, (int)(tin * 2 * MMF_NLM_T), 0, &full[slot]);
      if constexpr (kLoadArrays == 2) tma_load_2d(s + arr_elems * sizeof(cpx), &mapB, (int)(tile * 2 * MMF_NLM_T), 0, &full[slot]);
      if constexpr (kLoadTable) tma_load_2d(s + tab_off, &mapC, (int)(tile * MMF_NLM_T), 0, &full[slot]);
    }
    for (int jj = (j > MMF_NLM_SLOTS ? j - MMF_NLM_SLOTS : 0); jj < j; ++jj) {  // drain
      const int slot = jj % MMF_NLM_SLOTS, use = jj / MMF_NLM_SLOTS;
      mbar_wait(&done[slot], use & 1);
      store_tile(blockIdx.x + jj * tstep, slot);
    }
    tma_store_wait_all();
    return;
  }

  // ------------------------------------------------------------------------------------------------ compute warps
  const int gthreads = 32 * NW;
  const int g = lane >> 2, q = lane & 3;
  const int a = warp * 8 + g;
  const bool valid = a < M;

  // this warp's slab of kappa as A fragments: kf[ks] = kappa[a][4 ks + q]
  double kf[NK];
  const int krow = GROUPED ? warp * 8 + g : a;   // GROUPED: row of the distinct-row matrix this lane's fragments hold
  const bool kvalid = GROUPED ? krow < p.G : valid;
#pragma unroll
  for (int ks = 0; ks < NK; ++ks) {
    const int b = 4 * ks + q;
    kf[ks] = (kvalid && b < M) ? p.kappa[(long long)krow * M + b] : 0.0;
  }
  const int grp = (GROUPED && valid) ? p.group_of[a] : 0;
  // S = kappa P for this lane's mode and samples 2q, 2q + 1 (after the barrier that published P)
  auto contract = [&](const double* Pbuf, double& s0, double& s1) {
    if constexpr (GROUPED) {
      if (warp * 8 < p.G) {   // warp-uniform
        double t0, t1;
        nlm_contract<NK>(kf, Pbuf, g, q, t0, t1);
        if (kvalid) *reinterpret_cast<double2*>(Sg + krow * MMF_NLM_PSTRIDE + 2 * q) = make_double2(t0, t1);
      }
      group_barrier(1, gthreads);
      const double2 sv = *reinterpret_cast<const double2*>(Sg + grp * MMF_NLM_PSTRIDE + 2 * q);
      s0 = sv.x;
      s1 = sv.y;
    } else {
      nlm_contract<NK>(kf, Pbuf, g, q, s0, s1);
    }
  };
  const double third = 1.0 / 3.0, sixth = 1.0 / 6.0;
  const int e0 = (2 * a) * MMF_NLM_T + 2 * q;  // this lane's elements: rows 2a (x), 2a+1 (y), samples 2q, 2q+1

  int j = 0;
  for (long long tile = blockIdx.x; tile < p.ntiles; tile += tstep, ++j) {
    const int slot = j % MMF_NLM_SLOTS;
    cpx* sx = reinterpret_cast<cpx*>(smem_raw + slot * slot_bytes);
    cpx* sy = sx + arr_elems;
    double* P1 = TWO_ROUNDS ? Pb0 : ((j & 1) ? Pb1 : Pb0);
    mbar_wait(&full[slot], (j / MMF_NLM_SLOTS) & 1);

    cpx x[2][2], y[2][2], u[2][2];
#pragma unroll
    for (int pol = 0; pol < 2; ++pol)
#pragma unroll
      for (int i = 0; i < 2; ++i) {
        x[pol][i] = valid ? sx[e0 + pol * MMF_NLM_T + i] : make_double2(0.0, 0.0);
        if constexpr (NARR == 2 && MODE != NLM_ENTER) y[pol][i] = valid ? sy[e0 + pol * MMF_NLM_T + i] : make_double2(0.0, 0.0);
        if constexpr (MODE == NLM_S23) u[pol][i] = axpy(0.5, y[pol][i], x[pol][i]);
        else if constexpr (MODE == NLM_AGR_ITJ) u[pol][i] = y[pol][i];   // |A|^2 at z + h: from the previous iterate
        else u[pol][i] = x[pol][i];
      }
    if constexpr (MODE == NLM_AGR_IT1) {  // no contraction: Y <- exp(i T) X, element by element
      if (valid) {
        const double2 th = *reinterpret_cast<const double2*>(smem_raw + slot * slot_bytes + tab_off +
                                                             (a * MMF_NLM_T + 2 * q) * sizeof(double));
        double sn[2], cs[2];
        sincos(th.x, &sn[0], &cs[0]);
        sincos(th.y, &sn[1], &cs[1]);
#pragma unroll
        for (int pol = 0; pol < 2; ++pol)
#pragma unroll
          for (int i = 0; i < 2; ++i) sx[e0 + pol * MMF_NLM_T + i] = cmul(x[pol][i], make_double2(cs[i], sn[i]));
      }
      fence_proxy_async_smem();
      __syncwarp();
      if (lane == 0) mbar_arrive(&done[slot]);
      continue;
    }
    if constexpr (MODE == NLM_RK4) {
      cpx acc[2][2];
#pragma unroll
      for (int r = 0; r < 4; ++r) {
        double* Pr = (r & 1) ? Pb1 : Pb0;
        if (valid)
          *reinterpret_cast<double2*>(Pr + a * MMF_NLM_PSTRIDE + 2 * q) =
              make_double2(power2(u[0][0], u[1][0]), power2(u[0][1], u[1][1]));
        group_barrier(1, gthreads);
        double sr[2];
        contract(Pr, sr[0], sr[1]);
#pragma unroll
        for (int pol = 0; pol < 2; ++pol)
#pragma unroll
          for (int i = 0; i < 2; ++i) {
            const cpx k = times_ig(u[pol][i], p.hg * sr[i]);  // k_{r+1} = h N(u) u
            const cpx xx = x[pol][i];
            if (r == 0) acc[pol][i] = axpy(sixth, k, xx);
            else acc[pol][i] = axpy((r == 3) ? sixth : third, k, acc[pol][i]);
            if (r < 3) u[pol][i] = axpy((r == 2) ? 1.0 : 0.5, k, xx);
          }
      }
      if (valid) {
#pragma unroll
        for (int pol = 0; pol < 2; ++pol)
#pragma unroll
          for (int i = 0; i < 2; ++i) sx[e0 + pol * MMF_NLM_T + i] = acc[pol][i];
      }
      fence_proxy_async_smem();
      __syncwarp();
      if (lane == 0) mbar_arrive(&done[slot]);
      continue;
    }
    // ---- round 1 ---------------------------------------------------------------------------------------------
    if (valid)
      *reinterpret_cast<double2*>(P1 + a * MMF_NLM_PSTRIDE + 2 * q) =
          make_double2(power2(u[0][0], u[1][0]), power2(u[0][1], u[1][1]));
    group_barrier(1, gthreads);
    double s[2];
    contract(P1, s[0], s[1]);
    const double g1[2] = {p.hg * s[0], p.hg * s[1]};

    if constexpr (MODE == NLM_AGR_S0 || MODE == NLM_AGR_ITJ) {
      double2* tt = reinterpret_cast<double2*>(smem_raw + slot * slot_bytes + tab_off + (a * MMF_NLM_T + 2 * q) * sizeof(double));
      if (valid) {
        if constexpr (MODE == NLM_AGR_S0) {
          *tt = make_double2(g1[0], g1[1]);   // T = h gamma S(A(z))
        } else {
          const double2 t0 = *tt;
          double sn[2], cs[2];
          sincos(0.5 * (t0.x + g1[0]), &sn[0], &cs[0]);   // (h gamma / 2) [S(A(z)) + S(A_{j-1}(z + h))]
          sincos(0.5 * (t0.y + g1[1]), &sn[1], &cs[1]);
#pragma unroll
          for (int pol = 0; pol < 2; ++pol)
#pragma unroll
            for (int i = 0; i < 2; ++i) sy[e0 + pol * MMF_NLM_T + i] = cmul(x[pol][i], make_double2(cs[i], sn[i]));
        }
      }
    } else if constexpr (MODE == NLM_PLAIN || MODE == NLM_ENTER) {
      cpx* so = (MODE == NLM_ENTER) ? sy : sx;  // ENTER keeps the field in the first array of the slot
      if (valid) {
#pragma unroll
        for (int pol = 0; pol < 2; ++pol)
#pragma unroll
          for (int i = 0; i < 2; ++i) so[e0 + pol * MMF_NLM_T + i] = times_ig(u[pol][i], g1[i]);
      }
    } else if constexpr (MODE == NLM_FINAL || MODE == NLM_EXIT) {
      if (valid) {
#pragma unroll
        for (int pol = 0; pol < 2; ++pol)
#pragma unroll
          for (int i = 0; i < 2; ++i) {
            const cpx an = axpy(sixth, times_ig(u[pol][i], g1[i]), y[pol][i]);
            sx[e0 + pol * MMF_NLM_T + i] = make_double2(p.gain * an.x, p.gain * an.y);
          }
      }
    } else {
      // ---- round 2 -------------------------------------------------------------------------------------------
      cpx v[2][2];  // S23: u3 = X + k2/2;  FINAL_NEXT: the new field A(z+h)
#pragma unroll
      for (int pol = 0; pol < 2; ++pol)
#pragma unroll
        for (int i = 0; i < 2; ++i) {
          const cpx k = times_ig(u[pol][i], g1[i]);  // k2 resp. k4
          if constexpr (MODE == NLM_S23) {
            v[pol][i] = axpy(0.5, k, x[pol][i]);
          } else {
            const cpx an = axpy(sixth, k, y[pol][i]);
            v[pol][i] = make_double2(p.gain * an.x, p.gain * an.y);   // the lumped amplifier acts before the next N
          }
        }
      if (valid)
        *reinterpret_cast<double2*>(Pb1 + a * MMF_NLM_PSTRIDE + 2 * q) =
            make_double2(power2(v[0][0], v[1][0]), power2(v[0][1], v[1][1]));
      group_barrier(1, gthreads);
      double s2[2];
      contract(Pb1, s2[0], s2[1]);
      const double g2[2] = {p.hg * s2[0], p.hg * s2[1]};
      if (valid) {
#pragma unroll
        for (int pol = 0; pol < 2; ++pol)
#pragma unroll
          for (int i = 0; i < 2; ++i) {
            const int o = e0 + pol * MMF_NLM_T + i;
            const cpx kk = times_ig(v[pol][i], g2[i]);  // k3 resp. the next bracket
            if constexpr (MODE == NLM_S23) {
              const cpx k2 = times_ig(u[pol][i], g1[i]);
              const cpx xx = x[pol][i], yy = y[pol][i];
              sx[o] = cadd(xx, kk);
              sy[o] = make_double2(xx.x + sixth * yy.x + third * k2.x + third * kk.x,
                                   xx.y + sixth * yy.y + third * k2.y + third * kk.y);
            } else {
              sx[o] = v[pol][i];
              sy[o] = kk;
            }
          }
      }
    }
    // results are in the slot: hand it to the producer for the TMA store
    fence_proxy_async_smem();
    __syncwarp();
    if (lane == 0) mbar_arrive(&done[slot]);
  }
}

}  // namespace mmf
