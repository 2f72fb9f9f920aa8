// tmem_exchange.cuh — the warp-local exchange of a 4096-point transform through TENSOR MEMORY instead of shared memory.
//
// Why.  Pass B (k_rows, fft_kernels.cuh) keeps its shared-memory pipe busy 71 % of the time with five exchanges of 16 B
// each way per point at 128 B per clock per SM (profiles/r2a_ncu_full_cfg4.md).  Tensor memory is a second on-chip
// store with a datapath of its own (bench.py --probes, profiles/r2b_probes.json: tcgen05.st 32x32b moves 840 B per clock
// per SM, tcgen05.ld at least 330, against 114-128 for LDS.128 and SHFL), but with that shape a thread only reaches its
// own lane.  The 16x256b shape is the
// exception: thread T of a warp reads (writes) lanes 8 q + (T >> 2) (+ 16 h for the second instruction) and, of every
// group of four 64-bit columns, column (T & 3) (layout determined with a probe kernel).  A store with one shape
// followed by a load with the other therefore MOVES data between the lanes of a warp:
//   store 32x32b (thread L writes doubles d = 0..15 of its lane), load 16x256b:
//       thread T receives, as value (h, q, g), what thread L = 16 h + 8 q + (T >> 2) wrote as double 4 g + (T & 3).
//   In index bits: the two top lane bits of the writer become register bits, the two low register bits of the writer
//   become the two low lane bits of the reader, the other three lane bits shift up by two.
// Two such trips exchange four lane bits with four register bits — the 16 x 16 transpose between the second and the
// third radix-16 stage of a 4096-point transform (whose values stay inside a warp), with no shared-memory traffic.
// The reverse (store 16x256b, load 32x32b) undoes a trip; the inverse transform uses it.
//
// Layouts of the 12 index bits f of a tile (warp = f[11:9] throughout; reg = the 4-bit register index):
//   stage 2:  lane = (f3 f2 f1 f0 f8), reg = (f7 f6 f5 f4)            -- what the exchange through shared memory delivers
//   trip   :  lane = (f1 f0 f8 f5 f4), reg = (f3 f2 f7 f6)
//   trip   :  lane = (f8 f5 f4 f7 f6), reg = (f1 f0 f3 f2)  -> renamed to reg = (f3 f2 f1 f0) = the stage-3 digit
// Real and imaginary parts travel as two column blocks (columns [0,32) and [32,64) of the warp's exchange buffer).
#pragma once
#include "async_copy.cuh"
#include "fft_core.cuh"

namespace mmf {

#define MMF_R16(a, o) "r"(a[o + 0]), "r"(a[o + 1]), "r"(a[o + 2]), "r"(a[o + 3]), "r"(a[o + 4]), "r"(a[o + 5]), \
    "r"(a[o + 6]), "r"(a[o + 7]), "r"(a[o + 8]), "r"(a[o + 9]), "r"(a[o + 10]), "r"(a[o + 11]), "r"(a[o + 12]),   \
    "r"(a[o + 13]), "r"(a[o + 14]), "r"(a[o + 15])
#define MMF_W16(a, o) "=r"(a[o + 0]), "=r"(a[o + 1]), "=r"(a[o + 2]), "=r"(a[o + 3]), "=r"(a[o + 4]), "=r"(a[o + 5]), \
    "=r"(a[o + 6]), "=r"(a[o + 7]), "=r"(a[o + 8]), "=r"(a[o + 9]), "=r"(a[o + 10]), "=r"(a[o + 11]), "=r"(a[o + 12]),  \
    "=r"(a[o + 13]), "=r"(a[o + 14]), "=r"(a[o + 15])
#define MMF_RW16(a, o) "+r"(a[o + 0]), "+r"(a[o + 1]), "+r"(a[o + 2]), "+r"(a[o + 3]), "+r"(a[o + 4]), "+r"(a[o + 5]), \
    "+r"(a[o + 6]), "+r"(a[o + 7]), "+r"(a[o + 8]), "+r"(a[o + 9]), "+r"(a[o + 10]), "+r"(a[o + 11]), "+r"(a[o + 12]),  \
    "+r"(a[o + 13]), "+r"(a[o + 14]), "+r"(a[o + 15])

// 32 consecutive columns of the thread's own lane
__device__ __forceinline__ void tmem_st_32x32b_x32(uint32_t taddr, const int (&w)[32]) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,"
      "%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31,%32};\n" ::"r"(taddr),
      MMF_R16(w, 0), MMF_R16(w, 16));
}
__device__ __forceinline__ void tmem_ld_32x32b_x32(int (&w)[32], uint32_t taddr) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,"
      "%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];\n"
      : MMF_W16(w, 0), MMF_W16(w, 16)
      : "r"(taddr));
}
// 16 lanes x 32 columns: register 4 g + 2 q + w <-> lane 8 q + (T >> 2), column 8 g + 2 (T & 3) + w
__device__ __forceinline__ void tmem_st_16x256b_x4(uint32_t taddr, const int (&w)[16]) {
  asm volatile(
      "tcgen05.st.sync.aligned.16x256b.x4.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};\n" ::"r"(taddr),
      MMF_R16(w, 0));
}
__device__ __forceinline__ void tmem_ld_16x256b_x4(int (&w)[16], uint32_t taddr) {
  asm volatile(
      "tcgen05.ld.sync.aligned.16x256b.x4.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];\n"
      : MMF_W16(w, 0)
      : "r"(taddr));
}
// wait for this thread's tensor-memory loads; names the registers so that no use of them is scheduled ahead of it
__device__ __forceinline__ void tmem_wait_ld16(int (&w)[16]) {
  asm volatile("tcgen05.wait::ld.sync.aligned;\n" : MMF_RW16(w, 0));
}
__device__ __forceinline__ void tmem_wait_ld32(int (&w)[32]) {
  asm volatile("tcgen05.wait::ld.sync.aligned;\n" : MMF_RW16(w, 0), MMF_RW16(w, 16));
}

// forward trip (store 32x32b, load 16x256b): v[j] of lane L arrives as v[8 h + 4 q + g] of lane T, where
// L = 16 h + 8 q + (T >> 2) and j = 4 g + (T & 3).   xa: the warp's 64-column exchange buffer (lane base of its quarter).
__device__ __forceinline__ void tmem_trip_fwd(cpx (&v)[16], uint32_t xa) {
  {
    int re[32], im[32];
#pragma unroll
    for (int j = 0; j < 16; ++j) {
      re[2 * j] = __double2loint(v[j].x);
      re[2 * j + 1] = __double2hiint(v[j].x);
      im[2 * j] = __double2loint(v[j].y);
      im[2 * j + 1] = __double2hiint(v[j].y);
    }
    tmem_st_32x32b_x32(xa, re);
    tmem_st_32x32b_x32(xa + 32, im);
  }
  tmem_wait_st();
  int a[2][16], b[2][16];  // [h][4 g + 2 q + w]: real parts, imaginary parts
  tmem_ld_16x256b_x4(a[0], xa);
  tmem_ld_16x256b_x4(a[1], xa + (16u << 16));
  tmem_ld_16x256b_x4(b[0], xa + 32);
  tmem_ld_16x256b_x4(b[1], xa + 32 + (16u << 16));
  tmem_wait_ld16(a[0]);
  tmem_wait_ld16(a[1]);
  tmem_wait_ld16(b[0]);
  tmem_wait_ld16(b[1]);
#pragma unroll
  for (int h = 0; h < 2; ++h)
#pragma unroll
    for (int q = 0; q < 2; ++q)
#pragma unroll
      for (int g = 0; g < 4; ++g)
        v[8 * h + 4 * q + g] = make_double2(__hiloint2double(a[h][4 * g + 2 * q + 1], a[h][4 * g + 2 * q]),
                                            __hiloint2double(b[h][4 * g + 2 * q + 1], b[h][4 * g + 2 * q]));
}

// reverse trip (store 16x256b, load 32x32b): v[8 h + 4 q + g] of lane T arrives as v[4 g + (T & 3)] of lane
// 16 h + 8 q + (T >> 2) — the inverse of tmem_trip_fwd.
__device__ __forceinline__ void tmem_trip_rev(cpx (&v)[16], uint32_t xa) {
  {
    int a[2][16], b[2][16];
#pragma unroll
    for (int h = 0; h < 2; ++h)
#pragma unroll
      for (int q = 0; q < 2; ++q)
#pragma unroll
        for (int g = 0; g < 4; ++g) {
          const cpx x = v[8 * h + 4 * q + g];
          a[h][4 * g + 2 * q] = __double2loint(x.x);
          a[h][4 * g + 2 * q + 1] = __double2hiint(x.x);
          b[h][4 * g + 2 * q] = __double2loint(x.y);
          b[h][4 * g + 2 * q + 1] = __double2hiint(x.y);
        }
    tmem_st_16x256b_x4(xa, a[0]);
    tmem_st_16x256b_x4(xa + (16u << 16), a[1]);
    tmem_st_16x256b_x4(xa + 32, b[0]);
    tmem_st_16x256b_x4(xa + 32 + (16u << 16), b[1]);
  }
  tmem_wait_st();
  int re[32], im[32];
  tmem_ld_32x32b_x32(re, xa);
  tmem_ld_32x32b_x32(im, xa + 32);
  tmem_wait_ld32(re);
  tmem_wait_ld32(im);
#pragma unroll
  for (int j = 0; j < 16; ++j)
    v[j] = make_double2(__hiloint2double(re[2 * j + 1], re[2 * j]), __hiloint2double(im[2 * j + 1], im[2 * j]));
}

// ---- the 4096-point chains of pass B with the second exchange in tensor memory ---------------------------------------
// Thread t of a group (warp = t >> 5, lane = t & 31).  Stage 1 keeps the layout of fft_core.cuh (registers = f[11:8],
// thread = f[7:0]); stages 2 and 3 use the lane assignments listed at the top of this file.
struct Tm12 {
  int base1;   // stage 1: t
  int base2;   // stage 2: warp << 9 | (lane & 1) << 8 | lane >> 1
  int tv;      // stage 3: f[11:4] of the thread's values = warp << 5 | l4 << 4 | l1 << 3 | l0 << 2 | l3 << 1 | l2
};
__device__ __forceinline__ Tm12 tm12_layout(int t) {
  const int lane = t & 31, warp = t >> 5;
  Tm12 L;
  L.base1 = t;
  L.base2 = (warp << 9) | ((lane & 1) << 8) | (lane >> 1);
  L.tv = (warp << 5) | (lane & 16) | ((lane & 3) << 2) | ((lane >> 2) & 3);
  return L;
}
// The exchange between stages 1 and 2 stays in shared memory; with the stage-2 lanes above a quarter warp reads
// f[1:0] x f8, so the bank swizzle also folds bit 8 in (the stage-1 side, consecutive f, is conflict-free regardless).
__device__ __forceinline__ int swz12(int f) { return f ^ ((f >> 4) & 7) ^ ((f >> 6) & 4); }
template <int LO>
__device__ __forceinline__ void tile_lds12(cpx (&v)[16], const cpx* __restrict__ s, int base) {
#pragma unroll
  for (int j = 0; j < 16; ++j) v[j] = s[swz12(base | (j << LO))];
}
template <int LO>
__device__ __forceinline__ void tile_sts12(const cpx (&v)[16], cpx* __restrict__ s, int base) {
#pragma unroll
  for (int j = 0; j < 16; ++j) s[swz12(base | (j << LO))] = v[j];
}
// v[(g << 2) | (h << 1) | q] <- v[(h << 3) | (q << 2) | g]  (register renaming) and its inverse
__device__ __forceinline__ void tm12_rename_fwd(cpx (&v)[16]) {
  cpx w[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) w[i] = v[i];
#pragma unroll
  for (int h = 0; h < 2; ++h)
#pragma unroll
    for (int q = 0; q < 2; ++q)
#pragma unroll
      for (int g = 0; g < 4; ++g) v[(g << 2) | (h << 1) | q] = w[(h << 3) | (q << 2) | g];
}
__device__ __forceinline__ void tm12_rename_inv(cpx (&v)[16]) {
  cpx w[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) w[i] = v[i];
#pragma unroll
  for (int h = 0; h < 2; ++h)
#pragma unroll
    for (int q = 0; q < 2; ++q)
#pragma unroll
      for (int g = 0; g < 4; ++g) v[(h << 3) | (q << 2) | g] = w[(g << 2) | (h << 1) | q];
}

// Forward chain (DIF).  Entry: v in the stage-1 layout, taken by the caller from the tile TMA staged in s UNSWIZZLED:
// the first exchange write of thread t goes to slots swz12(t | j << 8), which differ from the slots t | j << 8 it read
// in bits [2:0] only, i.e. they were read by lanes of the same warp — a warp barrier orders the two, no group barrier.
// Exit: v[j] = slot (tv << 4 | j), digit-reversed order.
template <int SIGN>
__device__ __forceinline__ void fft12_dif_tm(cpx (&v)[16], cpx* __restrict__ s, const Tm12& L, const cpx* __restrict__ tab,
                                             int bar, uint32_t xa) {
  stage_math<12, 0, 8, 4, SIGN, true>(v, L.base1, tab + tw_offset(12, 12, 3));
  __syncwarp();
  tile_sts12<8>(v, s, L.base1);
  group_barrier(bar, MMF_GROUP_THREADS);
  tile_lds12<4>(v, s, L.base2);
  stage_math<12, 0, 4, 4, SIGN, true>(v, L.base2, tab + tw_offset(12, 8, 2));
  tmem_trip_fwd(v, xa);
  tmem_trip_fwd(v, xa);
  tm12_rename_fwd(v);
  stage_math<12, 0, 0, 4, SIGN, true>(v, 0, tab);
}
// Inverse chain (DIT), the adjoint of the forward chain with the opposite SIGN.  Exit: v in the stage-1 layout.
template <int SIGN>
__device__ __forceinline__ void fft12_dit_tm(cpx (&v)[16], cpx* __restrict__ s, const Tm12& L, const cpx* __restrict__ tab,
                                             int bar, uint32_t xa) {
  stage_math<12, 0, 0, 4, SIGN, false>(v, 0, tab);
  tm12_rename_inv(v);
  tmem_trip_rev(v, xa);
  tmem_trip_rev(v, xa);
  stage_math<12, 0, 4, 4, SIGN, false>(v, L.base2, tab + tw_offset(12, 8, 2));
  tile_sts12<4>(v, s, L.base2);
  group_barrier(bar, MMF_GROUP_THREADS);
  tile_lds12<8>(v, s, L.base1);
  stage_math<12, 0, 8, 4, SIGN, false>(v, L.base1, tab + tw_offset(12, 12, 3));
}

}  // namespace mmf
