// fft_core.cuh — register-level and shared-memory FFT building blocks (fp64 complex), sm_100a.
//
// Role in the path: rows a1/a3 of the hot-path table (forward / inverse transform of every field, PAPER.md:107
// "fast Fourier transforms ... rows are aligned linear in the memory"; Eq. 6 PAPER.md:75-88 needs exp(h/2 L)
// four times per step).  Design:
//   * a "tile" is 2^12 complex values worked on by one GROUP of 256 threads; every thread owns 16 values
//     (64 registers) and performs radix-2..16 butterflies on them;
//   * a transform of 2^LOGP points is split into NST = ceil(LOGP/4) digits.  The FIRST stage takes its 16 values
//     from the tile TMA staged in shared memory and the LAST stage leaves them in registers for the epilogue
//     (spectral multiply, inter-pass twiddle); the same shared-memory slot is the exchange buffer BETWEEN stages
//     (one STS.128 + one LDS.128 per value per exchange, one group barrier per exchange);
//   * decimation in frequency on the way to the spectrum, the exact adjoint (decimation in time) on the way back,
//     so no bit-reversal pass exists: the spectrum stays in digit-reversed slot order, the last forward stage and
//     the first inverse stage share one register layout, and the exp(h/2 L) table is stored in that order;
//   * the exchange buffer is XOR-swizzled (slot ^ ((slot >> 4) & 7)): every stage's LDS.128/STS.128 pattern is
//     bank-conflict free;
//   * inter-stage twiddles come from per-stage tables laid out [c][b] (c = output index of the butterfly, b = low
//     bits of the point index): lanes read consecutive or identical entries, one to four wavefronts per load
//     instead of a 32-way gather from a length-N table.
#pragma once
#include <cuda_runtime.h>

namespace mmf {

typedef double2 cpx;

__device__ __forceinline__ cpx cadd(cpx a, cpx b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ cpx csub(cpx a, cpx b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ cpx cmul(cpx a, cpx b) {
  return make_double2(fma(a.x, b.x, -a.y * b.y), fma(a.x, b.y, a.y * b.x));
}
// a * conj(b)
__device__ __forceinline__ cpx cmulc(cpx a, cpx b) {
  return make_double2(fma(a.x, b.x, a.y * b.y), fma(a.y, b.x, -a.x * b.y));
}
template <int SIGN>
__device__ __forceinline__ cpx cmul_s(cpx a, cpx w) {  // a * (SIGN > 0 ? w : conj(w))
  return SIGN > 0 ? cmul(a, w) : cmulc(a, w);
}

// multiply by exp(SIGN * 2 pi i * S16 / 16), S16 in [0, 8): constants of the 16th roots of unity
template <int S16, int SIGN>
__device__ __forceinline__ cpx mul_root16(cpx d) {
  constexpr double C8 = 0.92387953251128675613;  // cos(pi/8)
  constexpr double S8 = 0.38268343236508977173;  // sin(pi/8)
  constexpr double H = 0.70710678118654752440;   // sqrt(1/2)
  if constexpr (S16 == 0) {
    return d;
  } else if constexpr (S16 == 4) {
    return SIGN > 0 ? make_double2(-d.y, d.x) : make_double2(d.y, -d.x);
  } else if constexpr (S16 == 2) {  // (1 + s i)/sqrt2
    return SIGN > 0 ? make_double2((d.x - d.y) * H, (d.x + d.y) * H) : make_double2((d.x + d.y) * H, (d.y - d.x) * H);
  } else if constexpr (S16 == 6) {  // (-1 + s i)/sqrt2
    return SIGN > 0 ? make_double2(-(d.x + d.y) * H, (d.x - d.y) * H) : make_double2((d.y - d.x) * H, -(d.x + d.y) * H);
  } else {
    constexpr double wr = (S16 == 1) ? C8 : (S16 == 3) ? S8 : (S16 == 5) ? -S8 : -C8;
    constexpr double wi = (S16 == 1) ? S8 : (S16 == 3) ? C8 : (S16 == 5) ? C8 : S8;
    return cmul_s<SIGN>(d, make_double2(wr, wi));
  }
}

// Natural-order DFT of R = 2,4,8,16 values held in registers:  v[c] <- sum_a exp(SIGN 2 pi i a c / R) v[a].
// Radix-2 decimation in frequency, fully unrolled; the final re-ordering is register renaming.
template <int R, int SIGN>
struct Dft {
  template <int A>
  static __device__ __forceinline__ void split(const cpx (&v)[R], cpx (&u)[R / 2], cpx (&t)[R / 2]) {
    if constexpr (A < R / 2) {
      u[A] = cadd(v[A], v[A + R / 2]);
      t[A] = mul_root16<A * (16 / R), SIGN>(csub(v[A], v[A + R / 2]));
      split<A + 1>(v, u, t);
    }
  }
  static __device__ __forceinline__ void run(cpx (&v)[R]) {
    cpx u[R / 2], t[R / 2];
    split<0>(v, u, t);
    Dft<R / 2, SIGN>::run(u);
    Dft<R / 2, SIGN>::run(t);
#pragma unroll
    for (int c = 0; c < R / 2; ++c) {
      v[2 * c] = u[c];
      v[2 * c + 1] = t[c];
    }
  }
};
template <int SIGN>
struct Dft<1, SIGN> {
  static __device__ __forceinline__ void run(cpx (&)[1]) {}
};

#define MMF_TILE_LOG 12        // complex values per group tile (2^12 = 64 KiB of exchange buffer)
#define MMF_GROUP_THREADS 256  // 2^(MMF_TILE_LOG - 4)

__host__ __device__ __forceinline__ constexpr int swz(int f) { return f ^ ((f >> 4) & 7); }

// Split of a length-2^LOGN transform into NST = ceil(LOGN/4) digits, most significant first:
// digit i has LR = ceil(remaining / stages_left) bits.
__host__ __device__ constexpr int nstages(int logn) { return (logn + 3) / 4; }
__host__ __device__ constexpr int stage_lr(int remain, int nst) { return (remain + nst - 1) / nst; }
// digit widths of the last and the last-but-one stage
__host__ __device__ constexpr int last_lr(int remain, int nst) {
  return nst <= 1 ? remain : last_lr(remain - stage_lr(remain, nst), nst - 1);
}
__host__ __device__ constexpr int prev_lr(int remain, int nst) {
  return nst <= 1 ? 0 : nst == 2 ? stage_lr(remain, 2) : prev_lr(remain - stage_lr(remain, nst), nst - 1);
}

// Slot p (digits d1 d2 ... most significant first, radices r1 r2 ...) holds bin k = d1 + r1 d2 + r1 r2 d3 + ...
template <int REMAIN, int NST>
__host__ __device__ __forceinline__ constexpr int slot_to_bin(int p) {
  if constexpr (NST == 0) {
    return 0;
  } else {
    constexpr int LR = stage_lr(REMAIN, NST);
    constexpr int LM = REMAIN - LR;
    return (p >> LM) + (slot_to_bin<LM, NST - 1>(p & ((1 << LM) - 1)) << LR);
  }
}
template <int LOGN>
__host__ __device__ __forceinline__ constexpr int slot_to_bin(int p) {
  return slot_to_bin<LOGN, nstages(LOGN)>(p);
}

// ---- per-stage twiddle tables ---------------------------------------------------------------------------------------
// The stage that transforms an LR-bit digit with LOGM point-index bits below it multiplies output c of the
// butterfly at low index b by exp(+-2 pi i b c / 2^(LR+LOGM)).  Table of one stage: entry [(c-1) << LOGM | b],
// c = 1 .. 2^LR - 1, b < 2^LOGM (stages with LOGM = 0 have none).  Tables of all stages are concatenated, most
// significant digit first.  (The host fills them with the same recursion, mmf_api.cu.)
// COMPACT stages (radix 16 over 256 points below, the one big table: 61 KB): only c = 1, 2, 3 (rows 0-2) and
// c = 4, 8, 12 (rows 3-5) are stored and w^(b (4 c1 + c0)) = w^(4 b c1) w^(b c0) costs one more product for the nine
// mixed entries — 24 KB instead of 61 KB of shared memory, and 6 instead of 15 table reads per thread.
__host__ __device__ constexpr bool tw_compact(int lr, int logm) { return lr == 4 && logm == 8; }
__host__ __device__ constexpr int tw_stage_entries(int lr, int logm) {
  return logm > 0 ? ((tw_compact(lr, logm) ? 6 : ((1 << lr) - 1)) << logm) : 0;
}
__host__ __device__ constexpr int tw_total_entries(int remain, int nst) {
  return nst <= 0 ? 0
                  : tw_stage_entries(stage_lr(remain, nst), remain - stage_lr(remain, nst)) +
                        tw_total_entries(remain - stage_lr(remain, nst), nst - 1);
}
__host__ __device__ constexpr int tw_offset(int logp, int remain, int nst) {
  return tw_total_entries(logp, nstages(logp)) - tw_total_entries(remain, nst);
}

// ---- register layout of a stage -------------------------------------------------------------------------------------
// A tile is 2^LOGTOT values = [batch][point (LOGP bits)][column (LOGW bits)], flat index f.  In the stage whose digit
// sits at point bits [LOGM+LR-1 : LOGM], thread t owns f_j = base | (j << LO), j = 0..15, with
// LO = min(LOGM + LOGW, LOGTOT - 4) and base = t with four zero bits inserted at position LO.
__host__ __device__ constexpr int stage_lo(int logm, int logw, int logtot) {
  return (logm + logw < logtot - 4) ? (logm + logw) : (logtot - 4);
}
template <int LO>
__device__ __forceinline__ int stage_base(int t) {
  return ((t >> LO) << (LO + 4)) | (t & ((1 << LO) - 1));
}
template <int LO>
__device__ __forceinline__ void tile_lds(cpx (&v)[16], const cpx* __restrict__ s, int base) {
#pragma unroll
  for (int j = 0; j < 16; ++j) v[j] = s[swz(base | (j << LO))];
}
template <int LO>
__device__ __forceinline__ void tile_sts(const cpx (&v)[16], cpx* __restrict__ s, int base) {
#pragma unroll
  for (int j = 0; j < 16; ++j) s[swz(base | (j << LO))] = v[j];
}

__device__ __forceinline__ void group_barrier(int id, int nthreads) {
  asm volatile("bar.sync %0, %1;\n" ::"r"(id), "r"(nthreads) : "memory");
}
// Synchronisation of the exchange between two stage layouts LOA, LOB.  The thread index is the flat index f with the
// 4 register bits at [LO, LO+4) removed; when both register fields lie below bit 9, f[9:11] is thread bits [5:7] in
// both layouts, i.e. every value stays inside its warp and __syncwarp is enough — the warps of a group then drift
// apart between the group-wide exchanges, and one warp's shared-memory phase overlaps another's arithmetic.
template <int LOA, int LOB>
__device__ __forceinline__ void exchange_barrier(int id) {
  if constexpr (LOA <= 5 && LOB <= 5) __syncwarp();
  else group_barrier(id, MMF_GROUP_THREADS);
}

// x[c] *= w^(SIGN b c), c = 1 .. R-1, from this stage's table (full: row c-1; compact: see tw_compact)
template <int R, int LR, int LOGM, int SIGN>
__device__ __forceinline__ void stage_twiddle(cpx (&x)[R], const cpx* __restrict__ tab, int b) {
  if constexpr (tw_compact(LR, LOGM)) {
    cpx lo[4], hi[4];
#pragma unroll
    for (int i = 1; i < 4; ++i) {
      lo[i] = tab[((i - 1) << LOGM) | b];
      hi[i] = tab[((i + 2) << LOGM) | b];
    }
#pragma unroll
    for (int c = 1; c < R; ++c) {
      const int c0 = c & 3, c1 = c >> 2;
      const cpx w = c1 == 0 ? lo[c0] : c0 == 0 ? hi[c1] : cmul(hi[c1], lo[c0]);
      x[c] = cmul_s<SIGN>(x[c], w);
    }
  } else {
#pragma unroll
    for (int c = 1; c < R; ++c) x[c] = cmul_s<SIGN>(x[c], tab[((c - 1) << LOGM) | b]);
  }
}

// One stage on the 16 registers of a thread.
//   DIF:  x <- Dft(x) then x[c] *= w_L^(SIGN b c)        (L = 2^(LR+LOGM), b = point index mod 2^LOGM)
//   DIT:  x[c] *= w_L^(SIGN b c) then x <- Dft(x)        (the adjoint of the DIF stage of opposite SIGN)
// tab = this stage's twiddle table (see above), exp(+2 pi i b c / L).
template <int LOGTOT, int LOGW, int LOGM, int LR, int SIGN, bool DIF>
__device__ __forceinline__ void stage_math(cpx (&v)[16], int base, const cpx* __restrict__ tab) {
  constexpr int SH = LOGM + LOGW;
  constexpr int LO = stage_lo(LOGM, LOGW, LOGTOT);
  constexpr int R = 1 << LR;
  constexpr int DSH = SH - LO;
#pragma unroll
  for (int q = 0; q < 16 / R; ++q) {
    const int jq = ((q >> DSH) << (DSH + LR)) | (q & ((1 << DSH) - 1));
    cpx x[R];
#pragma unroll
    for (int a = 0; a < R; ++a) x[a] = v[jq | (a << DSH)];
    const int b = ((base | (jq << LO)) >> LOGW) & ((1 << LOGM) - 1);
    if constexpr (DIF) {
      Dft<R, SIGN>::run(x);
      if constexpr (LOGM > 0) stage_twiddle<R, LR, LOGM, SIGN>(x, tab, b);
    } else {
      if constexpr (LOGM > 0) stage_twiddle<R, LR, LOGM, SIGN>(x, tab, b);
      Dft<R, SIGN>::run(x);
    }
#pragma unroll
    for (int a = 0; a < R; ++a) v[jq | (a << DSH)] = x[a];
  }
}

// Forward chain (DIF, most significant digit first).  Entry: v in the layout of stage (REMAIN, NST) — for the first
// call REMAIN = LOGP, NST = nstages(LOGP), loaded by the caller from global memory.  Exit: v in the layout of the
// last stage (LOGM = 0), values in digit-reversed slot order.  s = this group's exchange buffer, tab = the
// concatenated tables of the LOGP-point transform, bar = the group's named-barrier id.
// FENCE: also synchronise after the last exchange read (needed when the caller's next use of the buffer does not
// start with the slots this thread read last, i.e. when the chain is not followed by its adjoint).
// PRESYNC: also synchronise before the FIRST exchange write (needed when the caller took v from the exchange buffer
// itself UNSWIZZLED — a tile staged there by TMA — so that nobody overwrites a value not yet read).  A WARP barrier is
// enough: thread t then read the slots base | j << LO and writes swz(base | j << LO), and the swizzle changes bits
// [2:0] of a slot only — lane or register bits, never warp bits — so the slots a thread overwrites were read by
// lanes of its own warp.
template <int LOGTOT, int LOGP, int LOGW, int REMAIN, int NST, int SIGN, bool FENCE, bool PRESYNC = false>
__device__ __forceinline__ void fft_dif(cpx (&v)[16], cpx* __restrict__ s, int t, const cpx* __restrict__ tab, int bar) {
  constexpr int LR = stage_lr(REMAIN, NST), LOGM = REMAIN - LR, LO = stage_lo(LOGM, LOGW, LOGTOT);
  const int base = stage_base<LO>(t);
  stage_math<LOGTOT, LOGW, LOGM, LR, SIGN, true>(v, base, tab + tw_offset(LOGP, REMAIN, NST));
  if constexpr (NST > 1) {
    constexpr int LR2 = stage_lr(LOGM, NST - 1), LO2 = stage_lo(LOGM - LR2, LOGW, LOGTOT);
    if constexpr (PRESYNC && REMAIN == LOGP) __syncwarp();
    tile_sts<LO>(v, s, base);
    exchange_barrier<LO, LO2>(bar);
    tile_lds<LO2>(v, s, stage_base<LO2>(t));
    if constexpr (FENCE && NST == 2) group_barrier(bar, MMF_GROUP_THREADS);
    fft_dif<LOGTOT, LOGP, LOGW, LOGM, NST - 1, SIGN, FENCE, PRESYNC>(v, s, t, tab, bar);
  }
}

// Inverse chain (DIT, least significant digit first): the adjoint of fft_dif with the opposite SIGN.  Entry: v in the
// layout of the last stage; exit: v in the layout of stage (REMAIN, NST) of the outermost call, natural order.
template <int LOGTOT, int LOGP, int LOGW, int REMAIN, int NST, int SIGN, bool FENCE, bool PRESYNC = false>
__device__ __forceinline__ void fft_dit(cpx (&v)[16], cpx* __restrict__ s, int t, const cpx* __restrict__ tab, int bar) {
  constexpr int LR = stage_lr(REMAIN, NST), LOGM = REMAIN - LR, LO = stage_lo(LOGM, LOGW, LOGTOT);
  const int base = stage_base<LO>(t);
  if constexpr (NST > 1) {
    constexpr int LR2 = stage_lr(LOGM, NST - 1), LO2 = stage_lo(LOGM - LR2, LOGW, LOGTOT);
    fft_dit<LOGTOT, LOGP, LOGW, LOGM, NST - 1, SIGN, false, PRESYNC>(v, s, t, tab, bar);
    if constexpr (PRESYNC && NST == 2) __syncwarp();
    tile_sts<LO2>(v, s, stage_base<LO2>(t));
    exchange_barrier<LO2, LO>(bar);
    tile_lds<LO>(v, s, base);
    if constexpr (FENCE) group_barrier(bar, MMF_GROUP_THREADS);
  }
  stage_math<LOGTOT, LOGW, LOGM, LR, SIGN, false>(v, base, tab + tw_offset(LOGP, REMAIN, NST));
}

}  // namespace mmf
