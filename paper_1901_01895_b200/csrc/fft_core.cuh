// fft_core.cuh — register-level and shared-memory FFT building blocks (fp64 complex), sm_100a.
//
// Role in the path: rows a1/a3 of the hot-path table (forward / inverse transform of every field, PAPER.md:107
// "fast Fourier transforms ... rows are aligned linear in the memory"; Eq. 6 PAPER.md:75-88 needs exp(h/2 L)
// four times per step).  Design:
//   * every thread owns 16 complex values (64 registers) and performs radix-2..16 butterflies on them;
//   * a tile of 2^LOGTOT complex values lives in shared memory; one "stage" reads 16 values per thread,
//     transforms one digit of the index and writes them back IN PLACE (decimation in frequency on the way to
//     the spectrum, the exact adjoint — decimation in time — on the way back), so no bit-reversal pass exists:
//     the spectrum simply stays in digit-reversed slot order and the exp(h/2 L) table is stored in that order;
//   * the 16 values a thread touches always span 4 contiguous index bits and the tile is XOR-swizzled
//     (slot ^ ((slot >> 4) & 7)) which makes every stage's LDS.128/STS.128 pattern bank-conflict free.
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

__device__ __forceinline__ int swz(int f) { return f ^ ((f >> 4) & 7); }

// Split of a length-2^LOGN transform into NST = ceil(LOGN/4) digits, most significant first:
// digit i has LR = ceil(remaining / stages_left) bits.
__host__ __device__ constexpr int nstages(int logn) { return (logn + 3) / 4; }
__host__ __device__ constexpr int stage_lr(int remain, int nst) { return (remain + nst - 1) / nst; }

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

// One in-place stage on a shared-memory tile of 2^LOGTOT values = 2^(LOGTOT-LOGW) transform points x 2^LOGW
// interleaved columns.  Transforms the LR-bit digit sitting at point-index bits [LOGM+LR-1 : LOGM].
//   DIF:  v <- Dft(v) then v[c] *= w_L^(SIGN b c)        (L = 2^(LR+LOGM), b = point index mod 2^LOGM)
//   DIT:  v[c] *= w_L^(SIGN b c) then v <- Dft(v)        (the adjoint of the DIF stage of opposite SIGN)
// tw[] holds exp(+2 pi i j / 2^LOGN) for j < 2^LOGN (LOGN = transform length; tile bits above LOGN + LOGW are a
// batch index).  t = thread index in [0, 2^(LOGTOT-4)).
template <int LOGTOT, int LOGN, int LOGW, int LOGM, int LR, int SIGN, bool DIF>
__device__ __forceinline__ void smem_stage(cpx* __restrict__ s, int t, const cpx* __restrict__ tw) {
  constexpr int SH = LOGM + LOGW;
  constexpr int LO = (SH < LOGTOT - 4) ? SH : (LOGTOT - 4);
  constexpr int R = 1 << LR;
  constexpr int DSH = SH - LO;
  constexpr int TWSH = LOGN - LR - LOGM;
  const int base = ((t >> LO) << (LO + 4)) | (t & ((1 << LO) - 1));
  cpx v[16];
#pragma unroll
  for (int j = 0; j < 16; ++j) v[j] = s[swz(base | (j << LO))];
#pragma unroll
  for (int q = 0; q < 16 / R; ++q) {
    const int jq = ((q >> DSH) << (DSH + LR)) | (q & ((1 << DSH) - 1));
    cpx x[R];
#pragma unroll
    for (int a = 0; a < R; ++a) x[a] = v[jq | (a << DSH)];
    const int b = ((base | (jq << LO)) >> LOGW) & ((1 << LOGM) - 1);
    if constexpr (DIF) {
      Dft<R, SIGN>::run(x);
      if constexpr (LOGM > 0) {
#pragma unroll
        for (int c = 1; c < R; ++c) x[c] = cmul_s<SIGN>(x[c], tw[(b * c) << TWSH]);
      }
    } else {
      if constexpr (LOGM > 0) {
#pragma unroll
        for (int c = 1; c < R; ++c) x[c] = cmul_s<SIGN>(x[c], tw[(b * c) << TWSH]);
      }
      Dft<R, SIGN>::run(x);
    }
#pragma unroll
    for (int a = 0; a < R; ++a) v[jq | (a << DSH)] = x[a];
  }
#pragma unroll
  for (int j = 0; j < 16; ++j) s[swz(base | (j << LO))] = v[j];
}

// All stages, most significant digit first (DIF, natural order in -> digit-reversed slots out) ...
template <int LOGTOT, int LOGN, int LOGW, int REMAIN, int NST, int SIGN>
__device__ __forceinline__ void smem_fft_dif(cpx* s, int t, const cpx* __restrict__ tw) {
  if constexpr (NST > 0) {
    constexpr int LR = stage_lr(REMAIN, NST);
    smem_stage<LOGTOT, LOGN, LOGW, REMAIN - LR, LR, SIGN, true>(s, t, tw);
    __syncthreads();
    smem_fft_dif<LOGTOT, LOGN, LOGW, REMAIN - LR, NST - 1, SIGN>(s, t, tw);
  }
}
// ... and least significant digit first (DIT, digit-reversed slots in -> natural order out).
template <int LOGTOT, int LOGN, int LOGW, int REMAIN, int NST, int SIGN>
__device__ __forceinline__ void smem_fft_dit(cpx* s, int t, const cpx* __restrict__ tw) {
  if constexpr (NST > 0) {
    constexpr int LR = stage_lr(REMAIN, NST);
    smem_fft_dit<LOGTOT, LOGN, LOGW, REMAIN - LR, NST - 1, SIGN>(s, t, tw);
    smem_stage<LOGTOT, LOGN, LOGW, REMAIN - LR, LR, SIGN, false>(s, t, tw);
    __syncthreads();
  }
}

}  // namespace mmf
