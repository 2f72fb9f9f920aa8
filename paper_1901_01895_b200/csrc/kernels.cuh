// kernels.cuh — the global kernels of the RK4IP hot path (sm_100a, fp64).
//
//   k_cols  passes A and C of the three-pass operator D = exp(h/2 L):  length-N1 transforms over the slow
//           (strided) index of a row viewed as an N1 x N2 matrix, plus the inter-pass twiddle W_N^(k1 n2).
//   k_rows  pass B: contiguous length-N2 transform -> multiply by the tabulated exp(h/2 L_a(w_k))/N ->
//           adjoint length-N2 transform, all inside one shared-memory residency.  For N <= 4096 this kernel
//           alone is D.
//   k_etab  fills the exp(h/2 L_a(w_k)) table in the slot order pass B consumes (double-double phase).
//   k_nl    the fused nonlinear kernel: mode powers, kappa contraction, nonlinear product and the RK4
//           stage combinations of Eq. (6b)-(6f) in one pass over a time tile of all 2M rows.
//
// Index algebra of D (forward sign +, reading R1 of DESIGN.md):  n = N2 n1 + n2,  k = k1 + N1 k2,
//   X[k1 + N1 k2] = sum_n2 W_N2^(k2 n2) [ W_N^(k1 n2) sum_n1 W_N1^(k1 n1) x[N2 n1 + n2] ]
// pass A does the inner sum and the twiddle, pass B the outer sum; the way back is the exact adjoint.
#pragma once
#include "fft_core.cuh"

namespace mmf {

// runtime version of slot_to_bin<LOGN> (same digit rule), used by table generation and the debug map
__host__ __device__ inline int slot_to_bin_rt(int logn, int p) {
  int remain = logn, nst = nstages(logn), k = 0, shift = 0;
  while (nst > 0) {
    const int lr = stage_lr(remain, nst), lm = remain - lr;
    k += (p >> lm) << shift;
    p &= (1 << lm) - 1;
    shift += lr;
    remain = lm;
    --nst;
  }
  return k;
}

// W_N^x = whi[x >> lb] * wlo[x & (2^lb - 1)]  (two small tables instead of one of N entries)
struct TwoLevelTw {
  const cpx* __restrict__ whi;
  const cpx* __restrict__ wlo;
  int lb;
  __device__ __forceinline__ cpx get(long long x) const {
    return cmul(whi[x >> lb], wlo[x & ((1LL << lb) - 1)]);
  }
};

// ---------------------------------------------------------------------------------------------------- pass A / C
// grid = (N2 / W, 2M, nbuf); block = 2^(LOGN1 + LOGW - 4).  DIR 0: pass A (DIF, sign +, then twiddle);
// DIR 1: pass C (conjugate twiddle, then DIT, sign -).
template <int LOGN1, int LOGW, int DIR>
__global__ void __launch_bounds__(1 << (LOGN1 + LOGW - 4))
k_cols(cpx* __restrict__ X0, cpx* __restrict__ X1, const cpx* __restrict__ tw1, TwoLevelTw tw, int logn2) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cpx* s = reinterpret_cast<cpx*>(smem_raw);
  constexpr int LOGTOT = LOGN1 + LOGW;
  constexpr int NT = 1 << (LOGTOT - 4);
  const int t = threadIdx.x;
  const int n2_0 = blockIdx.x << LOGW;
  const long long N = 1LL << (LOGN1 + logn2);
  cpx* base = (blockIdx.z ? X1 : X0) + (long long)blockIdx.y * N + n2_0;
#pragma unroll
  for (int j = 0; j < 16; ++j) {
    const int f = j * NT + t;
    const int pos = f >> LOGW, c = f & ((1 << LOGW) - 1);
    cpx v = base[((long long)pos << logn2) | c];
    if constexpr (DIR == 1) {
      const long long x = (long long)slot_to_bin<LOGN1>(pos) * (n2_0 + c);
      v = cmulc(v, tw.get(x));
    }
    s[swz(f)] = v;
  }
  __syncthreads();
  if constexpr (DIR == 0)
    smem_fft_dif<LOGTOT, LOGN1, LOGW, LOGN1, nstages(LOGN1), +1>(s, t, tw1);
  else
    smem_fft_dit<LOGTOT, LOGN1, LOGW, LOGN1, nstages(LOGN1), -1>(s, t, tw1);
#pragma unroll
  for (int j = 0; j < 16; ++j) {
    const int f = j * NT + t;
    const int pos = f >> LOGW, c = f & ((1 << LOGW) - 1);
    cpx v = s[swz(f)];
    if constexpr (DIR == 0) {
      const long long x = (long long)slot_to_bin<LOGN1>(pos) * (n2_0 + c);
      v = cmul(v, tw.get(x));
    }
    base[((long long)pos << logn2) | c] = v;
  }
}

// -------------------------------------------------------------------------------------------------------- pass B
// A "chunk" is one contiguous run of N2 values (memory row p1 of field row r: chunk = r * N1 + p1).
// grid = (ceil(nchunks / 2^LOGB), 1, nbuf); block = 2^(LOGN2 + LOGB - 4).  MODE 0: transform, * E, adjoint
// transform.  MODE 1: transform only (debug entry point).
template <int LOGN2, int LOGB, int MODE>
__global__ void __launch_bounds__(1 << (LOGN2 + LOGB - 4))
k_rows(cpx* __restrict__ X0, cpx* __restrict__ X1, const cpx* __restrict__ E, const cpx* __restrict__ tw2,
       long long nchunks, int logn1) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cpx* s = reinterpret_cast<cpx*>(smem_raw);
  constexpr int LOGTOT = LOGN2 + LOGB;
  constexpr int NT = 1 << (LOGTOT - 4);
  const int t = threadIdx.x;
  const long long chunk0 = (long long)blockIdx.x << LOGB;
  cpx* base = (blockIdx.z ? X1 : X0) + (chunk0 << LOGN2);
#pragma unroll
  for (int j = 0; j < 16; ++j) {
    const int f = j * NT + t;
    if (chunk0 + (f >> LOGN2) < nchunks) s[swz(f)] = base[f];
  }
  __syncthreads();
  smem_fft_dif<LOGTOT, LOGN2, 0, LOGN2, nstages(LOGN2), +1>(s, t, tw2);
  if constexpr (MODE == 0) {
#pragma unroll
    for (int j = 0; j < 16; ++j) {
      const int f = j * NT + t;
      const long long ch = chunk0 + (f >> LOGN2);
      if (ch < nchunks) {
        const long long mode = ch >> (logn1 + 1);
        const long long p1 = ch & ((1LL << logn1) - 1);
        const cpx e = E[(((mode << logn1) + p1) << LOGN2) + (f & ((1 << LOGN2) - 1))];
        s[swz(f)] = cmul(s[swz(f)], e);
      }
    }
    __syncthreads();
    smem_fft_dit<LOGTOT, LOGN2, 0, LOGN2, nstages(LOGN2), -1>(s, t, tw2);
  }
#pragma unroll
  for (int j = 0; j < 16; ++j) {
    const int f = j * NT + t;
    if (chunk0 + (f >> LOGN2) < nchunks) base[f] = s[swz(f)];
  }
}

// ------------------------------------------------------------------------------------- exp(h/2 L) table, slot order
// double-double helpers (error-free transformations; ~106-bit phase so that the reduced angle is exact to fp64)
struct dd {
  double hi, lo;
};
__host__ __device__ inline dd dd_quick(double a, double b) {
  const double s = a + b;
  return dd{s, b - (s - a)};
}
__host__ __device__ inline dd dd_two_sum(double a, double b) {
  const double s = a + b, bb = s - a;
  return dd{s, (a - (s - bb)) + (b - bb)};
}
__host__ __device__ inline dd dd_two_prod(double a, double b) {
  const double p = a * b;
  return dd{p, fma(a, b, -p)};
}
__host__ __device__ inline dd dd_add(dd a, dd b) {
  dd s = dd_two_sum(a.hi, b.hi);
  dd t = dd_two_sum(a.lo, b.lo);
  s.lo += t.hi;
  s = dd_quick(s.hi, s.lo);
  s.lo += t.lo;
  return dd_quick(s.hi, s.lo);
}
__host__ __device__ inline dd dd_mul(dd a, dd b) {
  dd p = dd_two_prod(a.hi, b.hi);
  p.lo += a.hi * b.lo + a.lo * b.hi;
  return dd_quick(p.hi, p.lo);
}
__host__ __device__ inline dd dd_mul_d(dd a, double b) {
  dd p = dd_two_prod(a.hi, b);
  p.lo += a.lo * b;
  return dd_quick(p.hi, p.lo);
}
__host__ __device__ inline dd dd_div_d(dd a, double b) {
  const double q1 = a.hi / b;
  dd r = dd_add(a, dd_mul_d(dd{-q1, 0.0}, b));
  const double q2 = r.hi / b;
  r = dd_add(r, dd_mul_d(dd{-q2, 0.0}, b));
  const double q3 = r.hi / b;
  dd q = dd_quick(q1, q2);
  return dd_add(q, dd{q3, 0.0});
}

#define MMF_MAXK 8
struct EtabParams {
  dd coef[MMF_MAXK];  // filled per mode on the device from cbase: hh * beta_n / n!
  dd wstep;           // 2 pi / (N dt)
  dd twopi;
  double amp;         // exp(-alpha hh / 2) / N
  int K, logn1, logn2;
};

// E[mode][slot] = amp * exp(i * sum_n coef_n(mode) * w_k^n),  k = bin held by slot (p1, q).
// coefs: device array [M][K] of dd.  grid = (N / 256, M), block = 256.
__global__ void k_etab(cpx* __restrict__ E, const dd* __restrict__ coefs, EtabParams P) {
  const long long N = 1LL << (P.logn1 + P.logn2);
  const long long slot = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (slot >= N) return;
  const int mode = blockIdx.y;
  const int p1 = (int)(slot >> P.logn2), q = (int)(slot & ((1LL << P.logn2) - 1));
  const long long k = (long long)slot_to_bin_rt(P.logn1, p1) + ((long long)slot_to_bin_rt(P.logn2, q) << P.logn1);
  const long long ks = (k < N / 2) ? k : k - N;  // Nyquist bin takes the negative frequency
  const dd w = dd_mul_d(P.wstep, (double)ks);
  const dd* c = coefs + (long long)mode * P.K;
  dd ph = c[P.K - 1];
  for (int n = P.K - 2; n >= 0; --n) ph = dd_add(dd_mul(ph, w), c[n]);
  // reduce modulo 2 pi in double-double, then first-order correction for the low word
  const double nrev = rint(ph.hi / P.twopi.hi);
  dd r = dd_add(ph, dd_mul_d(P.twopi, -nrev));
  double sn, cs;
  sincos(r.hi, &sn, &cs);
  const double sr = fma(cs, r.lo, sn), cr = fma(-sn, r.lo, cs);
  E[(long long)mode * N + slot] = make_double2(P.amp * cr, P.amp * sr);
}

// slot -> bin map for the debug entry point.  grid = N/256
__global__ void k_slot_map(long long* __restrict__ idx, int logn1, int logn2) {
  const long long N = 1LL << (logn1 + logn2);
  const long long slot = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (slot >= N) return;
  const int p1 = (int)(slot >> logn2), q = (int)(slot & ((1LL << logn2) - 1));
  idx[slot] = (long long)slot_to_bin_rt(logn1, p1) + ((long long)slot_to_bin_rt(logn2, q) << logn1);
}

// SPEC[r][bin(slot)] = X[r][slot]   (debug: natural-order spectrum).  grid = (N/256, 2M)
__global__ void k_unpermute(const cpx* __restrict__ X, cpx* __restrict__ SPEC, int logn1, int logn2) {
  const long long N = 1LL << (logn1 + logn2);
  const long long slot = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (slot >= N) return;
  const int p1 = (int)(slot >> logn2), q = (int)(slot & ((1LL << logn2) - 1));
  const long long k = (long long)slot_to_bin_rt(logn1, p1) + ((long long)slot_to_bin_rt(logn2, q) << logn1);
  SPEC[(long long)blockIdx.y * N + k] = X[(long long)blockIdx.y * N + slot];
}

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
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double* P1 = reinterpret_cast<double*>(smem_raw);
  double* P2 = P1 + (size_t)p.M * MMF_NL_T;
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
          const cpx an = make_double2(fma(sixth, k.x, z.x), fma(sixth, k.y, z.y));
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
