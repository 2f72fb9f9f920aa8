// rk4ip_oracle.cpp — CPU ORACLE. TEST INFRASTRUCTURE ONLY.
//
// A plain, slow, obviously-correct fp64 implementation of the RK4IP step for the multimode
// Manakov/NLSE, written from the paper (arXiv 1901.01895; citations are PAPER.md:<line>).
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// build, load or call this file.  It shares no code, header, table generator or helper with the
// CUDA path under paper_1901_01895_b200/csrc/, and nothing in the product imports it.
//
// What is computed (every function cites the passage it follows):
//   Eq. (1)  PAPER.md:35-37   dA_a/dz = L A_a + i*gamma*(sum_b kappa_ab |A_b|^2) A_a,
//                             L = -alpha/2 + i*sum_n (i^n/n!) beta_{n,a} d^n/dt^n
//   Eq. (6)  PAPER.md:75-88   the RK4IP step (6a)-(6f) with separation distance z' = z + h/2
//   layout   PAPER.md:95,107  2M x N complex matrix, row-major, one row per spatial/polarisation mode
//
// Readings taken where the paper is silent or garbled:
//   R1  Fourier sign: the time-domain operator of Eq. (1) is the authority.  With
//       A(t) = sum_w At(w) exp(-i w t) one gets dAt/dz = (-alpha/2 + i sum_n beta_n w^n/n!) At,
//       so "to frequency" is X_k = sum_n x_n exp(+2 pi i k n/N) and back carries exp(-...)/N.
//   R2  sum_{n=0} runs over the K coefficients the caller supplies (n = 0..K-1).
//   R3  Eq. (6b): k1 = exp(h/2 L)[ h N(A) A ]  (operator applied to the product).
//   R4  Eq. (6e): k4 = h N(u4) u4 with u4 = exp(h/2 L)[A_I + k3].
//   R5  |A_b|^2 of a Jones vector = |A_bx|^2 + |A_by|^2; rows 2a, 2a+1 are the x, y polarisations of mode a.
//   R7  the Nyquist bin k = N/2 takes the negative frequency.
//
// Pins (tests/test_oracle_pins.py, -m "not gpu"): direct-DFT and library-FFT agreement, tone eigenvalue
// exp(h L(W)), circular delay for beta_1, exact nonlinear phase rotation, energy decay exp(-alpha z),
// soliton shape, 4th-order convergence against an independent adaptive integrator, integer exactness,
// composition.  No function here is "parity unpinned".
//
// Noise loading (section 6: "White noise is added to the signals before the receiver, setting the optical
// signal-to-noise ratio (OSNR) to 20 dB"; reading R18 in DESIGN.md): philox4x32_10 (the counter-based generator of
// Salmon, Moraes, Dror, Shaw, "Parallel random numbers: as easy as 1, 2, 3", SC'11, written from its definition),
// gaussian_pair (Box-Muller) and add_noise.  Pins (tests/test_oracle_noise_pins.py): the generator's published
// known-answer vectors bit for bit, uniform-to-unit-interval mapping limits, mean / variance / whiteness / normality of
// the added field within stated statistical bounds, the realised OSNR of a known-power field, the zero-noise limit,
// stream independence of the matrix size.
//
// Numerical hygiene: twiddles and the dispersion phase are evaluated per index in long double
// (never by recurrence); no -ffast-math.

#include <cmath>
#include <complex>
#include <cstdint>
#include <cstring>
#include <thread>
#include <vector>

namespace {

typedef std::complex<double> cplx;
const long double PI_L = 3.141592653589793238462643383279502884L;

bool is_pow2(long long n) { return n >= 1 && (n & (n - 1)) == 0; }

// run f(i) for i in [0, count) on up to nthreads std::threads (contiguous blocks; items are independent)
template <class F>
void parallel_for(long long count, int nthreads, F f) {
  if (nthreads < 1) nthreads = 1;
  if (nthreads == 1 || count < 2) {
    for (long long i = 0; i < count; ++i) f(i);
    return;
  }
  if ((long long)nthreads > count) nthreads = (int)count;
  std::vector<std::thread> pool;
  for (int w = 0; w < nthreads; ++w) {
    long long lo = count * w / nthreads, hi = count * (w + 1) / nthreads;
    pool.emplace_back([lo, hi, &f]() { for (long long i = lo; i < hi; ++i) f(i); });
  }
  for (auto& t : pool) t.join();
}

// exp(sign * 2 pi i p / N) for 0 <= p < N, in long double.  The angle is folded into the first octant with exact
// integer arithmetic before sinl/cosl are called, so multiples of a quarter turn give exactly 0 and +-1 and the
// table has the symmetries of the unit circle.
void unit_root(long long p, long long N, int sign, long double* c, long double* s) {
  long long q = 8 * p;            // position in eighths of a turn, scaled by N
  int oct = (int)(q / N);         // octant 0..7
  long long rem = q - (long long)oct * N;   // 0 <= rem < N, angle inside the octant = (rem/N) * (pi/4)
  long double a;                  // folded angle in [0, pi/4]
  if (oct & 1) a = (PI_L / 4.0L) * ((long double)(N - rem) / (long double)N);
  else         a = (PI_L / 4.0L) * ((long double)rem / (long double)N);
  long double ca = cosl(a), sa = sinl(a);
  if (rem == 0 && !(oct & 1)) { ca = 1.0L; sa = 0.0L; }
  long double cc, ss;
  switch (oct) {
    case 0: cc = ca;  ss = sa;  break;
    case 1: cc = sa;  ss = ca;  break;
    case 2: cc = -sa; ss = ca;  break;
    case 3: cc = -ca; ss = sa;  break;
    case 4: cc = -ca; ss = -sa; break;
    case 5: cc = -sa; ss = -ca; break;
    case 6: cc = sa;  ss = -ca; break;
    default: cc = ca; ss = -sa; break;
  }
  *c = cc;
  *s = (sign >= 0) ? ss : -ss;
}

// The plain definition of the discrete Fourier sum, O(N^2):  out_k = sum_n in_n exp(sign * 2 pi i k n / N).
// (Definition of the DFT; sign = +1 is "to frequency" under reading R1.)
void dft_direct(const cplx* in, cplx* out, long long N, int sign) {
  for (long long k = 0; k < N; ++k) {
    long double sr = 0.0L, si = 0.0L;
    for (long long n = 0; n < N; ++n) {
      long long p = (k * n) % N;  // exact integer phase index
      long double c, s;
      unit_root(p, N, sign, &c, &s);
      sr += (long double)in[n].real() * c - (long double)in[n].imag() * s;
      si += (long double)in[n].real() * s + (long double)in[n].imag() * c;
    }
    out[k] = cplx((double)sr, (double)si);
  }
}

// Textbook iterative radix-2 decimation-in-time FFT (bit reversal, then log2 N butterfly stages),
// unnormalised, same sum as dft_direct.  Twiddle j is exp(sign * 2 pi i j / N) from sinl/cosl.
void fft_radix2(cplx* x, long long N, int sign) {
  if (N < 2) return;
  int lg = 0;
  while ((1LL << lg) < N) ++lg;
  for (long long i = 0; i < N; ++i) {
    long long r = 0;
    for (int b = 0; b < lg; ++b) if (i & (1LL << b)) r |= 1LL << (lg - 1 - b);
    if (r > i) std::swap(x[i], x[r]);
  }
  std::vector<cplx> w(N / 2);
  for (long long j = 0; j < N / 2; ++j) {
    long double c, s;
    unit_root(j, N, sign, &c, &s);
    w[j] = cplx((double)c, (double)s);
  }
  for (long long len = 2; len <= N; len <<= 1) {
    long long half = len / 2, step = N / len;
    for (long long base = 0; base < N; base += len) {
      for (long long j = 0; j < half; ++j) {
        cplx t = w[j * step] * x[base + j + half];
        cplx u = x[base + j];
        x[base + j] = u + t;
        x[base + j + half] = u - t;
      }
    }
  }
}

// Angular frequency of bin k (reading R7): w_k = 2 pi k'/(N dt), k' = k for k < N/2, else k - N.
long double omega_of_bin(long long k, long long N, double dt) {
  long long ks = (k < N / 2) ? k : k - N;
  return 2.0L * PI_L * (long double)ks / ((long double)N * (long double)dt);
}

// exp(hh * L_a(w_k)) with L_a(w) = -alpha/2 + i * sum_{n=0}^{K-1} beta_{n,a} w^n / n!   (Eq. 1; R1, R2)
// hh is the distance the factor advances (h/2 inside a step).  Long double throughout, rounded once.
cplx linear_factor(long double w, double hh, double alpha, const double* beta_a, int K) {
  long double phase = 0.0L, wn = 1.0L, fact = 1.0L;
  for (int n = 0; n < K; ++n) {
    if (n > 0) { wn *= w; fact *= (long double)n; }
    phase += (long double)beta_a[n] * wn / fact;
  }
  phase *= (long double)hh;
  long double amp = expl(-(long double)alpha * (long double)hh / 2.0L);
  return cplx((double)(amp * cosl(phase)), (double)(amp * sinl(phase)));
}

// E[a][k] for all modes and bins.
void linear_table(cplx* E, int M, long long N, double dt, double hh, double alpha, const double* beta, int K,
                  int nthreads) {
  parallel_for((long long)M, nthreads, [&](long long a) {
    for (long long k = 0; k < N; ++k)
      E[a * N + k] = linear_factor(omega_of_bin(k, N, dt), hh, alpha, beta + a * K, K);
  });
}

// D(x) = exp(hh L) x for every row: to frequency (sign +), multiply by E_a[k], back (sign -) and 1/N.
// Row r belongs to mode a = r/2 (R5).  (Eq. 6a "exp(h/2 L) . A"; linear step per row)
void apply_D(cplx* x, int M, long long N, const cplx* E, int nthreads) {
  parallel_for(2LL * M, nthreads, [&](long long r) {
    cplx* row = x + r * N;
    const cplx* Ea = E + (r / 2) * N;
    fft_radix2(row, N, +1);
    for (long long k = 0; k < N; ++k) row[k] *= Ea[k];
    fft_radix2(row, N, -1);
    double inv = 1.0 / (double)N;
    for (long long k = 0; k < N; ++k) row[k] *= inv;
  });
}

// out_{a,p}[t] = (i * hgamma * S_a[t]) * u_{a,p}[t],  S_a[t] = sum_b kappa_ab P_b[t],  P_b = |u_bx|^2 + |u_by|^2
// (Eq. 1 nonlinear part; h N(u) u of Eq. 6b-e with hgamma = h*gamma).  b ascending, plain loops.
void nonlinear(const cplx* u, cplx* out, int M, long long N, double hgamma, const double* kappa, int nthreads) {
  const long long BLK = 4096;
  long long nblk = (N + BLK - 1) / BLK;
  parallel_for(nblk, nthreads, [&](long long blk) {
    std::vector<double> P(M);
    long long t0 = blk * BLK, t1 = std::min(N, t0 + BLK);
    for (long long t = t0; t < t1; ++t) {
      for (int b = 0; b < M; ++b) {
        cplx ux = u[(2LL * b) * N + t], uy = u[(2LL * b + 1) * N + t];
        P[b] = (ux.real() * ux.real() + ux.imag() * ux.imag()) + (uy.real() * uy.real() + uy.imag() * uy.imag());
      }
      for (int a = 0; a < M; ++a) {
        double S = 0.0;
        for (int b = 0; b < M; ++b) S += kappa[(long long)a * M + b] * P[b];
        double g = hgamma * S;
        for (int p = 0; p < 2; ++p) {
          cplx v = u[(2LL * a + p) * N + t];
          out[(2LL * a + p) * N + t] = cplx(-g * v.imag(), g * v.real());  // (i g) * v
        }
      }
    }
  });
}

// The paper's own data structure (Fig. 2): one coupling coefficient per PAIR OF POLARISATION MODES,
// "a matrix of 2M x 2M elements".  Row r = 2a + p of the field is polarisation mode r:
//   out_r[t] = (i * hgamma * S_r[t]) * u_r[t],   S_r[t] = sum_{s=0}^{2M-1} kappa2[r][s] |u_s[t]|^2      (s ascending)
// The Manakov form of nonlinear() is the special case kappa2[2a+p][2b+q] = kappa_ab.
void nonlinear_general(const cplx* u, cplx* out, int M, long long N, double hgamma, const double* kappa2, int nthreads) {
  const long long BLK = 4096;
  const int R = 2 * M;
  long long nblk = (N + BLK - 1) / BLK;
  parallel_for(nblk, nthreads, [&](long long blk) {
    std::vector<double> P(R);
    long long t0 = blk * BLK, t1 = std::min(N, t0 + BLK);
    for (long long t = t0; t < t1; ++t) {
      for (int s = 0; s < R; ++s) {
        cplx v = u[(long long)s * N + t];
        P[s] = v.real() * v.real() + v.imag() * v.imag();
      }
      for (int r = 0; r < R; ++r) {
        double S = 0.0;
        for (int s = 0; s < R; ++s) S += kappa2[(long long)r * R + s] * P[s];
        double g = hgamma * S;
        cplx v = u[(long long)r * N + t];
        out[(long long)r * N + t] = cplx(-g * v.imag(), g * v.real());  // (i g) * v
      }
    }
  });
}

// N of Eq. (1) in either form: kappa is [M][M] (Manakov, general = false) or [2M][2M] (general = true)
void apply_N(const cplx* u, cplx* out, int M, long long N, double hgamma, const double* kappa, bool general,
             int nthreads) {
  if (general) nonlinear_general(u, out, M, N, hgamma, kappa, nthreads);
  else nonlinear(u, out, M, N, hgamma, kappa, nthreads);
}

// One RK4IP step, Eq. (6a)-(6f) in the paper's order and notation (R3, R4).
// E is the table for hh = h/2.  Seven full-size buffers, nothing fused or reordered.
void rk4ip_step(cplx* A, int M, long long N, const cplx* E, double hgamma, const double* kappa, bool general,
                int nthreads, cplx* AI, cplx* k1, cplx* k2, cplx* k3, cplx* k4, cplx* tmp) {
  const long long tot = 2LL * M * N;
  // (6a) A_I = exp(h/2 L) A
  std::memcpy((void*)AI, (const void*)A, sizeof(cplx) * tot);
  apply_D(AI, M, N, E, nthreads);
  // (6b) k1 = exp(h/2 L) [ h N(A) A ]
  apply_N(A, k1, M, N, hgamma, kappa, general, nthreads);
  apply_D(k1, M, N, E, nthreads);
  // (6c) k2 = h N(A_I + k1/2) [A_I + k1/2]
  for (long long i = 0; i < tot; ++i) tmp[i] = AI[i] + k1[i] / 2.0;
  apply_N(tmp, k2, M, N, hgamma, kappa, general, nthreads);
  // (6d) k3 = h N(A_I + k2/2) [A_I + k2/2]
  for (long long i = 0; i < tot; ++i) tmp[i] = AI[i] + k2[i] / 2.0;
  apply_N(tmp, k3, M, N, hgamma, kappa, general, nthreads);
  // (6e) k4 = h N( exp(h/2 L)[A_I + k3] ) exp(h/2 L)[A_I + k3]
  for (long long i = 0; i < tot; ++i) tmp[i] = AI[i] + k3[i];
  apply_D(tmp, M, N, E, nthreads);
  apply_N(tmp, k4, M, N, hgamma, kappa, general, nthreads);
  // (6f) A(z+h) = exp(h/2 L)[A_I + k1/6 + k2/3 + k3/3] + k4/6
  for (long long i = 0; i < tot; ++i) tmp[i] = AI[i] + k1[i] / 6.0 + k2[i] / 3.0 + k3[i] / 3.0;
  apply_D(tmp, M, N, E, nthreads);
  for (long long i = 0; i < tot; ++i) A[i] = tmp[i] + k4[i] / 6.0;
}

// One symmetric split step with a Runge-Kutta nonlinear substep ("SSFM-RK4": Eq. 4 PAPER.md:58-61 with the nonlinear
// part "solved ... with explicit schemes like the Runge-Kutta method"), written out in that order:
//   A <- exp(h/2 L) A;   A <- classical RK4 over h of dA/dz = N(A) A (Eq. 1 without its linear part);   A <- exp(h/2 L) A
// E is the table for hh = h/2; hgamma = h*gamma, so nonlinear() returns h N(u) u.  Plain buffers, nothing fused.
void ssfm_rk4_step(cplx* A, int M, long long N, const cplx* E, double hgamma, const double* kappa, int nthreads,
                   cplx* k1, cplx* k2, cplx* k3, cplx* k4, cplx* tmp) {
  const long long tot = 2LL * M * N;
  apply_D(A, M, N, E, nthreads);
  nonlinear(A, k1, M, N, hgamma, kappa, nthreads);
  for (long long i = 0; i < tot; ++i) tmp[i] = A[i] + k1[i] / 2.0;
  nonlinear(tmp, k2, M, N, hgamma, kappa, nthreads);
  for (long long i = 0; i < tot; ++i) tmp[i] = A[i] + k2[i] / 2.0;
  nonlinear(tmp, k3, M, N, hgamma, kappa, nthreads);
  for (long long i = 0; i < tot; ++i) tmp[i] = A[i] + k3[i];
  nonlinear(tmp, k4, M, N, hgamma, kappa, nthreads);
  for (long long i = 0; i < tot; ++i) A[i] = A[i] + k1[i] / 6.0 + k2[i] / 3.0 + k3[i] / 3.0 + k4[i] / 6.0;
  apply_D(A, M, N, E, nthreads);
}

// S_a[t] = sum_b kappa_ab P_b[t],  P_b = |u_bx|^2 + |u_by|^2  (the real factor of N = i gamma S, Eq. 1)
// for every mode a and sample t; S is [M][N] doubles.  Same plain loops and summation order as nonlinear().
void mode_phase_rate(const cplx* u, double* S, int M, long long N, const double* kappa, int nthreads) {
  const long long BLK = 4096;
  long long nblk = (N + BLK - 1) / BLK;
  parallel_for(nblk, nthreads, [&](long long blk) {
    std::vector<double> P(M);
    long long t0 = blk * BLK, t1 = std::min(N, t0 + BLK);
    for (long long t = t0; t < t1; ++t) {
      for (int b = 0; b < M; ++b) {
        cplx ux = u[(2LL * b) * N + t], uy = u[(2LL * b + 1) * N + t];
        P[b] = (ux.real() * ux.real() + ux.imag() * ux.imag()) + (uy.real() * uy.real() + uy.imag() * uy.imag());
      }
      for (int a = 0; a < M; ++a) {
        double acc = 0.0;
        for (int b = 0; b < M; ++b) acc += kappa[(long long)a * M + b] * P[b];
        S[(long long)a * N + t] = acc;
      }
    }
  });
}

// One symmetric split step with the ITERATIVE nonlinear part ("SSFM-Agrawal": Eq. 4, "solved by an
// iterative approach as described in [6]" PAPER.md:63; "requires the computation of |A|^2 once at the position z for
// the first iteration and at the position z + h for every following iteration" PAPER.md:111).  Reading R14:
// the integral of Eq. (4) by the trapezoidal rule, int_z^{z+h} N(z') dz' ~ (h/2) [N(z) + N(z+h)] with N = i gamma S
// (a multiplication in the time domain); N(z+h) is not known, so
//   iteration 1:      N(z+h) := N(z)                        A_1 = D( exp(i h gamma S(A(z)))                  D A(z) )
//   iteration j >= 2: N(z+h) from A_{j-1}                   A_j = D( exp(i (h gamma / 2) [S(A(z)) + S(A_{j-1})]) D A(z) )
// and A(z+h) = A_niter.  D = exp(h/2 L), E its table (hh = h/2).  S0, S1 are [M][N] doubles, B and Y full fields.
void ssfm_agrawal_step(cplx* A, int M, long long N, const cplx* E, double hgamma, const double* kappa, int niter,
                       int nthreads, cplx* B, cplx* Y, double* S0, double* S1) {
  const long long tot = 2LL * M * N;
  mode_phase_rate(A, S0, M, N, kappa, nthreads);            // |A|^2 "once at the position z"
  std::memcpy((void*)B, (const void*)A, sizeof(cplx) * tot);
  apply_D(B, M, N, E, nthreads);                            // exp(h/2 L) A(z)
  for (int it = 1; it <= niter; ++it) {
    if (it > 1) mode_phase_rate(Y, S1, M, N, kappa, nthreads);   // |A|^2 "at the position z + h"
    for (long long r = 0; r < 2LL * M; ++r) {
      const double *s0 = S0 + (r / 2) * N, *s1 = S1 + (r / 2) * N;
      for (long long t = 0; t < N; ++t) {
        const double theta = (it == 1) ? hgamma * s0[t] : 0.5 * hgamma * (s0[t] + s1[t]);
        Y[r * N + t] = B[r * N + t] * cplx(std::cos(theta), std::sin(theta));
      }
    }
    apply_D(Y, M, N, E, nthreads);                          // exp(h/2 L)
  }
  std::memcpy((void*)A, (const void*)Y, sizeof(cplx) * tot);
}


// ------------------------------------------------------------------------------------------------ noise loading
// Philox-4x32 with 10 rounds (Salmon et al., SC'11, section 3.3 / Table 2): the state is four 32-bit words c0..c3, the
// key two words k0, k1.  One round: (hi0, lo0) = M0 * c0, (hi1, lo1) = M1 * c2 (32 x 32 -> 64-bit products), then
//   c0' = hi1 ^ c1 ^ k0,  c1' = lo1,  c2' = hi0 ^ c3 ^ k1,  c3' = lo0;
// between rounds the key is bumped by the Weyl constants W0 (golden ratio), W1 (sqrt(3) - 1).
void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  const uint64_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
  const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    if (round > 0) {
      k0 += W0;
      k1 += W1;
    }
    const uint64_t p0 = M0 * c0, p1 = M1 * c2;
    const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0, hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    const uint32_t n0 = hi1 ^ c1 ^ k0, n1 = lo1, n2 = hi0 ^ c3 ^ k1, n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// Two 32-bit words -> a double in the OPEN interval (0, 1): the top 52 bits k of (hi : lo), u = (k + 1/2) 2^-52.
// Every value is exactly representable (k + 1/2 has at most 53 significant bits); smallest 2^-53, largest 1 - 2^-53.
double unit_open(uint32_t hi, uint32_t lo) {
  const uint64_t k = ((uint64_t)hi << 20) | (uint64_t)(lo >> 12);
  return ((double)k + 0.5) * 0x1p-52;
}

// The complex standard normal sample (E|z|^2 = 1, real and imaginary part independent N(0, 1/2)) of row r, sample t
// under `seed`: counter = (t low word, t high word, r, 0), key = (seed low word, seed high word); Box-Muller on
// u1 = unit_open(w0, w1), u2 = unit_open(w2, w3):  z = sqrt(-ln u1) (cos 2 pi u2 + i sin 2 pi u2).
cplx noise_unit_sample(uint64_t seed, uint32_t row, uint64_t t) {
  const uint32_t ctr[4] = {(uint32_t)t, (uint32_t)(t >> 32), row, 0u};
  const uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
  uint32_t w[4];
  philox4x32_10(ctr, key, w);
  const double u1 = unit_open(w[0], w[1]), u2 = unit_open(w[2], w[3]);
  const double rad = std::sqrt(-std::log(u1));
  const long double ang = 6.283185307179586476925286766559005768L * (long double)u2;
  return cplx(rad * (double)cosl(ang), rad * (double)sinl(ang));
}

// PAPER.md:255 with reading R18.  For every spatial mode a:
//   P_a     = (1/N) sum_t (|A_ax(t)|^2 + |A_ay(t)|^2)          mean signal power of the mode, both polarisations [W]
//   P_ch    = P_a / nch                                         per wavelength channel (nch channels share the mode)
//   N0      = P_ch / (2 B_ref OSNR)                             noise power spectral density PER POLARISATION: the OSNR
//                                                               counts the noise of both polarisations in B_ref
//   sigma^2 = N0 / dt                                           variance of one complex sample of one polarisation: white
//                                                               over the whole simulated band 1/dt
//   A_{a,p}(t) += sigma_a z_{2a+p}(t),  z = noise_unit_sample.
// power_out[a] = P_a (of the field BEFORE the noise).  OSNR = 10^(osnr_db/10); osnr_db = +inf adds nothing.
void add_noise(cplx* A, int M, long long N, double dt, double osnr_db, double ref_bw, int nch, uint64_t seed,
               double* power_out) {
  const double osnr = std::pow(10.0, osnr_db / 10.0);
  for (int a = 0; a < M; ++a) {
    double sum = 0.0;
    for (int p = 0; p < 2; ++p)
      for (long long t = 0; t < N; ++t) sum += std::norm(A[(size_t)(2 * a + p) * N + t]);
    const double P = sum / (double)N;
    power_out[a] = P;
    const double sigma = std::sqrt(P / (double)nch / (2.0 * ref_bw * osnr) / dt);
    if (!(sigma > 0.0)) continue;
    for (int p = 0; p < 2; ++p)
      for (long long t = 0; t < N; ++t)
        A[(size_t)(2 * a + p) * N + t] += sigma * noise_unit_sample(seed, (uint32_t)(2 * a + p), (uint64_t)t);
  }
}

}  // namespace

extern "C" {

// All complex arrays are interleaved (re, im) doubles.  Return 0 on success, -1 on bad arguments.

int orc_dft(const double* in, double* out, long long N, int sign) {
  if (!in || !out || N < 1 || (sign != 1 && sign != -1)) return -1;
  dft_direct((const cplx*)in, (cplx*)out, N, sign);
  return 0;
}

int orc_fft(double* x, long long N, int sign) {
  if (!x || !is_pow2(N) || (sign != 1 && sign != -1)) return -1;
  fft_radix2((cplx*)x, N, sign);
  return 0;
}

int orc_omega(double* w, long long N, double dt) {
  if (!w || N < 1 || !(dt > 0)) return -1;
  for (long long k = 0; k < N; ++k) w[k] = (double)omega_of_bin(k, N, dt);
  return 0;
}

// E[M][N] complex: exp(hh * L_a(w_k)); beta is [M][K] row-major, beta[a*K+n] = beta_{n,a}.
int orc_linear_table(double* E, int M, long long N, double dt, double hh, double alpha, const double* beta, int K,
                     int nthreads) {
  if (!E || !beta || M < 1 || K < 1 || !is_pow2(N) || !(dt > 0)) return -1;
  linear_table((cplx*)E, M, N, dt, hh, alpha, beta, K, nthreads);
  return 0;
}

// x[2M][N] <- exp(hh L) x, E from orc_linear_table with the same hh.
int orc_apply_D(double* x, int M, long long N, const double* E, int nthreads) {
  if (!x || !E || M < 1 || !is_pow2(N)) return -1;
  apply_D((cplx*)x, M, N, (const cplx*)E, nthreads);
  return 0;
}

// out[2M][N] = (i * hgamma * sum_b kappa_ab P_b) * u;  kappa is [M][M] row-major, kappa[a*M+b] = kappa_ab.
int orc_nonlinear(const double* u, double* out, int M, long long N, double hgamma, const double* kappa,
                  int nthreads) {
  if (!u || !out || !kappa || M < 1 || N < 1) return -1;
  nonlinear((const cplx*)u, (cplx*)out, M, N, hgamma, kappa, nthreads);
  return 0;
}

// A[2M][N] advanced nsteps RK4IP steps of size h, in place.
int orc_rk4ip(double* A, int M, long long N, double dt, double h, double alpha, const double* beta, int K,
              double gamma, const double* kappa, int nsteps, int nthreads) {
  if (!A || !beta || !kappa || M < 1 || K < 1 || !is_pow2(N) || !(dt > 0) || nsteps < 0) return -1;
  if (nsteps == 0) return 0;
  const long long tot = 2LL * M * N;
  std::vector<cplx> E((size_t)M * N), AI(tot), k1(tot), k2(tot), k3(tot), k4(tot), tmp(tot);
  linear_table(E.data(), M, N, dt, h / 2.0, alpha, beta, K, nthreads);
  for (int s = 0; s < nsteps; ++s)
    rk4ip_step((cplx*)A, M, N, E.data(), h * gamma, kappa, false, nthreads, AI.data(), k1.data(), k2.data(), k3.data(),
               k4.data(), tmp.data());
  return 0;
}

// A link of nspans fibre spans (section 6: "two 80 km spans ... After each span, the fiber losses are
// compensated by a noiseless amplifier with flat-gain profile"): each span is steps_per_span RK4IP steps of size h,
// followed by the lumped amplifier A <- gain * A (gain = the AMPLITUDE factor, the same for every mode and frequency;
// exp(alpha L_span / 2) compensates the loss exactly).  general != 0: kappa is the [2M][2M] matrix.
int orc_rk4ip_spans(double* A, int M, long long N, double dt, double h, double alpha, const double* beta, int K,
                    double gamma, const double* kappa, int general, int nspans, int steps_per_span, double gain,
                    int nthreads) {
  if (!A || !beta || !kappa || M < 1 || K < 1 || !is_pow2(N) || !(dt > 0) || nspans < 0 || steps_per_span < 1) return -1;
  const long long tot = 2LL * M * N;
  std::vector<cplx> E((size_t)M * N), AI(tot), k1(tot), k2(tot), k3(tot), k4(tot), tmp(tot);
  linear_table(E.data(), M, N, dt, h / 2.0, alpha, beta, K, nthreads);
  cplx* a = (cplx*)A;
  for (int sp = 0; sp < nspans; ++sp) {
    for (int s = 0; s < steps_per_span; ++s)
      rk4ip_step(a, M, N, E.data(), h * gamma, kappa, general != 0, nthreads, AI.data(), k1.data(), k2.data(), k3.data(),
                 k4.data(), tmp.data());
    for (long long i = 0; i < tot; ++i) a[i] *= gain;      // the lumped amplifier at the end of the span
  }
  return 0;
}

// out[2M][N] = (i * hgamma * sum_s kappa2[r][s] |u_s|^2) * u_r;  kappa2 is [2M][2M] row-major.
int orc_nonlinear_general(const double* u, double* out, int M, long long N, double hgamma, const double* kappa2,
                          int nthreads) {
  if (!u || !out || !kappa2 || M < 1 || N < 1) return -1;
  nonlinear_general((const cplx*)u, (cplx*)out, M, N, hgamma, kappa2, nthreads);
  return 0;
}

// orc_rk4ip with the general per-polarisation coupling matrix kappa2 [2M][2M].
int orc_rk4ip_general(double* A, int M, long long N, double dt, double h, double alpha, const double* beta, int K,
                      double gamma, const double* kappa2, int nsteps, int nthreads) {
  if (!A || !beta || !kappa2 || M < 1 || K < 1 || !is_pow2(N) || !(dt > 0) || nsteps < 0) return -1;
  if (nsteps == 0) return 0;
  const long long tot = 2LL * M * N;
  std::vector<cplx> E((size_t)M * N), AI(tot), k1(tot), k2(tot), k3(tot), k4(tot), tmp(tot);
  linear_table(E.data(), M, N, dt, h / 2.0, alpha, beta, K, nthreads);
  for (int s = 0; s < nsteps; ++s)
    rk4ip_step((cplx*)A, M, N, E.data(), h * gamma, kappa2, true, nthreads, AI.data(), k1.data(), k2.data(), k3.data(),
               k4.data(), tmp.data());
  return 0;
}

// A[2M][N] advanced nsteps SSFM-RK4 steps of size h (symmetric split step, Eq. 4), in place.
int orc_ssfm_rk4(double* A, int M, long long N, double dt, double h, double alpha, const double* beta, int K,
                 double gamma, const double* kappa, int nsteps, int nthreads) {
  if (!A || !beta || !kappa || M < 1 || K < 1 || !is_pow2(N) || !(dt > 0) || nsteps < 0) return -1;
  if (nsteps == 0) return 0;
  const long long tot = 2LL * M * N;
  std::vector<cplx> E((size_t)M * N), k1(tot), k2(tot), k3(tot), k4(tot), tmp(tot);
  linear_table(E.data(), M, N, dt, h / 2.0, alpha, beta, K, nthreads);
  for (int s = 0; s < nsteps; ++s)
    ssfm_rk4_step((cplx*)A, M, N, E.data(), h * gamma, kappa, nthreads, k1.data(), k2.data(), k3.data(), k4.data(),
                  tmp.data());
  return 0;
}

// A[2M][N] advanced nsteps SSFM-Agrawal steps of size h with niter >= 1 iterations each (Eq. 4, reading R14), in place.
int orc_ssfm_agrawal(double* A, int M, long long N, double dt, double h, double alpha, const double* beta, int K,
                     double gamma, const double* kappa, int nsteps, int niter, int nthreads) {
  if (!A || !beta || !kappa || M < 1 || K < 1 || !is_pow2(N) || !(dt > 0) || nsteps < 0 || niter < 1) return -1;
  if (nsteps == 0) return 0;
  const long long tot = 2LL * M * N;
  std::vector<cplx> E((size_t)M * N), B(tot), Y(tot);
  std::vector<double> S0((size_t)M * N), S1((size_t)M * N);
  linear_table(E.data(), M, N, dt, h / 2.0, alpha, beta, K, nthreads);
  for (int s = 0; s < nsteps; ++s)
    ssfm_agrawal_step((cplx*)A, M, N, E.data(), h * gamma, kappa, niter, nthreads, B.data(), Y.data(), S0.data(),
                      S1.data());
  return 0;
}

// noise loading: the generator alone (for its known-answer pins) and the whole operation
int orc_philox4x32_10(const uint32_t* ctr, const uint32_t* key, uint32_t* out) {
  if (!ctr || !key || !out) return -1;
  philox4x32_10(ctr, key, out);
  return 0;
}

int orc_noise_unit(double* z, unsigned long long seed, unsigned row, unsigned long long t0, long long count) {
  if (!z || count < 0) return -1;
  for (long long i = 0; i < count; ++i) {
    const cplx v = noise_unit_sample(seed, row, t0 + (uint64_t)i);
    z[2 * i] = v.real();
    z[2 * i + 1] = v.imag();
  }
  return 0;
}

int orc_add_noise(double* A, int M, long long N, double dt, double osnr_db, double ref_bw, int nch,
                  unsigned long long seed, double* power_out) {
  if (!A || !power_out || M < 1 || N < 1 || !(dt > 0) || !(ref_bw > 0) || nch < 1 || std::isnan(osnr_db)) return -1;
  add_noise(reinterpret_cast<cplx*>(A), M, N, dt, osnr_db, ref_bw, nch, seed, power_out);
  return 0;
}

}  // extern "C"
