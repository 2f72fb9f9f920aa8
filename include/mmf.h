/* mmf.h — C ABI of the B200-native RK4IP propagator for the multimode Manakov/NLSE.
 *
 * Source of truth for what is computed: arXiv 1901.01895 ("the paper"; citations are PAPER.md:<line> of the
 * extracted text) — Eq. (1) PAPER.md:35-37 (model), Eq. (6a)-(6f) PAPER.md:75-88 (the RK4IP step), data layout
 * PAPER.md:95,107 (2M x N complex matrix, row-major, one row per spatial/polarisation mode).  Readings taken where
 * the paper is silent or garbled are listed in DESIGN.md ("Readings").
 *
 * Conventions
 *   - Units are the caller's: dt in [T], h in [L]; alpha in 1/[L] is the linear POWER attenuation (the amplitude
 *     decays as exp(-alpha z/2), Eq. 1); beta_n in [T]^n/[L]; gamma in 1/(W [L]) with |A|^2 in W.
 *   - Field layout: A[2M][N] complex128, interleaved (re, im), row-major; row r = 2a + p is polarisation p (0 = x,
 *     1 = y) of spatial mode a.  |A_b|^2 of Eq. (1) is |A_bx|^2 + |A_by|^2 (Manakov).
 *   - Fourier convention (Eq. 1 is written in the time domain; it fixes the convention): A(t) = sum_k At_k
 *     exp(-i w_k t), w_k = 2 pi k'/(N dt), k' = k for k < N/2 and k - N otherwise (the Nyquist bin is negative);
 *     then L_a(w) = -alpha/2 + i sum_{n=0}^{K-1} beta_{n,a} w^n / n!  and beta_1 > 0 DELAYS the field.
 *   - Every function returns MMF_OK (0) or a negative error code; nothing throws, prints or keeps global state.
 *     Plans are independent; one plan must not be used from two streams at once.
 *   - "device" pointers are CUDA device pointers of the current device; "host" pointers are ordinary memory.
 *   - Functions taking a stream only ENQUEUE work on it (no allocation, no synchronisation) unless stated.
 */
#ifndef MMF_H_
#define MMF_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define MMF_OK      0
#define MMF_EINVAL -1   /* bad argument (null pointer, size, non-finite parameter, unset/small workspace, alignment) */
#define MMF_ENOMEM -2   /* host or device allocation failed */
#define MMF_ECUDA  -3   /* CUDA runtime / launch error */
#define MMF_ETOOBIG -4  /* mmf_apply_nonlinear_static only: M * N * 8 bytes exceed MMF_STATIC_SCRATCH_BYTES */

typedef struct mmf_plan mmf_plan; /* opaque */

/* Create a plan for M spatial modes x 2 polarisations x N samples.
 *   out    host, receives the plan.
 *   M >= 1; N a power of two, 16 <= N <= 2^24; dt > 0 sample spacing; h step size (Eq. 6: separation z' = z+h/2).
 *   alpha  power attenuation (Eq. 1, "-alpha/2").
 *   beta   host, [M][K] row-major, beta[a*K + n] = beta_{n,a}, n = 0..K-1 (Eq. 1 Taylor coefficients), 1 <= K <= 8.
 *   gamma  Kerr coefficient (Eq. 1).
 *   kappa  host, [M][M] row-major, kappa[a*M + b] = kappa_ab (Eq. 1; need not be symmetric).
 * beta and kappa are copied; the plan owns its small device tables (kappa, twiddles). */
int mmf_plan_create(mmf_plan **out, int M, long long N, double dt, double h, double alpha, const double *beta, int K,
                    double gamma, const double *kappa);

/* Same, with the GENERAL coupling matrix the paper's implementation stores (Fig. 2: "a matrix of
 * 2M x 2M elements", one coefficient per pair of polarisation modes):
 *   kappa2  host, [2M][2M] row-major, kappa2[r*2M + s] couples row s (= 2b + q) into row r (= 2a + p):
 *           N_r = i gamma sum_s kappa2[r][s] |A_s|^2.  Need not be symmetric.  kappa2[2a+p][2b+q] = kappa_ab is Eq. (1).
 * Requires M <= 120 (MMF_EINVAL otherwise).  Such a plan runs mmf_propagate, mmf_propagate_host and mmf_apply_*;
 * the split-step entry points return MMF_EINVAL for it.  Workspace: three more field buffers (four when N > 4096). */
int mmf_plan_create_general(mmf_plan **out, int M, long long N, double dt, double h, double alpha, const double *beta,
                            int K, double gamma, const double *kappa2);

/* Bytes of device workspace the plan needs: one more full-field buffer when N <= 4096, two when N > 4096 (three resp.
 * four when M > 120) plus the tabulated exp(h/2 L_a(w_k)) of Eq. (6a) (one row per mode), plus for N <= 4096 a real
 * [M][N] table for mmf_propagate_ssfm_agrawal.  The caller allocates it
 * (e.g. a torch uint8 tensor), 256-byte aligned, and keeps it alive while the plan is used.  Note: for N > 4096 the
 * library works on copies in an internal (blocked) sample order; A_dev is read in the natural order documented above
 * by the first kernel of a call and written in it by the last one. */
size_t mmf_plan_workspace_bytes(const mmf_plan *plan);

/* Attach the workspace and fill the plan's tables in it (enqueues kernels on `cuda_stream`, a cudaStream_t passed
 * as void*; 0 = default stream).  Must precede mmf_propagate / mmf_apply_*. */
int mmf_plan_set_workspace(mmf_plan *plan, void *ws_dev, size_t bytes, void *cuda_stream);

/* Advance A by nsteps RK4IP steps of size h, Eq. (6a)-(6f), in place.
 *   A_dev  device, [2M][N] complex128 (layout above), 16-byte aligned.  nsteps >= 0 (0 is a no-op).
 * Calling with n1 then n2 steps equals one call with n1+n2 steps.  For N = 4096 and M <= 4 the whole call is one
 * kernel (a thread-block cluster with the field in distributed shared memory; MMF_SMALL_CLUSTER=0 in the environment
 * selects the kernel-per-stage plan instead; the two agree to rounding — <= 1e-13 relative L2 per field in the tests —
 * not bit for bit, because the cluster kernel sums kappa_ab P_b in a per-warp rotated mode order).  On MMF_ECUDA (a launch failed mid-sequence) the
 * contents of A_dev and of the workspace are unspecified: the caller must restore the field before retrying. */
int mmf_propagate(mmf_plan *plan, void *A_dev, int nsteps, void *cuda_stream);

/* A link of nspans fibre spans (section 6: "After each span, the fiber losses are compensated by a
 * noiseless amplifier with flat-gain profile"): nspans x steps_per_span RK4IP steps, and after the last step of every
 * span A <- gain * A (gain = AMPLITUDE factor, the same for all modes and frequencies; exp(alpha h steps_per_span / 2)
 * compensates the span loss exactly).  The multiplication rides on the last kernel of the span: no extra pass.
 * nspans >= 0, steps_per_span >= 1, gain finite.  Equals mmf_propagate(steps_per_span) + a scaling, nspans times. */
int mmf_propagate_spans(mmf_plan *plan, void *A_dev, int nspans, int steps_per_span, double gain, void *cuda_stream);

/* Advance A by nsteps SYMMETRIC SPLIT STEPS of size h with a Runge-Kutta nonlinear substep ("SSFM-RK4": Eq. 4
 * PAPER.md:58-61 with the nonlinear part solved by classical RK4), in place:
 *   A <- exp(h/2 L) A;  A <- RK4 over h of dA/dz = N(A) A;  A <- exp(h/2 L) A        (globally O(h^2)).
 * Same arguments and layout as mmf_propagate; runs on the same transform kernels and one fused nonlinear kernel that
 * evaluates all four N per sample tile (2 F of traffic).  Requires M <= 120 (MMF_EINVAL otherwise). */
int mmf_propagate_ssfm(mmf_plan *plan, void *A_dev, int nsteps, void *cuda_stream);

/* Advance A by nsteps symmetric split steps with the ITERATIVE nonlinear part ("SSFM-Agrawal": Eq. 4 PAPER.md:58-61,
 * "solved by an iterative approach as described in [6]" PAPER.md:63, "|A|^2 once at the position z for the first
 * iteration and at the position z + h for every following iteration" PAPER.md:111), in place.  Per step, with
 * S_a(u) = sum_b kappa_ab |u_b|^2 and the integral of Eq. (4) by the trapezoidal rule:
 *   B = exp(h/2 L) A(z);  A_1 = exp(h/2 L)[exp(i h gamma S(A(z))) B];
 *   A_j = exp(h/2 L)[exp(i (h gamma/2) (S(A(z)) + S(A_{j-1}))) B], j = 2..niter;  A(z+h) = A_niter.   (globally O(h^2))
 * niter >= 1 (2 is the textbook choice).  Same arguments, layout and M <= 120 restriction as mmf_propagate_ssfm. */
int mmf_propagate_ssfm_agrawal(mmf_plan *plan, void *A_dev, int nsteps, int niter, void *cuda_stream);

/* Same, for a HOST field: copies A_host to an internal slot of the workspace-adjacent device buffer `A_dev_scratch`
 * (device, [2M][N] complex128, caller-owned), propagates, copies back and SYNCHRONISES the stream.  A_host should be
 * page-locked for full copy bandwidth.  This is the end-to-end entry point bench.py times. */
int mmf_propagate_host(mmf_plan *plan, void *A_host, void *A_dev_scratch, int nsteps, void *cuda_stream);

/* A stream of nfields HOST fields through one plan (e.g. a launch-power sweep of one fibre): field i propagates on
 * `cuda_stream` while field i + 1 is copied in and field i - 1 is copied out on two internal copy streams, over the two
 * device buffers A_dev0 / A_dev1 (device, [2M][N] complex128 each, caller-owned; A_dev1 may be null when nfields == 1).
 *   A_hosts  host array of nfields host pointers, each [2M][N] complex128, page-locked for the copies to overlap.
 * Every field is advanced nsteps RK4IP steps in place (in its host buffer).  SYNCHRONISES before returning.
 * (One field alone cannot hide its copies: the first transform of a step needs the whole time axis of every row.) */
int mmf_propagate_host_batch(mmf_plan *plan, void *const *A_hosts, int nfields, void *A_dev0, void *A_dev1, int nsteps,
                             void *cuda_stream);

/* ROW-SHARDED propagation (sections 4.1-4.3: every process holds whole rows of the signal matrix and
 * "the squared absolute values have to be shared between the GPUs" once per evaluation of N, four times per step).
 * A shard plan describes ONE rank: its M_local modes mode0 .. mode0 + M_local - 1 of a fibre with M_total modes.
 *   beta        host, [M_local][K]: the rank's own modes.
 *   kappa_rows  host, [M_local][M_total] row-major: rows mode0 .. of the fibre's kappa (all columns).
 * Workspace (mmf_plan_workspace_bytes): three field buffers of the rank's size (four when N > 4096) + its E table.
 * One RK4IP step is the sequence below, driven by the caller with ITS collective between powers and apply
 * (paper_1901_01895_b200/sharded.py does it with torch.distributed; the library itself never communicates):
 *   mmf_shard_begin(A)                         the rank's rows [2 M_local][N]; A stays attached until mmf_shard_end
 *   powers(0); all-gather; apply(0)            Y <- h N(A) A                                  (bracket of Eq. 6b)
 *   per step:  linear(0)                       A_I = D A, k1 = D Y                            (6a), (6b)
 *              powers(1); all-gather; apply(1) k2 = h N(A_I + k1/2)(A_I + k1/2)               (6c)
 *              powers(2); all-gather; apply(2) k3 (6d) and the brackets of (6e), (6f)
 *              linear(1)                       u4 = D(A_I + k3), D(bracket)                   (6e), (6f)
 *              powers(3); all-gather; apply(3, gain)   A <- gain (D(bracket) + h N(u4) u4 / 6)   (6e), (6f)
 *              powers(0); all-gather; apply(0) for the next step (not after the last one)
 *   mmf_shard_end()                            the result is in A
 * mmf_shard_powers / mmf_shard_apply work on a TIME CHUNK: samples t_first .. t_first + t_count - 1 (the whole axis:
 *   0, N), with P_dev (device, [M_total][t_count] doubles, row-major) the chunk's own power block.  powers writes rows
 *   mode0 .. mode0 + M_local - 1: P[b][t - t_first] = |u_bx(t)|^2 + |u_by(t)|^2, u the argument of the stage's N; the
 *   caller's all-gather fills the other rows; apply reads all of them.  Chunks let the gather of one chunk overlap
 *   the kernels of its neighbours.  For N > 4096 the sample index is the library's internal (blocked)
 *   order — the same on every rank, since it depends on N only.  stage: 0..3 as listed.
 * Size bound, checked by mmf_plan_create_shard (MMF_EINVAL): the apply kernel keeps the rank's kappa rows, a power tile
 *   and a result tile in one SM's shared memory, 8 (M_total MP + 32 M_total + 32 MP) <= 232 448 bytes with MP = M_local
 *   rounded up to a multiple of 4 (e.g. M_total = 240: M_local <= 80, three ranks or more; M_total = 120: any split).
 * Shard plans accept only the mmf_shard_* calls, mmf_apply_linear and the timing / debug calls. */
int mmf_plan_create_shard(mmf_plan **out, int M_local, int M_total, int mode0, long long N, double dt, double h,
                          double alpha, const double *beta, int K, double gamma, const double *kappa_rows);
int mmf_shard_begin(mmf_plan *plan, void *A_dev, void *cuda_stream);
int mmf_shard_powers(mmf_plan *plan, int stage, void *P_dev, long long t_first, long long t_count, void *cuda_stream);
int mmf_shard_apply(mmf_plan *plan, int stage, const void *P_dev, long long t_first, long long t_count, double gain,
                    void *cuda_stream);
int mmf_shard_linear(mmf_plan *plan, int which, void *cuda_stream);
int mmf_shard_end(mmf_plan *plan, void *cuda_stream);

/* Stage-level entry points (each is a row group of the hot path; used by the parity tests).
 * mmf_apply_linear:    X <- exp(h/2 L) X  (Eq. 6a: transform, multiply by exp(h/2 L_a(w_k)), transform back), in place.
 * mmf_apply_nonlinear: OUT <- h N(U) U = i h gamma (sum_b kappa_ab |U_b|^2) U_a   (Eq. 1 / the bracket of Eq. 6b).
 *                      U and OUT are device [2M][N] complex128 and may alias exactly (OUT == U) or not at all. */
int mmf_apply_linear(mmf_plan *plan, void *X_dev, void *cuda_stream);
int mmf_apply_nonlinear(mmf_plan *plan, const void *U_dev, void *OUT_dev, void *cuda_stream);

/* NOISE LOADING (section 6: "White noise is added to the signals before the receiver, setting the optical
 * signal-to-noise ratio (OSNR) to 20 dB"; the reading of that sentence is R18 in DESIGN.md).  Adds complex circular white
 * Gaussian noise, independent per row and sample, to the field in place; needs no plan and no workspace.
 *   A_dev     device, [2M][N] complex128 in the natural layout documented at the top, 16-byte aligned; any N >= 1.
 *   dt        sample spacing [T];  ref_bw  the OSNR's reference bandwidth [1/T] (12.5 GHz = 0.1 nm by convention);
 *   osnr_db   requested OSNR in dB (+infinity: nothing is added);  nch >= 1  wavelength channels carried by a mode.
 *   seed      selects the noise stream.  The sample of (seed, row, t) comes from Philox-4x32-10 with counter
 *             (t low word, t high word, row, 0) and key (seed low word, seed high word) and Box-Muller on two 52-bit
 *             uniforms: it does not depend on M, N or the launch, so any sub-block can be reproduced.
 *   mode_power_dev  device, [M] doubles, OUTPUT: P_a = mean over t of |A_ax|^2 + |A_ay|^2 of the field BEFORE the noise.
 * Per spatial mode a: noise density per polarisation N0 = P_a / (nch 2 ref_bw OSNR) (the OSNR counts the noise of both
 * polarisations inside ref_bw against the power of one channel), white over the simulated band 1/dt, i.e. variance
 * sigma_a^2 = N0 / dt per complex sample; A_{a,p}(t) += sigma_a z(seed, 2a+p, t) with E|z|^2 = 1.  Enqueues two kernels
 * (mode powers: one read of the field; noise: one read and one write).  M <= 32767.
 * mmf_debug_noise_words: the generator alone — words_dev (device, 16-byte aligned) receives the four 32-bit Philox
 * output words of samples t0 .. t0 + count - 1 of `row`, [count][4] uint32. */
int mmf_add_noise(void *A_dev, int M, long long N, double dt, double osnr_db, double ref_bw, int nch,
                  unsigned long long seed, double *mode_power_dev, void *cuda_stream);
int mmf_debug_noise_words(unsigned long long seed, unsigned row, unsigned long long t0, long long count, void *words_dev,
                          void *cuda_stream);

/* The nonlinear operator for callers that CANNOT ALLOCATE device memory: OUT <- h N(U) U of Eq. (1), as
 * mmf_apply_nonlinear computes it, but without a plan and without a workspace.
 *   Who needs it: a host program that took all of HBM for its own pool at start-up (any later cudaMalloc fails there),
 *   a framework whose caching allocator must see every device byte, and code in a latency-critical loop, where the
 *   device-wide synchronisation inside cudaMalloc / cudaFree is not acceptable.  mmf_plan_create and a torch-allocated
 *   workspace are out of reach for all three; this call needs neither, and itself calls no cudaMalloc, cudaFree or
 *   allocating library routine.
 *   M >= 1 modes, N >= 1 samples (any N, no transform is involved), h and gamma finite;
 *   kappa_dev  DEVICE, [M][M] row-major doubles, kappa_dev[a*M + b] = kappa_ab (the caller's memory, not copied);
 *   U_dev      device, [2M][N] complex128, the layout documented at the top, 16-byte aligned;
 *   OUT_dev    device, same shape; may be U_dev itself or must not overlap it at all.
 * It runs the two-kernel form of the paper's Listing 1 (powers to global memory as a real [M][N]
 * matrix, then contraction and product); the power matrix goes to a file-scope `static __device__` array of
 * MMF_STATIC_SCRATCH_BYTES (4 MiB), so M * N <= 524 288 (config 0: 8 192, config 1: 393 216 fit; 120 modes up to
 * N = 4096).  A larger problem returns MMF_ETOOBIG and launches nothing.  Consequences of the static array:
 *   - each GPU on which the library's code gets loaded gives up those 4 MiB until the process ends;
 *   - every call on a device uses the same array.  A call writes all the entries it reads, so leftovers of the
 *     previous call do no harm and nothing needs clearing, but calls that can overlap on the GPU (different streams or
 *     host threads) race: issue them into one stream or order them with events;
 *   - the first call on each device looks up the array's device address (cudaGetSymbolAddress, with that device
 *     current) and may trigger the loading of the module.  Make that first call during set-up, before you begin any
 *     stream capture.  Later calls only enqueue two kernels on `cuda_stream`.
 * Results agree with mmf_apply_nonlinear to rounding (the sum over b runs in ascending order here, in tensor-core
 * fragment order there); on integer-valued data both are exact. */
#define MMF_STATIC_SCRATCH_BYTES (4u << 20)
int mmf_apply_nonlinear_static(int M, long long N, double h, double gamma, const double *kappa_dev, const void *U_dev,
                               void *OUT_dev, void *cuda_stream);

/* Debug / test entry points.
 * mmf_debug_forward:  SPEC <- the plain forward transform of every row of X, SPEC[r][k] = sum_n X[r][n] exp(+2 pi i k n/N),
 *                     written in NATURAL bin order (the hot path never materialises this order).  X is destroyed.
 * mmf_debug_freq_index: host int64 array idx[N]; idx[s] = the bin k that slot s of the plan's internal (permuted)
 *                     spectrum layout holds.  Must be a permutation of 0..N-1.  Synchronises. */
int mmf_debug_forward(mmf_plan *plan, void *X_dev, void *SPEC_dev, void *cuda_stream);
int mmf_debug_freq_index(mmf_plan *plan, long long *idx_host);

/* Number of kernel launches this plan has enqueued since creation (bench.py's gpu_launches). */
long long mmf_plan_launch_count(const mmf_plan *plan);

/* Mode groups (section 6: "The modes form strongly coupled groups of modes ... This is taken into account
 * by choosing the appropriate nonlinear coupling coefficients kappa"; Table 2: 15 groups for 120 modes).  When the
 * kappa given to mmf_plan_create has only G distinct rows (exact equality; every mode of a group couples to the others
 * alike), G <= 32 and 2 G <= M, the contraction runs on the G distinct rows and every mode picks its group's result:
 * G M instead of M M products per time sample, the same values bit for bit.  Returns G, or 0 when the plan contracts
 * the dense matrix (also with MMF_GROUPED=0 in the environment at plan creation). */
int mmf_plan_groups(const mmf_plan *plan);

/* Per-kernel timing for bench.py's roofline.  mmf_plan_set_timing(plan, 1) makes every later launch of
 * this plan be bracketed by a pair of CUDA events on the launching stream (and drops earlier records; at most 65536
 * launches are recorded, later ones run unrecorded); (plan, 0) switches it off.  While it is on, small problems run
 * launch by launch instead of from their captured graphs, and without programmatic dependent launch.  mmf_plan_get_timing SYNCHRONISES on the recorded events of kernel class `kclass`
 * (0 <= kclass < mmf_kernel_class_count()) and returns their summed device time [ms], their number, and the
 * ALGORITHMIC bytes of one such launch, averaged over the recorded ones (full-field reads + writes; tables excluded). */
int mmf_plan_set_timing(mmf_plan *plan, int enable);
int mmf_kernel_class_count(void);
const char *mmf_kernel_class_name(int kclass);
int mmf_plan_get_timing(mmf_plan *plan, int kclass, double *total_ms, long long *launches, double *alg_bytes);

/* Frees the plan and its device tables (not the workspace, which the caller owns). */
int mmf_plan_destroy(mmf_plan *plan);

/* Static, human-readable text for a status code; for MMF_ECUDA the last CUDA error string seen by this thread. */
const char *mmf_status_string(int status);

/* Library version string. */
const char *mmf_version(void);

#ifdef __cplusplus
}
#endif
#endif /* MMF_H_ */
