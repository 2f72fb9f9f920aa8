// mmf_api.cu — the C ABI of include/mmf.h: plan management, table generation and the per-step launch sequence.
// The product path: every step of the hot path runs in the kernels of fft_kernels.cuh / nl_tma.cuh / nl_simt.cuh;
// there is no CPU fallback.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <mutex>
#include <vector>

#include "../../include/mmf.h"
#include "fft_kernels.cuh"
#include "nl_tma.cuh"
#include "nl_simt.cuh"
#include "nl_general.cuh"
#include "nl_shard.cuh"
#include "small_cluster.cuh"

using namespace mmf;

namespace {

thread_local char g_cuda_msg[256] = "CUDA error";

int cuda_fail(cudaError_t e) {
  snprintf(g_cuda_msg, sizeof(g_cuda_msg), "CUDA error: %s", cudaGetErrorString(e));
  return MMF_ECUDA;
}
#define CU(call)                                \
  do {                                          \
    cudaError_t e__ = (call);                   \
    if (e__ != cudaSuccess) return cuda_fail(e__); \
  } while (0)

constexpr int kGroups = 2;  // independent 256-thread groups per persistent transform CTA

// exp(2 pi i p / n) for 0 <= p < n (n a power of two), long double with the angle folded to [0, pi/4] first,
// so that the table is exactly symmetric and quarter turns are exact.  (Written independently of the oracle.)
void root_of_unity(long long p, long long n, double* re, double* im) {
  static const long double TWO_PI = 6.283185307179586476925286766559005768L;
  p %= n;
  const long long quarter = n / 4;
  long double c, s;
  if (n < 8) {  // n = 1, 2, 4: all values exact
    static const int C4[4] = {1, 0, -1, 0}, S4[4] = {0, 1, 0, -1};
    const int q = (int)(p * (4 / n));
    *re = C4[q];
    *im = S4[q];
    return;
  }
  const int quad = (int)(p / quarter);
  long long r = p % quarter;  // angle r/n turns inside the quadrant, 0 <= r < n/4
  bool swap = false;
  if (r > quarter / 2) {  // fold about the diagonal of the quadrant
    r = quarter - r;
    swap = true;
  }
  if (r == 0) {
    c = 1.0L;
    s = 0.0L;
  } else if (2 * r == quarter && !swap) {
    c = s = 0.707106781186547524400844362104849039L;
  } else {
    const long double ang = TWO_PI * (long double)r / (long double)n;
    c = cosl(ang);
    s = sinl(ang);
  }
  if (swap) {
    const long double tmp = c;
    c = s;
    s = tmp;
  }
  long double cr, ci;
  switch (quad) {
    case 0: cr = c; ci = s; break;
    case 1: cr = -s; ci = c; break;
    case 2: cr = -c; ci = -s; break;
    default: cr = s; ci = -c; break;
  }
  *re = (double)cr;
  *im = (double)ci;
}

// stage twiddle tables of a 2^logp-point transform in the order fft_core.cuh reads them: stages most significant
// digit first, stage (lr, logm) holding exp(2 pi i b c / 2^(lr+logm)) at [(c-1) << logm | b].
int upload_stage_tables(cpx** dptr, int logp) {
  std::vector<cpx> h;
  int remain = logp, nst = nstages(logp);
  while (nst > 0) {
    const int lr = stage_lr(remain, nst), logm = remain - lr;
    if (logm > 0)
      for (int c = 1; c < (1 << lr); ++c) {
        if (tw_compact(lr, logm) && !(c < 4 || (c & 3) == 0)) continue;  // rows c = 1, 2, 3, 4, 8, 12 only
        for (int b = 0; b < (1 << logm); ++b) {
          cpx w;
          root_of_unity((long long)b * c, 1LL << (lr + logm), &w.x, &w.y);
          h.push_back(w);
        }
      }
    remain = logm;
    --nst;
  }
  if ((int)h.size() != tw_total_entries(logp, nstages(logp))) return MMF_EINVAL;
  if (h.empty()) h.push_back(make_double2(1.0, 0.0));
  CU(cudaMalloc((void**)dptr, sizeof(cpx) * h.size()));
  CU(cudaMemcpy(*dptr, h.data(), sizeof(cpx) * h.size(), cudaMemcpyHostToDevice));
  return MMF_OK;
}

size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

}  // namespace

struct mmf_plan {
  int M = 0, K = 0, logn = 0, logn1 = 0, logn2 = 0;
  int nlm_nk = -1;   // k-steps of the tensor-path nonlinear kernel; -1: M too large, legacy kernels (4 buffers)
  bool general = false;  // kappa is the general [2M][2M] per-polarisation matrix (k_nlg, four-buffer plan)
  // row-sharded plan (mmf_plan_create_shard): M = the rank's own modes, kappa = its [M][M_total] rows
  int M_total = 0, mode0 = 0;
  cpx* shard_X = nullptr;   // the rank's field while a sharded propagation is open (mmf_shard_begin .. mmf_shard_end)
  void* shard_A = nullptr;
  int num_sms = 148;
  int device = 0;    // the device the plan's tables live on; every call must be made with it current
  long long N = 0;
  double dt = 0, h = 0, alpha = 0, gamma = 0;
  std::vector<double> beta, kappa;
  double* d_kappa = nullptr;
  cpx *d_tw1 = nullptr, *d_tw2 = nullptr, *d_ipt = nullptr;
  dd* d_coefs = nullptr;
  unsigned char* ws = nullptr;
  size_t ws_bytes = 0, field_bytes = 0;
  cpx *Y = nullptr, *Z = nullptr, *W = nullptr, *V = nullptr, *E = nullptr;
  double* T = nullptr;  // N <= 4096: the table of mmf_propagate_ssfm_agrawal (workspace)
  // launch plan ("small-problem launch plan"): everything a launch needs besides its arguments is computed once per plan —
  // tensor maps per (kind, buffer), the dynamic shared-memory attribute and the occupancy per kernel — and the step
  // body of small problems is replayed from a captured CUDA graph
  struct MapEntry { int kind; const void* base; int aux; CUtensorMap map; };
  std::vector<MapEntry> map_cache;
  struct OccEntry { const void* kern; int threads; size_t smem; int occ; };
  std::vector<OccEntry> occ_cache;
  bool dry_run = false;              // launch helpers prepare (attributes, maps) but do not launch
  bool pdl = true;                   // launch with programmatic stream serialization (async_copy.cuh); MMF_PDL=0 disables
  int small_cluster = -1;            // whole-propagation cluster kernel (small_cluster.cuh): -1 untested, 0 no, 1 yes
  // mode groups (nl_tma.cuh GROUPED): kappa has only G distinct rows; 0 = dense contraction
  int G = 0;
  double* d_kappa_g = nullptr;       // [G][M]
  int* d_group_of = nullptr;         // [M]
  cudaStream_t cap_stream = nullptr; // capture stream of the step-body graphs
  struct GraphEntry { const void* X; const void* Y; int reps; long long nlaunch; cudaGraphExec_t exec; };
  std::vector<GraphEntry> graphs;
  long long launches = 0;
  // optional per-launch CUDA-event timing (mmf_plan_set_timing): one (start, stop) pair per launch
  bool timing = false;
  std::vector<cudaEvent_t> ev;       // 2 per recorded launch
  std::vector<int> ev_class;         // kernel class of each recorded launch
  std::vector<double> ev_bytes;      // algorithmic bytes of each recorded launch (full-field reads + writes)
};

namespace {

// ---- kernel classes (for mmf_plan_get_timing) ----------------------------------------------------------------------
enum { KC_COLS_FWD = 0, KC_ROWS, KC_COLS_INV, KC_NL_PLAIN, KC_NL_STAGE2, KC_NL_STAGE3, KC_NL_FINAL, KC_NL_FINAL_NEXT,
       KC_NLM_PLAIN, KC_NLM_S23, KC_NLM_FINAL, KC_NLM_FINAL_NEXT, KC_NLM_RK4, KC_NLM_ENTER, KC_NLM_EXIT, KC_NLM_AGR_S0,
       KC_NLM_AGR_IT1, KC_NLM_AGR_ITJ, KC_PERM, KC_NLG_PLAIN, KC_NLG_STAGE2, KC_NLG_STAGE3, KC_NLG_FINAL, KC_SHARD_POW, KC_SHARD_APPLY, KC_SMALL, KC_COUNT };
const char* const kc_names[KC_COUNT] = {"k_cols<fwd>", "k_rows", "k_cols<inv>", "k_nl<plain>", "k_nl<stage2>",
                                        "k_nl<stage3>", "k_nl<final>", "k_nl<final_next>", "k_nlm<plain>",
                                        "k_nlm<s23>", "k_nlm<final>", "k_nlm<final_next>", "k_nlm<rk4>", "k_nlm<enter>",
                                        "k_nlm<exit>", "k_nlm<agr_s0>", "k_nlm<agr_it1>", "k_nlm<agr_itj>", "k_perm",
                                        "k_nlg<plain>", "k_nlg<stage2>", "k_nlg<stage3>", "k_nlg<final>", "k_shard_pow",
                                        "k_shard_apply", "k_small"};

// event bracket around one launch when timing is on (events go on the launching stream)
constexpr size_t kMaxTimedLaunches = 1 << 16;
struct LaunchTimer {
  mmf_plan* p;
  cudaStream_t st;
  cudaEvent_t stop = nullptr;
  // nfields = full-field copies the launch reads plus writes (its algorithmic traffic in units of F)
  LaunchTimer(mmf_plan* p_, int kclass, double nfields, cudaStream_t st_) : p(p_), st(st_) {
    if (!p->timing || p->ev_class.size() >= kMaxTimedLaunches) return;   // bounded: later launches go unrecorded
    cudaEvent_t a = nullptr;
    if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&stop) != cudaSuccess) { stop = nullptr; return; }
    p->ev.push_back(a);
    p->ev.push_back(stop);
    p->ev_class.push_back(kclass);
    p->ev_bytes.push_back(nfields * (double)p->field_bytes);
    cudaEventRecord(a, st);
  }
  ~LaunchTimer() {
    if (stop) cudaEventRecord(stop, st);
  }
};

// Every kernel of the propagation paths goes through here: with programmatic stream serialization the grid may start
// while its predecessor in the stream drains (its prologue — barrier init, tensor-memory allocation, constant tables —
// overlaps that tail; griddepcontrol.wait in the kernel orders everything that touches the predecessor's output).
// Off while per-launch events are being recorded (the events must bracket whole kernels).
template <class... KArgs, class... Args>
cudaError_t launch_kernel(const mmf_plan* p, void (*kern)(KArgs...), unsigned grid, unsigned block, size_t smem,
                          cudaStream_t st, Args&&... args) {
  cudaLaunchConfig_t cfg;
  memset(&cfg, 0, sizeof(cfg));
  cfg.gridDim = dim3(grid, 1, 1);
  cfg.blockDim = dim3(block, 1, 1);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = (p->pdl && !p->timing) ? 1 : 0;
  return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}

void clear_events(mmf_plan* p) {
  for (cudaEvent_t e : p->ev) cudaEventDestroy(e);
  p->ev.clear();
  p->ev_class.clear();
  p->ev_bytes.clear();
}

// cuTensorMapEncodeTiled through the runtime's driver entry point query (no link-time dependency on libcuda)
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn encode_tiled_fn() {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void* ptr = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ptr, cudaEnableDefault, &qres) == cudaSuccess &&
        qres == cudaDriverEntryPointSuccess)
      fn = (EncodeTiledFn)ptr;
  }
  return fn;
}

// 2-D tensor map of a field buffer seen as doubles [nrows_outer][2 * inner complex], box = (2 W doubles) x boxrows
int strided_tile_map(const void* base, cuuint64_t inner_cpx, cuuint64_t nrows_outer, int logw, cuuint32_t boxrows,
                     CUtensorMap* map) {
  EncodeTiledFn enc = encode_tiled_fn();
  if (!enc) {
    snprintf(g_cuda_msg, sizeof(g_cuda_msg), "CUDA error: cuTensorMapEncodeTiled is unavailable");
    return MMF_ECUDA;
  }
  const cuuint64_t gdim[2] = {2 * inner_cpx, nrows_outer};
  const cuuint64_t gstride[1] = {sizeof(cpx) * inner_cpx};
  const cuuint32_t box[2] = {(cuuint32_t)2 << logw, boxrows};
  const cuuint32_t estr[2] = {1, 1};
  const CUresult r = enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, const_cast<void*>(base), gdim, gstride, box, estr,
                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                         CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    snprintf(g_cuda_msg, sizeof(g_cuda_msg), "CUDA error: cuTensorMapEncodeTiled failed (%d)", (int)r);
    return MMF_ECUDA;
  }
  return MMF_OK;
}

// BLOCKED order (fft_kernels.cuh), the column tile of passes A / C: pitch rows of WB complex values, rows x N2/WB x N1
// of them; box = W adjacent columns x min(N1, 256) rows
int blocked_cols_map_build(const mmf_plan* p, const void* base, CUtensorMap* map) {
  const int logw = MMF_TILE_LOG - p->logn1, logwb = block_logw(p->logn1);
  return strided_tile_map(base, 1ULL << logwb, ((cuuint64_t)(2 * p->M)) << (p->logn2 - logwb + p->logn1), logw,
                          p->logn1 > 8 ? 256u : (1u << p->logn1), map);
}

// BLOCKED order, the chunk of pass B: pitch rows of one block (N1 WB complex values), rows x N2/WB of them;
// box = the WB values of one (block, p1) x min(N2/WB, 256) blocks
int blocked_rows_map_build(const mmf_plan* p, const void* base, CUtensorMap* map) {
  const int logwb = block_logw(p->logn1), lognb = p->logn2 - logwb;
  return strided_tile_map(base, 1ULL << (p->logn1 + logwb), ((cuuint64_t)(2 * p->M)) << lognb, logwb,
                          lognb > 8 ? 256u : (1u << lognb), map);
}

// ---- launch-plan caches --------------------------------------------------------------------------------------------
enum { MAP_COLS = 0, MAP_ROWS, MAP_TILE, MAP_TABLE, MAP_NATURAL };
int field_tile_map_build(const mmf_plan* p, const void* base, CUtensorMap* map, int boxrows);
int table_tile_map_build(const mmf_plan* p, const void* base, CUtensorMap* map);

// the tensor map of `kind` over the buffer at `base` (aux: box rows of MAP_TILE), encoded once per plan and buffer
int cached_map(mmf_plan* p, int kind, const void* base, int aux, CUtensorMap* out) {
  for (const auto& e : p->map_cache)
    if (e.kind == kind && e.base == base && e.aux == aux) {
      *out = e.map;
      return MMF_OK;
    }
  mmf_plan::MapEntry e;
  e.kind = kind; e.base = base; e.aux = aux;
  int rc = MMF_EINVAL;
  switch (kind) {
    case MAP_COLS: rc = blocked_cols_map_build(p, base, &e.map); break;
    case MAP_ROWS: rc = blocked_rows_map_build(p, base, &e.map); break;
    case MAP_TILE: rc = field_tile_map_build(p, base, &e.map, aux); break;
    case MAP_TABLE: rc = table_tile_map_build(p, base, &e.map); break;
    case MAP_NATURAL: {
      const int logwb = block_logw(p->logn1);
      rc = strided_tile_map(base, 1ULL << p->logn2, ((cuuint64_t)(2 * p->M)) << p->logn1, logwb,
                            1u << (MMF_TILE_LOG - logwb), &e.map);
      break;
    }
    default: break;
  }
  if (rc != MMF_OK) return rc;
  if (p->map_cache.size() >= 64) p->map_cache.erase(p->map_cache.begin());   // callers that cycle through many buffers
  p->map_cache.push_back(e);
  *out = e.map;
  return MMF_OK;
}
int blocked_cols_map(mmf_plan* p, const void* base, CUtensorMap* map) { return cached_map(p, MAP_COLS, base, 0, map); }
int blocked_rows_map(mmf_plan* p, const void* base, CUtensorMap* map) { return cached_map(p, MAP_ROWS, base, 0, map); }
int field_tile_map(mmf_plan* p, const void* base, CUtensorMap* map, int boxrows = 0) {
  return cached_map(p, MAP_TILE, base, boxrows, map);
}
int table_tile_map(mmf_plan* p, const void* base, CUtensorMap* map) { return cached_map(p, MAP_TABLE, base, 0, map); }

// cudaFuncAttributeMaxDynamicSharedMemorySize.  The attribute belongs to the (kernel, device) pair, not to a plan, and
// several kernels' dynamic shared memory depends on plan values (M, G, the shard sizes), so two live plans can share an
// instantiation with different needs.  The library therefore keeps, process-wide, the largest value it has set per
// kernel and device and only ever RAISES it: a launch with a smaller need is covered by the larger opt-in, and no plan
// can lower the limit under another one.  (A per-plan "done" flag is only a shortcut in front of the shared record.)
struct SmemAttr {
  const void* kern;
  int device;
  size_t bytes;
};
std::mutex g_smem_attr_mutex;
std::vector<SmemAttr> g_smem_attr;

template <class K>
int ensure_smem(mmf_plan* p, K kern, size_t smem) {
  const void* key = reinterpret_cast<const void*>(kern);
  std::lock_guard<std::mutex> lock(g_smem_attr_mutex);
  for (SmemAttr& a : g_smem_attr)
    if (a.kern == key && a.device == p->device) {
      if (smem <= a.bytes) return MMF_OK;
      CU(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
      a.bytes = smem;
      return MMF_OK;
    }
  CU(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  g_smem_attr.push_back({key, p->device, smem});
  return MMF_OK;
}
template <class K>
int cached_occupancy(mmf_plan* p, K kern, int threads, size_t smem, int* occ) {
  const void* key = reinterpret_cast<const void*>(kern);
  for (const auto& e : p->occ_cache)
    if (e.kern == key && e.threads == threads && e.smem == smem) {
      *occ = e.occ;
      return MMF_OK;
    }
  CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(occ, kern, threads, smem));
  p->occ_cache.push_back({key, threads, smem, *occ});
  return MMF_OK;
}
#define MMF_ENSURE_SMEM(kern, smem)                          \
  do {                                                       \
    const int rc__ = ensure_smem(p, kern, smem);             \
    if (rc__ != MMF_OK) return rc__;                         \
  } while (0)

// ---- launch helpers ----------------------------------------------------------------------------------------------
template <int LOGN1, int DIR>
int launch_cols_t(mmf_plan* p, cpx* X0, cpx* X1, int nbuf, cudaStream_t st) {
  constexpr size_t smem = cols_smem_bytes<LOGN1>();
  constexpr int LOGW = MMF_TILE_LOG - LOGN1;
  auto kern = k_cols<LOGN1, DIR, kGroups>;
  MMF_ENSURE_SMEM(kern, smem);
  ColsParams q;
  q.twtab = p->d_tw1; q.ipt = p->d_ipt;
  q.logn2 = p->logn2; q.logwb = block_logw(LOGN1); q.nrows = 2 * p->M; q.nbuf = nbuf;
  CUtensorMap map0, map1;
  int rc;
  if ((rc = blocked_cols_map(p, X0, &map0)) != MMF_OK) return rc;
  if ((rc = blocked_cols_map(p, nbuf > 1 ? X1 : X0, &map1)) != MMF_OK) return rc;
  const long long tiles = ((long long)nbuf * 2 * p->M) << (p->logn2 - LOGW);
  long long grid = tiles < p->num_sms ? tiles : p->num_sms;
  if (p->dry_run) return MMF_OK;
  LaunchTimer lt(p, DIR == 0 ? KC_COLS_FWD : KC_COLS_INV, 2 * nbuf, st);
  CU(launch_kernel(p, kern, (unsigned)grid, MMF_GROUP_THREADS * kGroups, smem, st, map0, map1, q));
  p->launches++;
  return MMF_OK;
}

template <int DIR>
int launch_cols(mmf_plan* p, cpx* X0, cpx* X1, int nbuf, cudaStream_t st) {
  switch (p->logn1) {
#ifndef MMF_LEAN_BUILD   // MMF_LEAN_BUILD: config-4 instantiations only (quick builds for kernel experiments)
    case 6: return launch_cols_t<6, DIR>(p, X0, X1, nbuf, st);
    case 8: return launch_cols_t<8, DIR>(p, X0, X1, nbuf, st);
    case 12: return launch_cols_t<12, DIR>(p, X0, X1, nbuf, st);
#endif
    case 10: return launch_cols_t<10, DIR>(p, X0, X1, nbuf, st);
    default: return MMF_EINVAL;
  }
}

// X0 / X1: the field buffers (tiled order unless SINGLE); OUT: MODE 1 only, receives the slot-order spectrum
template <int LOGN2, int MODE, bool SINGLE>
int launch_rows_t(mmf_plan* p, cpx* X0, cpx* X1, int nbuf, cpx* OUT, cudaStream_t st) {
  constexpr size_t smem = rows_smem_bytes<LOGN2>();
  constexpr int LOGB = MMF_TILE_LOG - LOGN2;
  auto kern = k_rows<LOGN2, MODE, SINGLE, kGroups>;
  MMF_ENSURE_SMEM(kern, smem);
  RowsParams q;
  q.X0 = X0; q.X1 = nbuf > 1 ? X1 : X0; q.OUT = OUT; q.E = p->E; q.twtab = p->d_tw2;
  CUtensorMap map0, map1;
  memset(&map0, 0, sizeof(map0));
  memset(&map1, 0, sizeof(map1));
  if (!SINGLE) {
    int rc;
    if ((rc = blocked_rows_map(p, q.X0, &map0)) != MMF_OK) return rc;
    if ((rc = blocked_rows_map(p, q.X1, &map1)) != MMF_OK) return rc;
  }
  q.nchunks = (2LL * p->M) << p->logn1;
  q.logn1 = p->logn1; q.nbuf = nbuf; q.M = p->M;
  const long long items = SINGLE ? ((q.nchunks + (1 << LOGB) - 1) >> LOGB) : ((long long)p->M << (p->logn1 - LOGB));
  long long grid = items < p->num_sms ? items : p->num_sms;
  if (p->dry_run) return MMF_OK;
  LaunchTimer lt(p, KC_ROWS, 2 * nbuf, st);
  CU(launch_kernel(p, kern, (unsigned)grid, MMF_GROUP_THREADS * kGroups, smem, st, map0, map1, q));
  p->launches++;
  return MMF_OK;
}

template <int MODE>
int launch_rows(mmf_plan* p, cpx* X0, cpx* X1, int nbuf, cpx* OUT, cudaStream_t st) {
  if (p->logn1 == 0) {
    switch (p->logn2) {
#define MMF_ROWS_CASE(L) case L: return launch_rows_t<L, MODE, true>(p, X0, X1, nbuf, OUT, st);
#ifndef MMF_LEAN_BUILD
      MMF_ROWS_CASE(4) MMF_ROWS_CASE(5) MMF_ROWS_CASE(6) MMF_ROWS_CASE(7) MMF_ROWS_CASE(8) MMF_ROWS_CASE(9)
      MMF_ROWS_CASE(10) MMF_ROWS_CASE(11)
#endif
      MMF_ROWS_CASE(12)
#undef MMF_ROWS_CASE
      default: return MMF_EINVAL;
    }
  }
  switch (p->logn2) {
#define MMF_ROWS_CASE(L) case L: return launch_rows_t<L, MODE, false>(p, X0, X1, nbuf, OUT, st);
#ifndef MMF_LEAN_BUILD
    MMF_ROWS_CASE(6) MMF_ROWS_CASE(7) MMF_ROWS_CASE(8) MMF_ROWS_CASE(9) MMF_ROWS_CASE(10) MMF_ROWS_CASE(11)
#endif
    MMF_ROWS_CASE(12)
#undef MMF_ROWS_CASE
    default: return MMF_EINVAL;
  }
}

// D on one or two full-field buffers: exp(h/2 L) in place (rows a1-a3 of the hot path).  For N > 4096 the buffers are
// in the BLOCKED order (fft_kernels.cuh); to_tiled / to_natural convert on the way in and out of a propagation.
int apply_D(mmf_plan* p, cpx* X0, cpx* X1, int nbuf, cudaStream_t st) {
  int rc;
  if (p->logn1 > 0 && (rc = launch_cols<0>(p, X0, X1, nbuf, st)) != MMF_OK) return rc;
  if ((rc = launch_rows<0>(p, X0, X1, nbuf, nullptr, st)) != MMF_OK) return rc;
  if (p->logn1 > 0 && (rc = launch_cols<1>(p, X0, X1, nbuf, st)) != MMF_OK) return rc;
  return MMF_OK;
}

// DIR 0: blocked <- natural (out of place);  DIR 1: natural <- blocked.  Only for N > 4096 (logn1 > 0).
template <int DIR>
int launch_perm(mmf_plan* p, cpx* natural, cpx* blocked, cudaStream_t st) {
  constexpr size_t smem = 3 * (sizeof(cpx) << MMF_TILE_LOG) + 64;
  auto kern = k_perm<DIR>;
  MMF_ENSURE_SMEM(kern, smem);
  const int logwb = block_logw(p->logn1);
  CUtensorMap mapn;  // natural order: memory rows of N2 values, box = one block's WB columns x 4096 / WB rows
  int rc;
  if ((rc = cached_map(p, MAP_NATURAL, natural, 0, &mapn)) != MMF_OK) return rc;
  PermParams q;
  q.blocked = blocked; q.logn1 = p->logn1; q.logn2 = p->logn2; q.logwb = logwb; q.nrows = 2 * p->M;
  const long long tiles = ((long long)2 * p->M) << (p->logn1 + p->logn2 - MMF_TILE_LOG);
  long long grid = tiles < p->num_sms ? tiles : p->num_sms;
  if (p->dry_run) return MMF_OK;
  LaunchTimer lt(p, KC_PERM, 2, st);
  CU(launch_kernel(p, kern, (unsigned)grid, 32, smem, st, mapn, q));
  p->launches++;
  return MMF_OK;
}
int to_tiled(mmf_plan* p, cpx* natural, cpx* tiled, cudaStream_t st) { return launch_perm<0>(p, natural, tiled, st); }
int to_natural(mmf_plan* p, cpx* tiled, cpx* natural, cudaStream_t st) { return launch_perm<1>(p, natural, tiled, st); }

size_t nl_smem_bytes(const mmf_plan* p) { return sizeof(double) * 2 * (size_t)p->M * MMF_NL_T; }

template <int MODE>
int launch_nl(mmf_plan* p, cpx* X, cpx* Y, cpx* Z, cpx* W, cudaStream_t st, double gain = 1.0) {
  auto kern = k_nl<MODE>;
  const size_t smem = nl_smem_bytes(p);
  MMF_ENSURE_SMEM(kern, smem);
  NlParams q;
  q.X = X; q.Y = Y; q.Z = Z; q.W = W;
  q.kappa = p->d_kappa;
  q.hg = p->h * p->gamma;
  q.gain = gain;
  q.M = p->M;
  q.N = p->N;
  const unsigned grid = (unsigned)((p->N + MMF_NL_T - 1) / MMF_NL_T);
  if (p->dry_run) return MMF_OK;
  LaunchTimer lt(p, KC_NL_PLAIN + MODE, MODE == NL_PLAIN ? 2 : MODE == NL_STAGE2 ? 3 : MODE == NL_STAGE3 ? 5 : MODE == NL_FINAL ? 3 : 4, st);
  CU(launch_kernel(p, kern, grid, MMF_NL_T * MMF_NL_WARPS, smem, st, q));
  p->launches++;
  return MMF_OK;
}

// ---- fused nonlinear kernel on the fp64 tensor path (M <= MMF_NLM_MAXM) ------------------------------------------
constexpr int kNlmNk[] = {1, 2, 3, 4, 6, 8, 9, 12, 16, 20, 24, 28, 30, 32};

int nlm_pick_nk(int M) {
  const int need = (M + 3) / 4;
  for (int nk : kNlmNk)
    if (nk >= need) return nk;
  return -1;
}

// tensor map of a field buffer [2M][N] complex128 seen as doubles [2M][2N], box = (8 samples = 16 doubles) x 2M rows
int field_tile_map_build(const mmf_plan* p, const void* base, CUtensorMap* map, int boxrows) {
  EncodeTiledFn enc = encode_tiled_fn();
  if (!enc) {
    snprintf(g_cuda_msg, sizeof(g_cuda_msg), "CUDA error: cuTensorMapEncodeTiled is unavailable");
    return MMF_ECUDA;
  }
  const cuuint64_t gdim[2] = {(cuuint64_t)(2 * p->N), (cuuint64_t)(2 * p->M)};
  const cuuint64_t gstride[1] = {(cuuint64_t)p->N * sizeof(cpx)};
  const cuuint32_t box[2] = {2 * MMF_NLM_T, (cuuint32_t)(boxrows > 0 ? boxrows : 2 * p->M)};
  const cuuint32_t estr[2] = {1, 1};
  const CUresult r = enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, const_cast<void*>(base), gdim, gstride, box, estr,
                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                         CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    snprintf(g_cuda_msg, sizeof(g_cuda_msg), "CUDA error: cuTensorMapEncodeTiled failed (%d)", (int)r);
    return MMF_ECUDA;
  }
  return MMF_OK;
}

// tensor map of the real table T [M][N] doubles (the SSFM-Agrawal modes), box = 8 samples x M rows
int table_tile_map_build(const mmf_plan* p, const void* base, CUtensorMap* map) {
  EncodeTiledFn enc = encode_tiled_fn();
  if (!enc) {
    snprintf(g_cuda_msg, sizeof(g_cuda_msg), "CUDA error: cuTensorMapEncodeTiled is unavailable");
    return MMF_ECUDA;
  }
  const cuuint64_t gdim[2] = {(cuuint64_t)p->N, (cuuint64_t)p->M};
  const cuuint64_t gstride[1] = {(cuuint64_t)p->N * sizeof(double)};
  const cuuint32_t box[2] = {MMF_NLM_T, (cuuint32_t)p->M};
  const cuuint32_t estr[2] = {1, 1};
  const CUresult r = enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, const_cast<void*>(base), gdim, gstride, box, estr,
                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                         CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    snprintf(g_cuda_msg, sizeof(g_cuda_msg), "CUDA error: cuTensorMapEncodeTiled failed (%d)", (int)r);
    return MMF_ECUDA;
  }
  return MMF_OK;
}

// PLAIN: A = U, B = OUT; ENTER: A = the caller's field (natural order), B = X, C = Y; EXIT: A = X, B = Y, C = the
// caller's field; AGR_*: A = X, B = Y, C = the real table T; other modes: A = X, B = Y (C unused).
template <int NK, int MODE>
int launch_nlm_t(mmf_plan* p, const cpx* A, cpx* B, cpx* C, cudaStream_t st, double gain) {
  constexpr int NARR = nlm_narr<MODE>();
  // mode groups: the grouped kernel where its extra S rows still fit beside the ring (they do not for the largest
  // three-array split-step slots at M = 120 with many groups: those launches contract the dense matrix)
  const bool grouped = p->G > 0 && nlt_smem_bytes(p->M, NK, NARR, nlm_has_table<MODE>(), p->G) <= 227 * 1024;
  auto kern = grouped ? k_nlt<NK, MODE, 1> : k_nlt<NK, MODE, 0>;
  NltParams q;
  q.kappa = grouped ? p->d_kappa_g : p->d_kappa;
  q.group_of = p->d_group_of;
  q.G = grouped ? p->G : 0;
  q.hg = p->h * p->gamma;
  q.gain = gain;
  q.M = p->M;
  q.NW = (p->M + 7) / 8;
  q.ntiles = p->N / MMF_NLM_T;
  q.logn1 = p->logn1; q.logn2 = p->logn2; q.logwb = block_logw(p->logn1);
  CUtensorMap mapA, mapB, mapC;
  int rc;
  if ((rc = field_tile_map(p, A, &mapA)) != MMF_OK) return rc;
  if ((rc = field_tile_map(p, B, &mapB)) != MMF_OK) return rc;
  if constexpr (nlm_has_table<MODE>()) {
    if (!C) return MMF_EINVAL;
    if ((rc = table_tile_map(p, C, &mapC)) != MMF_OK) return rc;
  } else if ((rc = field_tile_map(p, C ? C : B, &mapC)) != MMF_OK) return rc;
  const size_t smem = nlt_smem_bytes(p->M, NK, NARR, nlm_has_table<MODE>(), q.G);
  const int threads = 32 * (q.NW + 1);
  MMF_ENSURE_SMEM(kern, smem);
  int occ = 1;
  if ((rc = cached_occupancy(p, kern, threads, smem, &occ)) != MMF_OK) return rc;
  if (occ < 1) return MMF_EINVAL;
  long long grid = (long long)p->num_sms * occ;        // persistent: every resident CTA walks its own tile list
  if (grid > q.ntiles) grid = q.ntiles;
  constexpr double kFields = (MODE == NLM_PLAIN || MODE == NLM_RK4) ? 2 : (MODE == NLM_S23 || MODE == NLM_FINAL_NEXT) ? 4
                             : MODE == NLM_AGR_S0 ? 1.25 : MODE == NLM_AGR_IT1 ? 2.25 : MODE == NLM_AGR_ITJ ? 3.25 : 3;
  if (p->dry_run) return MMF_OK;
  LaunchTimer lt(p, KC_NLM_PLAIN + MODE, kFields, st);
  CU(launch_kernel(p, kern, (unsigned)grid, (unsigned)threads, smem, st, mapA, mapB, mapC, q));
  p->launches++;
  return MMF_OK;
}

template <int MODE>
int launch_nlm(mmf_plan* p, const cpx* A, cpx* B, cudaStream_t st, cpx* C = nullptr, double gain = 1.0) {
  switch (p->nlm_nk) {
#define MMF_NLM_CASE(NKV) case NKV: return launch_nlm_t<NKV, MODE>(p, A, B, C, st, gain);
#ifndef MMF_LEAN_BUILD
    MMF_NLM_CASE(2) MMF_NLM_CASE(3) MMF_NLM_CASE(4) MMF_NLM_CASE(6) MMF_NLM_CASE(8) MMF_NLM_CASE(9)
    MMF_NLM_CASE(12) MMF_NLM_CASE(16) MMF_NLM_CASE(20) MMF_NLM_CASE(24) MMF_NLM_CASE(28)
    MMF_NLM_CASE(32)
#endif
    MMF_NLM_CASE(1) MMF_NLM_CASE(30)
#undef MMF_NLM_CASE
    default: return MMF_EINVAL;
  }
}

// a plan's tables, workspace and tensor maps belong to one device: refuse calls made with another one current
bool on_plan_device(const mmf_plan* p) {
  int dev = -1;
  return cudaGetDevice(&dev) == cudaSuccess && dev == p->device;
}

// ---- general per-polarisation coupling (k_nlg): F0 / F1 full-tile inputs, Hin own-rows input, Ho0 / Ho1 outputs ------
template <int MODE>
int launch_nlg(mmf_plan* p, const cpx* F0, const cpx* F1, const cpx* Hin, cpx* Ho0, cpx* Ho1, cudaStream_t st,
               double gain = 1.0) {
  auto kern = k_nlg<MODE>;
  NlgParams q;
  q.kappa2 = p->d_kappa;
  q.hg = p->h * p->gamma;
  q.gain = gain;
  q.M = p->M;
  q.NW = (p->M + 7) / 8;
  q.nchunk = (2 * p->M + 15) / 16;
  q.ntiles = p->N / MMF_NLM_T;
  CUtensorMap mF0, mF1, mHin, mHo0, mHo1;
  int rc;
  if ((rc = field_tile_map(p, F0, &mF0)) != MMF_OK) return rc;
  if ((rc = field_tile_map(p, F1 ? F1 : F0, &mF1)) != MMF_OK) return rc;
  if ((rc = field_tile_map(p, Hin ? Hin : F0, &mHin, p->M)) != MMF_OK) return rc;
  if ((rc = field_tile_map(p, Ho0, &mHo0, p->M)) != MMF_OK) return rc;
  if ((rc = field_tile_map(p, Ho1 ? Ho1 : Ho0, &mHo1, p->M)) != MMF_OK) return rc;
  const size_t smem = nlg_smem_bytes(p->M, q.nchunk, nlg_nfull<MODE>(), nlg_half_in<MODE>());
  MMF_ENSURE_SMEM(kern, smem);
  long long pairs = p->num_sms / 2;                      // persistent: CTA pairs (the two halves of the rows)
  if (pairs > q.ntiles) pairs = q.ntiles;
  if (pairs < 1) pairs = 1;
  constexpr double kFields = MODE == NLG_PLAIN ? 2 : MODE == NLG_STAGE2 ? 3 : MODE == NLG_STAGE3 ? 5 : 3;
  if (p->dry_run) return MMF_OK;
  LaunchTimer lt(p, KC_NLG_PLAIN + MODE, kFields, st);
  CU(launch_kernel(p, kern, (unsigned)(2 * pairs), (unsigned)(32 * (q.NW + 1)), smem, st, mF0, mF1, mHin, mHo0, mHo1, q));
  p->launches++;
  return MMF_OK;
}

// The whole propagation in one cluster kernel (small_cluster.cuh): N = 4096, M <= MMF_SMALL_MAXM, Manakov kappa.
typedef void (*SmallKernel)(SmallParams);
SmallKernel small_kernel(int M) {
  switch (M) {
    case 1: return k_small<1>;
    case 2: return k_small<2>;
    case 3: return k_small<3>;
    case 4: return k_small<4>;
    default: return nullptr;
  }
}
bool small_cluster_usable(mmf_plan* p) {
  if (p->small_cluster >= 0) return p->small_cluster == 1;
  p->small_cluster = 0;
  const char* e = getenv("MMF_SMALL_CLUSTER");
  if (e && e[0] == '0') return false;
  if (p->logn != MMF_SMALL_LOGN || p->M > MMF_SMALL_MAXM || p->general || p->M_total > 0) return false;
  const int T = 4 * p->M;
  SmallKernel k_small = small_kernel(p->M);
  if (cudaFuncSetAttribute(k_small, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)small_smem_bytes()) != cudaSuccess ||
      (T > 8 && cudaFuncSetAttribute(k_small, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) != cudaSuccess)) {
    cudaGetLastError();
    return false;
  }
  cudaLaunchConfig_t cfg;
  memset(&cfg, 0, sizeof(cfg));
  cfg.gridDim = dim3(T, 1, 1);
  cfg.blockDim = dim3(MMF_SMALL_THREADS, 1, 1);
  cfg.dynamicSmemBytes = small_smem_bytes();
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = T; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  int nclusters = 0;
  if (cudaOccupancyMaxActiveClusters(&nclusters, k_small, &cfg) != cudaSuccess || nclusters < 1) {
    cudaGetLastError();
    return false;
  }
  p->small_cluster = 1;
  return true;
}

int launch_small(mmf_plan* p, cpx* A, int nsteps, int span, double gain, cudaStream_t st) {
  SmallParams q;
  q.A = A; q.E = p->E; q.twtab = p->d_tw2; q.kappa = p->d_kappa;
  q.hg = p->h * p->gamma; q.gain = gain;
  q.M = p->M; q.nsteps = nsteps; q.span = span;
  const int T = 4 * p->M;
  cudaLaunchConfig_t cfg;
  memset(&cfg, 0, sizeof(cfg));
  cfg.gridDim = dim3(T, 1, 1);
  cfg.blockDim = dim3(MMF_SMALL_THREADS, 1, 1);
  cfg.dynamicSmemBytes = small_smem_bytes();
  cfg.stream = st;
  cudaLaunchAttribute attr[2];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = T; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
  attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[1].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = (p->pdl && !p->timing) ? 2 : 1;
  LaunchTimer lt(p, KC_SMALL, 2, st);
  CU(cudaLaunchKernelEx(&cfg, small_kernel(p->M), q));
  p->launches++;
  return MMF_OK;
}

bool finite_all(const double* v, size_t n) {
  for (size_t i = 0; i < n; ++i)
    if (!std::isfinite(v[i])) return false;
  return true;
}

void free_tables(mmf_plan* p) {
  clear_events(p);
  for (auto& g : p->graphs) cudaGraphExecDestroy(g.exec);
  p->graphs.clear();
  if (p->cap_stream) cudaStreamDestroy(p->cap_stream);
  p->cap_stream = nullptr;
  cudaFree(p->d_kappa);
  cudaFree(p->d_kappa_g);
  cudaFree(p->d_group_of);
  cudaFree(p->d_tw1);
  cudaFree(p->d_tw2);
  cudaFree(p->d_ipt);
  cudaFree(p->d_coefs);
}

}  // namespace

namespace {
template <int STAGE>
int launch_shard(mmf_plan* p, bool pow, double* P_all, long long t_first, long long t_count, double gain, cudaStream_t st) {
  ShardParams q;
  q.X = p->shard_X; q.Y = p->Y; q.Z = p->Z; q.W = p->W;
  q.kappa_rows = p->d_kappa; q.P_all = P_all;
  q.hg = p->h * p->gamma; q.gain = gain;
  q.M_local = p->M; q.M_total = p->M_total; q.mode0 = p->mode0; q.N = p->N;
  q.t_first = t_first; q.t_count = t_count;
  const double frac = (double)t_count / (double)p->N;   // of the launch's full-axis traffic
  const unsigned grid = (unsigned)((t_count + MMF_SH_T - 1) / MMF_SH_T);
  if (pow) {
    LaunchTimer lt(p, KC_SHARD_POW, frac * (STAGE == SH_PLAIN || STAGE == SH_FINAL ? 1.0 : 2.0), st);
    CU(launch_kernel(p, k_shard_pow<STAGE>, grid, MMF_SH_T * MMF_SH_WARPS, 0, st, q));
  } else {
    const size_t smem = shard_apply_smem_bytes(p->M, p->M_total);
    if (smem > 227 * 1024) return MMF_EINVAL;
    auto kern = k_shard_apply<STAGE>;
    MMF_ENSURE_SMEM(kern, smem);
    int occ = 1;
    int rc = cached_occupancy(p, kern, MMF_SH_T * MMF_SH_WARPS, smem, &occ);
    if (rc != MMF_OK) return rc;
    if (occ < 1) return MMF_EINVAL;
    unsigned pgrid = (unsigned)(p->num_sms * occ);   // persistent: kappa goes to shared memory once per CTA
    if (pgrid > grid) pgrid = grid;
    LaunchTimer lt(p, KC_SHARD_APPLY, frac * (STAGE == SH_PLAIN ? 2 : STAGE == SH_STAGE2 ? 3 : STAGE == SH_STAGE3 ? 5 : 3), st);
    CU(launch_kernel(p, kern, pgrid, MMF_SH_T * MMF_SH_WARPS, smem, st, q));
  }
  p->launches++;
  return MMF_OK;
}
int shard_stage(mmf_plan* p, int stage, bool pow, double* P_all, long long t_first, long long t_count, double gain,
                cudaStream_t st) {
  if (t_first < 0 || t_count < 1 || t_first + t_count > p->N) return MMF_EINVAL;
  switch (stage) {
    case SH_PLAIN: return launch_shard<SH_PLAIN>(p, pow, P_all, t_first, t_count, gain, st);
    case SH_STAGE2: return launch_shard<SH_STAGE2>(p, pow, P_all, t_first, t_count, gain, st);
    case SH_STAGE3: return launch_shard<SH_STAGE3>(p, pow, P_all, t_first, t_count, gain, st);
    case SH_FINAL: return launch_shard<SH_FINAL>(p, pow, P_all, t_first, t_count, gain, st);
    default: return MMF_EINVAL;
  }
}
bool shard_ready(const mmf_plan* p) { return p && p->M_total > 0 && p->ws && on_plan_device(p); }
}  // namespace

namespace mmf {
// For the library's other translation units (nl_static.cu): keep the text of a CUDA error for mmf_status_string.
int note_cuda_error(cudaError_t e) { return cuda_fail(e); }
}  // namespace mmf

extern "C" {

const char* mmf_version(void) { return "mmf-b200 0.1"; }

const char* mmf_status_string(int status) {
  switch (status) {
    case MMF_OK: return "ok";
    case MMF_EINVAL: return "invalid argument";
    case MMF_ENOMEM: return "out of memory";
    case MMF_ECUDA: return g_cuda_msg;
    case MMF_ETOOBIG: return "problem too large for the static scratch array (M * N * 8 > MMF_STATIC_SCRATCH_BYTES)";
    default: return "unknown status";
  }
}

static int plan_create_impl(mmf_plan** out, int M, long long N, double dt, double h, double alpha, const double* beta,
                            int K, double gamma, const double* kappa, bool general, int M_total = 0, int mode0 = 0);

int mmf_plan_create(mmf_plan** out, int M, long long N, double dt, double h, double alpha, const double* beta, int K,
                    double gamma, const double* kappa) {
  return plan_create_impl(out, M, N, dt, h, alpha, beta, K, gamma, kappa, false);
}

int mmf_plan_create_general(mmf_plan** out, int M, long long N, double dt, double h, double alpha, const double* beta,
                            int K, double gamma, const double* kappa2) {
  return plan_create_impl(out, M, N, dt, h, alpha, beta, K, gamma, kappa2, true);
}

int mmf_plan_create_shard(mmf_plan** out, int M_local, int M_total, int mode0, long long N, double dt, double h,
                          double alpha, const double* beta, int K, double gamma, const double* kappa_rows) {
  if (M_local < 1 || mode0 < 0 || M_total < M_local || mode0 + M_local > M_total) return MMF_EINVAL;
  return plan_create_impl(out, M_local, N, dt, h, alpha, beta, K, gamma, kappa_rows, false, M_total, mode0);
}

static int plan_create_impl(mmf_plan** out, int M, long long N, double dt, double h, double alpha, const double* beta,
                            int K, double gamma, const double* kappa, bool general, int M_total, int mode0) {
  if (!out) return MMF_EINVAL;
  *out = nullptr;
  if (!beta || !kappa || M < 1 || K < 1 || K > MMF_MAXK) return MMF_EINVAL;
  if (N < 16 || N > (1LL << 24) || (N & (N - 1)) != 0) return MMF_EINVAL;
  if (!(dt > 0) || !std::isfinite(dt) || !std::isfinite(h) || !std::isfinite(alpha) || !std::isfinite(gamma))
    return MMF_EINVAL;
  const bool shard = M_total > 0;
  const size_t KD = general ? 2 * (size_t)M : (size_t)M;   // kappa is KD x KC
  const size_t KC = shard ? (size_t)M_total : KD;
  if (general && M > MMF_NLG_MAXM) return MMF_EINVAL;       // the general kernel keeps an M x 2M slab in tensor memory
  if (!finite_all(beta, (size_t)M * K) || !finite_all(kappa, KD * KC)) return MMF_EINVAL;
  if (sizeof(double) * 2 * KC * MMF_NL_T > 227 * 1024) return MMF_EINVAL;  // mode-power tile must fit one SM
  // a shard plan's apply kernel keeps the rank's kappa rows, a power tile and a result tile in one SM's shared memory:
  // refuse here, not at the first mmf_shard_apply in the middle of a step (include/mmf.h states the bound)
  if (shard && shard_apply_smem_bytes(M, M_total) > 227 * 1024) return MMF_EINVAL;
  mmf_plan* p = new (std::nothrow) mmf_plan;
  if (!p) return MMF_ENOMEM;
  p->M = M; p->K = K; p->N = N; p->dt = dt; p->h = h; p->alpha = alpha; p->gamma = gamma;
  p->beta.assign(beta, beta + (size_t)M * K);
  p->kappa.assign(kappa, kappa + KD * KC);
  p->general = general;
  p->M_total = M_total;
  p->mode0 = mode0;
  {
    const char* e = getenv("MMF_PDL");
    if (e && e[0] == '0') p->pdl = false;
  }
  int logn = 0;
  while ((1LL << logn) < N) ++logn;
  p->logn = logn;
  // N = N1 N2: pass B (the FP64- and L1-heaviest pass: two transforms) gets the shorter transform where possible
  if (logn <= MMF_TILE_LOG) p->logn1 = 0;
  else if (logn == 13) p->logn1 = 6;
  else if (logn <= 15) p->logn1 = 8;
  else if (logn <= 20) p->logn1 = 8;   // N2 <= 2^12; the 256-byte segments of W = 16 columns stream best
  else if (logn <= 22) p->logn1 = 10;
  else p->logn1 = 12;
  p->logn2 = logn - p->logn1;
  p->nlm_nk = (!general && !shard && M <= MMF_NLM_MAXM) ? nlm_pick_nk(M) : -1;   // shard plans: four-buffer plan
  {
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) == cudaSuccess) p->device = dev;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && sms > 0) p->num_sms = sms;
  }
  p->field_bytes = sizeof(cpx) * 2 * (size_t)M * (size_t)N;
  int rc = MMF_OK;
  do {
    cudaError_t e = cudaMalloc((void**)&p->d_kappa, sizeof(double) * KD * KC);
    if (e != cudaSuccess) { rc = (e == cudaErrorMemoryAllocation) ? MMF_ENOMEM : cuda_fail(e); break; }
    e = cudaMemcpy(p->d_kappa, kappa, sizeof(double) * KD * KC, cudaMemcpyHostToDevice);
    if (e != cudaSuccess) { rc = cuda_fail(e); break; }
    if (p->nlm_nk > 0) {
      // mode groups: if kappa has few DISTINCT rows (exact equality), the contraction runs on those (nl_tma.cuh GROUPED)
      const char* eg = getenv("MMF_GROUPED");
      std::vector<int> group_of(M), rep;
      for (int a = 0; a < M; ++a) {
        int gfound = -1;
        for (size_t gi = 0; gi < rep.size() && gfound < 0; ++gi)
          if (memcmp(kappa + (size_t)a * M, kappa + (size_t)rep[gi] * M, sizeof(double) * M) == 0) gfound = (int)gi;
        if (gfound < 0) {
          gfound = (int)rep.size();
          rep.push_back(a);
        }
        group_of[a] = gfound;
      }
      const int G = (int)rep.size();
      if (!(eg && eg[0] == '0') && G <= MMF_NLM_MAXG && 2 * G <= M) {
        std::vector<double> kg((size_t)G * M);
        for (int gi = 0; gi < G; ++gi) memcpy(kg.data() + (size_t)gi * M, kappa + (size_t)rep[gi] * M, sizeof(double) * M);
        e = cudaMalloc((void**)&p->d_kappa_g, sizeof(double) * kg.size());
        if (e != cudaSuccess) { rc = (e == cudaErrorMemoryAllocation) ? MMF_ENOMEM : cuda_fail(e); break; }
        e = cudaMemcpy(p->d_kappa_g, kg.data(), sizeof(double) * kg.size(), cudaMemcpyHostToDevice);
        if (e != cudaSuccess) { rc = cuda_fail(e); break; }
        e = cudaMalloc((void**)&p->d_group_of, sizeof(int) * M);
        if (e != cudaSuccess) { rc = (e == cudaErrorMemoryAllocation) ? MMF_ENOMEM : cuda_fail(e); break; }
        e = cudaMemcpy(p->d_group_of, group_of.data(), sizeof(int) * M, cudaMemcpyHostToDevice);
        if (e != cudaSuccess) { rc = cuda_fail(e); break; }
        p->G = G;
      }
    }
    if ((rc = upload_stage_tables(&p->d_tw2, p->logn2)) != MMF_OK) break;
    if (p->logn1 > 0) {
      if ((rc = upload_stage_tables(&p->d_tw1, p->logn1)) != MMF_OK) break;
      // inter-pass table (fft_kernels.cuh): per column tile, W_N^(k1(pos0(t)) n2(t)) for the 256 threads of a group
      // and the steps W_N^(wA n2), W_N^(wB n2) of the exponent along the registers of the last pass-A stage
      const int nst1 = nstages(p->logn1), lrl = last_lr(p->logn1, nst1), lrp = prev_lr(p->logn1, nst1);
      const long long wA = 1LL << (p->logn1 - lrl);
      const long long wB = (lrl == 4) ? 8 * wA : 1LL << (p->logn1 - lrl - lrp);
      if (lrl < 3 || lrl > 4) { rc = MMF_EINVAL; break; }
      const int logw = MMF_TILE_LOG - p->logn1, W = 1 << logw, ipt = ipt_row_entries(logw);
      const long long nct = 1LL << (p->logn2 - logw);
      std::vector<cpx> h((size_t)nct * ipt);
      for (long long ct = 0; ct < nct; ++ct) {
        cpx* row = h.data() + (size_t)ct * ipt;
        for (int t = 0; t < 256; ++t) {
          const long long k1 = slot_to_bin_rt(p->logn1, 16 * (t >> logw)), n2 = ct * W + (t & (W - 1));
          root_of_unity(k1 * n2, N, &row[t].x, &row[t].y);
        }
        for (int c = 0; c < W; ++c) {
          root_of_unity(wA * (ct * W + c), N, &row[256 + c].x, &row[256 + c].y);
          root_of_unity(wB * (ct * W + c), N, &row[256 + W + c].x, &row[256 + W + c].y);
        }
      }
      cudaError_t e2 = cudaMalloc((void**)&p->d_ipt, sizeof(cpx) * h.size());
      if (e2 != cudaSuccess) { rc = (e2 == cudaErrorMemoryAllocation) ? MMF_ENOMEM : cuda_fail(e2); break; }
      e2 = cudaMemcpy(p->d_ipt, h.data(), sizeof(cpx) * h.size(), cudaMemcpyHostToDevice);
      if (e2 != cudaSuccess) { rc = cuda_fail(e2); break; }
    }
    // per-mode phase coefficients hh * beta_n / n! in double-double (hh = h/2, Eq. 6a)
    std::vector<dd> coefs((size_t)M * K);
    for (int a = 0; a < M; ++a) {
      double fact = 1.0;
      for (int n = 0; n < K; ++n) {
        if (n > 0) fact *= n;
        coefs[(size_t)a * K + n] = dd_div_d(dd_two_prod(0.5 * h, beta[(size_t)a * K + n]), fact);
      }
    }
    e = cudaMalloc((void**)&p->d_coefs, sizeof(dd) * coefs.size());
    if (e != cudaSuccess) { rc = cuda_fail(e); break; }
    e = cudaMemcpy(p->d_coefs, coefs.data(), sizeof(dd) * coefs.size(), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) { rc = cuda_fail(e); break; }
  } while (0);
  if (rc != MMF_OK) {
    free_tables(p);
    delete p;
    return rc;
  }
  *out = p;
  return MMF_OK;
}

size_t mmf_plan_workspace_bytes(const mmf_plan* p) {
  if (!p) return 0;
  const size_t F = align_up(p->field_bytes, 256);
  const size_t E = align_up(sizeof(cpx) * (size_t)p->M * (size_t)p->N, 256);
  // tensor-path plan: one more field buffer; DFMA plan (M > 120): three, plus one to hold the field in tiled order
  // (N > 4096, tensor path: two, the field and the second buffer both live in the workspace in blocked order)
  // N <= 4096 (field sizes of KiB..MiB): also the real table T [M][N] of mmf_propagate_ssfm_agrawal; for N > 4096 T
  // lives in the caller's field buffer, which is free between the entry and the exit conversion
  const size_t T = p->logn1 > 0 ? 0 : align_up(sizeof(double) * (size_t)p->M * (size_t)p->N, 256);
  return (p->nlm_nk > 0 ? (p->logn1 > 0 ? 2 : 1) : (p->logn1 > 0 ? 4 : 3)) * F + E + T;
}

int mmf_plan_set_workspace(mmf_plan* p, void* ws_dev, size_t bytes, void* cuda_stream) {
  if (!p || !ws_dev || !on_plan_device(p)) return MMF_EINVAL;
  if (bytes < mmf_plan_workspace_bytes(p) || ((size_t)ws_dev & 255) != 0) return MMF_EINVAL;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const size_t F = align_up(p->field_bytes, 256);
  p->ws = (unsigned char*)ws_dev;
  p->ws_bytes = bytes;
  p->Y = (cpx*)(p->ws);
  if (p->nlm_nk > 0) {
    p->W = p->V = nullptr;
    p->Z = p->logn1 > 0 ? (cpx*)(p->ws + F) : nullptr;  // second blocked-order buffer
    p->E = (cpx*)(p->ws + (p->logn1 > 0 ? 2 : 1) * F);
  } else {
    p->Z = (cpx*)(p->ws + F);
    p->W = (cpx*)(p->ws + 2 * F);
    p->V = p->logn1 > 0 ? (cpx*)(p->ws + 3 * F) : nullptr;
    p->E = (cpx*)(p->ws + (p->logn1 > 0 ? 4 : 3) * F);
  }
  p->T = p->logn1 > 0 ? nullptr : (double*)((unsigned char*)p->E + align_up(sizeof(cpx) * (size_t)p->M * (size_t)p->N, 256));
  EtabParams P;
  memset(&P, 0, sizeof(P));
  static const dd TWO_PI_DD = {6.283185307179586232e+00, 2.449293598294706414e-16};
  P.twopi = TWO_PI_DD;
  P.wstep = dd_div_d(TWO_PI_DD, (double)p->N * p->dt);
  P.amp = std::exp(-p->alpha * p->h / 4.0) / (double)p->N;
  P.K = p->K;
  P.logn1 = p->logn1;
  P.logn2 = p->logn2;
  dim3 grid((unsigned)((p->N + 255) / 256), (unsigned)p->M);
  k_etab<<<grid, 256, 0, st>>>(p->E, p->d_coefs, P);
  p->launches++;
  CU(cudaGetLastError());
  return MMF_OK;
}

namespace {

// one interior RK4IP step of the tensor-path plan: D(X,Y); S23; D(X,Y); FINAL_NEXT  (Eq. 6a-6f + the next 6b bracket)
int step_body(mmf_plan* p, cpx* X, cpx* Y, cudaStream_t st, double gain = 1.0) {
  int rc;
  if ((rc = apply_D(p, X, Y, 2, st)) != MMF_OK) return rc;
  if ((rc = launch_nlm<NLM_S23>(p, X, Y, st)) != MMF_OK) return rc;
  if ((rc = apply_D(p, X, Y, 2, st)) != MMF_OK) return rc;
  return launch_nlm<NLM_FINAL_NEXT>(p, X, Y, st, nullptr, gain);
}

// Small problems are bound by launch latency (hard part 6): their step body is captured once per
// (X, Y, reps) into a CUDA graph and replayed.  Large ones gain nothing and launch directly.
constexpr size_t kGraphMaxFieldBytes = (size_t)64 << 20;
constexpr int kGraphReps = 16;

cudaGraphExec_t body_graph(mmf_plan* p, cpx* X, cpx* Y, int reps, long long* nlaunch) {
  for (const auto& g : p->graphs)
    if (g.X == X && g.Y == Y && g.reps == reps) {
      *nlaunch = g.nlaunch;
      return g.exec;
    }
  if (!p->cap_stream && cudaStreamCreateWithFlags(&p->cap_stream, cudaStreamNonBlocking) != cudaSuccess) {
    p->cap_stream = nullptr;
    return nullptr;
  }
  p->dry_run = true;   // attributes, occupancy and tensor maps: everything that is not a stream operation, up front
  int rc = step_body(p, X, Y, p->cap_stream);
  p->dry_run = false;
  if (rc != MMF_OK) return nullptr;
  const long long before = p->launches;
  if (cudaStreamBeginCapture(p->cap_stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
    cudaGetLastError();
    return nullptr;
  }
  for (int i = 0; i < reps && rc == MMF_OK; ++i) rc = step_body(p, X, Y, p->cap_stream);
  cudaGraph_t graph = nullptr;
  const cudaError_t e = cudaStreamEndCapture(p->cap_stream, &graph);
  const long long n = p->launches - before;
  p->launches = before;   // nothing ran yet: replays are counted when they are enqueued
  cudaGraphExec_t exec = nullptr;
  if (rc != MMF_OK || e != cudaSuccess || !graph || cudaGraphInstantiate(&exec, graph, 0) != cudaSuccess) {
    cudaGetLastError();
    if (graph) cudaGraphDestroy(graph);
    return nullptr;
  }
  cudaGraphDestroy(graph);
  if (p->graphs.size() >= 8) {  // callers that cycle through many field buffers: keep the newest
    cudaGraphExecDestroy(p->graphs.front().exec);
    p->graphs.erase(p->graphs.begin());
  }
  p->graphs.push_back({X, Y, reps, n, exec});
  *nlaunch = n;
  return exec;
}

// nbody interior steps, from graphs where that pays, else launch by launch
int run_bodies(mmf_plan* p, cpx* X, cpx* Y, int nbody, cudaStream_t st) {
  int rc;
  cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
  const bool graphs = !p->timing && nbody >= 2 && p->field_bytes <= kGraphMaxFieldBytes &&
                      cudaStreamIsCapturing(st, &cs) == cudaSuccess && cs == cudaStreamCaptureStatusNone;
  if (graphs) {
    for (const int reps : {kGraphReps, 1}) {
      if (nbody < reps) continue;
      long long n = 0;
      cudaGraphExec_t exec = body_graph(p, X, Y, reps, &n);
      if (!exec) break;       // capture unavailable: the direct path below takes the rest
      for (; nbody >= reps; nbody -= reps) {
        CU(cudaGraphLaunch(exec, st));
        p->launches += n;
      }
    }
  }
  for (; nbody > 0; --nbody)
    if ((rc = step_body(p, X, Y, st)) != MMF_OK) return rc;
  return MMF_OK;
}

}  // namespace

// nsteps RK4IP steps; span > 0: after every span-th step the new field is multiplied by `gain` (lumped amplifier)
static int propagate_impl(mmf_plan* p, void* A_dev, int nsteps, int span, double gain, void* cuda_stream) {
  if (!p || !A_dev || nsteps < 0 || ((size_t)A_dev & 15) != 0) return MMF_EINVAL;
  if (!p->ws || !on_plan_device(p) || p->M_total > 0) return MMF_EINVAL;   // shard plans: the mmf_shard_* calls
  if (nsteps == 0) return MMF_OK;
  auto gain_of = [&](int s) { return (span > 0 && (s + 1) % span == 0) ? gain : 1.0; };   // gain applied by step s
  cudaStream_t st = (cudaStream_t)cuda_stream;
  cpx* A = (cpx*)A_dev;
  const bool tiled = p->logn1 > 0;  // N > 4096: every kernel below works in the blocked order (fft_kernels.cuh)
  int rc;
  if (p->nlm_nk > 0) {
    // two full-field buffers X, Y.  N <= 4096: the caller's buffer and the workspace's.  N > 4096: both in the
    // workspace, in blocked order; the first and the last nonlinear kernel read / write the caller's buffer in its
    // natural order, so the layout conversions cost no pass of their own.
    if (!tiled && small_cluster_usable(p)) return launch_small(p, A, nsteps, span, gain, st);   // one kernel for the call
    cpx *X = tiled ? p->Y : A, *Y = tiled ? p->Z : p->Y;
    // per step: D(X,Y); S23 in place; D(X,Y); FINAL(+NEXT)
    if (tiled) rc = launch_nlm<NLM_ENTER>(p, A, X, st, Y);               // X <- A, Y <- h N(A) A   (6b bracket)
    else rc = launch_nlm<NLM_PLAIN>(p, X, Y, st);
    if (rc != MMF_OK) return rc;
    for (int s = 0; s < nsteps - 1;) {                                            // all steps but the last
      int plain = 0;                                                              // steps without an amplifier after them
      while (s + plain < nsteps - 1 && gain_of(s + plain) == 1.0) ++plain;
      if ((rc = run_bodies(p, X, Y, plain, st)) != MMF_OK) return rc;
      s += plain;
      if (s < nsteps - 1) {
        if ((rc = step_body(p, X, Y, st, gain_of(s))) != MMF_OK) return rc;     // the last step of a span
        ++s;
      }
    }
    const double gl = gain_of(nsteps - 1);
    if ((rc = apply_D(p, X, Y, 2, st)) != MMF_OK) return rc;                      // (6a) A_I, (6b) k1
    if ((rc = launch_nlm<NLM_S23>(p, X, Y, st)) != MMF_OK) return rc;    // (6c), (6d), brackets of 6e/6f
    if ((rc = apply_D(p, X, Y, 2, st)) != MMF_OK) return rc;                      // (6e) argument, (6f) first term
    if (tiled) rc = launch_nlm<NLM_EXIT>(p, X, Y, st, A, gl);            // (6e)+(6f) into the caller's buffer
    else rc = launch_nlm<NLM_FINAL>(p, X, Y, st, nullptr, gl);
    return rc;
  }
  cpx *X = A, *Y = p->Y, *Z = p->Z, *W = p->W;
  if (tiled) {
    if ((rc = to_tiled(p, A, p->V, st)) != MMF_OK) return rc;
    X = p->V;
  }
  if (p->general) {
    // general coupling: one N evaluation per launch, every launch writes a buffer nobody reads in it (nl_general.cuh)
    if ((rc = launch_nlg<NLG_PLAIN>(p, X, nullptr, nullptr, Y, nullptr, st)) != MMF_OK) return rc;   // Y <- h N(A) A
    for (int s = 0; s < nsteps; ++s) {
      if ((rc = apply_D(p, X, Y, 2, st)) != MMF_OK) return rc;                                        // (6a), (6b)
      if ((rc = launch_nlg<NLG_STAGE2>(p, X, Y, nullptr, Z, nullptr, st)) != MMF_OK) return rc;      // (6c) Z <- k2
      if ((rc = launch_nlg<NLG_STAGE3>(p, X, Z, Y, W, Y, st)) != MMF_OK) return rc;                  // (6d), brackets
      if ((rc = apply_D(p, W, Y, 2, st)) != MMF_OK) return rc;                                        // (6e) arg, (6f)
      if ((rc = launch_nlg<NLG_FINAL>(p, W, nullptr, Y, X, nullptr, st, gain_of(s))) != MMF_OK) return rc;   // (6e) + (6f)
      if (s + 1 < nsteps && (rc = launch_nlg<NLG_PLAIN>(p, X, nullptr, nullptr, Y, nullptr, st)) != MMF_OK) return rc;
    }
    if (tiled && (rc = to_natural(p, X, A, st)) != MMF_OK) return rc;
    return MMF_OK;
  }
  // the bracket of Eq. (6b) for the first step; later steps get it from NL_FINAL_NEXT
  if ((rc = launch_nl<NL_PLAIN>(p, X, Y, Z, W, st)) != MMF_OK) return rc;
  for (int s = 0; s < nsteps; ++s) {
    if ((rc = apply_D(p, X, Y, 2, st)) != MMF_OK) return rc;               // (6a) A_I, (6b) k1
    if ((rc = launch_nl<NL_STAGE2>(p, X, Y, Z, W, st)) != MMF_OK) return rc;  // (6c) k2
    if ((rc = launch_nl<NL_STAGE3>(p, X, Y, Z, W, st)) != MMF_OK) return rc;  // (6d) k3 and both brackets
    if ((rc = apply_D(p, W, Z, 2, st)) != MMF_OK) return rc;               // (6e) argument, (6f) first term
    if (s + 1 < nsteps) rc = launch_nl<NL_FINAL_NEXT>(p, X, Y, Z, W, st, gain_of(s));  // (6e)+(6f), and next (6b) bracket
    else rc = launch_nl<NL_FINAL>(p, X, Y, Z, W, st, gain_of(s));
    if (rc != MMF_OK) return rc;
  }
  if (tiled && (rc = to_natural(p, X, A, st)) != MMF_OK) return rc;
  return MMF_OK;
}

int mmf_propagate(mmf_plan* p, void* A_dev, int nsteps, void* cuda_stream) {
  return propagate_impl(p, A_dev, nsteps, 0, 1.0, cuda_stream);
}

int mmf_propagate_spans(mmf_plan* p, void* A_dev, int nspans, int steps_per_span, double gain, void* cuda_stream) {
  if (nspans < 0 || steps_per_span < 1 || !std::isfinite(gain)) return MMF_EINVAL;
  if ((long long)nspans * steps_per_span > 0x7fffffffLL) return MMF_EINVAL;
  return propagate_impl(p, A_dev, nspans * steps_per_span, steps_per_span, gain, cuda_stream);
}

int mmf_propagate_ssfm(mmf_plan* p, void* A_dev, int nsteps, void* cuda_stream) {
  if (!p || !A_dev || nsteps < 0 || ((size_t)A_dev & 15) != 0) return MMF_EINVAL;
  if (!p->ws || p->nlm_nk <= 0 || !on_plan_device(p)) return MMF_EINVAL;  // the fused RK4 substep exists on the tensor path only (M <= 120)
  if (nsteps == 0) return MMF_OK;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  cpx *A = (cpx*)A_dev, *X = A;
  const bool tiled = p->logn1 > 0;
  int rc;
  if (tiled) {
    if ((rc = to_tiled(p, A, p->Y, st)) != MMF_OK) return rc;
    X = p->Y;
  }
  for (int s = 0; s < nsteps; ++s) {
    if ((rc = apply_D(p, X, X, 1, st)) != MMF_OK) return rc;              // exp(h/2 L)
    if ((rc = launch_nlm<NLM_RK4>(p, X, X, st)) != MMF_OK) return rc;     // RK4 over h of dA/dz = N(A) A
    if ((rc = apply_D(p, X, X, 1, st)) != MMF_OK) return rc;              // exp(h/2 L)
  }
  if (tiled && (rc = to_natural(p, X, A, st)) != MMF_OK) return rc;
  return MMF_OK;
}

int mmf_propagate_ssfm_agrawal(mmf_plan* p, void* A_dev, int nsteps, int niter, void* cuda_stream) {
  if (!p || !A_dev || nsteps < 0 || niter < 1 || ((size_t)A_dev & 15) != 0) return MMF_EINVAL;
  if (!p->ws || p->nlm_nk <= 0 || !on_plan_device(p)) return MMF_EINVAL;  // tensor-path nonlinear kernel only (M <= 120)
  if (nsteps == 0) return MMF_OK;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  cpx* A = (cpx*)A_dev;
  const bool tiled = p->logn1 > 0;
  // two field buffers that swap roles every step (X: the field at z, then exp(h/2 L) A(z); Y: the iterate) and the
  // real table T = h gamma S(A(z)).  N > 4096: both buffers in the workspace (blocked order), T in the caller's buffer.
  cpx *X = tiled ? p->Y : A, *Y = tiled ? p->Z : p->Y;
  double* T = tiled ? (double*)A : p->T;
  int rc;
  if (tiled && (rc = to_tiled(p, A, X, st)) != MMF_OK) return rc;
  for (int s = 0; s < nsteps; ++s) {
    if ((rc = launch_nlm<NLM_AGR_S0>(p, X, X, st, (cpx*)T)) != MMF_OK) return rc;      // |A|^2 "once at the position z"
    if ((rc = apply_D(p, X, X, 1, st)) != MMF_OK) return rc;                            // exp(h/2 L) A(z)
    if ((rc = launch_nlm<NLM_AGR_IT1>(p, X, Y, st, (cpx*)T)) != MMF_OK) return rc;     // iteration 1: N(z+h) := N(z)
    if ((rc = apply_D(p, Y, Y, 1, st)) != MMF_OK) return rc;                            // exp(h/2 L)
    for (int it = 2; it <= niter; ++it) {
      if ((rc = launch_nlm<NLM_AGR_ITJ>(p, X, Y, st, (cpx*)T)) != MMF_OK) return rc;   // |A|^2 at z + h from the iterate
      if ((rc = apply_D(p, Y, Y, 1, st)) != MMF_OK) return rc;
    }
    cpx* t = X; X = Y; Y = t;
  }
  if (tiled) return to_natural(p, X, A, st);
  if (X != A) CU(cudaMemcpyAsync(A, X, p->field_bytes, cudaMemcpyDeviceToDevice, st));
  return MMF_OK;
}

// A stream of host fields through one plan: the copies of field i + 1 (in) and of field i - 1 (out) run on two copy
// streams while field i propagates, over two device buffers that alternate.  One field alone cannot hide its copies:
// the first transform needs the whole time axis of every row, the last one produces it.
int mmf_propagate_host_batch(mmf_plan* p, void* const* A_hosts, int nfields, void* A_dev0, void* A_dev1, int nsteps,
                             void* cuda_stream) {
  if (!p || !A_hosts || nfields < 0 || !A_dev0 || nsteps < 0 || !on_plan_device(p)) return MMF_EINVAL;
  if (nfields > 1 && (!A_dev1 || A_dev1 == A_dev0)) return MMF_EINVAL;
  for (int i = 0; i < nfields; ++i)
    if (!A_hosts[i]) return MMF_EINVAL;
  if (nfields == 0) return MMF_OK;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  void* dev[2] = {A_dev0, A_dev1};
  if (nfields == 1) {  // nothing to overlap with: everything in order on the caller's stream
    CU(cudaMemcpyAsync(dev[0], A_hosts[0], p->field_bytes, cudaMemcpyHostToDevice, st));
    const int rc = mmf_propagate(p, dev[0], nsteps, cuda_stream);
    if (rc != MMF_OK) return rc;
    CU(cudaMemcpyAsync(A_hosts[0], dev[0], p->field_bytes, cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    return MMF_OK;
  }
  cudaStream_t sin = nullptr, sout = nullptr;
  cudaEvent_t ev_start = nullptr, in_done[2] = {nullptr, nullptr}, comp_done[2] = {nullptr, nullptr},
              out_done[2] = {nullptr, nullptr};
  int rc = MMF_OK;
  auto fail = [&](cudaError_t e) { if (e != cudaSuccess && rc == MMF_OK) rc = cuda_fail(e); return e != cudaSuccess; };
  do {
    if (fail(cudaStreamCreateWithFlags(&sin, cudaStreamNonBlocking)) ||
        fail(cudaStreamCreateWithFlags(&sout, cudaStreamNonBlocking)) ||
        fail(cudaEventCreateWithFlags(&ev_start, cudaEventDisableTiming)))
      break;
    bool bad = false;
    for (int b = 0; b < 2 && !bad; ++b)
      bad = fail(cudaEventCreateWithFlags(&in_done[b], cudaEventDisableTiming)) ||
            fail(cudaEventCreateWithFlags(&comp_done[b], cudaEventDisableTiming)) ||
            fail(cudaEventCreateWithFlags(&out_done[b], cudaEventDisableTiming));
    if (bad) break;
    // the copy streams start after the work already enqueued on the caller's stream
    if (fail(cudaEventRecord(ev_start, st)) || fail(cudaStreamWaitEvent(sin, ev_start, 0)) ||
        fail(cudaStreamWaitEvent(sout, ev_start, 0)))
      break;
    auto copy_in = [&](int i) {
      const int b = i & 1;
      if (i >= 2 && fail(cudaStreamWaitEvent(sin, out_done[b], 0))) return;   // field i - 2 has left this buffer
      if (fail(cudaMemcpyAsync(dev[b], A_hosts[i], p->field_bytes, cudaMemcpyHostToDevice, sin))) return;
      fail(cudaEventRecord(in_done[b], sin));
    };
    copy_in(0);
    for (int i = 0; i < nfields && rc == MMF_OK; ++i) {
      const int b = i & 1;
      if (i + 1 < nfields) copy_in(i + 1);
      if (rc != MMF_OK || fail(cudaStreamWaitEvent(st, in_done[b], 0))) break;
      if ((rc = mmf_propagate(p, dev[b], nsteps, cuda_stream)) != MMF_OK) break;
      if (fail(cudaEventRecord(comp_done[b], st)) || fail(cudaStreamWaitEvent(sout, comp_done[b], 0)) ||
          fail(cudaMemcpyAsync(A_hosts[i], dev[b], p->field_bytes, cudaMemcpyDeviceToHost, sout)) ||
          fail(cudaEventRecord(out_done[b], sout)))
        break;
    }
    // the call returns with every field back on the host; the caller's stream is ordered after the last copy out
    if (sout) fail(cudaStreamSynchronize(sout));
    if (sin) fail(cudaStreamSynchronize(sin));
    fail(cudaStreamSynchronize(st));
  } while (0);
  if (rc != MMF_OK) {  // drain whatever was enqueued before the failure
    if (sin) cudaStreamSynchronize(sin);
    if (sout) cudaStreamSynchronize(sout);
    cudaStreamSynchronize(st);
  }
  for (int b = 0; b < 2; ++b) {
    if (in_done[b]) cudaEventDestroy(in_done[b]);
    if (comp_done[b]) cudaEventDestroy(comp_done[b]);
    if (out_done[b]) cudaEventDestroy(out_done[b]);
  }
  if (ev_start) cudaEventDestroy(ev_start);
  if (sin) cudaStreamDestroy(sin);
  if (sout) cudaStreamDestroy(sout);
  return rc;
}

int mmf_propagate_host(mmf_plan* p, void* A_host, void* A_dev_scratch, int nsteps, void* cuda_stream) {
  void* one[1] = {A_host};
  return mmf_propagate_host_batch(p, A_host ? one : nullptr, 1, A_dev_scratch, nullptr, nsteps, cuda_stream);
}

int mmf_apply_linear(mmf_plan* p, void* X_dev, void* cuda_stream) {
  if (!p || !X_dev || !p->ws || ((size_t)X_dev & 15) != 0 || !on_plan_device(p)) return MMF_EINVAL;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  cpx* X = (cpx*)X_dev;
  if (p->logn1 == 0) return apply_D(p, X, X, 1, st);
  int rc;  // N > 4096: through the tiled order, with the workspace's field buffer as the working copy
  if ((rc = to_tiled(p, X, p->Y, st)) != MMF_OK) return rc;
  if ((rc = apply_D(p, p->Y, p->Y, 1, st)) != MMF_OK) return rc;
  return to_natural(p, p->Y, X, st);
}

int mmf_apply_nonlinear(mmf_plan* p, const void* U_dev, void* OUT_dev, void* cuda_stream) {
  if (!p || !U_dev || !OUT_dev || (((size_t)U_dev | (size_t)OUT_dev) & 15) != 0 || !on_plan_device(p)) return MMF_EINVAL;
  if (p->M_total > 0) return MMF_EINVAL;   // a shard sees only its own rows
  if (p->general) {
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (U_dev != OUT_dev) return launch_nlg<NLG_PLAIN>(p, (const cpx*)U_dev, nullptr, nullptr, (cpx*)OUT_dev, nullptr, st);
    if (!p->ws) return MMF_EINVAL;   // in place: through the workspace (a CTA reads rows its partner writes)
    int rc = launch_nlg<NLG_PLAIN>(p, (const cpx*)U_dev, nullptr, nullptr, p->Y, nullptr, st);
    if (rc != MMF_OK) return rc;
    CU(cudaMemcpyAsync(OUT_dev, p->Y, p->field_bytes, cudaMemcpyDeviceToDevice, st));
    return MMF_OK;
  }
  if (p->nlm_nk > 0) return launch_nlm<NLM_PLAIN>(p, (const cpx*)U_dev, (cpx*)OUT_dev, (cudaStream_t)cuda_stream);
  return launch_nl<NL_PLAIN>(p, (cpx*)U_dev, (cpx*)OUT_dev, nullptr, nullptr, (cudaStream_t)cuda_stream);
}

// ---- row-sharded propagation: stage entry points, sequenced by paper_1901_01895_b200/sharded.py ----

int mmf_shard_begin(mmf_plan* p, void* A_dev, void* cuda_stream) {
  if (!shard_ready(p) || !A_dev || ((size_t)A_dev & 15) != 0 || p->shard_A) return MMF_EINVAL;
  p->shard_A = A_dev;
  p->shard_X = (cpx*)A_dev;
  if (p->logn1 > 0) {   // N > 4096: the rank's rows go to the blocked order the transform kernels work in
    const int rc = to_tiled(p, (cpx*)A_dev, p->V, (cudaStream_t)cuda_stream);
    if (rc != MMF_OK) { p->shard_A = nullptr; return rc; }
    p->shard_X = p->V;
  }
  return MMF_OK;
}

int mmf_shard_powers(mmf_plan* p, int stage, void* P_dev, long long t_first, long long t_count, void* cuda_stream) {
  if (!shard_ready(p) || !p->shard_A || !P_dev || ((size_t)P_dev & 7) != 0) return MMF_EINVAL;
  return shard_stage(p, stage, true, (double*)P_dev, t_first, t_count, 1.0, (cudaStream_t)cuda_stream);
}

int mmf_shard_apply(mmf_plan* p, int stage, const void* P_dev, long long t_first, long long t_count, double gain,
                    void* cuda_stream) {
  if (!shard_ready(p) || !p->shard_A || !P_dev || ((size_t)P_dev & 7) != 0 || !std::isfinite(gain)) return MMF_EINVAL;
  return shard_stage(p, stage, false, (double*)P_dev, t_first, t_count, gain, (cudaStream_t)cuda_stream);
}

int mmf_shard_linear(mmf_plan* p, int which, void* cuda_stream) {
  if (!shard_ready(p) || !p->shard_A || which < 0 || which > 1) return MMF_EINVAL;
  return which == 0 ? apply_D(p, p->shard_X, p->Y, 2, (cudaStream_t)cuda_stream)     // (6a) A_I, (6b) k1
                    : apply_D(p, p->W, p->Z, 2, (cudaStream_t)cuda_stream);           // (6e) argument, (6f) first term
}

int mmf_shard_end(mmf_plan* p, void* cuda_stream) {
  if (!shard_ready(p) || !p->shard_A) return MMF_EINVAL;
  int rc = MMF_OK;
  if (p->logn1 > 0) rc = to_natural(p, p->shard_X, (cpx*)p->shard_A, (cudaStream_t)cuda_stream);
  p->shard_A = nullptr;
  p->shard_X = nullptr;
  return rc;
}

int mmf_debug_forward(mmf_plan* p, void* X_dev, void* SPEC_dev, void* cuda_stream) {
  if (!p || !X_dev || !SPEC_dev || X_dev == SPEC_dev || !on_plan_device(p)) return MMF_EINVAL;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int rc;
  cpx *X = (cpx*)X_dev, *S = (cpx*)SPEC_dev;
  if (p->logn1 > 0) {
    // SPEC holds the working copy in tiled order; pass B leaves the slot-order spectrum in X (chunk-contiguous)
    if ((rc = to_tiled(p, X, S, st)) != MMF_OK) return rc;
    if ((rc = launch_cols<0>(p, S, S, 1, st)) != MMF_OK) return rc;
    if ((rc = launch_rows<1>(p, S, S, 1, X, st)) != MMF_OK) return rc;
  } else {
    if ((rc = launch_rows<1>(p, X, X, 1, X, st)) != MMF_OK) return rc;
  }
  dim3 grid((unsigned)((p->N + 255) / 256), (unsigned)(2 * p->M));
  k_unpermute<<<grid, 256, 0, st>>>((const cpx*)X_dev, (cpx*)SPEC_dev, p->logn1, p->logn2);
  p->launches++;
  CU(cudaGetLastError());
  return MMF_OK;
}

int mmf_debug_freq_index(mmf_plan* p, long long* idx_host) {
  if (!p || !idx_host || !on_plan_device(p)) return MMF_EINVAL;
  long long* d = nullptr;
  CU(cudaMalloc((void**)&d, sizeof(long long) * (size_t)p->N));
  k_slot_map<<<(unsigned)((p->N + 255) / 256), 256>>>(d, p->logn1, p->logn2);
  p->launches++;
  cudaError_t e = cudaMemcpy(idx_host, d, sizeof(long long) * (size_t)p->N, cudaMemcpyDeviceToHost);
  cudaFree(d);
  if (e != cudaSuccess) return cuda_fail(e);
  return MMF_OK;
}

long long mmf_plan_launch_count(const mmf_plan* p) { return p ? p->launches : 0; }

int mmf_plan_groups(const mmf_plan* p) { return p ? p->G : 0; }

int mmf_plan_set_timing(mmf_plan* p, int enable) {
  if (!p) return MMF_EINVAL;
  clear_events(p);
  p->timing = enable != 0;
  return MMF_OK;
}

int mmf_kernel_class_count(void) { return KC_COUNT; }

const char* mmf_kernel_class_name(int kclass) { return (kclass >= 0 && kclass < KC_COUNT) ? kc_names[kclass] : ""; }

int mmf_plan_get_timing(mmf_plan* p, int kclass, double* total_ms, long long* launches, double* alg_bytes) {
  if (!p || kclass < 0 || kclass >= KC_COUNT || !total_ms || !launches || !alg_bytes) return MMF_EINVAL;
  double tot = 0.0, bytes = 0.0, bsum = 0.0;
  long long n = 0;
  for (size_t i = 0; i < p->ev_class.size(); ++i) {
    if (p->ev_class[i] != kclass) continue;
    bsum += p->ev_bytes[i];
    CU(cudaEventSynchronize(p->ev[2 * i + 1]));
    float ms = 0.f;
    CU(cudaEventElapsedTime(&ms, p->ev[2 * i], p->ev[2 * i + 1]));
    tot += ms;
    ++n;
  }
  // algorithmic bytes of one launch: the average over the recorded launches of this class
  bytes = n > 0 ? bsum / (double)n : 0.0;
  *total_ms = tot;
  *launches = n;
  *alg_bytes = bytes;
  return MMF_OK;
}

int mmf_plan_destroy(mmf_plan* p) {
  if (!p) return MMF_EINVAL;
  free_tables(p);
  delete p;
  return MMF_OK;
}

}  // extern "C"
