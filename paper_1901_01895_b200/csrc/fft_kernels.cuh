// fft_kernels.cuh — the transform kernels of the RK4IP hot path (sm_100a, fp64): rows a1-a3 of the hot-path table.
//
//   k_cols  passes A and C of the three-pass operator D = exp(h/2 L) (Eq. 6a):  length-N1 transforms
//           over the slow (strided) index of a row viewed as an N1 x N2 matrix, plus the inter-pass twiddle
//           W_N^(k1 n2).
//   k_rows  pass B: contiguous length-N2 transform -> multiply by the tabulated exp(h/2 L_a(w_k))/N -> adjoint
//           length-N2 transform, the spectrum never leaving the SM.  For N <= 4096 this kernel alone is D.
//   k_etab  fills the exp(h/2 L_a(w_k)) table in the order pass B consumes it (double-double phase).
//
// Index algebra of D (forward sign +, reading R1 of DESIGN.md):  n = N2 n1 + n2,  k = k1 + N1 k2,
//   X[k1 + N1 k2] = sum_n2 W_N2^(k2 n2) [ W_N^(k1 n2) sum_n1 W_N1^(k1 n1) x[N2 n1 + n2] ]
// pass A does the inner sum and the twiddle, pass B the outer sum; the way back is the exact adjoint.
//
// Execution model: persistent CTAs (one per SM) of G independent groups of 256 threads.  A group owns one 64 KiB
// exchange buffer and walks its own list of 4096-point tiles (fft_core.cuh); groups of a CTA share the stage
// twiddle tables in shared memory and run out of phase, so that one group's exchanges overlap the other's
// butterflies.  Tiles travel between HBM and shared memory as TMA bulk copies through a three-slot ring (the slot is
// also the group's exchange buffer); no compute warp issues a global load or store.
#pragma once
#include "async_copy.cuh"
#include "fft_core.cuh"
#include "tmem_exchange.cuh"

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

// The stage tables of a transform travel to shared memory as ONE bulk copy issued by the CTA's first thread right after
// the barrier initialisation (no thread-level loads, and the copy overlaps the rest of the prologue and the first
// tile loads); every thread waits on its mbarrier once, before the first table read.
template <int ENTRIES>
__device__ __forceinline__ void request_stage_tables(cpx* __restrict__ tab, const cpx* __restrict__ src, uint64_t* tabbar) {
  if constexpr (ENTRIES > 0) {
    mbar_arrive_expect_tx(tabbar, ENTRIES * (int)sizeof(cpx));
    bulk_load_1d(tab, src, ENTRIES * (int)sizeof(cpx), tabbar);
  }
}
template <int ENTRIES>
__device__ __forceinline__ void await_stage_tables(uint64_t* tabbar) {
  if constexpr (ENTRIES > 0) mbar_wait(tabbar, 0);
}

// ---------------------------------------------------------------------------------------------------- pass A / C
// Inter-pass table (filled by the host, mmf_api.cu): one row of 256 + 2 W entries per column tile ct,
//   [t]           W_N^(k1(pos0(t)) n2(t)),  pos0(t) = 16 (t >> LOGW) the first slot thread t holds after the last
//                 pass-A stage, n2(t) = ct W + (t & (W - 1)) its column;
//   [256 + c]     W_N^(wA n2),  [256 + W + c]  W_N^(wB n2),  n2 = ct W + c: the steps of the exponent along the
//                 16 registers of that layout, k1(pos0 + j) = k1(pos0) + wA (j & 7) + wB (j >> 3).
// The row travels to shared memory with the tile (one bulk copy), so the kernel makes no global load of its own.
__host__ __device__ constexpr int ipt_row_entries(int logw) { return 256 + (2 << logw); }

struct ColsParams {
  const cpx* __restrict__ twtab;  // stage tables of the N1-point transform
  const cpx* __restrict__ ipt;    // inter-pass table [N2 / W][256 + 2 W]
  int logn2, logwb, nrows, nbuf;
};

// BLOCKED field layout (the order every kernel between mmf_propagate's entry and exit works in when N > 4096).
// A row of N = N1 N2 samples, n = N2 n1 + n2 with n2 = WB ctb + cb (WB = 2^logwb = max(W, 16) columns per block), is
// stored as [ctb][n1][cb]: position (ctb N1 + n1) WB + cb.  Measured with a pure TMA copy: in the
// natural order the tile of passes A / C (64-byte segments at 64 KiB pitch) streams at 4.7 TB/s and the contiguous
// chunk of pass B at 6.3; in the blocked order the A / C tile (64-byte segments at 256-byte pitch inside one
// contiguous block) streams at 5.2 TB/s and the chunk of pass B (256-byte segments) at 5.9 — and pass B, bound by
// its arithmetic, needs only 3.7.  The nonlinear kernels act on every time sample alike and never see the
// difference (8 consecutive positions are still 8 time samples, the same for every row).  k_perm converts a buffer
// between the natural and the blocked order on the way in and out.
__host__ __device__ constexpr int block_logw(int logn1) { return (MMF_TILE_LOG - logn1) > 4 ? (MMF_TILE_LOG - logn1) : 4; }

// v[j] *= W_N^(k1(pos0 + j) n2)  (or its conjugate): the 16 factors are t0 sA^(j&7) sB^(j>>3) — three look-ups per
// thread and short product chains (depth <= 4).
template <bool CONJ>
__device__ __forceinline__ void apply_interpass(cpx (&v)[16], cpx t0, cpx sA, cpx sB) {
  const cpx t1 = cmul(t0, sB);
  cpx pw[8];
  pw[1] = sA;
  pw[2] = cmul(sA, sA);
  pw[3] = cmul(pw[2], sA);
  pw[4] = cmul(pw[2], pw[2]);
  pw[5] = cmul(pw[4], sA);
  pw[6] = cmul(pw[4], pw[2]);
  pw[7] = cmul(pw[4], pw[3]);
  v[0] = CONJ ? cmulc(v[0], t0) : cmul(v[0], t0);
  v[8] = CONJ ? cmulc(v[8], t1) : cmul(v[8], t1);
#pragma unroll
  for (int e = 1; e < 8; ++e) {
    const cpx a = cmul(t0, pw[e]), b = cmul(t1, pw[e]);
    v[e] = CONJ ? cmulc(v[e], a) : cmul(v[e], a);
    v[8 + e] = CONJ ? cmulc(v[8 + e], b) : cmul(v[8 + e], b);
  }
}

// un-swizzled tile access: the layout TMA writes / reads (tile element f at slot f)
template <int LO>
__device__ __forceinline__ void tile_lds_linear(cpx (&v)[16], const cpx* __restrict__ s, int base) {
#pragma unroll
  for (int j = 0; j < 16; ++j) v[j] = s[base | (j << LO)];
}
template <int LO>
__device__ __forceinline__ void tile_sts_linear(const cpx (&v)[16], cpx* __restrict__ s, int base) {
#pragma unroll
  for (int j = 0; j < 16; ++j) s[base | (j << LO)] = v[j];
}

// number of tile slots of the pass A / C ring: three where the stage tables leave room (N1 <= 2^10), else two
__host__ __device__ constexpr int cols_slots(int logn1) { return logn1 <= 10 ? 3 : 2; }
template <int LOGN1>
__host__ __device__ constexpr size_t cols_smem_bytes() {
  constexpr int TWN = tw_total_entries(LOGN1, nstages(LOGN1));
  return sizeof(cpx) * (((size_t)cols_slots(LOGN1) << MMF_TILE_LOG) +
                        (size_t)cols_slots(LOGN1) * ipt_row_entries(MMF_TILE_LOG - LOGN1) + ((TWN + 7) & ~7)) + 64;
}

// grid = persistent (<= one CTA per SM); block = 512 = two groups of 256.  DIR 0: pass A (DIF, sign +, then twiddle);
// DIR 1: pass C (conjugate twiddle, then DIT, sign -).  A tile is N1 points x W = 2^(12 - LOGN1) adjacent columns of
// one field row: in the blocked layout the box (2 W doubles, N1 rows) at (2 W (ct % (WB/W)), (row N2/WB + ct / (WB/W)) N1)
// of the 2-D tensor map (inner = 2 WB doubles, outer = rows x N2/WB x N1), moved in boxes of <= 256 rows.
// Data movement is asynchronous and off the LSU pipe: the CTA's tiles t = 0, 1, 2, ... rotate through S ring slots
// (slot t % S), tile t is worked on by group t % 2 IN its slot (the slot is also the group's exchange buffer), and the
// group's first thread stores it and then refills the slot its previous tile vacated with tile t - 2 + S, which the
// other group picks up half a tile period later.  map0 / map1: the two field buffers.
template <int LOGN1, int DIR, int G>
__global__ void __launch_bounds__(MMF_GROUP_THREADS* G, 1)
k_cols(const __grid_constant__ CUtensorMap map0, const __grid_constant__ CUtensorMap map1, ColsParams p) {
  static_assert(G == 2, "two groups alternate over the ring");
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  constexpr int LOGW = MMF_TILE_LOG - LOGN1, W = 1 << LOGW;
  constexpr int NST = nstages(LOGN1);
  constexpr int TWN = tw_total_entries(LOGN1, NST);
  constexpr int LR1 = stage_lr(LOGN1, NST), LO1 = stage_lo(LOGN1 - LR1, LOGW, MMF_TILE_LOG);  // first-stage layout
  constexpr int LOL = stage_lo(0, LOGW, MMF_TILE_LOG);                                        // last-stage layout
  constexpr int S = cols_slots(LOGN1);
  constexpr int TILE_BYTES = (int)sizeof(cpx) << MMF_TILE_LOG;
  constexpr int RB = LOGN1 > 8 ? 256 : (1 << LOGN1);  // rows per TMA box
  constexpr int NBOX = (1 << LOGN1) / RB;
  constexpr int BOX_BYTES = RB * W * (int)sizeof(cpx);
  constexpr int IPT = ipt_row_entries(LOGW);
  static_assert(NST >= 2, "the ring protocol assumes at least one exchange");
  cpx* ring = reinterpret_cast<cpx*>(smem_raw);
  cpx* ipts = ring + ((size_t)S << MMF_TILE_LOG);
  cpx* tab = ipts + S * IPT;
  uint64_t* full = reinterpret_cast<uint64_t*>(tab + ((TWN + 7) & ~7));
  uint64_t* done = full + S;
  uint64_t* tabbar = done + G;
  pdl_launch_dependents();
  if (threadIdx.x == 0) {
#pragma unroll
    for (int i = 0; i < S; ++i) mbar_init(&full[i], 1);
#pragma unroll
    for (int i = 0; i < G; ++i) mbar_init(&done[i], MMF_GROUP_THREADS);
    mbar_init(tabbar, 1);
    mbar_init_fence();
    request_stage_tables<TWN>(tab, p.twtab, tabbar);
    tma_prefetch_desc(&map0);
    tma_prefetch_desc(&map1);
  }
  __syncthreads();
  pdl_wait();                            // the field buffers are the predecessor's output; the tables above are not
  const int grp = threadIdx.x / MMF_GROUP_THREADS, t = threadIdx.x % MMF_GROUP_THREADS;
  const bool elect = t == 0;
  const int bar = 1 + grp;
  const int logn2 = p.logn2;
  const long long nct = 1LL << (logn2 - LOGW);
  const long long total = nct * p.nrows * p.nbuf;
  const long long ntile = total > blockIdx.x ? (total - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;

  // tensor-map coordinates of the CTA's tile tt (blocked layout), its buffer and its column tile
  const int logsub = p.logwb - LOGW;  // column tiles per block
  auto tile_coords = [&](long long tt, int& c0, int& c1, const CUtensorMap*& m, long long& ct) {
    const long long u = blockIdx.x + tt * gridDim.x;
    ct = u & (nct - 1);
    const long long rb = u >> (logn2 - LOGW);
    c0 = (int)(ct & ((1 << logsub) - 1)) << (LOGW + 1);                                       // doubles
    c1 = (int)((((rb % p.nrows) << (logn2 - p.logwb)) + (ct >> logsub)) << LOGN1);            // pitch row
    m = (rb / p.nrows) ? &map1 : &map0;
  };
  auto issue_load = [&](long long tt) {
    int c0, c1;
    const CUtensorMap* m;
    long long ct;
    tile_coords(tt, c0, c1, m, ct);
    const int b = (int)(tt % S);
    mbar_arrive_expect_tx(&full[b], TILE_BYTES + IPT * (int)sizeof(cpx));
    unsigned char* dst = smem_raw + (size_t)b * TILE_BYTES;
#pragma unroll
    for (int i = 0; i < NBOX; ++i) tma_load_2d(dst + i * BOX_BYTES, m, c0, c1 + i * RB, &full[b]);
    bulk_load_1d(ipts + b * IPT, p.ipt + ct * IPT, IPT * (int)sizeof(cpx), &full[b]);
  };
  auto issue_store = [&](long long tt) {
    int c0, c1;
    const CUtensorMap* m;
    long long ct;
    tile_coords(tt, c0, c1, m, ct);
    const unsigned char* src = smem_raw + (size_t)(tt % S) * TILE_BYTES;
#pragma unroll
    for (int i = 0; i < NBOX; ++i) tma_store_2d(m, c0, c1 + i * RB, src + i * BOX_BYTES);
    tma_store_commit();
  };

  if (threadIdx.x == 0)
    for (long long tt = 0; tt < S && tt < ntile; ++tt) issue_load(tt);
  await_stage_tables<TWN>(tabbar);

  const int base1 = stage_base<LO1>(t), basel = stage_base<LOL>(t);
  const int c = t & (W - 1);
  int it = 0;
  for (long long tt = grp; tt < ntile; tt += G, ++it) {
    const int b = (int)(tt % S);
    cpx* s = ring + ((size_t)b << MMF_TILE_LOG);
    const cpx* ip = ipts + b * IPT;
    // the slot this group's previous tile (tt - 2) left: refill it with tile tt - 2 + S once its store has read it
    const bool refill = elect && tt >= G && tt - G + S < ntile;
    if (S == 2 && refill) {
      tma_store_wait_read();
      issue_load(tt - G + S);
    }
    mbar_wait(&full[b], (uint32_t)((tt / S) & 1));
    cpx v[16];
    if constexpr (DIR == 0) {
      tile_lds_linear<LO1>(v, s, base1);
      if (S > 2 && refill) {
        tma_store_wait_read();
        issue_load(tt - G + S);
      }
      fft_dif<MMF_TILE_LOG, LOGN1, LOGW, LOGN1, NST, +1, false, true>(v, s, t, tab, bar);
      apply_interpass<false>(v, ip[t], ip[256 + c], ip[256 + W + c]);
      __syncwarp();  // the unswizzled slots written next were read, swizzled, by lanes of this warp (fft_core.cuh, PRESYNC)
      tile_sts_linear<LOL>(v, s, basel);
    } else {
      tile_lds_linear<LOL>(v, s, basel);
      const cpx t0 = ip[t], sA = ip[256 + c], sB = ip[256 + W + c];
      if (S > 2 && refill) {
        tma_store_wait_read();
        issue_load(tt - G + S);
      }
      apply_interpass<true>(v, t0, sA, sB);
      fft_dit<MMF_TILE_LOG, LOGN1, LOGW, LOGN1, NST, -1, false, true>(v, s, t, tab, bar);
      __syncwarp();
      tile_sts_linear<LO1>(v, s, base1);
    }
    // hand the finished tile to the async proxy: every thread's writes are fenced, the first thread stores
    fence_proxy_async_smem();
    mbar_arrive(&done[grp]);
    if (elect) {
      mbar_wait(&done[grp], (uint32_t)(it & 1));
      issue_store(tt);
    }
  }
  if (elect) tma_store_wait_all();
}

// ---------------------------------------------------------------------------------------- natural <-> blocked order
// A copy through a three-slot ring driven by one thread per CTA; DIR 0: natural -> blocked, DIR 1: blocked ->
// natural.  A tile is RT = 4096 / WB consecutive memory rows n1 of one block: in the natural buffer the box
// (2 WB doubles = 256-byte segments, RT rows) of the map (inner = 2 N2 doubles, outer = rows x N1), in the blocked
// buffer 64 KiB of contiguous memory.  mmf_propagate runs it once on the way in and once on the way out.
// grid = persistent, block = 32.
struct PermParams {
  cpx* blocked;
  int logn1, logn2, logwb, nrows;
};
template <int DIR>
__global__ void __launch_bounds__(32, 1) k_perm(const __grid_constant__ CUtensorMap mapn, PermParams p) {
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  constexpr int S = 3;
  constexpr int TILE_BYTES = (int)sizeof(cpx) << MMF_TILE_LOG;
  uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw + S * TILE_BYTES);
  pdl_launch_dependents();
  if (threadIdx.x != 0) return;
#pragma unroll
  for (int i = 0; i < S; ++i) mbar_init(&full[i], 1);
  mbar_init_fence();
  tma_prefetch_desc(&mapn);
  pdl_wait();
  const int logrt = MMF_TILE_LOG - p.logwb;                 // rows per tile
  const int lognb = p.logn2 - p.logwb;                      // blocks per row
  const int logtb = p.logn1 - logrt;                        // tiles per block
  const long long total = (long long)p.nrows << (lognb + logtb);
  const long long ntile = total > blockIdx.x ? (total - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
  // tile u = (row, block ctb, row group i): natural box coordinates and blocked address
  auto coords = [&](long long tt, int& c0, int& c1, cpx*& g) {
    const long long u = blockIdx.x + tt * gridDim.x;
    const long long ctb = u & ((1LL << lognb) - 1), i = (u >> lognb) & ((1LL << logtb) - 1), row = u >> (lognb + logtb);
    c0 = (int)(ctb << (p.logwb + 1));
    c1 = (int)((row << p.logn1) + (i << logrt));
    g = p.blocked + ((((row << lognb) + ctb) << p.logn1) << p.logwb) + (i << MMF_TILE_LOG);
  };
  auto load = [&](long long tt) {
    int c0, c1;
    cpx* g;
    coords(tt, c0, c1, g);
    const int b = (int)(tt % S);
    unsigned char* sl = smem_raw + (size_t)b * TILE_BYTES;
    mbar_arrive_expect_tx(&full[b], TILE_BYTES);
    if constexpr (DIR == 0) tma_load_2d(sl, &mapn, c0, c1, &full[b]);
    else bulk_load_1d(sl, g, TILE_BYTES, &full[b]);
  };
  for (long long tt = 0; tt < S - 1 && tt < ntile; ++tt) load(tt);
  for (long long tt = 0; tt < ntile; ++tt) {
    const int b = (int)(tt % S);
    if (tt + S - 1 < ntile) {  // the slot of tile tt - 1: refill it once its store has read it
      if (tt >= 1) tma_store_wait_read();
      load(tt + S - 1);
    }
    mbar_wait(&full[b], (uint32_t)((tt / S) & 1));
    int c0, c1;
    cpx* g;
    coords(tt, c0, c1, g);
    const unsigned char* sl = smem_raw + (size_t)b * TILE_BYTES;
    if constexpr (DIR == 0) bulk_store_1d(g, sl, TILE_BYTES);
    else tma_store_2d(&mapn, c0, c1, sl);
    tma_store_commit();
  }
  tma_store_wait_all();
}

// -------------------------------------------------------------------------------------------------------- pass B
// A "chunk" is one contiguous run of N2 values (memory row p1 of field row r: chunk = r * N1 + p1); a tile is
// 2^(12 - LOGN2) consecutive chunks = 64 KiB of contiguous memory.  The exp(h/2 L) table holds, per (mode, p1) chunk,
// its N2 entries in the register order of the last forward stage: entry [(q & 15) << (LOGN2 - 4) | (q >> 4)] belongs
// to slot q, so that lanes read consecutive entries.
struct RowsParams {
  cpx* X0;                        // SINGLE: the field buffers (natural order); else unused (tensor maps)
  cpx* X1;
  cpx* OUT;                       // MODE 1: where the slot-order spectrum goes (chunk-contiguous)
  const cpx* __restrict__ E;
  const cpx* __restrict__ twtab;  // stage tables of the N2-point transform
  long long nchunks;              // per buffer: 2 M N1
  int logn1, nbuf, M;
};

#define MMF_ROWS_SLOTS 3
template <int LOGN2>
__host__ __device__ constexpr size_t rows_smem_bytes() {
  constexpr int TWN = tw_total_entries(LOGN2, nstages(LOGN2));
  return sizeof(cpx) * (((size_t)MMF_ROWS_SLOTS << MMF_TILE_LOG) + ((TWN + 7) & ~7)) + 64;
}

// MODE 0: transform, * E, adjoint transform (in place).  MODE 1: forward transform only, output in slot order
// (debug entry point).  SINGLE: N1 = 1 (the whole of D in this kernel; tiles may be ragged and hold several rows).
// Order of work: an item is (mode a, tile of chunks); its 2 nbuf sub-tiles (polarisation x buffer) share one piece of
// the table and are done back to back by the same group, so the table comes from HBM once.  The CTA's items
// j = 0, 1, ... (item blockIdx.x + j gridDim.x) go to group j % 2.
// Data movement: as in k_cols — the CTA's tiles tt = 0, 1, ... (group tt % 2, sub-tile (tt / 2) % sub of item
// 2 (tt / (2 sub)) + tt % 2) rotate through three 64 KiB ring slots that are also the exchange buffers; a tile is one
// bulk copy each way, issued by the group's first thread: contiguous (cp.async.bulk) when N <= 4096, else — blocked
// layout — chunk p1 of a row is the box (2 WB doubles) x (N2 / WB rows) at (2 WB p1, row N2 / WB) of the 2-D tensor
// map (inner = 2 N1 WB doubles = one block, outer = rows x N2 / WB), moved in boxes of <= 256 rows; the box lands as
// [ctb][cb] = the chunk in n2 order.  The sub-tiles of an odd last item alternate between the groups, so the
// rotation has no holes.  map0 / map1: the two field buffers (unused when SINGLE).
template <int LOGN2, int MODE, bool SINGLE, int G>
__global__ void __launch_bounds__(MMF_GROUP_THREADS* G, 1)
k_rows(const __grid_constant__ CUtensorMap map0, const __grid_constant__ CUtensorMap map1, RowsParams p) {
  static_assert(G == 2, "two groups alternate over the ring");
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  constexpr int LOGB = MMF_TILE_LOG - LOGN2;
  constexpr int NST = nstages(LOGN2);
  constexpr int TWN = tw_total_entries(LOGN2, NST);
  constexpr int LR1 = stage_lr(LOGN2, NST), LO1 = stage_lo(LOGN2 - LR1, 0, MMF_TILE_LOG);
  constexpr int S = MMF_ROWS_SLOTS;
  constexpr int TILE_BYTES = (int)sizeof(cpx) << MMF_TILE_LOG;
  cpx* ring = reinterpret_cast<cpx*>(smem_raw);
  cpx* tab = ring + ((size_t)S << MMF_TILE_LOG);
  uint64_t* full = reinterpret_cast<uint64_t*>(tab + ((TWN + 7) & ~7));
  uint64_t* done = full + S;
  // The E values of a thread are the same for all sub-tiles of an item (polarisations x buffers): they are fetched
  // into tensor memory (64 columns of the thread's own lane) at the top of the item's first tile — while no tile is
  // held in registers, so all 16 loads are in flight at once — and every sub-tile reads them back from there: no
  // global-load latency inside a transform, no LSU traffic, no shared memory (none is left).
  constexpr bool ECACHE = MODE == 0;
  // 4096-point transforms: the exchange between the last two stages goes through tensor memory (tmem_exchange.cuh),
  // 64 more columns per warp
  constexpr bool TMX = LOGN2 == 12;
  constexpr uint32_t WARP_COLS = TMX ? 128 : 64;
  constexpr uint32_t TMEM_COLS = 4 * WARP_COLS;  // 4 warps share a lane quarter
  uint32_t* tmem_word = reinterpret_cast<uint32_t*>(done + G);
  uint64_t* tabbar = done + G + 1;
  if (threadIdx.x == 0) {
#pragma unroll
    for (int i = 0; i < S; ++i) mbar_init(&full[i], 1);
#pragma unroll
    for (int i = 0; i < G; ++i) mbar_init(&done[i], MMF_GROUP_THREADS);
    mbar_init(tabbar, 1);
    mbar_init_fence();
    request_stage_tables<TWN>(tab, p.twtab, tabbar);
  }
  if constexpr (ECACHE || TMX) {
    if (threadIdx.x < 32) {
      __syncwarp();  // reconverge after the single-thread block above: tcgen05.alloc is .sync.aligned
      tmem_alloc(tmem_word, TMEM_COLS);
    }
    tmem_fence_before_sync();
  }
  __syncthreads();
  // Dependents are released only now, with the tensor-memory columns in hand: a successor that allocates tensor memory
  // ahead of its own griddepcontrol.wait could otherwise land on this SM, take the columns first and then wait for a
  // grid whose CTA here is still blocked in tcgen05.alloc.  A kernel signals once it holds every blocking resource.
  pdl_launch_dependents();
  pdl_wait();                            // the field buffers (and, after plan set-up, the E table) come from predecessors
  uint32_t taddr = 0;   // this warp's columns: [0, 64) the E values of the item, [64, 128) the exchange buffer (TMX)
  if constexpr (ECACHE || TMX) {
    tmem_fence_after_sync();
    const uint32_t warp = threadIdx.x >> 5;
    taddr = *tmem_word + (((warp & 3) * 32) << 16) + (warp >> 2) * WARP_COLS;
  }
  int cached_item = -1;
  const int grp = threadIdx.x / MMF_GROUP_THREADS, t = threadIdx.x % MMF_GROUP_THREADS;
  const bool elect = t == 0;
  const int bar = 1 + grp;
  const int base1 = stage_base<LO1>(t);
  const Tm12 lay = tm12_layout(t);
  const int tl = TMX ? lay.tv : t;                   // slot >> 4 of this thread's last-stage values
  const int cht = (tl << 4) >> LOGN2;                // their chunk (inside the tile)
  const int tq = tl & ((1 << (LOGN2 - 4)) - 1);
  const int logn1 = p.logn1;
  const int logsub = (SINGLE ? 0 : 1) + (p.nbuf > 1 ? 1 : 0);   // sub-tiles per item: nbuf (SINGLE) or 2 nbuf
  const long long items = SINGLE ? ((p.nchunks + (1 << LOGB) - 1) >> LOGB) : ((long long)p.M << (logn1 - LOGB));
  const long long nitem = items > blockIdx.x ? (items - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;  // this CTA's
  const long long npaired = (nitem >> 1) << (logsub + 1);        // tiles of the items done in pairs (one per group)
  const long long ntile = npaired + ((nitem & 1) << logsub);     // an odd last item: its sub-tiles alternate groups

  // geometry of the CTA's tile tt: first chunk, buffer, item
  auto tile_geom = [&](long long tt, long long& chunk0, int& buf, long long& item) {
    long long j;
    int sidx;
    if (tt < npaired) {
      const long long q = tt >> 1;
      j = ((q >> logsub) << 1) + (tt & 1);
      sidx = (int)(q & ((1 << logsub) - 1));
    } else {
      j = nitem - 1;
      sidx = (int)(tt - npaired);
    }
    item = blockIdx.x + j * gridDim.x;
    if constexpr (SINGLE) {
      chunk0 = item << LOGB;
      buf = sidx;
    } else {
      const long long a = item >> (logn1 - LOGB), tau = item & ((1LL << (logn1 - LOGB)) - 1);
      chunk0 = ((2 * a + (sidx & 1)) << logn1) + (tau << LOGB);
      buf = sidx >> 1;
    }
  };
  auto tile_bytes = [&](long long chunk0) -> uint32_t {
    if constexpr (SINGLE) {
      const long long left = (p.nchunks - chunk0) << LOGN2;
      return (uint32_t)(left < (1LL << MMF_TILE_LOG) ? left * (long long)sizeof(cpx) : TILE_BYTES);
    } else {
      return TILE_BYTES;
    }
  };
  // blocked layout: the boxes of one chunk (block width, boxes per chunk and rows per box depend on N1)
  const int logwb = SINGLE ? 0 : block_logw(logn1);
  const int lognb = LOGN2 - logwb;                                 // blocks (pitch rows) per chunk
  auto chunk_boxes = [&](long long chunk, int buf, unsigned char* sl, uint64_t* bar) {
    const CUtensorMap* m = buf ? &map1 : &map0;
    const int rbr = lognb > 8 ? 256 : (1 << lognb), nboxc = (1 << lognb) / rbr;
    const int box_bytes = (rbr << logwb) * (int)sizeof(cpx);
    const int c0 = (int)(chunk & ((1LL << logn1) - 1)) << (logwb + 1);
    const int c1 = (int)(chunk >> logn1) << lognb;
    for (int i = 0; i < nboxc; ++i) {
      if (bar) tma_load_2d(sl + i * box_bytes, m, c0, c1 + i * rbr, bar);
      else tma_store_2d(m, c0, c1 + i * rbr, sl + i * box_bytes);
    }
  };
  auto issue_load = [&](long long tt) {
    long long chunk0, item;
    int buf;
    tile_geom(tt, chunk0, buf, item);
    const int b = (int)(tt % S);
    const uint32_t bytes = tile_bytes(chunk0);
    mbar_arrive_expect_tx(&full[b], bytes);
    if constexpr (SINGLE) {
      bulk_load_1d(smem_raw + (size_t)b * TILE_BYTES, (buf ? p.X1 : p.X0) + (chunk0 << LOGN2), bytes, &full[b]);
    } else {
      for (int q = 0; q < (1 << LOGB); ++q)
        chunk_boxes(chunk0 + q, buf, smem_raw + (size_t)b * TILE_BYTES + ((size_t)q << LOGN2) * sizeof(cpx), &full[b]);
    }
    if constexpr (!SINGLE && MODE == 0) {
      // first sub-tile of an item (polarisation x of buffer 0): pull the item's piece of the table into L2
      if (buf == 0 && ((chunk0 >> logn1) & 1) == 0) {
        const long long a = item >> (logn1 - LOGB), tau = item & ((1LL << (logn1 - LOGB)) - 1);
        bulk_prefetch_l2(p.E + (((a << logn1) + (tau << LOGB)) << LOGN2), TILE_BYTES);
      }
    }
  };

  if (threadIdx.x == 0) {
    if constexpr (!SINGLE) {
      tma_prefetch_desc(&map0);
      tma_prefetch_desc(&map1);
    }
    for (long long tt = 0; tt < S && tt < ntile; ++tt) issue_load(tt);
  }
  await_stage_tables<TWN>(tabbar);

  // Only the tile number stays live across the transforms: geometry is recomputed where it is needed (the table
  // pointer after the forward chain, the store address by the first thread) to keep the 16 values in registers.
  const int ntile_i = (int)ntile;
  for (int tt = grp; tt < ntile_i; tt += G) {
    // the slot this group's previous tile (tt - 2) left: refill it with tile tt + 1 once its store has read it
    const bool refill = elect && tt >= G && tt - G + S < ntile_i;
    const int b = tt % S;
    cpx* s = ring + ((size_t)b << MMF_TILE_LOG);
    if constexpr (ECACHE) {
      // First tile of an item: fetch the thread's 16 E values into tensor memory NOW, while no tile is held in
      // registers — all 16 loads in flight at once (one latency per item instead of one per pair of values), and
      // every sub-tile of the item reads them back from there.
      long long chunk0, item;
      int buf;
      tile_geom(tt, chunk0, buf, item);
      if ((int)item != cached_item) {  // uniform over the group
        long long ech;  // table chunk of this thread's last-stage values
        bool live = true;
        if constexpr (SINGLE) {
          ech = (chunk0 + cht) >> 1;   // chunk = row, table chunk = mode
          live = chunk0 + cht < p.nchunks;  // ragged last tile: rows that do not exist (never stored)
        } else {
          const long long a = item >> (logn1 - LOGB), tau = item & ((1LL << (logn1 - LOGB)) - 1);
          ech = (a << logn1) + (tau << LOGB) + cht;
        }
        const cpx* e = p.E + (ech << LOGN2) + tq;
        cpx ev[16];
#pragma unroll
        for (int j = 0; j < 16; ++j) ev[j] = live ? __ldg(e + (j << (LOGN2 - 4))) : make_double2(1.0, 0.0);
#pragma unroll
        for (int c = 0; c < 8; ++c) {
          const cpx pr[2] = {ev[2 * c], ev[2 * c + 1]};
          tmem_st_c2(taddr + 8 * c, pr);
        }
        tmem_wait_st();
        cached_item = (int)item;
      }
    }
    mbar_wait(&full[b], (uint32_t)((tt / S) & 1));
    cpx v[16];
    tile_lds_linear<LO1>(v, s, base1);
    if (refill) {
      tma_store_wait_read();
      issue_load(tt - G + S);
    }
    if constexpr (TMX) fft12_dif_tm<+1>(v, s, lay, tab, bar, taddr + 64);
    else fft_dif<MMF_TILE_LOG, LOGN2, 0, LOGN2, NST, +1, MODE == 1, true>(v, s, t, tab, bar);
    if constexpr (MODE == 0) {
      if constexpr (ECACHE) {   // the item's E values are in tensor memory (loaded at the top of the item's first tile)
#pragma unroll
        for (int hb = 0; hb < 2; ++hb) {   // two batches of eight: two tensor-memory latencies per tile
          int wa[4][8];
#pragma unroll
          for (int c = 0; c < 4; ++c) tmem_ld_issue8(wa[c], taddr + 32 * hb + 8 * c);
#pragma unroll
          for (int c = 0; c < 4; ++c) tmem_ld_wait8(wa[c]);
#pragma unroll
          for (int c = 0; c < 4; ++c) {
            cpx ev[2];
            tmem_words_to_c2(ev, wa[c]);
            v[8 * hb + 2 * c] = cmul(v[8 * hb + 2 * c], ev[0]);
            v[8 * hb + 2 * c + 1] = cmul(v[8 * hb + 2 * c + 1], ev[1]);
          }
        }
      }
      if constexpr (TMX) fft12_dit_tm<-1>(v, s, lay, tab, bar, taddr + 64);
      else fft_dit<MMF_TILE_LOG, LOGN2, 0, LOGN2, NST, -1, false>(v, s, t, tab, bar);
      // the unswizzled slots written next were read, in the last exchange, swizzled by lanes of the same warp (the
      // swizzles touch bits [2:0] of a slot only): a warp barrier orders the two
      __syncwarp();
      tile_sts_linear<LO1>(v, s, base1);
      fence_proxy_async_smem();
      mbar_arrive(&done[grp]);
      if (elect) {
        long long chunk0, item;
        int buf;
        tile_geom(tt, chunk0, buf, item);
        mbar_wait(&done[grp], (uint32_t)((tt >> 1) & 1));
        if constexpr (SINGLE) {
          bulk_store_1d((buf ? p.X1 : p.X0) + (chunk0 << LOGN2), s, tile_bytes(chunk0));
        } else {
          for (int q = 0; q < (1 << LOGB); ++q)
            chunk_boxes(chunk0 + q, buf, reinterpret_cast<unsigned char*>(s + ((size_t)q << LOGN2)), nullptr);
        }
        tma_store_commit();
      }
    } else {
      long long chunk0, item;
      int buf;
      tile_geom(tt, chunk0, buf, item);
      if (!SINGLE || chunk0 + cht < p.nchunks) {
        cpx* g = p.OUT + (chunk0 << LOGN2);
#pragma unroll
        for (int j = 0; j < 16; ++j) g[(tl << 4) + j] = v[j];
      }
      group_barrier(bar, MMF_GROUP_THREADS);  // the slot may be refilled
    }
  }
  if (elect) tma_store_wait_all();
  if constexpr (ECACHE || TMX) {
    tmem_fence_before_sync();
    __syncthreads();
    if (threadIdx.x < 32) tmem_dealloc(*tmem_word, TMEM_COLS);
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
  dd wstep;    // 2 pi / (N dt)
  dd twopi;
  double amp;  // exp(-alpha hh / 2) / N
  int K, logn1, logn2;
};

// E[mode][p1][perm(q)] = amp * exp(i * sum_n coef_n(mode) * w_k^n),  k = bin held by slot (p1, q),
// perm(q) = (q & 15) << (logn2 - 4) | (q >> 4)  (the order k_rows reads).
// coefs: device array [M][K] of dd, hh * beta_n / n!.  grid = (N / 256, M), block = 256.
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
  const int qp = ((q & 15) << (P.logn2 - 4)) | (q >> 4);
  E[(long long)mode * N + ((long long)p1 << P.logn2) + qp] = make_double2(P.amp * cr, P.amp * sr);
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

}  // namespace mmf
