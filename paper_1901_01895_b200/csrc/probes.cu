// probes.cu — measurement probes behind `bench.py --probes` ("the builder MEASURES DFMA/DMMA peak ...
// and uses the measured value").  They are NOT on the hot path: they produce the denominators DESIGN.md §6 quotes —
// the fp64 issue peak of the plain and the tensor (DMMA) path, and the HBM bandwidth a pure TMA copy reaches with the
// exact access pattern (box shape, pitch, ring depth) of each product kernel.
#include <cstdio>
#include <cstring>

#include "../../include/mmf_probes.h"
#include "async_copy.cuh"
#include "tmem_exchange.cuh"

using namespace mmf;

namespace {

// ---- fp64 issue rate: a register-only instruction stream, ILP independent chains per thread ------------------------
// KIND 0: DADD x = x + y        1: DMUL x = x * y        2: DFMA x = fma(y, z, x) (three distinct register operands)
// KIND 3: DFMA x = fma(x, y, y) (two distinct)           4: butterfly t = x + y, y = x - y (2 DADD)
template <int ILP, int KIND>
__global__ void __launch_bounds__(1024, 1) k_probe_fp64(double* out, int iters, const double* in) {
  double x[ILP], y[ILP], z[ILP];
#pragma unroll
  for (int i = 0; i < ILP; ++i) {
    x[i] = in[(threadIdx.x + i) & 1023];
    y[i] = in[(threadIdx.x + 64 + i) & 1023];
    z[i] = in[(threadIdx.x + 128 + i) & 1023];
  }
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int r = 0; r < 8; ++r) {
#pragma unroll
      for (int i = 0; i < ILP; ++i) {
        if (KIND == 0) x[i] = x[i] + y[i];
        else if (KIND == 1) x[i] = x[i] * y[i];
        else if (KIND == 2) x[i] = fma(y[i], z[i], x[i]);
        else if (KIND == 3) x[i] = fma(x[i], y[i], y[i]);
        else {
          const double t = x[i] + y[i];
          y[i] = x[i] - y[i];
          x[i] = t;
        }
      }
    }
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < ILP; ++i) s += x[i] + y[i] + z[i];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// KIND 5: mma.sync.m8n8k4.f64 (SASS DMMA), CH independent accumulator chains per warp
template <int CH>
__global__ void __launch_bounds__(1024, 1) k_probe_dmma(double* out, int iters, const double* in) {
  double c[CH][2], a[CH], b[CH];
#pragma unroll
  for (int i = 0; i < CH; ++i) {
    c[i][0] = c[i][1] = 0;
    a[i] = in[(threadIdx.x + i) & 1023];
    b[i] = in[(threadIdx.x + 64 + i) & 1023];
  }
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int r = 0; r < 8; ++r)
#pragma unroll
      for (int i = 0; i < CH; ++i)
        asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                     : "+d"(c[i][0]), "+d"(c[i][1])
                     : "d"(a[i]), "d"(b[i]));
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < CH; ++i) s += c[i][0] + c[i][1];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// ---- pure TMA copy through the product kernels' ring: load tile -> slot -> store the tile back in place -----------
struct CopyParams {
  long long ntiles;
  int nct_log, nbox, rb, box_bytes, c0_mul, c1_mul, slots, bulk;
};
__global__ void __launch_bounds__(32, 1) k_probe_copy(const __grid_constant__ CUtensorMap map, CopyParams p, char* base) {
  extern __shared__ __align__(1024) unsigned char smem[];
  const int S = p.slots;
  const int slot_bytes = p.nbox * p.box_bytes;
  uint64_t* full = reinterpret_cast<uint64_t*>(smem + (size_t)S * slot_bytes);
  if (threadIdx.x != 0) return;
  for (int i = 0; i < S; ++i) mbar_init(&full[i], 1);
  mbar_init_fence();
  const long long n = p.ntiles > blockIdx.x ? (p.ntiles - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
  auto coords = [&](long long j, int& c0, int& c1) {
    const long long u = blockIdx.x + j * gridDim.x;
    const long long ct = u & ((1LL << p.nct_log) - 1), rb = u >> p.nct_log;
    c0 = (int)(ct * p.c0_mul);
    c1 = (int)(rb * p.c1_mul);
  };
  auto load = [&](long long j) {
    int c0, c1;
    coords(j, c0, c1);
    const int b = (int)(j % S);
    mbar_arrive_expect_tx(&full[b], slot_bytes);
    if (p.bulk) bulk_load_1d(smem + (size_t)b * slot_bytes, base + (blockIdx.x + j * gridDim.x) * (long long)slot_bytes, slot_bytes, &full[b]);
    else
      for (int i = 0; i < p.nbox; ++i)
        tma_load_2d(smem + (size_t)b * slot_bytes + (size_t)i * p.box_bytes, &map, c0, c1 + i * p.rb, &full[b]);
  };
  for (long long j = 0; j < S - 1 && j < n; ++j) load(j);
  for (long long j = 0; j < n; ++j) {
    const int b = (int)(j % S);
    if (j + S - 1 < n) {  // the slot of tile j - 1: refill it once its store has read it
      if (j >= 1) tma_store_wait_read();
      load(j + S - 1);
    }
    mbar_wait(&full[b], (uint32_t)((j / S) & 1));
    int c0, c1;
    coords(j, c0, c1);
    if (p.bulk) bulk_store_1d(base + (blockIdx.x + j * gridDim.x) * (long long)slot_bytes, smem + (size_t)b * slot_bytes, slot_bytes);
    else
      for (int i = 0; i < p.nbox; ++i) tma_store_2d(&map, c0, c1 + i * p.rb, smem + (size_t)b * slot_bytes + (size_t)i * p.box_bytes);
    tma_store_commit();
  }
  tma_store_wait_all();
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

template <class K>
int time_kernel(K launch, int reps, double* ms_out) {
  cudaEvent_t e0, e1;
  if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return MMF_ECUDA;
  launch();  // warm-up
  if (cudaDeviceSynchronize() != cudaSuccess) return MMF_ECUDA;
  cudaEventRecord(e0);
  for (int i = 0; i < reps; ++i) launch();
  cudaEventRecord(e1);
  const cudaError_t e = cudaDeviceSynchronize();
  float ms = 0.f;
  cudaEventElapsedTime(&ms, e0, e1);
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  if (e != cudaSuccess || cudaGetLastError() != cudaSuccess) return MMF_ECUDA;
  *ms_out = (double)ms / reps;
  return MMF_OK;
}

// ---- on-chip data movement and stage arithmetic: what an exchange of a 4096-point tile costs each way ---------------
// One CTA of `threads` threads per SM; every thread works on 16 complex values (the register tile of fft_core.cuh).
// KIND 0: tcgen05.ld 32x32b.x32 + wait (128 B per thread)     1: tcgen05.st 32x32b.x32 (+ wait per four)
// KIND 2: LDS.128 x 8 (128 B per thread)                      3: SHFL.BFLY b32 x 32 (128 B per thread)
// KIND 4: tmem_trip_fwd   5: tmem_trip_rev   (tmem_exchange.cuh: a 2-bit lane <-> register exchange of the 16 values)
// KIND 6: the warp-local exchange through shared memory (16 STS.128, warp barrier, 16 LDS.128, warp barrier)
// KIND 7: the group-wide exchange (16 STS.128, group barrier, 16 LDS.128, group barrier; groups of 256 threads)
// KIND 8: a radix-16 stage on registers only    9: a radix-16 stage with its 15 twiddles from a shared-memory table
// clk_out: clock64 ticks per operation of the CTA's first thread (all warps run the same loop concurrently).
template <int KIND>
__global__ void __launch_bounds__(512, 1) k_probe_onchip(int iters, double* out, long long* clk) {
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  __shared__ uint32_t tw;
  cpx* sbuf = reinterpret_cast<cpx*>(smem_raw);
  if (threadIdx.x < 32) tmem_alloc(&tw, 512);
  tmem_fence_before_sync();
  for (int i = threadIdx.x; i < 2 * 4096; i += blockDim.x) sbuf[i] = make_double2(0.6, 0.8);
  __syncthreads();
  tmem_fence_after_sync();
  const uint32_t warp = threadIdx.x >> 5;
  const uint32_t xa = tw + (((warp & 3) * 32) << 16) + (warp >> 2) * 128;
  const int grp = threadIdx.x >> 8, t = threadIdx.x & 255;
  cpx* s = sbuf + ((size_t)grp << 12);
  const Tm12 L = tm12_layout(t);
  cpx v[16];
#pragma unroll
  for (int j = 0; j < 16; ++j) v[j] = make_double2(1e-3 * (threadIdx.x + j), 1e-3 * j);
  int w[32];
#pragma unroll
  for (int j = 0; j < 32; ++j) w[j] = threadIdx.x + j;
  const long long t0 = clock64();
  for (int it = 0; it < iters; ++it) {
    if constexpr (KIND == 0) {
      int q[32];
      tmem_ld_32x32b_x32(q, xa + 32 * (it & 3));
      tmem_wait_ld32(q);
#pragma unroll
      for (int j = 0; j < 32; ++j) w[j] ^= q[j];   // every loaded word is consumed
    } else if constexpr (KIND == 1) {
      tmem_st_32x32b_x32(xa + 32 * (it & 3), w);
      if ((it & 3) == 3) tmem_wait_st();
      w[0] += it;
    } else if constexpr (KIND == 2) {
      const uint4* q = reinterpret_cast<const uint4*>(smem_raw);
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        const uint4 x = q[(threadIdx.x + 512 * j + 37 * (it & 3) + (w[0] & 1)) & 8191];
        w[0] += x.x;
      }
    } else if constexpr (KIND == 3) {
#pragma unroll
      for (int j = 0; j < 32; ++j) w[j] = __shfl_xor_sync(0xffffffffu, w[j], 1 + (j & 15));
    } else if constexpr (KIND == 4) {
      tmem_trip_fwd(v, xa);
    } else if constexpr (KIND == 5) {
      tmem_trip_rev(v, xa);
    } else if constexpr (KIND == 6) {
      tile_sts<4>(v, s, stage_base<4>(t));
      __syncwarp();
      tile_lds<0>(v, s, stage_base<0>(t));
      __syncwarp();
    } else if constexpr (KIND == 7) {
      tile_sts12<8>(v, s, L.base1);
      group_barrier(1 + grp, MMF_GROUP_THREADS);
      tile_lds12<4>(v, s, L.base2);
      group_barrier(1 + grp, MMF_GROUP_THREADS);
    } else if constexpr (KIND == 8) {
      stage_math<12, 0, 0, 4, +1, true>(v, 0, sbuf);
#pragma unroll
      for (int j = 0; j < 16; ++j) { v[j].x *= 0.25; v[j].y *= 0.25; }
    } else {
      stage_math<12, 0, 4, 4, +1, true>(v, t & 15, sbuf);
#pragma unroll
      for (int j = 0; j < 16; ++j) { v[j].x *= 0.25; v[j].y *= 0.25; }
    }
    if constexpr (KIND >= 4 && KIND <= 7) v[0].x += 1.0;
  }
  const long long t1 = clock64();
  double acc = 0;
#pragma unroll
  for (int j = 0; j < 16; ++j) acc += v[j].x + v[j].y;
#pragma unroll
  for (int j = 0; j < 32; ++j) acc += w[j];
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = acc;
  if (threadIdx.x == 0 && blockIdx.x == 0) clk[0] = t1 - t0;
  tmem_fence_before_sync();
  __syncthreads();
  if (threadIdx.x < 32) tmem_dealloc(tw, 512);
}

template <int KIND>
int run_onchip(int sms, int threads, int iters, double* out, long long* clk, double* ms_out) {
  const size_t smem = 2 * 4096 * sizeof(cpx);
  if (cudaFuncSetAttribute(k_probe_onchip<KIND>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
    return MMF_ECUDA;
  return time_kernel([&] { k_probe_onchip<KIND><<<sms, threads, smem>>>(iters, out, clk); }, 1, ms_out);
}

}  // namespace

extern "C" {

int mmf_probe_fp64(int kind, int threads, int iters, double* ms_out, double* thread_inst_out) {
  if (!ms_out || !thread_inst_out || threads < 32 || threads > 1024 || (threads & 31) || iters < 1) return MMF_EINVAL;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
    return MMF_ECUDA;
  double *out = nullptr, *in = nullptr;
  if (cudaMalloc((void**)&out, sizeof(double) * 1024 * (size_t)sms) != cudaSuccess) return MMF_ENOMEM;
  if (cudaMalloc((void**)&in, sizeof(double) * 1024) != cudaSuccess) { cudaFree(out); return MMF_ENOMEM; }
  cudaMemset(in, 0, sizeof(double) * 1024);
  constexpr int ILP = 8;
  int rc = MMF_EINVAL;
  double per_iter = 8.0 * ILP;  // thread-level instructions (KIND 5: warp-level DMMA per warp) per loop iteration
  switch (kind) {
    case 0: rc = time_kernel([&] { k_probe_fp64<ILP, 0><<<sms, threads>>>(out, iters, in); }, 3, ms_out); break;
    case 1: rc = time_kernel([&] { k_probe_fp64<ILP, 1><<<sms, threads>>>(out, iters, in); }, 3, ms_out); break;
    case 2: rc = time_kernel([&] { k_probe_fp64<ILP, 2><<<sms, threads>>>(out, iters, in); }, 3, ms_out); break;
    case 3: rc = time_kernel([&] { k_probe_fp64<ILP, 3><<<sms, threads>>>(out, iters, in); }, 3, ms_out); break;
    case 4: rc = time_kernel([&] { k_probe_fp64<ILP, 4><<<sms, threads>>>(out, iters, in); }, 3, ms_out); per_iter *= 2; break;
    case 5: rc = time_kernel([&] { k_probe_dmma<4><<<sms, threads>>>(out, iters, in); }, 3, ms_out); per_iter = 8.0 * 4; break;
    default: break;
  }
  cudaFree(out);
  cudaFree(in);
  // KIND 0-4: thread-level fp64 instructions of the whole launch; KIND 5: warp-level DMMA instructions
  *thread_inst_out = per_iter * (double)iters * (kind == 5 ? threads / 32 : threads) * sms;
  return rc;
}

int mmf_probe_tma_copy(void* buf_dev, size_t buf_bytes, unsigned long long dim0, unsigned long long dim1,
                       unsigned long long stride_bytes, unsigned box0, unsigned box1, int nbox, int nct_log, int c0_mul,
                       int c1_mul, long long ntiles, int slots, int bulk, int reps, double* ms_out, double* bytes_out) {
  if (!buf_dev || !ms_out || !bytes_out || nbox < 1 || slots < 2 || ntiles < 1 || reps < 1) return MMF_EINVAL;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
    return MMF_ECUDA;
  CUtensorMap map;
  memset(&map, 0, sizeof(map));
  CopyParams p;
  p.ntiles = ntiles; p.nct_log = nct_log; p.nbox = nbox; p.rb = (int)box1; p.c0_mul = c0_mul; p.c1_mul = c1_mul;
  p.slots = slots; p.bulk = bulk;
  p.box_bytes = (int)(box0 * box1 * sizeof(double));
  const size_t slot_bytes = (size_t)nbox * p.box_bytes;
  const size_t smem = slots * slot_bytes + 64;
  if (smem > 227 * 1024 || (slot_bytes & 15)) return MMF_EINVAL;
  if (bulk) {
    if ((size_t)ntiles * slot_bytes > buf_bytes) return MMF_EINVAL;
  } else {
    if (stride_bytes * dim1 > buf_bytes || dim0 * sizeof(double) > stride_bytes) return MMF_EINVAL;
    void* fp = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fp, cudaEnableDefault, &q) != cudaSuccess || !fp) return MMF_ECUDA;
    const cuuint64_t gdim[2] = {dim0, dim1};
    const cuuint64_t gs[1] = {stride_bytes};
    const cuuint32_t box[2] = {box0, box1};
    const cuuint32_t es[2] = {1, 1};
    if (((EncodeTiledFn)fp)(&map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, buf_dev, gdim, gs, box, es,
                            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return MMF_EINVAL;
  }
  if (cudaFuncSetAttribute(k_probe_copy, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return MMF_ECUDA;
  const long long grid = ntiles < sms ? ntiles : sms;
  const int rc = time_kernel([&] { k_probe_copy<<<(unsigned)grid, 32, smem>>>(map, p, (char*)buf_dev); }, reps, ms_out);
  *bytes_out = 2.0 * (double)ntiles * (double)slot_bytes;  // read + write
  return rc;
}

int mmf_probe_onchip(int kind, int threads, int iters, double* ms_out, double* clk_per_op_out) {
  if (!ms_out || !clk_per_op_out || iters < 1 || kind < 0 || kind > 9) return MMF_EINVAL;
  if (threads < 32 || threads > 512 || (threads & 31) || (kind == 7 && (threads & 255))) return MMF_EINVAL;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
    return MMF_ECUDA;
  double* out = nullptr;
  long long* clk = nullptr;
  if (cudaMalloc((void**)&out, sizeof(double) * 512 * (size_t)sms) != cudaSuccess) return MMF_ENOMEM;
  if (cudaMalloc((void**)&clk, sizeof(long long)) != cudaSuccess) { cudaFree(out); return MMF_ENOMEM; }
  int rc = MMF_EINVAL;
  switch (kind) {
#define MMF_ONCHIP_CASE(K) case K: rc = run_onchip<K>(sms, threads, iters, out, clk, ms_out); break;
    MMF_ONCHIP_CASE(0) MMF_ONCHIP_CASE(1) MMF_ONCHIP_CASE(2) MMF_ONCHIP_CASE(3) MMF_ONCHIP_CASE(4) MMF_ONCHIP_CASE(5)
    MMF_ONCHIP_CASE(6) MMF_ONCHIP_CASE(7) MMF_ONCHIP_CASE(8) MMF_ONCHIP_CASE(9)
#undef MMF_ONCHIP_CASE
    default: break;
  }
  long long h = 0;
  if (rc == MMF_OK && cudaMemcpy(&h, clk, sizeof(h), cudaMemcpyDeviceToHost) != cudaSuccess) rc = MMF_ECUDA;
  cudaFree(out);
  cudaFree(clk);
  *clk_per_op_out = (double)h / iters;
  return rc;
}

}  // extern "C"
