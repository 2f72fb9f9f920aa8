/* mmf_probes.h — C ABI of the MEASUREMENT PROBES behind `bench.py --probes` (the fp64 peak and the
 * access-pattern ceilings the rooflines in DESIGN.md section 6 are quoted against are MEASURED).  They are not part of
 * the product: they live in a library of their own, libmmf_probes.so (paper_1901_01895_b200/csrc/probes.cu), and
 * libmmf_b200.so neither contains nor needs them.  Status codes are those of mmf.h. */
#ifndef MMF_PROBES_H_
#define MMF_PROBES_H_

#include "mmf.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Each probe
 * allocates its own scratch (mmf_probe_tma_copy: the caller's), runs on the default stream and SYNCHRONISES.
 * mmf_probe_fp64:  a register-only fp64 instruction stream on every SM, `threads` per CTA (multiple of 32, <= 1024),
 *   kind 0 DADD, 1 DMUL, 2 DFMA with three distinct register operands, 3 DFMA with two, 4 add/sub butterfly (2 DADD),
 *   5 mma.sync.m8n8k4.f64 (DMMA; 512 flop per warp instruction).  Returns the time of one launch [ms] and the number
 *   of thread-level (kind 5: warp-level) instructions it executed.
 * mmf_probe_tma_copy:  a pure copy through the product kernels' shared-memory ring (TMA load tile -> slot -> TMA
 *   store in place, `slots` deep, one CTA per SM) over the device buffer buf_dev, seen as a 2-D fp64 tensor
 *   [dim1][dim0] with row pitch stride_bytes; tile u = (ct = u mod 2^nct_log, rb = u / 2^nct_log) is made of nbox
 *   boxes (box0 x box1) at coordinates (ct c0_mul, rb c1_mul + i box1).  bulk != 0: contiguous tiles of
 *   nbox box0 box1 doubles moved with cp.async.bulk instead.  Returns ms per launch and bytes moved (read + write).
 * mmf_probe_onchip:  what the on-chip data paths of the transform kernels cost, one CTA of `threads` threads (multiple
 *   of 32, <= 512) per SM, every thread on a register tile of 16 complex values: kind 0 tcgen05.ld 32x32b.x32 (128 B per
 *   thread), 1 tcgen05.st 32x32b.x32, 2 LDS.128 x 8, 3 SHFL.BFLY x 32 (128 B per thread each), 4 / 5 one forward /
 *   reverse tensor-memory trip (store 32x32b + load 16x256b or the reverse: a 2-bit lane <-> register exchange),
 *   6 the warp-local exchange through shared memory, 7 the group-wide exchange (threads = 256 or 512), 8 a radix-16
 *   stage on registers, 9 the same with its 15 twiddles from shared memory.  Returns ms per launch and the clock64
 *   ticks per operation seen by one thread while every warp of the CTA runs the same loop. */
int mmf_probe_fp64(int kind, int threads, int iters, double *ms_out, double *thread_inst_out);
int mmf_probe_onchip(int kind, int threads, int iters, double *ms_out, double *clk_per_op_out);
int mmf_probe_tma_copy(void *buf_dev, size_t buf_bytes, unsigned long long dim0, unsigned long long dim1,
                       unsigned long long stride_bytes, unsigned box0, unsigned box1, int nbox, int nct_log, int c0_mul,
                       int c1_mul, long long ntiles, int slots, int bulk, int reps, double *ms_out, double *bytes_out);

#ifdef __cplusplus
}
#endif
#endif /* MMF_PROBES_H_ */
