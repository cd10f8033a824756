/*
 * gwprobe.h -- C-ABI of the measurement-aid library csrc/libgwprobe.so (source: csrc/gw_probe.cu).
 *
 * NOT part of the product boundary (include/gwlnl.h, include/gwpop.h): these entry points measure the roofline
 * denominators that MEASURED_PEAKS.json does not hold -- SURVEY.md 8(d): "the builder must measure the peak with a
 * register-resident DFMA-chain microbenchmark in the same run" and "measure a pure-store ceiling too, since the
 * waveform kernel only writes" -- and are called by bench.py and `python -m paper_1904_02863_b200.probes` only.
 * Every function returns 0 or a negative code with the meaning of GW_ERR_* in gwlnl.h (-1 invalid argument,
 * -3 CUDA error, -4 not a compute-capability-10 device), allocates its own scratch buffer, enqueues on `cuda_stream`
 * (a cudaStream_t passed as void*) and synchronises before returning.
 */
#ifndef GWPROBE_H
#define GWPROBE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Register-resident fp64 rate microbenchmark on the current device (8 independent chains per thread, 64 warps
 * per SM): enqueues `n_iter` rounds of 64 instructions per thread and reports achieved fp64 FMA/s.  `mode` selects
 * the operand pattern: 0 = fma(v, imm, imm) (pipe peak); 1 = fma(a, b, v) with three distinct register operands;
 * 2 = three register operands of which one is shared by consecutive instructions; 3 = mma.sync m8n8k4 f64;
 * 4, 5 = mode 0 with 8 or 16 independent integer instructions beside every 8 DFMA.                        */
int gw_probe_fp64_fma_rate(int n_iter, int mode, double *fma_per_s, double *elapsed_ms, void *cuda_stream);

/* The SM clock that is actually running, in MHz (median over the SMs): one warp per SM spins for ~30 us of clock64()
 * between two reads of the nanosecond globaltimer.  Enqueued on `cuda_stream` right behind the timed work, it shows the
 * clock the preceding kernels ran at (NVML reports the requested clock; power management adjusts on a millisecond
 * scale).                                                                                                    */
int gw_probe_sm_clock(double *mhz_median, void *cuda_stream);

/* The floor of "one kernel timed alone between two CUDA events": median over n_rep of the event-to-event time of an
 * EMPTY kernel launched with the given grid, block and dynamic shared memory right behind other work on the stream.
 * On B200 this reads ~6 us whatever the launch shape; bench.py reports it beside every kernel-level time.      */
int gw_probe_launch_floor(int grid, int block, int dyn_smem_bytes, int n_rep, double *median_ms, void *cuda_stream);

/* Pure-store HBM bandwidth: `bytes` (far larger than the 126 MB L2) written once per pass with 16-byte streaming
 * stores by a grid of 8 CTAs per SM; best of `n_rep` passes after one warm-up pass.  GB/s = bytes / best time.   */
int gw_probe_store_bandwidth(int64_t bytes, int n_rep, double *gb_per_s, double *best_ms, void *cuda_stream);

/* Pure-load HBM bandwidth: `bytes` read once per pass with 16-byte streaming loads (four in flight per thread),
 * reduced in registers, nothing stored; best of `n_rep` passes after one warm-up pass.                       */
int gw_probe_load_bandwidth(int64_t bytes, int n_rep, double *gb_per_s, double *best_ms, void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* GWPROBE_H */
