/*
 * psg_bench.h -- measurement helpers of libpsg.so.  NOT part of the hot path of include/psg.h: bench.py and the tests
 * use them for roofline denominators ("FP32/SFU: must be measured first") and for the launch count the
 * bench line reports.  Same conventions as psg.h (extern "C", int status).
 */
#ifndef PSG_BENCH_H
#define PSG_BENCH_H

#include "psg.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Measured throughput of this device (register-only loops, CUDA-event timed, synchronises the device):
 * which = 0: FP32 FFMA lane-ops/s; 1: packed FFMA2 (f32x2) lane-ops/s (2 per lane per instruction);
 * 2: MUFU.EX2/s; 3: FP64 DFMA lane-ops/s; 4: F2F f32->f64->f32 round trips/s; 5: I2F.F32.S32/s;
 * 6: packed FADD2 lane-ops/s.  Denominators for the hill-sum roofline.
 * 7 / 8: hill evaluations/s of the BARE hill loop (k_hills' own inner loop on a shared-memory table, nothing
 * else; 2-D periodic / 3-D with 2 periodic CVs): the ceiling of the kernel's instruction mix.
 * 9: empty-kernel nodes/s of a replayed CUDA graph (1 / the launch floor t_floor of SURVEY.md 8(d), the bound of the
 *    latency-bound configs 0 and 2).
 * 10: binary64 exp() evaluations/s (the library routine on the FP64 pipe): the bound of the grid deposit (k_grid_deposit),
 *     of the interface CV (k_dti_mass, k_dti_apply) and of the binary64 hill terms (PSG_HILLS_F64).
 * 11: 1 / t where t = the time two event records bracket when the kernel between them is EMPTY and the stream has just
 *     flushed L2 with a 256 MiB memset -- the floor of bench.py's per-step timing protocol (about 6 us on B200; an event
 *     record drains the pipeline on both sides).
 * 100 + n: the same as 7 with only n passes of 1,024 hills (short-run behaviour). */
int psg_measure_alu_peak(int device, int which, double* ops_per_second_out);
/* Tuning knobs of the fused large-group step, for measurements: range_step_lag = items the position
 * producer of k_range_step may run ahead of the force group (0 = the default, 10); disable_range_step != 0 makes psg_step
 * take the separate kernels (k_range_moments, k_cv_eval, k_harmonic, k_apply_dense) instead. */
int psg_set_tuning(psg_ctx* ctx, int range_step_lag, int disable_range_step);
/* Launch counter: number of kernels this ctx has enqueued since creation (for bench.py's gpu_launches). */
long long psg_launch_count(const psg_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* PSG_BENCH_H */
