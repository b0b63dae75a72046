/*
 * shd_bench.h -- measurement tooling of libshd.so, kept apart from the hot-path boundary of shd.h:
 * per-kernel timers and counters that bench.py reads, and the two live peak probes behind its roofline denominators.
 */
#ifndef SHD_BENCH_H
#define SHD_BENCH_H
#include "shd.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Per-kernel device timing: with on != 0 every later shd_energy_grad / shd_smax records CUDA events on
 * the handle's stream around its launch groups; read the durations with shd_stat(h, 20..24). */
int shd_set_timing(shd_ctx* h, int on);

/* Introspection used by bench.py / tests (host scalars):
 *   what = 0 / 12: DFMAs the rho / gradient pass launches (padding included),
 *   what = 1: kernel launches of the last call, 2: padded (p,q) cell count of the rho pass,
 *   3: valid cell count, 4: bytes of device workspace, 5: particle splits of the rho pass,
 *   6: (p,q) tiles, 7: P, 8: Qn, 9: padded particle count, 10: particle blocks of the gradient
 *   pass, 11: q-steps walked by one gradient block, 13 / 17: segments of the gradient pass (FP64 / INT8),
 *   14 / 15: tiles / particle splits of the INT8 rho pass, 16: engine in use, 18: K-steps of the INT8 gradient pass,
 *   19: chunks per evaluation (shd_set_workspace), 25: particles per chunk, 26: bytes of per-particle tables,
 *   27: 1 when the engine is the library's own choice,
 *   28 / 29: SM clock in MHz INSIDE k_rho8 / k_grad8 during the last evaluation (clock64 against globaltimer in the
 *            issuing thread of CTA 0; under tensor load it is well below the clock nvidia-smi reports between kernels),
 *   20..24: milliseconds of the last call's launch groups (needs shd_set_timing):
 *           20 phasor tables (a1), 21 rho pass (a2), 22 finish (a3), 23 gradient operand, 24 gradient pass (a4). */
double shd_stat(const shd_ctx* h, int what);

/*
 * Measured FP64-pipe issue rate of the current device, the denominator of the "alu" roofline
 * (DESIGN.md "roofline").  kind = 0: dependent-DFMA chains, 1: DADD chains (8 per
 * thread, all SMs), 2: chains of the FP64 matrix instruction DMMA.8x8x4 (8 per warp; counted as 8 FMAs
 * per thread and instruction), the instruction the rho and gradient passes issue; runs for about
 * `seconds` (0 < seconds <= 10).  HOST out: instr_per_s[0] = best
 * launch, instr_per_s[1] = mean over the run (sustained), in thread-level FP64 instructions per
 * second.  Errors: SHD_EINVAL, SHD_ENOMEM, SHD_ECUDA.  Needs no handle.
 */
int shd_fp64_peak(int kind, double seconds, double instr_per_s[2]);

/*
 * INT8 tensor-core probe (an exact digit-sliced contraction on tcgen05.mma.kind::i8 would
 * replace the FP64 limb FMAs).  HOST out: *mismatches = wrong entries of a 128 x 64 x 128 s8 x s8 -> s32 product
 * computed by the 5th-generation tensor core (operands in shared memory, accumulator in TMEM) against the
 * integer product on the host (0 = exact); *tops = measured issue rate of M=128, N=256, K=32 instructions on
 * all SMs in tera-operations per second (2 per multiply-accumulate).  Needs no handle.
 */
int shd_i8_probe(double* tops, long* mismatches);

/*
 * FP64 and integer ALU work beside a tcgen05.mma.kind::i8 stream on the same SM (the measurement behind the integer
 * epilogue of k_grad8).  HOST out[8]: [0] cycles per DADD per warp, 16 warps of dependent chains alone;
 * [1] the same while a back-to-back M=128 N=256 K=32 stream runs on the SM; [2], [3] the same for IMAD chains;
 * [4] cycles per N = 256 instruction alone, [5] beside the DADD chains, [6] beside the IMAD chains; [7] SM clock in MHz
 * during the stream (clock64 against globaltimer).  Needs no handle.
 */
int shd_mix_probe(double out[8]);

#ifdef __cplusplus
}
#endif
#endif /* SHD_BENCH_H */
