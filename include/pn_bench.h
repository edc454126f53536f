/*
 * pn_bench.h -- C-ABI of libpn_bench.so: roofline-denominator probes for bench.py.  NOT part of the product library
 * (libpn.so, include/pn.h): nothing of the hot path lives here, and nothing in libpn.so depends on it.
 *
 * Each probe runs register-only chains of one arithmetic instruction on every SM of the current CUDA device and
 * returns the best of three timed launches (CUDA events on `cuda_stream`) as TFLOP/s, counting an FMA as 2 flops per
 * lane.  They give the measured counterpart of the nominal pipe peaks that DESIGN.md section 6 derives from the unit
 * counts (FP64: 64 lanes per SM; FP32: 128 lanes per SM) and the SM clock.
 *
 * Return value: 0 on success, -2 on a CUDA error (no device, launch failure).  Synchronous.
 */
#ifndef PN_BENCH_H_
#define PN_BENCH_H_

#ifdef __cplusplus
extern "C" {
#endif

/* sustained DFMA rate: the roofline denominator of the fp64 star-star pair kernels */
int pn_bench_fp64_peak(void* cuda_stream, double* tflops_host);

/* sustained FP32 FMA rate; packed = 0: scalar FFMA, packed = 1: the packed two-lane form fma.rn.f32x2 (FFMA2, one
   instruction for two FMAs per thread), which the fp32-pair kernels use */
int pn_bench_fp32_peak(void* cuda_stream, int packed, double* tflops_host);

/* Operand-bandwidth probes behind DESIGN.md section 6.1 (`python bench.py --probes`).  A stream of DFMAs in one-warp blocks,
   12 per SM; *cycles_host = SM cycles per DFMA warp-instruction and sub-partition at the rated clock (the issue limit is 2).
   kind 0: FP64 operand patterns, mode 0: two distinct register operands; 1: three; 2: pairs a += K d, b -= K d (d and K from
           the operand reuse cache in the second); 3: a three-register DFMA next to a one-register DMUL; 4: 1, 1, 3, 3.
   kind 1: a two-register DFMA stream with nx (0, 4 or 8) other-pipe instructions per 16 DFMA, mode 1: SHFL.IDX with the lane
           in a register (2 register reads); 2: SHFL.BFLY with an immediate mask (1); 3: IMAD (3); 4: MOV immediate (0);
           5: LOP3 with an immediate (1); 6: FADD (2); 7: LDS.128 (1). */
int pn_bench_operand_probe(void* cuda_stream, int kind, int mode, int nx, double* cycles_host);

#ifdef __cplusplus
}
#endif
#endif /* PN_BENCH_H_ */
