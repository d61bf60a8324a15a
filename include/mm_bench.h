/*
 * mm_bench.h -- measurement and self-test hooks of the moment-method library, built as a SEPARATE
 * shared object (paper_2401_15233_b200/libmm_bench.so, csrc/mm_bench.cu) so that the product library
 * (include/mm.h, libmm.so) keeps its contract of never allocating device memory.  These calls
 * cudaMalloc a few KB of scratch of their own and free it before returning.  Used by bench.py (roofline
 * denominator) and tests/ only.  Same status codes as mm.h (0 = ok, -1 invalid argument, -3 CUDA error).
 */
#ifndef MM_BENCH_H
#define MM_BENCH_H

#ifdef __cplusplus
extern "C" {
#endif

/* FP64 FMA peak of the current device, measured with a register-resident DFMA loop on `stream`
 * (cudaStream_t): 2 flop per FMA, best of `repeats` launches each of two forms of the loop -- multiplier and
 * addend loop-invariant registers (2.17 scheduler cycles per DFMA measured), and the multiplier an instruction
 * immediate (2.00 cycles, the pipe's issue rate) -- 16 independent chains per thread, 8 blocks of 256 threads
 * per SM.  This is the roofline denominator of this FP64-ALU-bound method;
 * MEASURED_PEAKS.json has no FP64 entry.  If sm_mhz != NULL it receives the SM clock during the probe,
 * from the kernel's own clock64() / globaltimer readings (MHz). */
int mm_measure_fp64_peak(void *stream, int repeats, double *tflops, double *sm_mhz);

/* Instruction rates of the FP64 pipe with operands the register-reuse cache cannot supply (the same launch shape
 * as mm_measure_fp64_peak; every instruction reads distinct registers of a 16-value ring), in 10^12 thread
 * instructions per second:  tinstr[0] DFMA d = fma(a, b, d) with three distinct registers, [1] DMUL, [2] DADD.
 * On B200 the DFMA of mm_measure_fp64_peak (multiplier and addend loop-invariant) and DMUL / DADD issue every 2
 * cycles per scheduler, a DFMA with three distinct register operands every 3: the realistic ceiling of code that is
 * not a polynomial in one variable. */
int mm_measure_fp64_operand_rates(void *stream, int repeats, double tinstr[3]);

/* Accuracy of the library's own elementary functions, measured on `stream` over n pseudo-random
 * arguments: max relative error in units of 2^-53 of
 * max_ulp[0] the branch-free reciprocal and [1] square root against IEEE (1e-30 .. 1e30),
 * [2] the tabulated a(P*), b(P*) of Eq 29c-d on (0, 3] against the direct formulas
 *     with libm pow / exp (whose own conditioning, P*^2 eps in the exponent, is ~10 units at P* = 3). */
int mm_selftest_fastmath(void *stream, int n, double max_ulp[3]);

#ifdef __cplusplus
}
#endif
#endif /* MM_BENCH_H */
