/* include/mem_bench.h -- FP64 issue microbenchmarks of libmem_b200.so, for bench.py --microbench and the
 * roofline discussion of DESIGN.md section 5.  Not part of the integrator's interface: a user of include/mem.h
 * needs none of these.  (mem_measure_fp64_peak, the roofline denominator of every bench line, is declared in
 * mem.h.)  Same conventions as mem.h: mem_status return codes, message in mem_last_error(). */
#ifndef MEM_B200_BENCH_H
#define MEM_B200_BENCH_H
#include "mem.h"

#ifdef __cplusplus
extern "C" {
#endif

/* The same measurement with three distinct 64-bit register operands per DFMA (x = fma(x, y, z), y and z in
 * registers): what the register file sustains for generic fused multiply-adds, about 2/3 of the figure
 * above on B200.  Reported beside the roofline as the ceiling of register-operand code. */
mem_status mem_measure_fp64_peak_rrr(int32_t repeats, double* tflops, void* cuda_stream);

/* The family of FP64 issue microbenchmarks behind the roofline discussion.  Every kind runs
 * 8 independent FP64 instruction chains per thread; *tflops = 2 * FP64 instructions / second / 1e12 (i.e. an FMA
 * counts 2 in every kind, so the figures compare instruction rates).  kind 0: DFMA with two uniform operands (=
 * mem_measure_fp64_peak); 1: DFMA with three register operands (= ..._rrr); 2: 5 DFMA : 2 DMUL : 1 DADD with
 * shuffled register operands; 3 / 4: kind 0 plus 8 / 16 independent integer instructions per 8 DFMAs; 5: DMUL and
 * 6: DADD with two register operands. */
mem_status mem_measure_fp64_rate(int32_t kind, int32_t repeats, double* tflops, void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* MEM_B200_BENCH_H */
