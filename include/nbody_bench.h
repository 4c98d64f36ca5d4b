/*
 * include/nbody_bench.h -- measurement helpers of libnbody.so that are NOT part of the method's API (bench.py and
 * the reports use them; see DESIGN.md section 6 for what the numbers are used for).  Same conventions as nbody.h.
 */
#ifndef NBODY_BENCH_H_
#define NBODY_BENCH_H_

#include "nbody.h"

#ifdef __cplusplus
extern "C" {
#endif

/* ------------------------------------------------------------------------------------------------------------
 * nbody_probe_peak -- chip micro-probes behind the roofline denominators of K_force (PAPER.md:49 quotes Tflop/s
 * per GPU as a fraction of peak; DESIGN.md section 6 says which peak).  Runs a loop of one instruction class on every
 * SM (2048 threads per SM, 8 independent chains per thread) for about `millis` ms and returns the achieved rate in
 * 1e12 thread-operations per second in tera_ops_host[0] and the SM clock in MHz measured inside that kernel
 * (clock64 / globaltimer) in tera_ops_host[1]; HOST array of 2.
 *   kind 0 = FFMA (fp32; one FFMA = ONE operation), 1 = DADD (fp64 add), 2 = F2F (fp64->fp32->fp64 round trip, 2 ops),
 *   3 = MUFU.RSQ, 4 = the literal difference pattern DADD + F2F + FADD (3 ops), 5 = packed FFMA2 with two fresh
 *   64-bit register operands, 6 = packed FFMA2 with three fresh operands (one FFMA2 = ONE operation = 4 flops),
 *   issue-port probes, one operation = the PAIR: 7 = FFMA2 + SHF (integer ALU pipe), 8 = FFMA2 + DADD (fp64 pipe),
 *   9 = FFMA2 + LDS.128 broadcast (+ 1 LOP3).  If the second instruction were hidden behind the FFMA2's second pipe
 *   cycle, kinds 7..9 would run at the rate of kind 5.
 * Synchronises.
 * ---------------------------------------------------------------------------------------------------------- */
int nbody_probe_peak(nbody_ctx *ctx, int kind, int millis, double *tera_ops_host);

#ifdef __cplusplus
}
#endif
#endif /* NBODY_BENCH_H_ */
