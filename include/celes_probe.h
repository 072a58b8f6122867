/* celes_probe.h -- FP32 throughput probes of libceles.so: measurement tools used by bench.py to calibrate the roofline
 * of the coupling kernel on the GPU and at the clocks of the run.  Not part of the method of arxiv 1706.02145 and not
 * needed by a user of celes.h.  Error codes are those of celes.h. */
#ifndef CELES_PROBE_H
#define CELES_PROBE_H

#ifdef __cplusplus
extern "C" {
#endif

/* FP32 peak probe: runs an FFMA-only kernel (independent chains, every SM) and reports the achieved
 * FLOP/s (2 flop per FMA).  variant 0: three-register FFMA; 1: FFMA with an immediate multiplicand;
 * 2: packed fma.rn.f32x2 (all three with operands that stay in the operand reuse cache); 3: packed fma.rn.f32x2 with
 * three register operands per instruction and none shared by consecutive instructions; 4: as 3 with the packed
 * multiplicand shared by eight consecutive instructions.  3 and 4 bracket what a stream shaped like the pair body
 * (coefficient x packed complex + packed accumulator) can sustain.  Synchronises the stream. */
int celes_fp32_peak_probe(int variant, int iters, double* flops_per_s, double* milliseconds, void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* CELES_PROBE_H */
