/*
 * frost_probe.h -- measurement probe, built into its own library libfrost_probe.so (bench only; not part
 * of libfrost_b200.so or of the C-ABI of include/frost.h).  Not a step of the path: bench.py uses it to
 * measure the FP64 issue rates the roofline of DESIGN.md section 5 is built on (MEASURED_PEAKS.json
 * carries no fp64 figure).
 */
#ifndef FROST_PROBE_H
#define FROST_PROBE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* FP64 issue-rate probes (register-only chains, 64 FP64 instructions per thread per iteration,
 * blocks_per_sm CTAs of 256 threads per SM).  mode: 0 DFMA with two loop-invariant operands,
 * 1 DADD, 2 DMUL, 3 mixed, 4 DFMA with three distinct register pairs, 5 DFMA triples sharing an
 * operand, 6 DFMA with an immediate, 7/8/9 a DADD stream plus integer-ALU / MUFU / LDS
 * instructions, 10/11 one dependent DFMA / DADD chain per thread (latency: run with blocks_per_sm = 1).
 * scratch: device buffer of >= num_SMs*blocks_per_sm*256 doubles (never written in
 * practice).  *out_instr (HOST, nullable) = thread-level FP64 instructions executed.  Timed with
 * CUDA events by bench.py --probe.  Launched on `stream` (cudaStream_t as
 * void*) of CUDA device `device`; returns 0, -1 (bad argument) or -2 (CUDA error).  Asynchronous. */
int frost_fp64_probe(int device, void *stream, int mode, int iters, int blocks_per_sm, double *scratch,
                     int64_t *out_instr);

#ifdef __cplusplus
}
#endif
#endif /* FROST_PROBE_H */
