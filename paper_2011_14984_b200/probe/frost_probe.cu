// frost_probe.cu -- register-only FP64 issue-rate probes (run on every SM).
// MEASURED_PEAKS.json has no fp64 entry, and the FP64 pipe of sm_100a turned out not to be a
// plain "one warp instruction per 2 cycles" unit: these probes measure what the sweep kernels
// are bounded by.  bench.py times modes 0/3 next to the headline
// number; `python bench.py --probe` prints the whole table.
//
// Built into its own library (libfrost_probe.so, bench only): not part of the product's C-ABI.
#include <cuda_runtime.h>

#include "frost_probe.h"

namespace frost {

// Every mode executes 64 FP64-pipe instructions per thread per iteration; all operands are
// thread-dependent so nothing is promoted to uniform registers.
template <int MODE>
__global__ void __launch_bounds__(256) fp64_probe_kernel(double *out, int iters, double seed) {
    __shared__ double4 sh[256];
    sh[threadIdx.x] = make_double4(seed, seed * 2, seed * 3, seed * 4);
    __syncthreads();
    double a[8], b[8], c[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        a[k] = seed + (double)(threadIdx.x + k) * 1e-6;
        b[k] = 1.0 - 1e-9 * (double)(k + 1 + threadIdx.x);
        c[k] = seed * 1e-3 * (double)(k + 1 + threadIdx.x);
    }
    double m0 = seed + threadIdx.x, m1 = seed * 3 + threadIdx.x;
    int ic[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) ic[k] = threadIdx.x + k;
    double sink = 0.0;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            if (MODE == 10 || MODE == 11) {   // ONE dependent chain per thread: 8 x 8 instructions = latency
#pragma unroll
                for (int k = 0; k < 8; ++k) a[0] = (MODE == 10) ? fma(a[0], b[0], c[0]) : a[0] + b[0];
                continue;
            }
            if (MODE == 5) {            // triples sharing one multiplicand, adjacent (operand reuse)
#pragma unroll
                for (int k = 0; k < 2; ++k) {
                    const double w = b[(r + k) & 7];
                    asm("fma.rn.f64 %0, %3, %4, %0;\n\tfma.rn.f64 %1, %3, %5, %1;\n\t"
                        "fma.rn.f64 %2, %3, %6, %2;"
                        : "+d"(a[3 * k]), "+d"(a[3 * k + 1]), "+d"(a[3 * k + 2])
                        : "d"(w), "d"(c[3 * k]), "d"(c[3 * k + 1]), "d"(c[3 * k + 2]));
                }
                a[6] = a[6] + b[6];
                a[7] = a[7] + b[7];
                continue;
            }
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                if (MODE == 0) a[k] = fma(a[k], b[0], c[0]);          // 1 RF read + 2 reused
                else if (MODE == 1) a[k] = a[k] + b[k];               // DADD, 2 register pairs
                else if (MODE == 2) a[k] = a[k] * b[k];               // DMUL, 2 register pairs
                else if (MODE == 3) a[k] = (r & 1) ? fma(a[k], a[k], c[k]) : ((r & 2) ? a[k] + b[k] : a[k] * b[k]);
                else if (MODE == 4) a[k] = fma(b[k], c[k], a[k]);     // DFMA, 3 distinct register pairs
                else if (MODE == 6) a[k] = fma(a[k], b[k], 1.5);      // DFMA, 2 register pairs + immediate
                else a[k] = a[k] + b[(k + r) & 7];                    // modes 7-9: DADD stream + extras
            }
            if ((r & 1) == 1) {          // extras once per 16 FP64 instructions
                if (MODE == 7) {         // 12 integer-ALU instructions
#pragma unroll
                    for (int x = 0; x < 4; ++x) ic[x] = (ic[x] ^ (ic[(x + 1) & 3] >> 3)) + it;
                }
                if (MODE == 8) {         // 2 MUFU.RSQ64H
                    asm volatile("rsqrt.approx.ftz.f64 %0, %0;" : "+d"(m0));
                    asm volatile("rsqrt.approx.ftz.f64 %0, %0;" : "+d"(m1));
                }
                if (MODE == 9) {         // 4 broadcast LDS.128
                    const double4 s0 = sh[(it * 8 + r) & 255], s1 = sh[(it * 8 + r + 1) & 255];
                    asm volatile("" ::"d"(s0.x), "d"(s0.y), "d"(s0.z), "d"(s0.w), "d"(s1.x), "d"(s1.y), "d"(s1.z), "d"(s1.w));
                }
            }
        }
    }
    double s = sink + m0 + m1;
#pragma unroll
    for (int k = 0; k < 8; ++k) s += a[k];
#pragma unroll
    for (int k = 0; k < 4; ++k) s += ic[k];
    if (s == 123.456) out[blockIdx.x * blockDim.x + threadIdx.x] = s;   // never true: keeps the chains
}

}  // namespace frost

extern "C" int frost_fp64_probe(int device, void *stream, int mode, int iters, int blocks_per_sm, double *scratch,
                                int64_t *out_instr) {
    using namespace frost;
    if (!scratch || iters < 1 || blocks_per_sm < 1 || mode < 0 || mode > 11) return -1;
    int prev = -1, sms = 0;
    if (cudaGetDevice(&prev) != cudaSuccess) return -2;
    if (prev != device && cudaSetDevice(device) != cudaSuccess) return -2;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device) != cudaSuccess) return -2;
    const int grid = sms * blocks_per_sm;
    cudaStream_t st = (cudaStream_t)stream;
#define FROST_PROBE_CASE(M) \
    case M: fp64_probe_kernel<M><<<grid, 256, 0, st>>>(scratch, iters, 0.5); break;
    switch (mode) {
        FROST_PROBE_CASE(0) FROST_PROBE_CASE(1) FROST_PROBE_CASE(2) FROST_PROBE_CASE(3)
        FROST_PROBE_CASE(4) FROST_PROBE_CASE(5) FROST_PROBE_CASE(6) FROST_PROBE_CASE(7)
        FROST_PROBE_CASE(8) FROST_PROBE_CASE(9) FROST_PROBE_CASE(10) FROST_PROBE_CASE(11)
    }
#undef FROST_PROBE_CASE
    if (out_instr) *out_instr = (int64_t)grid * 256 * (int64_t)iters * 64;   // thread-level FP64 instructions
    const cudaError_t e = cudaGetLastError();
    if (prev != device) cudaSetDevice(prev);
    return e == cudaSuccess ? 0 : -2;
}
