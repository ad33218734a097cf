// frost_probe.cu -- register-only FP64 issue-rate probe (DFMA / DADD / DMUL chains on every SM).
// MEASURED_PEAKS.json has no fp64 entry; bench.py times this kernel with CUDA events to obtain the
// sustained FP64-pipe rate the sweep rooflines are quoted against.
#include "frost_common.cuh"

namespace frost {

template <int MODE>
__global__ void __launch_bounds__(256) fp64_probe_kernel(double *out, int iters, double seed) {
    double a[8], b = seed, cst = 1.0 - seed * 1e-9;
#pragma unroll
    for (int k = 0; k < 8; ++k) a[k] = seed + (double)(threadIdx.x + k) * 1e-6;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 8; ++r) {
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                if (MODE == 0) a[k] = fma(a[k], cst, b);
                else if (MODE == 1) a[k] = a[k] + b;
                else if (MODE == 2) a[k] = a[k] * cst;
                else a[k] = (r & 1) ? fma(a[k], cst, b) : ((r & 2) ? a[k] + b : a[k] * cst);
            }
        }
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < 8; ++k) s += a[k];
    if (s == 123.456) out[blockIdx.x * blockDim.x + threadIdx.x] = s;   // never true: keeps the chains
}

}  // namespace frost

extern "C" int frost_fp64_probe(frost_ctx *c, int mode, int iters, int blocks_per_sm, double *scratch,
                                int64_t *out_instr) {
    using namespace frost;
    if (!c || !scratch || iters < 1 || blocks_per_sm < 1 || mode < 0 || mode > 3) return FROST_EINVAL;
    FROST_CUDA(c, cudaSetDevice(c->device));
    const int grid = c->num_sms * blocks_per_sm;
    switch (mode) {
        case 0: fp64_probe_kernel<0><<<grid, 256, 0, c->stream>>>(scratch, iters, 0.5); break;
        case 1: fp64_probe_kernel<1><<<grid, 256, 0, c->stream>>>(scratch, iters, 0.5); break;
        case 2: fp64_probe_kernel<2><<<grid, 256, 0, c->stream>>>(scratch, iters, 0.5); break;
        default: fp64_probe_kernel<3><<<grid, 256, 0, c->stream>>>(scratch, iters, 0.5); break;
    }
    if (out_instr) *out_instr = (int64_t)grid * 256 * (int64_t)iters * 64;   // thread-level FP64 instructions
    return check_launch(c);
}
