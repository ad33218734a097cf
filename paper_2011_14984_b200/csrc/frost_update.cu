// frost_update.cu -- the O(N), HBM-bound kernels of the path: gather/pack of the source and sink
// streams (step 1), kick / kick_sf and drift (Eq. 6), and the stable
// slow/fast partition (Eq. 29).
#include "frost_common.cuh"

namespace frost {

// out[k] = {x,y,z,m} of particle idx[k]; zero records for n_idx <= k < n_pad.  One 32-byte record
// per thread: two 16-byte stores, fully coalesced on the write side; reads are coalesced when idx
// is NULL or ascending-dense.
__global__ void pack_xm_kernel(const double *__restrict__ pos, const double *__restrict__ mass, int ld,
                               const int32_t *__restrict__ idx, int n_idx, int n_pad,
                               double4 *__restrict__ out, double wscale, int nan_pad,
                               double4 *__restrict__ zero_tail, int *__restrict__ eq_flag,
                               const int32_t *__restrict__ eq_ref) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n_pad) return;
    // the padding of the companion vector stream (accelerations written later by a reduction) is
    // zeroed here, so that no separate memset is needed
    if (zero_tail && k >= n_idx) zero_tail[k] = make_double4(0.0, 0.0, 0.0, 0.0);
    // 1: NaN (time-step streams: the candidate of a padding record drops out of every fmin); 2: far away
    // (force streams: a padding record must coincide with no particle, see SymGradientFast); 0: zeros
    const double fill = nan_pad == 1 ? __longlong_as_double(0x7ff8000000000000LL) : (nan_pad == 2 ? 1e150 : 0.0);
    double4 r = make_double4(fill, fill, fill, 0.0);
    if (k < n_idx) {
        const int i = idx ? idx[k] : k;
        r = make_double4(pos[i], pos[(size_t)ld + i], pos[2 * (size_t)ld + i], mass[i] * wscale);
        // equal-mass detection for the pair-symmetric sweeps (SymNewtonT<true>): bitwise comparison
        // against the first particle of the list eq_ref (NULL = particle 0)
        if (eq_flag && __double_as_longlong(mass[i]) != __double_as_longlong(mass[eq_ref ? eq_ref[0] : 0]))
            *eq_flag = 0;
    }
    out[k] = r;
}

// out[k] = {p_x, p_y, p_z, w} of particle idx[k] (accelerations or velocities); zero padding.
// w = 1.0, or with w_index the list position k in the low word (the time-step sweeps that enter their
// fast pairs into a union-find forest; position 0 is a valid value, so .w is not a "real record" flag).
__global__ void pack_vec_kernel(const double *__restrict__ planes, int ld,
                                const int32_t *__restrict__ idx, int n_idx, int n_pad,
                                double4 *__restrict__ out, int w_index) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n_pad) return;
    double4 r = make_double4(0.0, 0.0, 0.0, 0.0);
    if (k < n_idx) {
        const int i = idx ? idx[k] : k;
        r = make_double4(planes[i], planes[(size_t)ld + i], planes[2 * (size_t)ld + i],
                         w_index ? __hiloint2double(0, k) : 1.0);
    }
    out[k] = r;
}

// vec[k].w <- the component label of list position k in its low word (never read as a number)
__global__ void pack_label_kernel(const int *__restrict__ lab, int n_idx, int n_pad, double4 *__restrict__ vec) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n_pad) return;
    vec[k].w = __hiloint2double(0, k < n_idx ? lab[k] : -2);
}

__global__ void kick_kernel(double *__restrict__ vel, const double *__restrict__ acc,
                            const double *__restrict__ grad, int ld, const int32_t *__restrict__ idx,
                            int n_idx, double c, double kappa) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n_idx) return;
    const int i = idx ? idx[k] : k;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const size_t o = (size_t)d * ld + i;
        double a = acc[o];
        if (grad) a = fma(kappa, grad[o], a);
        vel[o] = fma(c, a, vel[o]);
    }
}

// kick followed by drift of the same particles in one pass (the two middle operator pairs of Alg. 2)
__global__ void kick_drift_kernel(double *__restrict__ pos, double *__restrict__ vel,
                                  const double *__restrict__ acc, const double *__restrict__ grad, int ld,
                                  const int32_t *__restrict__ idx, int n_idx, double ck, double kappa,
                                  double cd) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n_idx) return;
    const int i = idx ? idx[k] : k;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const size_t o = (size_t)d * ld + i;
        double a = acc[o];
        if (grad) a = fma(kappa, grad[o], a);
        const double v = fma(ck, a, vel[o]);
        vel[o] = v;
        pos[o] = fma(cd, v, pos[o]);
    }
}

__global__ void drift_kernel(double *__restrict__ pos, const double *__restrict__ vel, int ld,
                             const int32_t *__restrict__ idx, int n_idx, double c) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n_idx) return;
    const int i = idx ? idx[k] : k;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const size_t o = (size_t)d * ld + i;
        pos[o] = fma(c, vel[o], pos[o]);
    }
}

// Dense lists (idx == NULL): y[i] = fma(c, GRAD ? fma(kappa, g[i], x[i]) : x[i], y[i]) on the three planes --
// the kick (y = vel, x = acc, g = grad) and the drift (y = pos, x = vel) -- with four particles per thread
// (kDenseU = 2; two with the gradient term, whose third operand would otherwise cost the occupancy) as
// 16-byte accesses, every load issued before the first store.  Measured at N = 2^20, back to back over
// rotating buffers (bench.py other_rows; profiles/rows_ncu_r3.md): see there.  Same fma per element as the
// one-particle kernels: same bits.  The gather/pack kernel stays one record per thread: two records per
// thread store 64 contiguous bytes as strided 16-byte pieces and measured 15 % slower.
// n2 = n / 2 double2 per plane; an odd last particle is done by thread 0 of block 0.
constexpr int kDenseNT = 256;
template <bool GRAD, int kDenseU>
__global__ void __launch_bounds__(kDenseNT) update_dense_kernel(double *__restrict__ y, const double *__restrict__ x,
                                                               const double *__restrict__ g, int ld, int n,
                                                               double c, double kappa) {
    const int n2 = n >> 1, ld2 = ld >> 1;
    const int k0 = blockIdx.x * (kDenseNT * kDenseU) + threadIdx.x;
    double2 vy[3][kDenseU], vx[3][kDenseU], vg[3][kDenseU];
#pragma unroll
    for (int d = 0; d < 3; ++d)
#pragma unroll
        for (int u = 0; u < kDenseU; ++u) {
            const int k = k0 + u * kDenseNT;
            if (k < n2) {
                const size_t o = (size_t)d * ld2 + k;
                vx[d][u] = reinterpret_cast<const double2 *>(x)[o];
                if (GRAD) vg[d][u] = reinterpret_cast<const double2 *>(g)[o];
                vy[d][u] = reinterpret_cast<const double2 *>(y)[o];
            }
        }
#pragma unroll
    for (int d = 0; d < 3; ++d)
#pragma unroll
        for (int u = 0; u < kDenseU; ++u) {
            const int k = k0 + u * kDenseNT;
            if (k < n2) {
                double2 a = vx[d][u];
                if (GRAD) { a.x = fma(kappa, vg[d][u].x, a.x); a.y = fma(kappa, vg[d][u].y, a.y); }
                double2 r;
                r.x = fma(c, a.x, vy[d][u].x); r.y = fma(c, a.y, vy[d][u].y);
                reinterpret_cast<double2 *>(y)[(size_t)d * ld2 + k] = r;
            }
        }
    if ((n & 1) && blockIdx.x == 0 && threadIdx.x == 0) {
        const int i = n - 1;
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const size_t o = (size_t)d * ld + i;
            double a = x[o];
            if (GRAD) a = fma(kappa, g[o], a);
            y[o] = fma(c, a, y[o]);
        }
    }
}

__global__ void iota_kernel(int32_t *__restrict__ out, int n, int k0) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k < n) out[k] = k0 + k;
}

// planes[:, idx[k]] = 0 for the list positions k outside [lo, hi): the sinks another rank owns
__global__ void zero_outside_kernel(double *__restrict__ planes, int ld, const int32_t *__restrict__ idx,
                                    int n_idx, int lo, int hi) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n_idx || (k >= lo && k < hi)) return;
    const int i = idx ? idx[k] : k;
    planes[i] = 0.0; planes[(size_t)ld + i] = 0.0; planes[2 * (size_t)ld + i] = 0.0;
}

// ---- stable partition: count per block -> scan of block counts -> scatter ----------------------
constexpr int kPartBlock = 1024;

__device__ __forceinline__ int block_exclusive_scan_1024(int v, int *total) {
    __shared__ int warp_sums[32];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    int inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) warp_sums[w] = inc;
    __syncthreads();
    if (w == 0) {
        int s = warp_sums[lane];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, s, o);
            if (lane >= o) s += t;
        }
        warp_sums[lane] = s;
    }
    __syncthreads();
    const int base = (w > 0) ? warp_sums[w - 1] : 0;
    *total = warp_sums[31];
    __syncthreads();
    return base + inc - v;
}

__global__ void __launch_bounds__(kPartBlock)
part_count_kernel(const double *__restrict__ tau, const int32_t *__restrict__ idx, int n_idx,
                  double pivot, int *__restrict__ block_counts) {
    const int k = blockIdx.x * kPartBlock + threadIdx.x;
    int slow = 0;
    if (k < n_idx) slow = tau[idx ? idx[k] : k] >= pivot;
    const int c = __syncthreads_count(slow);
    if (threadIdx.x == 0) block_counts[blockIdx.x] = c;
}

// single block: exclusive scan of block_counts in place; counts[0] = |S|, counts[1] = |F|
__global__ void __launch_bounds__(kPartBlock)
part_scan_kernel(int *__restrict__ block_counts, int n_blocks, int n_idx, int *__restrict__ counts) {
    int carry = 0;
    for (int b0 = 0; b0 < n_blocks; b0 += kPartBlock) {
        const int b = b0 + threadIdx.x;
        const int v = (b < n_blocks) ? block_counts[b] : 0;
        int total;
        const int ex = block_exclusive_scan_1024(v, &total);
        if (b < n_blocks) block_counts[b] = carry + ex;
        carry += total;
    }
    if (threadIdx.x == 0) { counts[0] = carry; counts[1] = n_idx - carry; }
}

__global__ void __launch_bounds__(kPartBlock)
part_scatter_kernel(const double *__restrict__ tau, const int32_t *__restrict__ idx, int n_idx,
                    double pivot, const int *__restrict__ block_offsets,
                    int32_t *__restrict__ out_slow, int32_t *__restrict__ out_fast) {
    const int k = blockIdx.x * kPartBlock + threadIdx.x;
    int slow = 0, i = 0;
    if (k < n_idx) { i = idx ? idx[k] : k; slow = tau[i] >= pivot; }
    int total;
    const int ex = block_exclusive_scan_1024(slow, &total);
    if (k < n_idx) {
        const int slow_before = block_offsets[blockIdx.x] + ex;
        if (slow) out_slow[slow_before] = i;
        else out_fast[k - slow_before] = i;
    }
}

// ---- diagnostics (Eq. 23): T, U, P, L -------------------------
// One CTA; every thread keeps compensated (two-sum) partial sums over a strided subset, the CTA adds
// them in a fixed tree order -- deterministic, and accurate to ~1e-16 relative for N = 2^20.
struct Comp {
    double s, c;
    __device__ __forceinline__ void add(double v) {      // Neumaier
        const double t = s + v;
        c += (fabs(s) >= fabs(v)) ? (s - t) + v : (v - t) + s;
        s = t;
    }
};
constexpr int kDiagThreads = 1024;

__global__ void __launch_bounds__(kDiagThreads)
diag_kernel(const double *__restrict__ pos, const double *__restrict__ vel, const double *__restrict__ mass,
            const double *__restrict__ phi, int n, int ld, double *__restrict__ out8) {
    __shared__ double sh[2][8][kDiagThreads / 32];
    Comp q[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) q[k].s = q[k].c = 0.0;
    for (int i = threadIdx.x; i < n; i += kDiagThreads) {
        const double m = mass[i];
        const double x = pos[i], y = pos[(size_t)ld + i], z = pos[2 * (size_t)ld + i];
        const double vx = vel[i], vy = vel[(size_t)ld + i], vz = vel[2 * (size_t)ld + i];
        q[0].add(0.5 * m * fma(vz, vz, fma(vy, vy, vx * vx)));
        q[1].add(0.5 * m * phi[i]);
        q[2].add(m * vx); q[3].add(m * vy); q[4].add(m * vz);
        q[5].add(m * fma(y, vz, -z * vy));
        q[6].add(m * fma(z, vx, -x * vz));
        q[7].add(m * fma(x, vy, -y * vx));
    }
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        for (int o = 16; o > 0; o >>= 1) {     // fixed butterfly order
            const double s2 = __shfl_xor_sync(0xffffffffu, q[k].s, o);
            const double c2 = __shfl_xor_sync(0xffffffffu, q[k].c, o);
            q[k].add(s2); q[k].c += c2;
        }
        if (lane == 0) { sh[0][k][w] = q[k].s; sh[1][k][w] = q[k].c; }
    }
    __syncthreads();
    if (threadIdx.x < 8) {
        Comp t; t.s = t.c = 0.0;
        for (int ww = 0; ww < kDiagThreads / 32; ++ww) { t.add(sh[0][threadIdx.x][ww]); t.c += sh[1][threadIdx.x][ww]; }
        out8[threadIdx.x] = t.s + t.c;
    }
}

// ---- launchers ---------------------------------------------------------------------------------
// The dense kernels need an even plane stride and 16-byte aligned planes; lists below kDenseMin particles
// keep the one-particle kernels (more CTAs to spread over the SMs).
constexpr int kDenseMin = 65536;
static bool dense_ok(int ld, const void *a, const void *b, const void *c3) {
    return (ld & 1) == 0 && (((uintptr_t)a | (uintptr_t)b | (uintptr_t)c3) & 15u) == 0;
}
int launch_pack_xm(frost_ctx *c, int ld, const double *pos, const double *mass, const int32_t *idx,
                   int n_idx, int n_pad, double *out, double wscale, int nan_pad, double *zero_tail,
                   int *eq_flag, const int32_t *eq_ref) {
    if (n_pad <= 0) return FROST_OK;
    pack_xm_kernel<<<(n_pad + 255) / 256, 256, 0, c->stream>>>(pos, mass, ld, idx, n_idx, n_pad,
                                                             (double4 *)out, wscale, nan_pad,
                                                             (double4 *)zero_tail, eq_flag, eq_ref);
    return check_launch(c);
}

int launch_pack_vec(frost_ctx *c, int ld, const double *planes, const int32_t *idx, int n_idx,
                    int n_pad, double *out, int w_index) {
    if (n_pad <= 0) return FROST_OK;
    pack_vec_kernel<<<(n_pad + 255) / 256, 256, 0, c->stream>>>(planes, ld, idx, n_idx, n_pad,
                                                              (double4 *)out, w_index);
    return check_launch(c);
}

int launch_pack_label(frost_ctx *c, const int *lab, int n_idx, int n_pad, double *vec) {
    if (n_pad <= 0) return FROST_OK;
    pack_label_kernel<<<(n_pad + 255) / 256, 256, 0, c->stream>>>(lab, n_idx, n_pad, (double4 *)vec);
    return check_launch(c);
}

int launch_kick(frost_ctx *c, int ld, double *vel, const double *acc, const double *grad,
                const int32_t *idx, int n_idx, double cc, double kappa) {
    if (n_idx <= 0) return FROST_OK;
    const double *g = kappa != 0.0 ? grad : nullptr;
    if (!idx && n_idx >= kDenseMin && dense_ok(ld, vel, acc, g)) {
        const int n2 = n_idx >> 1;
        if (g) update_dense_kernel<true, 1><<<(n2 + kDenseNT - 1) / kDenseNT, kDenseNT, 0, c->stream>>>(vel, acc, g, ld, n_idx, cc, kappa);
        else update_dense_kernel<false, 2><<<(n2 + 2 * kDenseNT - 1) / (2 * kDenseNT), kDenseNT, 0, c->stream>>>(vel, acc, nullptr, ld, n_idx, cc, 0.0);
        return check_launch(c);
    }
    kick_kernel<<<(n_idx + 255) / 256, 256, 0, c->stream>>>(vel, acc, g, ld, idx, n_idx, cc, kappa);
    return check_launch(c);
}

int launch_kick_drift(frost_ctx *c, int ld, double *pos, double *vel, const double *acc, const double *grad,
                      const int32_t *idx, int n_idx, double ck, double kappa, double cd) {
    if (n_idx <= 0) return FROST_OK;
    kick_drift_kernel<<<(n_idx + 255) / 256, 256, 0, c->stream>>>(pos, vel, acc, kappa != 0.0 ? grad : nullptr,
                                                                ld, idx, n_idx, ck, kappa, cd);
    return check_launch(c);
}

int launch_drift(frost_ctx *c, int ld, double *pos, const double *vel, const int32_t *idx,
                 int n_idx, double cc) {
    if (n_idx <= 0) return FROST_OK;
    if (!idx && n_idx >= kDenseMin && dense_ok(ld, pos, vel, nullptr)) {
        const int n2 = n_idx >> 1;
        update_dense_kernel<false, 2><<<(n2 + 2 * kDenseNT - 1) / (2 * kDenseNT), kDenseNT, 0, c->stream>>>(pos, vel, nullptr, ld, n_idx, cc, 0.0);
        return check_launch(c);
    }
    drift_kernel<<<(n_idx + 255) / 256, 256, 0, c->stream>>>(pos, vel, ld, idx, n_idx, cc);
    return check_launch(c);
}

int launch_iota(frost_ctx *c, int32_t *out, int n, int k0) {
    if (n <= 0) return FROST_OK;
    iota_kernel<<<(n + 255) / 256, 256, 0, c->stream>>>(out, n, k0);
    return check_launch(c);
}

int launch_zero_outside(frost_ctx *c, int ld, double *planes, const int32_t *idx, int n_idx, int lo, int hi) {
    if (n_idx <= 0 || (lo <= 0 && hi >= n_idx)) return FROST_OK;
    zero_outside_kernel<<<(n_idx + 255) / 256, 256, 0, c->stream>>>(planes, ld, idx, n_idx, lo, hi);
    return check_launch(c);
}

int launch_partition(frost_ctx *c, const double *tau, const int32_t *idx, int n_idx,
                     double tau_pivot, int32_t *out_slow, int32_t *out_fast, int32_t *counts_host) {
    if (n_idx <= 0) { counts_host[0] = counts_host[1] = 0; return FROST_OK; }
    const int nb = (n_idx + kPartBlock - 1) / kPartBlock;
    FROST_TRY(ensure(c, c->blockcnt, (size_t)(nb + 2) * sizeof(int)));
    int *bc = (int *)c->blockcnt.p;
    int *dcounts = bc + nb;
    part_count_kernel<<<nb, kPartBlock, 0, c->stream>>>(tau, idx, n_idx, tau_pivot, bc);
    FROST_TRY(check_launch(c));
    part_scan_kernel<<<1, kPartBlock, 0, c->stream>>>(bc, nb, n_idx, dcounts);
    FROST_TRY(check_launch(c));
    part_scatter_kernel<<<nb, kPartBlock, 0, c->stream>>>(tau, idx, n_idx, tau_pivot, bc, out_slow,
                                                        out_fast);
    FROST_TRY(check_launch(c));
    FROST_CUDA(c, cudaMemcpyAsync(c->pinned_counts, dcounts, 2 * sizeof(int), cudaMemcpyDeviceToHost,
                                  c->stream));
    FROST_CUDA(c, cudaStreamSynchronize(c->stream));
    counts_host[0] = c->pinned_counts[0];
    counts_host[1] = c->pinned_counts[1];
    return FROST_OK;
}

int launch_diag(frost_ctx *c, int n, int ld, const double *pos, const double *vel, const double *mass,
                const double *phi, double *out8) {
    diag_kernel<<<1, kDiagThreads, 0, c->stream>>>(pos, vel, mass, phi, n, ld, out8);
    return check_launch(c);
}

}  // namespace frost
