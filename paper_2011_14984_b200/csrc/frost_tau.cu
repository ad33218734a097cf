// frost_tau.cu -- the time-step sweep of one hierarchy level (Eq. 49-54; assign_timesteps of Alg. 3,
// PAPER.md:592-593) with exact tile-level pruning.
//
// tau_i is a MINIMUM over pairs, and almost no pair defines it.  Every candidate obeys
//     c_ij >= min( eta t_ff / (1 + (3/2) eta (v/r) t_ff),  eta r v / ((1+eta) v^2 + eta mu / r) )
// (from s(q) >= 1/(1+|q|), |q_ff| <= (3/2) eta (v/r) t_ff, |q_fb| <= eta (1 + mu/(v^2 r)); the first
// bound grows with r and falls with v and mu, the second grows with r, falls with mu and is unimodal
// in v), so a whole block of pairs can be discarded when the bound, evaluated at the smallest
// distance, the extreme relative speeds and the largest mass sum the block allows, is not below any
// running minimum involved.  To make blocks compact the level's particles are put in Morton order
// first (the minimum does not depend on the order, so the result stays bitwise the same):
//
//   1. bounding box, 30-bit Morton keys, cub radix sort of (key, position in the list);
//   2. gather/pack of {x, G m} and {v} in that order, one bounding-box record per 32 particles
//      (position box, velocity box, min / max of G m; outward-rounded fp32), tau64[] = +inf;
//   3. pass 1: every A tile against its own (diagonal) block, one-sided -- after it every particle
//      has met its nearest neighbours and tau64 is close to final;
//   4. pass 2: the pair-symmetric rotation sweep of frost_sym.cu over the off-diagonal tile pairs
//      (the warps of a CTA take the chunks of a tile in round-robin order but are synchronised only
//      once per tile: the B-side minima go out by atomicMin, so nothing is combined in shared memory),
//      where a warp first tests its 32*KA resident particles' box against the box of the 32-particle
//      chunk it is about to meet and skips the chunk (32 rotation steps) if the bound allows;
//   5. both sides publish their minima with 64-bit atomicMin on the bit pattern (tau >= 0): the minimum
//      is exact whatever the order, so results are bitwise reproducible; tau64 doubles as the
//      shared upper bound that later blocks are tested against.
//
// The fp32 bound arithmetic uses strict one-sided comparisons, so overflow / underflow / NaN can only
// cause an evaluation, never a wrong skip; blocks whose |q| could exceed 1e8 (where s(q) itself
// loses digits) are always evaluated.
#include <cub/device/device_radix_sort.cuh>

#include "frost_pairs.cuh"

namespace frost {

constexpr int kTauNT = 128;          // threads per CTA = records per B tile
constexpr int kTauKA = 2;            // resident A particles per thread (A tile = 256); 4 / 2 / 1: 82 / 70 / 85 ms at N = 262144
constexpr int kTauWarps = kTauNT / 32;

struct __align__(16) TauBox {        // bounding record of 32 consecutive particles (64 bytes)
    float lo[3], hi[3], vlo[3], vhi[3], gmin, gmax, pad0, pad1;
};

struct TauParams {
    const double4 *xm, *vv;          // packed records in Morton order: {x,y,z,G m}, {vx,vy,vz,.}
    const TauBox *box;               // one per 32 records
    unsigned long long *tau64;       // bit patterns of the running minima (also the upper bounds)
    int n_tiles;                     // tiles of kTauNT records
    int seg_tiles;                   // B tiles per CTA (pass 2)
    int diag_only;                   // pass 1
    int prune;                       // 0: evaluate everything (tests)
    double eta_ff, eta_fb;
    // a split hierarchy entry (reading 24): every pair with a candidate below `pivot` is united
    // in the union-find forest over the SORTED positions; such a pair must never be discarded, so the
    // discard test then runs against max(running minimum, pivot)
    double pivot;                    // 0 when forest is NULL
    int *forest;
};

__device__ __forceinline__ double tau_from_bits(unsigned long long b) { return __longlong_as_double((long long)b); }
__device__ __forceinline__ void atomic_min_tau(unsigned long long *p, double v) {
    if (v == v) atomicMin(p, (unsigned long long)__double_as_longlong(v));    // v >= 0: bit order = value order
}

// ---- 1. bounding box of the level: one partial box per CTA, then one CTA over the partial boxes ---
// (pos = NULL: second stage, `idx`-less reduction of the n partial boxes stored as box6[b*6 + 0..5])
__global__ void __launch_bounds__(1024)
tau_bbox_kernel(const double *__restrict__ pos, int ld, const int32_t *__restrict__ idx, int n,
                const double *__restrict__ part_in, double *box6) {
    __shared__ double sh[6][32];
    double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300};
    if (!pos) {
        for (int b = threadIdx.x; b < n; b += 1024) {
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                lo[d] = fmin(lo[d], part_in[b * 6 + d]); hi[d] = fmax(hi[d], part_in[b * 6 + 3 + d]);
            }
        }
    }
    for (int k = blockIdx.x * 1024 + threadIdx.x; pos && k < n; k += gridDim.x * 1024) {
        const int i = idx ? idx[k] : k;
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const double x = pos[(size_t)d * ld + i];
            lo[d] = fmin(lo[d], x); hi[d] = fmax(hi[d], x);
        }
    }
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        for (int o = 16; o > 0; o >>= 1) {
            lo[d] = fmin(lo[d], __shfl_xor_sync(0xffffffffu, lo[d], o));
            hi[d] = fmax(hi[d], __shfl_xor_sync(0xffffffffu, hi[d], o));
        }
        if ((threadIdx.x & 31) == 0) { sh[d][threadIdx.x >> 5] = lo[d]; sh[3 + d][threadIdx.x >> 5] = hi[d]; }
    }
    __syncthreads();
    if (threadIdx.x < 6) {
        double v = sh[threadIdx.x][0];
        for (int w = 1; w < 32; ++w) v = threadIdx.x < 3 ? fmin(v, sh[threadIdx.x][w]) : fmax(v, sh[threadIdx.x][w]);
        box6[blockIdx.x * 6 + threadIdx.x] = v;
    }
}

__device__ __forceinline__ unsigned spread10(unsigned v) {      // 10 bits -> every third bit
    v = (v | (v << 16)) & 0x030000FFu;
    v = (v | (v << 8)) & 0x0300F00Fu;
    v = (v | (v << 4)) & 0x030C30C3u;
    v = (v | (v << 2)) & 0x09249249u;
    return v;
}

__global__ void tau_morton_kernel(const double *__restrict__ pos, int ld, const int32_t *__restrict__ idx, int n,
                                  const double *__restrict__ box6, unsigned *__restrict__ keys,
                                  int32_t *__restrict__ vals) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    const int i = idx ? idx[k] : k;
    unsigned key = 0;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const double lo = box6[d], w = box6[3 + d] - lo;
        double q = w > 0.0 ? (pos[(size_t)d * ld + i] - lo) / w * 1024.0 : 0.0;
        int c = (int)q;
        c = c < 0 ? 0 : (c > 1023 ? 1023 : c);
        key |= spread10((unsigned)c) << d;
    }
    keys[k] = key;
    vals[k] = k;
}

// sorted position -> global particle index
__global__ void tau_gather_idx_kernel(const int32_t *__restrict__ idx, const int32_t *__restrict__ perm, int n,
                                      int32_t *__restrict__ sidx) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k < n) sidx[k] = idx ? idx[perm[k]] : perm[k];
}

// ---- 2. one bounding record per 32 packed records; tau64 = +inf ------------------------------------
__global__ void tau_box_kernel(const double4 *__restrict__ xm, const double4 *__restrict__ vv, int n_pad,
                               TauBox *__restrict__ box, unsigned long long *__restrict__ tau64) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;       // n_pad is a multiple of 32
    if (k >= n_pad) return;
    tau64[k] = 0x7ff0000000000000ull;
    const double4 r = xm[k], v = vv[k];
    const bool real = r.x == r.x;                               // padding records carry NaN positions
    const double inf = __longlong_as_double(0x7ff0000000000000LL);
    double lo[7], hi[7];
    const double q[7] = {r.x, r.y, r.z, v.x, v.y, v.z, r.w};
#pragma unroll
    for (int d = 0; d < 7; ++d) {
        lo[d] = real ? q[d] : inf; hi[d] = real ? q[d] : -inf;
        for (int o = 16; o > 0; o >>= 1) {
            lo[d] = fmin(lo[d], __shfl_xor_sync(0xffffffffu, lo[d], o));
            hi[d] = fmax(hi[d], __shfl_xor_sync(0xffffffffu, hi[d], o));
        }
    }
    if ((threadIdx.x & 31) == 0) {
        TauBox b;
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            b.lo[d] = __double2float_rd(lo[d]); b.hi[d] = __double2float_ru(hi[d]);
            b.vlo[d] = __double2float_rd(lo[3 + d]); b.vhi[d] = __double2float_ru(hi[3 + d]);
        }
        b.gmin = __double2float_rd(lo[6]); b.gmax = __double2float_ru(hi[6]);
        b.pad0 = b.pad1 = 0.0f;
        box[k >> 5] = b;
    }
}

// Block constants of the discard test.  For a pair (i, j) of the two boxes let T = max of the two
// particles' running minima and v its relative speed.  With r >= r_lo, mu in [mu_lo, mu_hi]:
//   fly-by bound > T  <=  T (1+eta) v^2 - eta r v + T eta mu / r < 0, which holds for
//       1.3 T mu_hi / r_lo^2 < v < 0.79 eta r_lo / (T (1+eta))   if   T^2 < eta r_lo^3 / (6.3 (1+eta) mu_hi)
//   free-fall bound > T  <=  r_lo^3 eta_ff^2 (1-phi)^2 > mu_hi T^2,  phi = 1.185 eta_fb/(1+eta_fb)
//       (1.5 T v < phi r_lo by the upper speed limit)
//   |q| <= 1e8  <=  v^2 > mu_hi / (1e8 r_lo)  and  v^2 < 1e16 mu_lo / r_hi
// i.e. per pair:  T^2 < K,  v^2 T^2 < C,  v^2 > D T^2,  v^2 > V0,  v^2 < V1   (12 FP64 instructions
// with the 6 of v^2).  Relative speeds are not spatially coherent, so they are checked pair by pair;
// everything that depends on positions and masses is per block.  Strict comparisons: a NaN / inf /
// zero constant can only make the test fail.
struct TauConsts { double K, C, D, V0, V1; };

__device__ __forceinline__ bool tau_block_consts(const TauBox &A, const TauBox &B, float eff, float efb,
                                                 TauConsts *o) {
    float r2lo = 0.0f, r2hi = 0.0f;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const float g = fmaxf(0.0f, fmaxf(B.lo[d] - A.hi[d], A.lo[d] - B.hi[d]));
        const float f = fmaxf(fabsf(B.hi[d] - A.lo[d]), fabsf(A.hi[d] - B.lo[d]));
        r2lo = fmaf(g, g, r2lo); r2hi = fmaf(f, f, r2hi);
    }
    const float r_lo = sqrtf(r2lo) * 0.99999f, r_hi = sqrtf(r2hi) * 1.00001f;
    const float mu_hi = (A.gmax + B.gmax) * 1.00001f, mu_lo = (A.gmin + B.gmin) * 0.99999f;
    const float r3 = r_lo * r_lo * r_lo;
    const float phi = 1.185f * efb / (1.0f + efb);
    const float kff = eff * eff * (1.0f - phi) * (1.0f - phi) * r3 / mu_hi;
    const float kfb = efb * r3 / (6.3f * (1.0f + efb) * mu_hi);
    const float K = fminf(kff, kfb) * 0.999f;
    const float cc = 0.79f * efb * r_lo / (1.0f + efb);
    const float dd = 1.3f * mu_hi / (r_lo * r_lo);
    const float C = cc * cc * 0.999f, D = dd * dd * 1.002f;
    const float V0 = mu_hi / (1e8f * r_lo) * 1.002f, V1 = 1e16f * mu_lo / r_hi * 0.999f;
    o->K = (double)K; o->C = (double)C; o->D = (double)D; o->V0 = (double)V0; o->V1 = (double)V1;
    return (r_lo > 0.0f) && (phi < 0.9f) && (K > 0.0f) && (K < 3e38f) && (C > 0.0f) && (C < 3e38f) &&
           (D > 0.0f) && (D < 3e38f) && (V0 > 0.0f) && (V0 < 3e38f) && (V1 > 0.0f) && (V1 < 3e38f);
}

// the candidate of TimestepPolicy::pair (Eq. 49-54), once for both particles of the pair
__device__ __forceinline__ double tau_candidate(double x, double y, double z, double gm, double vx, double vy,
                                                double vz, const double4 &j0, const double4 &j1, double eta_ff,
                                                double eta_fb) {
    const double rx = j0.x - x, ry = j0.y - y, rz = j0.z - z;
    const double ux = j1.x - vx, uy = j1.y - vy, uz = j1.z - vz;
    const double r2 = fma(rz, rz, fma(ry, ry, rx * rx));
    const double v2 = fma(uz, uz, fma(uy, uy, ux * ux));
    const double rv = fma(rz, uz, fma(ry, uy, rx * ux));
    const double mu = gm + j0.w;
    const double ir = rsqrt_full(r2);
    const double iv = rsqrt_full(v2);
    const double ir2 = ir * ir;
    const double mir = mu * ir;
    const double t_ff = rsqrt_full(mir * ir2);
    const double t_fb = (r2 * ir) * iv;
    const double rvr2 = rv * ir2;
    const double q_ff = (rvr2 * t_ff) * (1.5 * eta_ff);
    const double f = rvr2 * t_fb;
    const double q_fb = fma(f, mir * (iv * iv), f) * eta_fb;
    const double c_ff = sym_factor(q_ff) * (t_ff * eta_ff);
    const double c_fb = sym_factor(q_fb) * (t_fb * eta_fb);
    return fmin(c_ff, c_fb);
}

// ---- 3./4. the sweep ------------------------------------------------------------------------------
// grid = (A tiles, segments); pass 1 (diag_only): the kTauKA B tiles of the A tile itself, one-sided;
// pass 2: the B tiles beyond the A tile, two-sided, with chunk-level pruning.
__global__ void __launch_bounds__(kTauNT, 4) tau_sym_kernel(const TauParams prm) {
    constexpr int NT = kTauNT, KA = kTauKA, TA = NT * KA;
    constexpr uint32_t kStageBytes = 2 * NT * kRecBytes;
    const int I = blockIdx.x;
    const int diag_end = (I + 1) * KA;
    const int tile0 = prm.diag_only ? I * KA : diag_end + blockIdx.y * prm.seg_tiles;
    const int tile_end = prm.diag_only ? diag_end : prm.n_tiles;
    if (tile0 >= tile_end || (prm.diag_only && blockIdx.y > 0)) return;
    const int ntiles = min(prm.diag_only ? KA : prm.seg_tiles, tile_end - tile0);

    extern __shared__ __align__(128) unsigned char smem_raw[];
    double4 *tiles = reinterpret_cast<double4 *>(smem_raw);                       // [kStages][2][NT]
    double *tbd2 = reinterpret_cast<double *>(smem_raw + kStages * kStageBytes);   // [2][NT] current minima of the tile
    TauBox *sbox2 = reinterpret_cast<TauBox *>(tbd2 + 2 * NT);                     // [2][kTauWarps]
    uint64_t *full = reinterpret_cast<uint64_t *>(sbox2 + 2 * kTauWarps);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < kStages; ++s) mbar_init(&full[s], 1);
        mbar_fence_init();
    }
    __syncthreads();
    auto issue = [&](int t) {
        const int s = t % kStages;
        mbar_expect_tx(&full[s], kStageBytes);
        double4 *dst = tiles + (size_t)s * 2 * NT;
        const size_t off = (size_t)(tile0 + t) * NT;
        bulk_g2s(dst, prm.xm + off, NT * kRecBytes, &full[s]);
        bulk_g2s(dst + NT, prm.vv + off, NT * kRecBytes, &full[s]);
    };
    if (tid == 0) {
        const int pre = min(kStages, ntiles);
        for (int t = 0; t < pre; ++t) issue(t);
    }

    // resident A particles and the bounding box of this warp's 32*KA of them
    double ax[KA], ay[KA], az[KA], agm[KA], avx[KA], avy[KA], avz[KA], at[KA];
    const int a_first = I * TA + tid;
    const double inf = __longlong_as_double(0x7ff0000000000000LL);
    TauBox A;
    {
        double lo[7], hi[7];
#pragma unroll
        for (int d = 0; d < 7; ++d) { lo[d] = inf; hi[d] = -inf; }
#pragma unroll
        for (int k = 0; k < KA; ++k) {
            const double4 r = prm.xm[a_first + k * NT], v = prm.vv[a_first + k * NT];
            ax[k] = r.x; ay[k] = r.y; az[k] = r.z; agm[k] = r.w; avx[k] = v.x; avy[k] = v.y; avz[k] = v.z;
            at[k] = tau_from_bits(prm.tau64[a_first + k * NT]);
            if (r.x == r.x) {
                const double q[7] = {r.x, r.y, r.z, v.x, v.y, v.z, r.w};
#pragma unroll
                for (int d = 0; d < 7; ++d) { lo[d] = fmin(lo[d], q[d]); hi[d] = fmax(hi[d], q[d]); }
            }
        }
#pragma unroll
        for (int d = 0; d < 7; ++d)
            for (int o = 16; o > 0; o >>= 1) {
                lo[d] = fmin(lo[d], __shfl_xor_sync(0xffffffffu, lo[d], o));
                hi[d] = fmax(hi[d], __shfl_xor_sync(0xffffffffu, hi[d], o));
            }
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            A.lo[d] = __double2float_rd(lo[d]); A.hi[d] = __double2float_ru(hi[d]);
            A.vlo[d] = __double2float_rd(lo[3 + d]); A.vhi[d] = __double2float_ru(hi[3 + d]);
        }
        A.gmin = __double2float_rd(lo[6]); A.gmax = __double2float_ru(hi[6]);
    }
    const float eff = (float)prm.eta_ff, efb = (float)prm.eta_fb;
    const int from = (lane + 31) & 31;

    for (int t = 0; t < ntiles; ++t) {
        const int s = t % kStages;
        const int tile = tile0 + t;
        const bool two_sided = !prm.diag_only;
        // stage the tile's bounding records and the current bounds of its particles (double-buffered by
        // tile parity: the warps are only synchronised once per tile and drift apart inside it)
        TauBox *sbox = sbox2 + (t & 1) * kTauWarps;
        double *tbd = tbd2 + (t & 1) * NT;
        if (tid < kTauWarps * 16)
            reinterpret_cast<float *>(sbox)[tid] = reinterpret_cast<const float *>(prm.box + (size_t)tile * kTauWarps)[tid];
        tbd[tid] = tau_from_bits(prm.tau64[(size_t)tile * NT + tid]);
        mbar_wait(&full[s], (uint32_t)(t / kStages) & 1u);
        __syncthreads();
        // every warp is past tile t-1: its stage can be refilled
        if (tid == 0 && t >= 1 && t - 1 + kStages < ntiles) issue(t - 1 + kStages);
        const double4 *t0 = tiles + (size_t)s * 2 * NT;
        for (int r = 0; r < kTauWarps; ++r) {
            const int c = (warp + r) % kTauWarps;
            double b = inf;
            bool skip = false;
            TauConsts tc;
            if (prm.prune && two_sided) skip = tau_block_consts(A, sbox[c], eff, efb, &tc);
            const double4 *c0 = t0 + c * 32, *c1 = c0 + NT;
            if (skip) {
                // block-level constants, pair-level check of the relative speed against the two
                // particles' own running minima; a pair that fails is evaluated in full
#pragma unroll 2
                for (int step = 0; step < 32; ++step) {
                    const int src = (lane - step) & 31;
                    const double4 j1 = c1[src];
                    const double tb = fmin(b, tbd[c * 32 + src]);        // the traveller's running minimum
                    bool ok = true;
#pragma unroll
                    for (int k = 0; k < KA; ++k) {
                        const double ux = j1.x - avx[k], uy = j1.y - avy[k], uz = j1.z - avz[k];
                        const double v2 = fma(uz, uz, fma(uy, uy, ux * ux));
                        const double T = fmax(fmax(at[k], tb), prm.pivot);
                        const double T2 = T * T;
                        ok = ok && (T2 < tc.K) && (v2 * T2 < tc.C) && (v2 > tc.D * T2) && (v2 > tc.V0) && (v2 < tc.V1);
                    }
                    if (!__all_sync(0xffffffffu, ok)) {
                        const double4 j0 = c0[src];
#pragma unroll
                        for (int k = 0; k < KA; ++k) {
                            const double cand = tau_candidate(ax[k], ay[k], az[k], agm[k], avx[k], avy[k], avz[k],
                                                              j0, j1, prm.eta_ff, prm.eta_fb);
                            at[k] = fmin(at[k], cand);
                            b = fmin(b, cand);
                            if (cand < prm.pivot) uf_union(prm.forest, a_first + k * NT, tile * NT + c * 32 + src);
                        }
                    }
                    b = __shfl_sync(0xffffffffu, b, from);
                }
            } else {
#pragma unroll 2
                for (int step = 0; step < 32; ++step) {
                    const int src = (lane - step) & 31;
                    const double4 j0 = c0[src], j1 = c1[src];
#pragma unroll
                    for (int k = 0; k < KA; ++k) {
                        const double cand = tau_candidate(ax[k], ay[k], az[k], agm[k], avx[k], avy[k], avz[k],
                                                          j0, j1, prm.eta_ff, prm.eta_fb);
                        at[k] = fmin(at[k], cand);
                        b = fmin(b, cand);
                        if (cand < prm.pivot) uf_union(prm.forest, a_first + k * NT, tile * NT + c * 32 + src);
                    }
                    b = __shfl_sync(0xffffffffu, b, from);
                }
            }
            // the chunk's particles collect their minima by atomicMin (exact in any order)
            if (two_sided && b < inf) atomic_min_tau(prm.tau64 + (size_t)tile * NT + c * 32 + lane, b);
        }
    }
#pragma unroll
    for (int k = 0; k < KA; ++k) atomic_min_tau(prm.tau64 + a_first + k * NT, at[k]);
}

// ---- 5. scatter tau and the bins -------------------------------------------------------------------
__global__ void tau_finish_kernel(const unsigned long long *__restrict__ tau64, const int32_t *__restrict__ sidx,
                                  int n, double tau_pivot, double *__restrict__ out_tau,
                                  int32_t *__restrict__ out_bin) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    const double tau = tau_from_bits(tau64[k]);
    const int g = sidx[k];
    out_tau[g] = tau;
    if (out_bin) {      // smallest k >= 0 with tau_pivot 2^-k <= tau (as reduce_tau_kernel)
        int b = 0;
        if (!(tau > 0.0)) b = 2000;
        else {
            double p = tau_pivot;
            while (p > tau && b < 2000) { p *= 0.5; ++b; }
        }
        out_bin[g] = b;
    }
}

// The forest over sorted positions -> a forest over LIST positions whose roots are the smallest list
// position of each component (what split_components expects): two passes over the sorted positions.
__global__ void tau_forest_min_kernel(const int *__restrict__ fs, const int32_t *__restrict__ perm, int n,
                                      int *__restrict__ minlist) {
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p < n) atomicMin(&minlist[uf_find(fs, p)], perm[p]);
}
__global__ void tau_forest_out_kernel(const int *__restrict__ fs, const int32_t *__restrict__ perm, int n,
                                      const int *__restrict__ minlist, int *__restrict__ forest_list) {
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p < n) forest_list[perm[p]] = minlist[uf_find(fs, p)];
}
__global__ void tau_forest_init_kernel(int *__restrict__ fs, int *__restrict__ minlist, int n_pad) {
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p < n_pad) { fs[p] = p; minlist[p] = 0x7fffffff; }
}

// Host driver.  prune = 0 evaluates every block (tests: the pruned result must be bitwise the same).
// forest != NULL (length >= n, over list positions): the fast pairs of the level (candidate < tau_pivot)
// are united in it -- the component search of a split hierarchy entry.
int tau_pruned(frost_ctx *c, int ld, const double *pos, const double *vel, const double *mass,
               const int32_t *idx, int n, double tau_pivot, double *out_tau, int32_t *out_bin, int prune,
               int *forest) {
    if (n <= 0) return FROST_OK;
    constexpr int TA = kTauNT * kTauKA;
    const int n_pad = round_up(n, TA);
    const int n_tiles = n_pad / kTauNT;
    // scratch: keys/vals (in, out), sorted index list, boxes, tau64, cub temp
    size_t cub_bytes = 0;
    cub::DeviceRadixSort::SortPairs(nullptr, cub_bytes, (const unsigned *)nullptr, (unsigned *)nullptr,
                                    (const int32_t *)nullptr, (int32_t *)nullptr, n, 0, 30, c->stream);
    const size_t o_keys = 0, o_keys2 = o_keys + (size_t)n_pad * 4, o_vals = o_keys2 + (size_t)n_pad * 4;
    const size_t o_vals2 = o_vals + (size_t)n_pad * 4, o_sidx = o_vals2 + (size_t)n_pad * 4;
    const size_t o_box6 = o_sidx + (size_t)n_pad * 4, o_boxes = o_box6 + 64;
    const size_t o_tau = o_boxes + (size_t)(n_pad / 32) * sizeof(TauBox);
    const size_t o_fs = o_tau + (size_t)n_pad * 8, o_min = o_fs + (forest ? (size_t)n_pad * 4 : 0);
    const size_t o_cub = o_min + (forest ? (size_t)n_pad * 4 : 0);
    FROST_TRY(ensure(c, c->tau_scratch, o_cub + cub_bytes + 256));
    FROST_TRY(ensure(c, c->recA_xm, (size_t)n_pad * kRecBytes));
    FROST_TRY(ensure(c, c->recA_v, (size_t)n_pad * kRecBytes));
    char *base = (char *)c->tau_scratch.p;
    unsigned *keys = (unsigned *)(base + o_keys), *keys2 = (unsigned *)(base + o_keys2);
    int32_t *vals = (int32_t *)(base + o_vals), *vals2 = (int32_t *)(base + o_vals2);
    int32_t *sidx = (int32_t *)(base + o_sidx);
    double *box6 = (double *)(base + o_box6);
    double *box_part = (double *)keys2;      // <= 256 partial boxes; keys2 is first written by the sort
    TauBox *boxes = (TauBox *)(base + o_boxes);
    unsigned long long *tau64 = (unsigned long long *)(base + o_tau);
    double *xm = (double *)c->recA_xm.p, *vv = (double *)c->recA_v.p;

    const int bb = (n + 8191) / 8192 < 256 ? (n + 8191) / 8192 : 256;       // 8 particles per thread
    if (bb > 1) {
        tau_bbox_kernel<<<bb, 1024, 0, c->stream>>>(pos, ld, idx, n, nullptr, box_part);
        FROST_TRY(check_launch(c));
        tau_bbox_kernel<<<1, 1024, 0, c->stream>>>(nullptr, 0, nullptr, bb, box_part, box6);
    } else {
        tau_bbox_kernel<<<1, 1024, 0, c->stream>>>(pos, ld, idx, n, nullptr, box6);
    }
    FROST_TRY(check_launch(c));
    tau_morton_kernel<<<(n + 255) / 256, 256, 0, c->stream>>>(pos, ld, idx, n, box6, keys, vals);
    FROST_TRY(check_launch(c));
    FROST_CUDA(c, cub::DeviceRadixSort::SortPairs(base + o_cub, cub_bytes, keys, keys2, vals, vals2, n, 0, 30,
                                                  c->stream));
    c->launches += 1;
    tau_gather_idx_kernel<<<(n + 255) / 256, 256, 0, c->stream>>>(idx, vals2, n, sidx);
    FROST_TRY(check_launch(c));
    FROST_TRY(launch_pack_xm(c, ld, pos, mass, sidx, n, n_pad, xm, c->G, 1));      // .w = G m, NaN padding
    FROST_TRY(launch_pack_vec(c, ld, vel, sidx, n, n_pad, vv));
    tau_box_kernel<<<n_pad / 256, 256, 0, c->stream>>>((const double4 *)xm, (const double4 *)vv, n_pad, boxes, tau64);
    FROST_TRY(check_launch(c));

    const size_t smem = (size_t)kStages * 2 * kTauNT * kRecBytes + 2 * kTauNT * sizeof(double) +
                        2 * kTauWarps * sizeof(TauBox) + kStages * sizeof(uint64_t);
    FROST_TRY(set_func_attr(c, tau_sym_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    TauParams prm{};
    prm.xm = (const double4 *)xm; prm.vv = (const double4 *)vv; prm.box = boxes; prm.tau64 = tau64;
    prm.n_tiles = n_tiles; prm.prune = prune; prm.eta_ff = c->eta_ff; prm.eta_fb = c->eta_fb;
    int *fs = (int *)(base + o_fs), *minlist = (int *)(base + o_min);
    prm.pivot = forest ? tau_pivot : 0.0; prm.forest = forest ? fs : nullptr;
    if (forest) {
        tau_forest_init_kernel<<<(n_pad + 255) / 256, 256, 0, c->stream>>>(fs, minlist, n_pad);
        FROST_TRY(check_launch(c));
    }
    const int a_tiles = n_pad / TA;
    prm.diag_only = 1; prm.seg_tiles = kTauKA;
    tau_sym_kernel<<<dim3(a_tiles, 1), kTauNT, smem, c->stream>>>(prm);
    FROST_TRY(check_launch(c));
    if (n_tiles > kTauKA) {
        // pass 2: ~16 waves of CTAs over the triangular tile-pair set
        const long long pairs = (long long)a_tiles * n_tiles - (long long)kTauKA * a_tiles * (a_tiles + 1) / 2;
        long long seg = pairs / (16LL * c->num_sms * 4);
        if (seg < 8) seg = 8;
        if (seg > n_tiles) seg = n_tiles;
        prm.diag_only = 0; prm.seg_tiles = (int)seg;
        const int segs = (int)((n_tiles - kTauKA + seg - 1) / seg);
        tau_sym_kernel<<<dim3(a_tiles, segs), kTauNT, smem, c->stream>>>(prm);
        FROST_TRY(check_launch(c));
    }
    if (forest) {
        tau_forest_min_kernel<<<(n + 255) / 256, 256, 0, c->stream>>>(fs, vals2, n, minlist);
        FROST_TRY(check_launch(c));
        tau_forest_out_kernel<<<(n + 255) / 256, 256, 0, c->stream>>>(fs, vals2, n, minlist, forest);
        FROST_TRY(check_launch(c));
    }
    tau_finish_kernel<<<(n + 255) / 256, 256, 0, c->stream>>>(tau64, sidx, n, tau_pivot, out_tau, out_bin);
    return check_launch(c);
}

}  // namespace frost
