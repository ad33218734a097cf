// frost_sweeps.cu -- the three all-pairs O(N_sink x N_source) fp64 sweeps:
// Newtonian accelerations (Eq. 24/42), gradient accelerations (Eq. 27/43/44) and the symmetrised
// time-step criterion (Eq. 49-54), for sm_100a.
//
// Design: sinks live in registers, K per thread; the packed source stream
// (32-byte records, contiguous in list order) is streamed global/L2 -> shared memory by 1-D TMA
// bulk copies (cp.async.bulk + mbarrier, SASS UBLKCP) through a kStages-deep ring; every warp
// reads each source record as broadcast LDS.128 and evaluates its K pairs on the FP64 pipe.  The
// source list is cut into slices (grid.y); each (sink block, slice) writes one partial per sink
// and a second kernel adds the partials in slice order -- deterministic, no float atomics.  The
// sweeps are FP64-issue bound, so everything that is not inherently fp64 (self-pair test, loop
// and address arithmetic) is kept off the FP64 pipe.
#include "frost_pairs.cuh"

namespace frost {

// ------------------------------------------------------------------------------------------------
// The sweep skeleton.  grid = (sink blocks, source slices); block = NT threads; K sinks per thread.
// ------------------------------------------------------------------------------------------------
template <class P, int K, int NT>
__global__ void __launch_bounds__(NT, (NT * K >= 512 ? 2 : 4))
sweep_kernel(const SweepParams prm) {
    constexpr int kWarps = NT / 32;
    constexpr uint32_t kStageBytes = P::kRecs * kTile * kRecBytes;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double4 *tiles = reinterpret_cast<double4 *>(smem_raw);            // [kStages][kRecs][kTile]
    uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw + kStages * kStageBytes);
    uint64_t *empty = full + kStages;

    const int tid = threadIdx.x;
    const int tile0 = blockIdx.y * prm.tiles_per_slice;
    const int ntiles = min(prm.tiles_per_slice, prm.n_tiles - tile0);

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < kStages; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], kWarps);
        }
        mbar_fence_init();
    }
    __syncthreads();

    auto issue = [&](int t) {   // producer: one thread fills stage t % kStages with tile tile0 + t
        const int s = t % kStages;
        mbar_expect_tx(&full[s], kStageBytes);
        double4 *dst = tiles + (size_t)s * P::kRecs * kTile;
        const size_t off = (size_t)(tile0 + t) * kTile;
        bulk_g2s(dst, prm.src0 + off, kTile * kRecBytes, &full[s]);
        if (P::kRecs == 2) bulk_g2s(dst + kTile, prm.src1 + off, kTile * kRecBytes, &full[s]);
    };
    if (tid == 0) {
        const int pre = min(kStages, ntiles);
        for (int t = 0; t < pre; ++t) issue(t);
    }

    typename P::Sink snk[K];
    typename P::Acc acc[K];
    const int sink0 = blockIdx.x * (NT * K) + tid;
#pragma unroll
    for (int k = 0; k < K; ++k) {
        P::load(snk[k], prm, sink0 + k * NT);
        P::init(acc[k]);
    }

    for (int t = 0; t < ntiles; ++t) {
        const int s = t % kStages;
        mbar_wait(&full[s], (uint32_t)(t / kStages) & 1u);
        const double4 *t0 = tiles + (size_t)s * P::kRecs * kTile;
        const double4 *t1 = t0 + (P::kRecs == 2 ? kTile : 0);
#pragma unroll 4
        for (int j = 0; j < kTile; ++j) {
            const double4 j0 = t0[j];
            const double4 j1 = (P::kRecs == 2) ? t1[j] : j0;
#pragma unroll
            for (int k = 0; k < K; ++k) P::pair(snk[k], acc[k], j0, j1, prm);
        }
        __syncwarp();
        if ((tid & 31) == 0) mbar_arrive(&empty[s]);
        // refill, lagging one tile so the producer warp rarely blocks on its siblings
        if (tid == 0 && t >= 1 && t - 1 + kStages < ntiles) {
            const int tp = t - 1;
            mbar_wait(&empty[tp % kStages], (uint32_t)(tp / kStages) & 1u);
            issue(tp + kStages);
        }
    }

    double *part = prm.partial + (size_t)blockIdx.y * P::kPlanes * prm.n_pad;
#pragma unroll
    for (int k = 0; k < K; ++k) P::store(acc[k], part, prm.n_pad, sink0 + k * NT);
}

// ------------------------------------------------------------------------------------------------
// Partial reduction + scatter.  One thread per sink, slices added in ascending order.
// ------------------------------------------------------------------------------------------------
__global__ void reduce_vec_kernel(const double *__restrict__ partial, int n_pad, int slices, int n_snk,
                                  double scale, const int32_t *__restrict__ idx, int ld,
                                  double *__restrict__ out, double4 *__restrict__ packed, int accumulate, int keep_w = 0) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_snk) return;
    double sx = 0.0, sy = 0.0, sz = 0.0;
    for (int s = 0; s < slices; ++s) {
        const double *p = partial + (size_t)s * 3 * n_pad;
        sx += p[i]; sy += p[n_pad + i]; sz += p[2 * n_pad + i];
    }
    sx *= scale; sy *= scale; sz *= scale;
    const int g = idx ? idx[i] : i;
    if (accumulate) { sx += out[g]; sy += out[(size_t)ld + g]; sz += out[2 * (size_t)ld + g]; }
    out[g] = sx; out[(size_t)ld + g] = sy; out[2 * (size_t)ld + g] = sz;
    if (packed) {
        if (keep_w) { double *q = (double *)(packed + i); q[0] = sx; q[1] = sy; q[2] = sz; }   // .w = label
        else packed[i] = make_double4(sx, sy, sz, 1.0);
    }
}

__global__ void reduce_tau_kernel(const double *__restrict__ partial, int n_pad, int slices, int n_set,
                                  const int32_t *__restrict__ idx, double tau_pivot,
                                  double *__restrict__ out_tau, int32_t *__restrict__ out_bin) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_set) return;
    double tau = partial[i];
    for (int s = 1; s < slices; ++s) tau = fmin(tau, partial[(size_t)s * n_pad + i]);
    const int g = idx ? idx[i] : i;
    out_tau[g] = tau;
    if (out_bin) {
        // smallest k >= 0 with tau_pivot 2^-k <= tau (halving is exact in binary floating point)
        int k = 0;
        if (!(tau > 0.0)) k = 2000;
        else {
            double p = tau_pivot;
            while (p > tau && k < 2000) { p *= 0.5; ++k; }
        }
        out_bin[g] = k;
    }
}

// ------------------------------------------------------------------------------------------------
// Launch planning
// ------------------------------------------------------------------------------------------------
struct Plan { int k, nt, sink_blocks, slices, tiles_per_slice, n_tiles; };

static Plan make_plan(const frost_ctx *c, int n_snk, int n_src, int max_k) {
    Plan pl;
    pl.n_tiles = (n_src + kTile - 1) / kTile;
    if (pl.n_tiles < 1) pl.n_tiles = 1;
    // sinks per thread: register blocking amortises the per-source LDS/loop/MUFU issue slots
    // (measured on B200: K=4 wins from ~32k sinks, K=2 from ~8k; below that K=1 with 128-thread
    // CTAs wastes the fewest lanes in the last sink block)
    int k = 1;
    if (n_snk >= 8192) k = 2;
    if (n_snk >= 32768) k = 4;
    if (c->tune_k > 0) k = c->tune_k;
    if (k > max_k) k = max_k;
    pl.k = k;
    pl.nt = (k == 1) ? 128 : 256;
    const int sb = pl.nt * pl.k;
    pl.sink_blocks = (n_snk + sb - 1) / sb;
    const int resident = c->num_sms * ((sb >= 512) ? 2 : 4);
    // slices: aim at >= 16 waves of work units
    int slices = 1;
    const long long want_units = 16LL * resident;
    if (pl.sink_blocks < want_units) slices = (int)((want_units + pl.sink_blocks - 1) / pl.sink_blocks);
    int max_slices = pl.n_tiles;      // down to one tile per slice: a sweep of a few thousand particles
    if (max_slices < 1) max_slices = 1;   // is bound by the serial work per thread, not by issue
    if (slices > max_slices) slices = max_slices;
    if (slices > 256) slices = 256;
    if (c->tune_slices > 0) slices = c->tune_slices < pl.n_tiles ? c->tune_slices : pl.n_tiles;
    pl.tiles_per_slice = (pl.n_tiles + slices - 1) / slices;
    pl.slices = (pl.n_tiles + pl.tiles_per_slice - 1) / pl.tiles_per_slice;
    return pl;
}

template <class P, int K, int NT>
static int launch_variant(frost_ctx *c, const SweepParams &prm, const Plan &pl) {
    const size_t smem = (size_t)kStages * P::kRecs * kTile * kRecBytes + 2 * kStages * sizeof(uint64_t);
    FROST_TRY(set_func_attr(c, sweep_kernel<P, K, NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    dim3 grid(pl.sink_blocks, pl.slices);
    sweep_kernel<P, K, NT><<<grid, NT, smem, c->stream>>>(prm);
    return check_launch(c);
}

template <class P>
static int launch_sweep(frost_ctx *c, const SweepParams &prm, const Plan &pl) {
    switch (pl.k) {
        case 1: return launch_variant<P, 1, 128>(c, prm, pl);
        case 2: return launch_variant<P, 2, 256>(c, prm, pl);
        case 4: return launch_variant<P, 4, 256>(c, prm, pl);
        default: return FROST_EINVAL;
    }
}

static int pad1024(int n) { return round_up(n > 0 ? n : 1, 1024); }

int sweep_newton(frost_ctx *c, const double *snk_xm, int n_snk, const double *src_xm, int n_src,
                 const int32_t *snk_idx, int ld, double *out_acc, double *snk_a_packed) {
    if (n_snk <= 0) return FROST_OK;
    const Plan pl = make_plan(c, n_snk, n_src, 4);
    const int n_pad = pad1024(n_snk);
    FROST_TRY(ensure(c, c->partial, (size_t)pl.slices * 3 * n_pad * sizeof(double)));
    SweepParams prm{};
    prm.snk0 = (const double4 *)snk_xm; prm.src0 = (const double4 *)src_xm;
    prm.snk1 = nullptr; prm.src1 = nullptr;
    prm.partial = (double *)c->partial.p; prm.n_pad = n_pad;
    prm.n_tiles = pl.n_tiles; prm.tiles_per_slice = pl.tiles_per_slice;
    // floor: keeps the unguarded rsqrt seed finite for the self pair (see NewtonPolicy::pair)
    prm.eps2 = c->eps2 > 0x1p-400 ? c->eps2 : 0x1p-400;
    prm.G = c->G; prm.eta_ff = c->eta_ff; prm.eta_fb = c->eta_fb;
    if (n_src <= 0) { prm.n_tiles = 0; }
    FROST_TRY(launch_sweep<NewtonPolicy>(c, prm, pl));
    reduce_vec_kernel<<<(n_snk + 255) / 256, 256, 0, c->stream>>>(
        (const double *)c->partial.p, n_pad, pl.slices, n_snk, c->G, snk_idx, ld, out_acc,
        (double4 *)snk_a_packed, c->accumulate);
    return check_launch(c);
}

int sweep_gradient(frost_ctx *c, const double *snk_xm, const double *snk_a, int n_snk,
                   const double *src_xm, const double *src_a, int n_src, const int32_t *snk_idx,
                   int ld, double *out_grad) {
    if (n_snk <= 0) return FROST_OK;
    const Plan pl = make_plan(c, n_snk, n_src, 2);
    const int n_pad = pad1024(n_snk);
    FROST_TRY(ensure(c, c->partial, (size_t)pl.slices * 3 * n_pad * sizeof(double)));
    SweepParams prm{};
    prm.snk0 = (const double4 *)snk_xm; prm.snk1 = (const double4 *)snk_a;
    prm.src0 = (const double4 *)src_xm; prm.src1 = (const double4 *)src_a;
    prm.partial = (double *)c->partial.p; prm.n_pad = n_pad;
    prm.n_tiles = pl.n_tiles; prm.tiles_per_slice = pl.tiles_per_slice;
    prm.eps2 = c->eps2; prm.G = c->G; prm.eta_ff = c->eta_ff; prm.eta_fb = c->eta_fb;
    if (n_src <= 0) { prm.n_tiles = 0; }
    FROST_TRY(launch_sweep<GradientPolicy>(c, prm, pl));
    reduce_vec_kernel<<<(n_snk + 255) / 256, 256, 0, c->stream>>>(
        (const double *)c->partial.p, n_pad, pl.slices, n_snk, 2.0 * c->G, snk_idx, ld, out_grad,
        nullptr, c->accumulate);
    return check_launch(c);
}

int sweep_timestep(frost_ctx *c, const double *xm, const double *v, int n_set, const int32_t *idx,
                   double tau_pivot, double *out_tau, int32_t *out_bin, int *forest) {
    if (n_set <= 0) return FROST_OK;
    const Plan pl = make_plan(c, n_set, n_set, 2);
    const int n_pad = pad1024(n_set);
    FROST_TRY(ensure(c, c->partial, (size_t)pl.slices * n_pad * sizeof(double)));
    SweepParams prm{};
    prm.snk0 = (const double4 *)xm; prm.snk1 = (const double4 *)v;
    prm.src0 = (const double4 *)xm; prm.src1 = (const double4 *)v;
    prm.partial = (double *)c->partial.p; prm.n_pad = n_pad;
    prm.n_tiles = pl.n_tiles; prm.tiles_per_slice = pl.tiles_per_slice;
    prm.eps2 = 0.0; prm.G = c->G; prm.eta_ff = c->eta_ff; prm.eta_fb = c->eta_fb;
    prm.pivot = tau_pivot; prm.forest = forest;
    if (forest) FROST_TRY(launch_sweep<TimestepEdgePolicy>(c, prm, pl));
    else FROST_TRY(launch_sweep<TimestepPolicy>(c, prm, pl));
    reduce_tau_kernel<<<(n_set + 255) / 256, 256, 0, c->stream>>>(
        (const double *)c->partial.p, n_pad, pl.slices, n_set, idx, tau_pivot, out_tau, out_bin);
    return check_launch(c);
}

// The inter-level kick of a split hierarchy entry needs a_i and g_i over the pairs of the entry's set
// whose component labels differ (reading 24).  One-sided self sweep of the list; the label
// stream shares the records of the packed accelerations.
int sweep_masked(frost_ctx *c, const double *xm, double *a_lab, int n_set, const int32_t *idx, int ld,
                 double *out_acc, double *out_grad, int accumulate) {
    if (n_set <= 0) return FROST_OK;
    const int n_pad = pad1024(n_set);
    for (int pass = 0; pass < 2; ++pass) {
        if ((pass == 0 && !out_acc) || (pass == 1 && !out_grad)) continue;
        const Plan pl = make_plan(c, n_set, n_set, pass == 0 ? 4 : 2);
        FROST_TRY(ensure(c, c->partial, (size_t)pl.slices * 3 * n_pad * sizeof(double)));
        SweepParams prm{};
        prm.snk0 = prm.src0 = (const double4 *)xm; prm.snk1 = prm.src1 = (const double4 *)a_lab;
        prm.partial = (double *)c->partial.p; prm.n_pad = n_pad;
        prm.n_tiles = pl.n_tiles; prm.tiles_per_slice = pl.tiles_per_slice;
        prm.G = c->G; prm.eta_ff = c->eta_ff; prm.eta_fb = c->eta_fb;
        if (pass == 0) {
            prm.eps2 = c->eps2 > 0x1p-400 ? c->eps2 : 0x1p-400;
            FROST_TRY(launch_sweep<MaskedNewtonPolicy>(c, prm, pl));
            // (with accumulate the packed stream would need the total, which only the planes hold: the
            //  caller re-packs before a gradient sweep)
            reduce_vec_kernel<<<(n_set + 255) / 256, 256, 0, c->stream>>>(
                (const double *)c->partial.p, n_pad, pl.slices, n_set, c->G, idx, ld, out_acc,
                accumulate ? nullptr : (double4 *)a_lab, accumulate, 1);
        } else {
            prm.eps2 = c->eps2;
            FROST_TRY(launch_sweep<MaskedGradientPolicy>(c, prm, pl));
            reduce_vec_kernel<<<(n_set + 255) / 256, 256, 0, c->stream>>>(
                (const double *)c->partial.p, n_pad, pl.slices, n_set, 2.0 * c->G, idx, ld, out_grad,
                nullptr, accumulate, 0);
        }
        FROST_TRY(check_launch(c));
    }
    return FROST_OK;
}

}  // namespace frost
