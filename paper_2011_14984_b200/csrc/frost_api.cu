// frost_api.cu -- the C-ABI of include/frost.h: argument checks, scratch, and the host-side
// sequencing of Alg. 2 (fsi) and Alg. 3 (hhs_fsi).  All arithmetic is in the kernels of
// frost_sweeps.cu / frost_update.cu.
#include <cstdio>
#include <new>

#include "frost_common.cuh"

using namespace frost;

// Packed record streams are zero-padded to a multiple of every tile size that reads them: 256-record
// source tiles and <= 1024-sink blocks of the one-sided sweeps, A tiles of 128 x KA records (KA = 2, 4, 6,
// 8) of the pair-symmetric sweeps.
static int pad_rec(int n) { return round_up(n > 0 ? n : 1, 3072); }

extern "C" {

int frost_create(frost_ctx **out, int device, void *stream) {
    if (!out) return FROST_EINVAL;
    *out = nullptr;
    int count = 0;
    if (cudaGetDeviceCount(&count) != cudaSuccess || device < 0 || device >= count) return FROST_ECUDA;
    frost_ctx *c = new (std::nothrow) frost_ctx();
    if (!c) return FROST_ENOMEM;
    c->device = device;
    DeviceGuard guard(c);
    if (!guard.ok) { delete c; return FROST_ECUDA; }
    c->stream = (cudaStream_t)stream;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) { delete c; return FROST_ECUDA; }
    c->num_sms = prop.multiProcessorCount;
    if (cudaMallocHost((void **)&c->pinned_counts, 4 * sizeof(int32_t)) != cudaSuccess) {
        delete c;
        return FROST_ENOMEM;
    }
    *out = c;
    return FROST_OK;
}

static void free_scratch(frost_ctx *c) {
    Buf *bufs[] = {&c->recA_xm, &c->recB_xm, &c->recA_v, &c->recB_v, &c->partial, &c->partialB, &c->tau_scratch, &c->symtot,
                   &c->acc, &c->grad, &c->tau, &c->blockcnt, &c->dev_stats, &c->shard_idx, &c->uf, &c->comp, &c->symflag, &c->eqflag};
    for (Buf *b : bufs) if (b->p) cudaFree(b->p);
    for (Buf &b : c->host_stage) if (b.p) cudaFree(b.p);
    for (int k = 0; k < FROST_MAX_LEVELS; ++k) {
        if (c->lvlS[k].p) cudaFree(c->lvlS[k].p);
        if (c->lvlF[k].p) cudaFree(c->lvlF[k].p);
        if (c->lvlC[k].p) cudaFree(c->lvlC[k].p);
    }
    if (c->pinned_counts) cudaFreeHost(c->pinned_counts);
}

int frost_destroy(frost_ctx *c) {
    if (!c) return FROST_EINVAL;
    DeviceGuard guard(c);
    cudaStreamSynchronize(c->stream);
    for (int k = 0; k < FROST_MAX_LEVELS; ++k) {
        if (frost_ctx *s = c->side[k]) {
            cudaStreamSynchronize(s->stream);
            free_scratch(s);
            cudaStreamDestroy(s->stream);
            delete s;
        }
        if (c->ev_fork[k]) cudaEventDestroy(c->ev_fork[k]);
        if (c->ev_join[k]) cudaEventDestroy(c->ev_join[k]);
    }
    free_scratch(c);
    delete c;
    return FROST_OK;
}

// The side context of hierarchy level k: its own stream and its own sweep scratch, the parent's
// parameters.  fsi(S, tau/2) of an entry at level k runs there while hhs_fsi(F, tau/2) recurses on the
// parent's stream (the two operators commute and touch disjoint particles).
static int side_ctx(frost_ctx *c, int level, frost_ctx **out) {
    frost_ctx *s = c->side[level];
    if (!s) {
        s = new (std::nothrow) frost_ctx();
        if (!s) return FROST_ENOMEM;
        s->device = c->device; s->num_sms = c->num_sms;
        if (cudaStreamCreateWithFlags(&s->stream, cudaStreamNonBlocking) != cudaSuccess) { delete s; return FROST_ECUDA; }
        FROST_CUDA(c, cudaEventCreateWithFlags(&c->ev_fork[level], cudaEventDisableTiming));
        FROST_CUDA(c, cudaEventCreateWithFlags(&c->ev_join[level], cudaEventDisableTiming));
        c->side[level] = s;
    }
    s->G = c->G; s->eps2 = c->eps2; s->eta_ff = c->eta_ff; s->eta_fb = c->eta_fb; s->max_depth = c->max_depth;
    s->tune_k = c->tune_k; s->tune_slices = c->tune_slices; s->tune_small = c->tune_small;
    s->tune_cluster = c->tune_cluster; s->tune_sym = c->tune_sym; s->split_max = c->split_max; s->kepler = c->kepler; s->tune_pair = c->tune_pair; s->tune_guard = c->tune_guard; s->tune_eqmass = c->tune_eqmass;
    s->sym_scratch = c->sym_scratch < ((size_t)1 << 30) ? c->sym_scratch : ((size_t)1 << 30);
    *out = s;
    return FROST_OK;
}

int frost_set_params(frost_ctx *c, double G, double eps2, double eta_ff, double eta_fb, int max_depth) {
    if (!c || !(eps2 >= 0.0) || !(eta_ff > 0.0) || !(eta_fb > 0.0) || max_depth < 1) return FROST_EINVAL;
    c->G = G; c->eps2 = eps2; c->eta_ff = eta_ff; c->eta_fb = eta_fb;
    c->max_depth = max_depth < FROST_MAX_LEVELS ? max_depth : FROST_MAX_LEVELS;
    return FROST_OK;
}

int frost_set_tuning(frost_ctx *c, int sinks_per_thread, int source_slices, int small_set_max,
                     int subtree_one_cta) {
    if (!c || subtree_one_cta < 0 || subtree_one_cta > 1) return FROST_EINVAL;
    c->tune_cluster = subtree_one_cta;
    if (small_set_max < -1 || small_set_max > small_max()) return FROST_EINVAL;
    c->tune_small = small_set_max;
    if (!(sinks_per_thread == 0 || sinks_per_thread == 1 || sinks_per_thread == 2 || sinks_per_thread == 4))
        return FROST_EINVAL;
    if (source_slices < 0) return FROST_EINVAL;
    c->tune_k = sinks_per_thread;
    c->tune_slices = source_slices;
    return FROST_OK;
}

int frost_set_symmetric(frost_ctx *c, int mode, int scratch_mib) {
    if (!c || mode < 0 || mode > 5 || scratch_mib < 0) return FROST_EINVAL;
    c->tune_sym = mode;
    c->sym_scratch = (size_t)(scratch_mib > 0 ? scratch_mib : 4096) << 20;
    return FROST_OK;
}

int frost_set_shard(frost_ctx *c, int rank, int world) {
    if (!c || world < 1 || rank < 0 || rank >= world) return FROST_EINVAL;
    c->shard_rank = rank; c->shard_world = world;
    return FROST_OK;
}

int frost_set_overlap(frost_ctx *c, int on) {
    if (!c || on < 0 || on > 1) return FROST_EINVAL;
    c->overlap = on;
    return FROST_OK;
}

int frost_set_split(frost_ctx *c, int split_max) {
    if (!c || split_max < 0) return FROST_EINVAL;
    c->split_max = split_max;
    return FROST_OK;
}

int frost_set_kepler(frost_ctx *c, int on) {
    if (!c || on < 0 || on > 1) return FROST_EINVAL;
    c->kepler = on;
    return FROST_OK;
}

int frost_set_equal_mass_path(frost_ctx *c, int on) {
    if (!c || on < 0 || on > 1) return FROST_EINVAL;
    c->tune_eqmass = on;
    return FROST_OK;
}

int frost_set_gradient_guard(frost_ctx *c, int on) {
    if (!c || on < 0 || on > 1) return FROST_EINVAL;
    c->tune_guard = on;
    return FROST_OK;
}

int frost_set_pair_path(frost_ctx *c, int on) {
    if (!c || on < 0 || on > 1) return FROST_EINVAL;
    c->tune_pair = on;
    return FROST_OK;
}

int64_t frost_launch_count(const frost_ctx *c) {
    if (!c) return -1;
    int64_t t = c->launches;
    for (int k = 0; k < FROST_MAX_LEVELS; ++k) if (c->side[k]) t += c->side[k]->launches;
    return t;
}
int frost_last_cuda_error(const frost_ctx *c) { return c ? c->last_cuda : 0; }
const char *frost_version(void) {
    static char buf[192];
    static const int n = snprintf(buf, sizeof(buf), "frost-b200 0.3 (sm_100a; pair-symmetric sweeps: %s)", frost::sym_geometry());
    (void)n;
    return buf;
}

const char *frost_strerror(int status) {
    switch (status) {
        case FROST_OK: return "ok";
        case FROST_EINVAL: return "invalid argument";
        case FROST_ECUDA: return "CUDA error (see frost_last_cuda_error)";
        case FROST_ENOMEM: return "out of memory";
        case FROST_EDEPTH: return "hierarchy deeper than max_depth";
        case FROST_ENONFINITE: return "non-finite input";
        case FROST_ELIMIT: return "more than 64 components above 1024 particles in one split entry (frost_set_split)";
        case FROST_ETOOBIG: return "n exceeds FROST_NOALLOC_MAX_N (frost_acc_noalloc has a fixed static scratch)";
        default: return "unknown status";
    }
}

}  // extern "C"

// Whether a sweep goes through the pair-symmetric kernels (frost_sym.cu).  They need enough tile
// pairs to fill the GPU (A tiles of 256 particles below 16384, B tiles of 128); measured crossovers
// on B200 against the one-sided sweeps with source slices: self Newton ~6000, gradient ~5000, time
// step ~4000 particles; mutual sweeps from ~1000 x 1000.  kind: 0 self force sweep, 1 mutual force
// sweep (nA = the larger set), 2 time-step sweep.
static bool use_sym(const frost_ctx *c, int nA, int nB, int kind) {
    if (c->tune_sym == 1) return false;
    if (c->tune_sym >= 2) return nA > 0 && nB > 0;
    if (kind == 0) return nA >= 6144;
    if (kind == 2) return nA >= 4096;
    return nA >= 1024 && (long long)nA * nB >= 1000000LL;
}

// This rank's contiguous block [lo, hi) of a list of k entries (frost_set_shard); larger blocks first.
static void shard_block(const frost_ctx *c, int k, int *lo, int *hi) {
    const int base = k / c->shard_world, rem = k % c->shard_world, r = c->shard_rank;
    *lo = r * base + (r < rem ? r : rem);
    *hi = *lo + base + (r < rem ? 1 : 0);
}

static int forces_impl_(frost_ctx *c, int n, int ld, const double *pos, const double *mass,
                       const int32_t *I, int nI, const int32_t *J, int nJ, double *acc, double *grad,
                       int flags) {
    if (!I) nI = n;
    if (!J) nJ = n;
    const bool mutual = (flags & FROST_MUTUAL) != 0;
    const bool self = (I == J) && (nI == nJ);
    const bool sharded = c->shard_world > 1;
    // sharded: the outputs are partial sums the caller adds across ranks, so the gradient sweep cannot
    // start from this call's own (partial) accelerations, and adding into out_* would count the old
    // content once per rank -- whichever kernels end up serving the sweep
    if (sharded && (((flags & FROST_ACC) && (flags & FROST_GRAD)) || (flags & FROST_ACCUMULATE))) return FROST_EINVAL;
    if (nI <= 0 && !(mutual && nJ > 0)) return FROST_OK;
    // (sharded one-sided sweeps read a block of the sink stream at an offset: one more tile of padding)
    const int padA = pad_rec(nI) + (sharded ? 1024 : 0), padB = pad_rec(nJ) + (sharded ? 1024 : 0);
    FROST_TRY(ensure(c, c->recA_xm, (size_t)padA * kRecBytes));
    FROST_TRY(ensure(c, c->recA_v, (size_t)padA * kRecBytes));
    double *Axm = (double *)c->recA_xm.p, *Av = (double *)c->recA_v.p;
    double *Bxm = Axm, *Bv = Av;
    // pair-symmetric sweeps (frost_sym.cu) serve both directions of every pair with one evaluation:
    // the self case, and the mutual case with the larger set as the register-resident A side
    const bool sym_self = self && use_sym(c, nI, nI, 0);
    const bool sym_mut = mutual && !self && use_sym(c, nI > nJ ? nI : nJ, nI > nJ ? nJ : nI, 1);
    // ... and have an equal-mass variant (one DMUL less per pair): the pack kernels clear the flag if any
    // mass of either list differs from the first one's
    int *eq = nullptr;
    if ((sym_self || sym_mut) && c->tune_eqmass) {
        FROST_TRY(ensure(c, c->eqflag, 256));
        eq = (int *)c->eqflag.p;
        FROST_CUDA(c, cudaMemsetAsync(eq, 1, sizeof(int), c->stream));
    }
    FROST_TRY(launch_pack_xm(c, ld, pos, mass, I, nI, padA, Axm, 1.0, 2, (flags & FROST_ACC) ? Av : nullptr, eq, I));
    if (!self) {
        FROST_TRY(ensure(c, c->recB_xm, (size_t)padB * kRecBytes));
        FROST_TRY(ensure(c, c->recB_v, (size_t)padB * kRecBytes));
        Bxm = (double *)c->recB_xm.p; Bv = (double *)c->recB_v.p;
        FROST_TRY(launch_pack_xm(c, ld, pos, mass, J, nJ, padB, Bxm, 1.0, 2, (flags & FROST_ACC) ? Bv : nullptr, eq, I));
    }
    c->eq_flag_cur = eq;
    if (sym_self || sym_mut) {
        const bool swap = sym_mut && nJ > nI;            // A = the larger set
        const double *Pxm = swap ? Bxm : Axm, *Qxm = swap ? Axm : Bxm;
        double *Pv = swap ? Bv : Av, *Qv = swap ? Av : Bv;
        const int32_t *Pi = swap ? J : I, *Qi = swap ? I : J;
        const int nP = swap ? nJ : nI, nQ = swap ? nI : nJ;
        if (flags & FROST_ACC) {
            FROST_TRY(sym_newton(c, Pxm, nP, Qxm, nQ, self, Pi, Qi, ld, acc, Pv, self ? nullptr : Qv));
        }
        if (flags & FROST_GRAD) {
            if (!(flags & FROST_ACC)) {
                FROST_TRY(launch_pack_vec(c, ld, acc, I, nI, padA, Av));
                if (!self) FROST_TRY(launch_pack_vec(c, ld, acc, J, nJ, padB, Bv));
            }
            FROST_TRY(sym_gradient(c, Pxm, Pv, nP, Qxm, Qv, nQ, self, Pi, Qi, ld, grad));
        }
        return FROST_OK;
    }
    // One-sided sweeps.  Sharded: each direction sweeps this rank's contiguous block of its sink list
    // against all sources and zeroes the outputs of the other sinks, so that the caller's sum over the
    // ranks is complete here too (each sink's sum then comes from one rank: bitwise the unsharded one).
    int loA = 0, hiA = nI, loB = 0, hiB = nJ;
    const int32_t *Ii = I, *Ji = J;
    if (sharded) {
        shard_block(c, nI, &loA, &hiA);
        shard_block(c, nJ, &loB, &hiB);
        if (!I || (!J && mutual)) {      // NULL = all particles: the block needs explicit indices
            FROST_TRY(ensure(c, c->shard_idx, (size_t)n * sizeof(int32_t)));
            FROST_TRY(launch_iota(c, (int32_t *)c->shard_idx.p, n, 0));
            if (!I) Ii = (const int32_t *)c->shard_idx.p;
            if (!J) Ji = (const int32_t *)c->shard_idx.p;
        }
    }
    const size_t oA = (size_t)4 * loA, oB = (size_t)4 * loB;
    if (flags & FROST_ACC) {
        FROST_TRY(sweep_newton(c, Axm + oA, hiA - loA, Bxm, nJ, Ii ? Ii + loA : nullptr, ld, acc, Av + oA));
        if (sharded) FROST_TRY(launch_zero_outside(c, ld, acc, I, nI, loA, hiA));
        if (mutual && !self) {
            FROST_TRY(sweep_newton(c, Bxm + oB, hiB - loB, Axm, nI, Ji ? Ji + loB : nullptr, ld, acc, Bv + oB));
            if (sharded) FROST_TRY(launch_zero_outside(c, ld, acc, J, nJ, loB, hiB));
        }
    }
    if (flags & FROST_GRAD) {
        if (!(flags & FROST_ACC)) FROST_TRY(launch_pack_vec(c, ld, acc, I, nI, padA, Av));
        if (!self && !((flags & FROST_ACC) && mutual))
            FROST_TRY(launch_pack_vec(c, ld, acc, J, nJ, padB, Bv));
        FROST_TRY(sweep_gradient(c, Axm + oA, Av + oA, hiA - loA, Bxm, Bv, nJ, Ii ? Ii + loA : nullptr, ld, grad));
        if (sharded) FROST_TRY(launch_zero_outside(c, ld, grad, I, nI, loA, hiA));
        if (mutual && !self) {
            FROST_TRY(sweep_gradient(c, Bxm + oB, Bv + oB, hiB - loB, Axm, Av, nI, Ji ? Ji + loB : nullptr, ld, grad));
            if (sharded) FROST_TRY(launch_zero_outside(c, ld, grad, J, nJ, loB, hiB));
        }
    }
    return FROST_OK;
}

static int forces_impl(frost_ctx *c, int n, int ld, const double *pos, const double *mass,
                       const int32_t *I, int nI, const int32_t *J, int nJ, double *acc, double *grad,
                       int flags) {
    // FROST_ACCUMULATE: the gradient sweep of the same call would start from this call's own
    // accelerations instead of the totals in out_acc
    if ((flags & FROST_ACCUMULATE) && (flags & FROST_ACC) && (flags & FROST_GRAD)) return FROST_EINVAL;
    c->accumulate = (flags & FROST_ACCUMULATE) ? 1 : 0;
    const int rc = forces_impl_(c, n, ld, pos, mass, I, nI, J, nJ, acc, grad, flags);
    c->accumulate = 0;
    c->eq_flag_cur = nullptr;
    return rc;
}

// forest != NULL (a split hierarchy entry): the sweep also unites the fast pairs -- candidate below
// tau_pivot -- in the union-find forest over list positions; every pair must then be evaluated, so the
// pruned sweep is not used.
static int timesteps_impl(frost_ctx *c, int n, int ld, const double *pos, const double *vel,
                          const double *mass, const int32_t *idx, int n_idx, double tau_pivot,
                          double *out_tau, int32_t *out_bin, int *forest = nullptr) {
    if (!idx) n_idx = n;
    if (n_idx <= 0) return FROST_OK;
    if (forest && c->tune_sym != 1 && c->tune_sym != 3 && n_idx >= 32768)     // pruned sweep with edge output
        return tau_pruned(c, ld, pos, vel, mass, idx, n_idx, tau_pivot, out_tau, out_bin, c->tune_sym != 4, forest);
    if (forest) {
        const int pad = pad_rec(n_idx);
        FROST_TRY(ensure(c, c->recA_xm, (size_t)pad * kRecBytes));
        FROST_TRY(ensure(c, c->recA_v, (size_t)pad * kRecBytes));
        double *xm = (double *)c->recA_xm.p, *v = (double *)c->recA_v.p;
        FROST_TRY(launch_iota(c, forest, n_idx, 0));
        FROST_TRY(launch_pack_xm(c, ld, pos, mass, idx, n_idx, pad, xm, c->G, 1));
        FROST_TRY(launch_pack_vec(c, ld, vel, idx, n_idx, pad, v, 1));
        if (c->tune_sym != 1 && n_idx >= 4096)
            return sym_timestep(c, xm, v, n_idx, idx, tau_pivot, out_tau, out_bin, forest);
        return sweep_timestep(c, xm, v, n_idx, idx, tau_pivot, out_tau, out_bin, forest);
    }
    // large levels: Morton order + exact block pruning (frost_tau.cu); tune_sym 3 = symmetric sweep
    // without pruning, 4 = the pruning machinery with pruning switched off, 5 = pruning at any size (tests)
    // (measured on B200 against the plain symmetric sweep: 1.3x at 65536, 2.4x at 262144, 2.8x at
    // 2^20 particles; break-even at ~30000, where the sort and the two passes start to dominate)
    if (c->tune_sym == 4 || c->tune_sym == 5 || (c->tune_sym != 1 && c->tune_sym != 3 && n_idx >= 32768))
        return tau_pruned(c, ld, pos, vel, mass, idx, n_idx, tau_pivot, out_tau, out_bin, c->tune_sym != 4);
    const int pad = pad_rec(n_idx);
    FROST_TRY(ensure(c, c->recA_xm, (size_t)pad * kRecBytes));
    FROST_TRY(ensure(c, c->recA_v, (size_t)pad * kRecBytes));
    double *xm = (double *)c->recA_xm.p, *v = (double *)c->recA_v.p;
    FROST_TRY(launch_pack_xm(c, ld, pos, mass, idx, n_idx, pad, xm, c->G, 1));   // .w = G m, NaN padding
    FROST_TRY(launch_pack_vec(c, ld, vel, idx, n_idx, pad, v));
    if (use_sym(c, n_idx, n_idx, 2)) return sym_timestep(c, xm, v, n_idx, idx, tau_pivot, out_tau, out_bin);
    return sweep_timestep(c, xm, v, n_idx, idx, tau_pivot, out_tau, out_bin);
}

static int small_threshold(const frost_ctx *c) { return c->tune_small < 0 ? small_max() : c->tune_small; }

// n_steps consecutive fsi steps (Alg. 2).  The trailing Newton sweep of one step is at the
// positions of the leading sweep of the next, so from the second step on the leading sweep is
// skipped: 3 all-pairs sweeps per step instead of 4, bitwise the same result.
// skip_leading: the context's acc planes already hold a^{SS} of this set at the current positions (the
// trailing sweep of an earlier fsi on the same set, nothing moved since): the first sweep is skipped.
static int fsi_impl(frost_ctx *c, int n, int ld, double *pos, double *vel, const double *mass,
                    const int32_t *idx, int n_idx, double dt, frost_hhs_stats *st, void *dev_stats,
                    int n_steps = 1, bool skip_leading = false) {
    if (!idx) n_idx = n;
    if (n_idx <= 0 || n_steps <= 0) return FROST_OK;
    if (n_idx <= small_threshold(c))     // device-resident, set in shared memory (row 11)
        return launch_small(c, 1, ld, pos, vel, mass, idx, n_idx, dt, 0, st ? dev_stats : nullptr, n_steps);
    FROST_TRY(ensure(c, c->acc, (size_t)3 * ld * sizeof(double)));
    FROST_TRY(ensure(c, c->grad, (size_t)3 * ld * sizeof(double)));
    double *acc = (double *)c->acc.p, *grad = (double *)c->grad.p;
    for (int k = 0; k < n_steps; ++k) {
        if (k == 0 && !skip_leading)
            FROST_TRY(forces_impl(c, n, ld, pos, mass, idx, n_idx, idx, n_idx, acc, nullptr, FROST_ACC));
        FROST_TRY(launch_kick_drift(c, ld, pos, vel, acc, nullptr, idx, n_idx, dt / 6.0, 0.0, dt / 2.0));
        FROST_TRY(forces_impl(c, n, ld, pos, mass, idx, n_idx, idx, n_idx, acc, grad, FROST_ACC | FROST_GRAD));
        FROST_TRY(launch_kick_drift(c, ld, pos, vel, acc, grad, idx, n_idx, 2.0 * dt / 3.0, dt * dt / 48.0,
                                    dt / 2.0));
        FROST_TRY(forces_impl(c, n, ld, pos, mass, idx, n_idx, idx, n_idx, acc, nullptr, FROST_ACC));
        FROST_TRY(launch_kick(c, ld, vel, acc, nullptr, idx, n_idx, dt / 6.0, 0.0));
    }
    if (st) {
        const int64_t np = (int64_t)n_idx * n_idx;
        st->pairs_newton += (2 * (int64_t)n_steps + 1) * np;
        st->pairs_gradient += (int64_t)n_steps * np;
    }
    return FROST_OK;
}

// fsi(S, h) of an entry at `level`.  With overlap on it is enqueued on the level's side stream after
// everything enqueued so far on the parent's stream (fork); join_side() makes the parent's stream
// wait for it.  Same kernels, same inputs, disjoint particles: bitwise the serial result.
// second: the second fsi(S, h) of the entry.  Between the two, S is only kicked (the recursion moves F),
// and the side context's acc planes are touched by nobody else: they still hold the trailing a^{SS} of
// the first call at the positions S still has, so the leading sweep of the second call is skipped --
// the same values, one all-pairs sweep of S less per entry.
static int fsi_side(frost_ctx *c, int level, int n, int ld, double *pos, double *vel, const double *mass,
                    const int32_t *S, int nS, double h, frost_hhs_stats *st, bool *forked, bool second = false) {
    *forked = false;
    if (nS <= 0) return FROST_OK;
    if (!c->overlap) return fsi_impl(c, n, ld, pos, vel, mass, S, nS, h, st, c->dev_stats.p);
    frost_ctx *s = nullptr;
    FROST_TRY(side_ctx(c, level, &s));
    FROST_CUDA(c, cudaEventRecord(c->ev_fork[level], c->stream));
    FROST_CUDA(c, cudaStreamWaitEvent(s->stream, c->ev_fork[level], 0));
    const int rc = fsi_impl(s, n, ld, pos, vel, mass, S, nS, h, st, c->dev_stats.p, 1, second);
    if (rc != FROST_OK) { c->last_cuda = s->last_cuda; return rc; }
    *forked = true;
    return FROST_OK;
}

static int join_side(frost_ctx *c, int level, bool forked) {
    if (!forked) return FROST_OK;
    FROST_CUDA(c, cudaEventRecord(c->ev_join[level], c->side[level]->stream));
    FROST_CUDA(c, cudaStreamWaitEvent(c->stream, c->ev_join[level], 0));
    return FROST_OK;
}

// The inter-level kick of one entry (Alg. 3's acc_sf_* + kick_sf; Eq. 41-44): masked = the entry was
// split into several components and the kicked pair set is "labels differ" over the whole set.
static int cross_kick(frost_ctx *c, int n, int ld, double *pos, double *vel, const double *mass,
                      const int32_t *set, int n_set, const int32_t *S, int nS, const int32_t *F, int nF,
                      const SplitInfo &si, bool with_g, double cc, double kappa) {
    double *acc = (double *)c->acc.p, *grad = (double *)c->grad.p;
    if (si.m > 1) {
        // P = S x F  u  G x R  u  { pairs of R in different components }, with G the largest component
        // above 1024 particles (if any) and R the rest of F: two pair-symmetric mutual sweeps and one
        // masked self sweep of R, the accelerations of all three added up before any gradient sweep
        // (Eq. 43-44 need the a of the whole pair set).  Every member of the set is a sink of at least
        // one overwriting sweep: S and F of the first (when S is not empty), else R and G.
        const int32_t *G = si.C + si.g_off;
        const int nG = si.g_size, nR = si.nR;
        const int pad = pad_rec(nR);
        for (int phase = 0; phase < (with_g ? 2 : 1); ++phase) {
            const int fl = phase == 0 ? FROST_ACC : FROST_GRAD;
            double *out = phase == 0 ? acc : grad;
            bool fresh = true;                                        // nothing written to `out` yet
            if (nS > 0) {
                FROST_TRY(forces_impl(c, n, ld, pos, mass, S, nS, F, nF, acc, grad, fl | FROST_MUTUAL));
                fresh = false;
            }
            if (nG > 0 && nR > 0) {
                FROST_TRY(forces_impl(c, n, ld, pos, mass, G, nG, si.R, nR, acc, grad,
                                      fl | FROST_MUTUAL | (fresh ? 0 : FROST_ACCUMULATE)));
                fresh = false;
            }
            if (nR > 0) {
                FROST_TRY(ensure(c, c->recA_xm, (size_t)pad * kRecBytes));
                FROST_TRY(ensure(c, c->recA_v, (size_t)pad * kRecBytes));
                double *xm = (double *)c->recA_xm.p, *av = (double *)c->recA_v.p;
                FROST_TRY(launch_pack_xm(c, ld, pos, mass, si.R, nR, pad, xm, 1.0, 0, av));
                if (phase == 1) FROST_TRY(launch_pack_vec(c, ld, acc, si.R, nR, pad, av));     // the total a of P
                FROST_TRY(launch_pack_label(c, si.labR, nR, pad, av));
                // pair-symmetric from the same size as the unmasked self sweeps, else one-sided
                if (use_sym(c, nR, nR, 0))
                    FROST_TRY(sym_masked(c, xm, av, nR, si.R, ld, phase == 0 ? out : nullptr,
                                         phase == 1 ? out : nullptr, fresh ? 0 : 1));
                else
                    FROST_TRY(sweep_masked(c, xm, av, nR, si.R, ld, phase == 0 ? out : nullptr,
                                           phase == 1 ? out : nullptr, fresh ? 0 : 1));
            }
        }
        return launch_kick(c, ld, vel, acc, with_g ? grad : nullptr, set, n_set, cc, kappa);
    }
    if (nS > 0 && nF > 0) {
        FROST_TRY(forces_impl(c, n, ld, pos, mass, S, nS, F, nF, acc, grad,
                              FROST_ACC | FROST_MUTUAL | (with_g ? FROST_GRAD : 0)));
        return launch_kick(c, ld, vel, acc, with_g ? grad : nullptr, set, n_set, cc, kappa);   // S u F
    }
    return FROST_OK;
}

static int hhs_rec(frost_ctx *c, int n, int ld, double *pos, double *vel, const double *mass,
                   const int32_t *set, int n_set, double tau_pivot, int level, frost_hhs_stats *st,
                   bool is_comp = false);

// hhs_fsi(C, tau/2) of every component of F (Alg. 3: hhs_fsi(F, tau/2))
static int recurse_fast(frost_ctx *c, int n, int ld, double *pos, double *vel, const double *mass,
                        const int32_t *F, int nF, const SplitInfo &si, double h, int level,
                        frost_hhs_stats *st) {
    if (si.m <= 1) return hhs_rec(c, n, ld, pos, vel, mass, F, nF, h, level + 1, st, si.split);
    FROST_TRY(launch_comp_batch(c, 1, ld, pos, vel, mass, si.C, si.desc_small, si.n_small_dev, si.n_small, h,
                                level + 1, c->dev_stats.p));
    FROST_TRY(launch_comp_batch(c, 0, ld, pos, vel, mass, si.C, si.desc_med, si.n_med_dev, si.n_med, h,
                                level + 1, c->dev_stats.p));
    for (int b = 0; b < si.n_big; ++b)
        FROST_TRY(hhs_rec(c, n, ld, pos, vel, mass, si.C + si.big_off[b], si.big_size[b], h, level + 1, st, true));
    return FROST_OK;
}

static int hhs_rec(frost_ctx *c, int n, int ld, double *pos, double *vel, const double *mass,
                   const int32_t *set, int n_set, double tau_pivot, int level, frost_hhs_stats *st,
                   bool is_comp) {
    if (n_set <= 0) return FROST_OK;
    if (level >= c->max_depth || level >= FROST_MAX_LEVELS) return FROST_EDEPTH;
    // the whole subtree on the device, asynchronously (row 11); a two-body component of a split entry
    // under frost_set_kepler goes there whatever the threshold (the propagator lives in that kernel)
    if (n_set <= small_threshold(c) || (is_comp && n_set == 2 && c->kepler && c->eps2 == 0.0))
        return launch_small(c, 0, ld, pos, vel, mass, set, n_set, tau_pivot, level, c->dev_stats.p, 1, is_comp);
    double *tau = (double *)c->tau.p;
    const bool split = c->split_max > 0 && n_set <= c->split_max;
    int *forest = nullptr;
    if (split) {
        FROST_TRY(ensure(c, c->uf, (size_t)pad_rec(n_set) * sizeof(int)));
        forest = (int *)c->uf.p;
    }
    FROST_TRY(timesteps_impl(c, n, ld, pos, vel, mass, set, n_set, tau_pivot, tau, nullptr, forest));
    FROST_TRY(ensure(c, c->lvlS[level], (size_t)n_set * sizeof(int32_t)));
    FROST_TRY(ensure(c, c->lvlF[level], (size_t)n_set * sizeof(int32_t)));
    int32_t *S = (int32_t *)c->lvlS[level].p, *F = (int32_t *)c->lvlF[level].p;
    int32_t cnt[2];
    FROST_TRY(launch_partition(c, tau, set, n_set, tau_pivot, S, F, cnt));
    const int nS = cnt[0], nF = cnt[1];
    SplitInfo si;
    si.split = split;
    si.m = nF > 0 ? 1 : 0;
    si.sumsq = (long long)nF * nF;
    if (split && nF > 0) {
        FROST_TRY(split_components(c, level, ld, tau, set, n_set, tau_pivot, forest, F, nF, &si));
        si.split = true;
        F = const_cast<int32_t *>(si.C);       // same members, components contiguous
    }
    if (st) {
        if (level > st->depth) st->depth = level;
        st->entries[level] += 1;
        st->n_slow[level] += nS;
        st->n_fast[level] += nF;
        st->n_comp[level] += si.m;
        st->pairs_timestep += (int64_t)n_set * n_set;
    }
    const double h = 0.5 * tau_pivot;
    bool forked = false;
    FROST_TRY(cross_kick(c, n, ld, pos, vel, mass, set, n_set, S, nS, F, nF, si, false, tau_pivot / 6.0, 0.0));
    FROST_TRY(fsi_side(c, level, n, ld, pos, vel, mass, S, nS, h, st, &forked));       // fsi(S, tau/2) ...
    FROST_TRY(recurse_fast(c, n, ld, pos, vel, mass, F, nF, si, h, level, st));         // ... || hhs_fsi(F, tau/2)
    FROST_TRY(join_side(c, level, forked));
    FROST_TRY(cross_kick(c, n, ld, pos, vel, mass, set, n_set, S, nS, F, nF, si, true, 2.0 * tau_pivot / 3.0,
                         tau_pivot * tau_pivot / 48.0));
    FROST_TRY(fsi_side(c, level, n, ld, pos, vel, mass, S, nS, h, st, &forked, true));
    FROST_TRY(recurse_fast(c, n, ld, pos, vel, mass, F, nF, si, h, level, st));
    FROST_TRY(join_side(c, level, forked));
    FROST_TRY(cross_kick(c, n, ld, pos, vel, mass, set, n_set, S, nS, F, nF, si, false, tau_pivot / 6.0, 0.0));
    if (st) {
        // ordered pairs of the kicked set: all but slow-slow and same-component pairs (2 |S| |F| unsplit)
        const int64_t cr = (int64_t)n_set * n_set - (int64_t)nS * nS - si.sumsq;
        st->pairs_newton += 3 * cr;
        st->pairs_gradient += cr;
    }
    return FROST_OK;
}

static bool bad_planes(int n, int ld) { return n < 0 || ld < n; }

extern "C" {

int frost_forces(frost_ctx *c, int n, int ld, const double *pos, const double *vel,
                 const double *mass, const int32_t *sink_idx, int n_sink,
                 const int32_t *source_idx, int n_source, double *out_acc, double *out_grad,
                 int flags) {
    (void)vel;
    if (!c || bad_planes(n, ld) || !pos || !mass || !out_acc) return FROST_EINVAL;
    if (!(flags & (FROST_ACC | FROST_GRAD)) || (flags & ~15)) return FROST_EINVAL;
    if ((flags & FROST_GRAD) && !out_grad) return FROST_EINVAL;
    if ((flags & FROST_MUTUAL) && ((sink_idx == nullptr) != (source_idx == nullptr))) return FROST_EINVAL;
    if ((sink_idx && n_sink < 0) || (source_idx && n_source < 0)) return FROST_EINVAL;
    if (n == 0) return FROST_OK;
    FROST_DEVICE(c);
    return forces_impl(c, n, ld, pos, mass, sink_idx, n_sink, source_idx, n_source, out_acc, out_grad, flags);
}

int frost_forces_host(frost_ctx *c, int n, int ld, const double *pos, const double *mass,
                      const int32_t *sink_idx, int n_sink, const int32_t *source_idx,
                      int n_source, double *out_acc, double *out_grad, int flags) {
    if (!c || bad_planes(n, ld) || !pos || !mass || !out_acc) return FROST_EINVAL;
    if (!(flags & (FROST_ACC | FROST_GRAD)) || (flags & ~15)) return FROST_EINVAL;
    if ((flags & FROST_GRAD) && !out_grad) return FROST_EINVAL;
    if ((flags & FROST_MUTUAL) && ((sink_idx == nullptr) != (source_idx == nullptr))) return FROST_EINVAL;
    if ((sink_idx && n_sink < 0) || (source_idx && n_source < 0)) return FROST_EINVAL;
    if (n == 0) return FROST_OK;
    FROST_DEVICE(c);
    const size_t pb = (size_t)3 * ld * sizeof(double);
    FROST_TRY(ensure(c, c->host_stage[0], pb));
    FROST_TRY(ensure(c, c->host_stage[1], (size_t)n * sizeof(double)));
    FROST_TRY(ensure(c, c->host_stage[2], pb));
    FROST_TRY(ensure(c, c->host_stage[3], pb));
    double *dpos = (double *)c->host_stage[0].p, *dmass = (double *)c->host_stage[1].p;
    double *dacc = (double *)c->host_stage[2].p, *dgrad = (double *)c->host_stage[3].p;
    int32_t *dI = nullptr, *dJ = nullptr;
    if (sink_idx) {
        FROST_TRY(ensure(c, c->host_stage[4], (size_t)(n_sink + 1) * sizeof(int32_t)));
        dI = (int32_t *)c->host_stage[4].p;
        FROST_CUDA(c, cudaMemcpyAsync(dI, sink_idx, (size_t)n_sink * sizeof(int32_t), cudaMemcpyHostToDevice, c->stream));
    }
    if (source_idx) {
        if (source_idx == sink_idx && n_source == n_sink) dJ = dI;
        else {
            FROST_TRY(ensure(c, c->host_stage[5], (size_t)(n_source + 1) * sizeof(int32_t)));
            dJ = (int32_t *)c->host_stage[5].p;
            FROST_CUDA(c, cudaMemcpyAsync(dJ, source_idx, (size_t)n_source * sizeof(int32_t), cudaMemcpyHostToDevice, c->stream));
        }
    }
    FROST_CUDA(c, cudaMemcpyAsync(dpos, pos, pb, cudaMemcpyHostToDevice, c->stream));
    FROST_CUDA(c, cudaMemcpyAsync(dmass, mass, (size_t)n * sizeof(double), cudaMemcpyHostToDevice, c->stream));
    // out_acc is an input when the gradient is requested on caller-provided accelerations or the sums
    // are accumulated, and entries outside the swept sets must come back untouched; when every
    // particle is a sink of an overwriting sweep the planes are pure outputs and are not uploaded
    const bool all_sinks = !sink_idx && ld == n;
    const bool accum = (flags & FROST_ACCUMULATE) != 0;
    if (!(all_sinks && (flags & FROST_ACC) && !accum))
        FROST_CUDA(c, cudaMemcpyAsync(dacc, out_acc, pb, cudaMemcpyHostToDevice, c->stream));
    if ((flags & FROST_GRAD) && !(all_sinks && !accum))
        FROST_CUDA(c, cudaMemcpyAsync(dgrad, out_grad, pb, cudaMemcpyHostToDevice, c->stream));
    FROST_TRY(forces_impl(c, n, ld, dpos, dmass, dI, n_sink, dJ, n_source, dacc, dgrad, flags));
    if (flags & FROST_ACC)
        FROST_CUDA(c, cudaMemcpyAsync(out_acc, dacc, pb, cudaMemcpyDeviceToHost, c->stream));
    if (flags & FROST_GRAD)
        FROST_CUDA(c, cudaMemcpyAsync(out_grad, dgrad, pb, cudaMemcpyDeviceToHost, c->stream));
    FROST_CUDA(c, cudaStreamSynchronize(c->stream));
    return FROST_OK;
}

int frost_timesteps(frost_ctx *c, int n, int ld, const double *pos, const double *vel,
                    const double *mass, const int32_t *idx, int n_idx, double tau_pivot,
                    double *out_tau, int32_t *out_bin) {
    if (!c || bad_planes(n, ld) || !pos || !vel || !mass || !out_tau) return FROST_EINVAL;
    if (idx && n_idx < 0) return FROST_EINVAL;
    if (out_bin && !(tau_pivot > 0.0)) return FROST_EINVAL;
    if (n == 0) return FROST_OK;
    FROST_DEVICE(c);
    return timesteps_impl(c, n, ld, pos, vel, mass, idx, n_idx, tau_pivot, out_tau, out_bin);
}

int frost_partition(frost_ctx *c, int n, const double *tau, const int32_t *idx, int n_idx,
                    double tau_pivot, int32_t *out_slow, int32_t *out_fast, int32_t *counts) {
    if (!c || n < 0 || !tau || !out_slow || !out_fast || !counts) return FROST_EINVAL;
    if (!idx) n_idx = n;
    if (n_idx < 0) return FROST_EINVAL;
    FROST_DEVICE(c);
    return launch_partition(c, tau, idx, n_idx, tau_pivot, out_slow, out_fast, counts);
}

int frost_kick(frost_ctx *c, int n, int ld, double *vel, const double *acc, const double *grad,
               const int32_t *idx, int n_idx, double cc, double kappa) {
    if (!c || bad_planes(n, ld) || !vel || !acc) return FROST_EINVAL;
    if (kappa != 0.0 && !grad) return FROST_EINVAL;
    if (!idx) n_idx = n;
    if (n_idx < 0) return FROST_EINVAL;
    FROST_DEVICE(c);
    return launch_kick(c, ld, vel, acc, grad, idx, n_idx, cc, kappa);
}

int frost_drift(frost_ctx *c, int n, int ld, double *pos, const double *vel, const int32_t *idx,
                int n_idx, double cc) {
    if (!c || bad_planes(n, ld) || !pos || !vel) return FROST_EINVAL;
    if (!idx) n_idx = n;
    if (n_idx < 0) return FROST_EINVAL;
    FROST_DEVICE(c);
    return launch_drift(c, ld, pos, vel, idx, n_idx, cc);
}

int frost_fsi_step(frost_ctx *c, int n, int ld, double *pos, double *vel, const double *mass,
                   const int32_t *idx, int n_idx, double dt) {
    if (!c || bad_planes(n, ld) || !pos || !vel || !mass) return FROST_EINVAL;
    if (idx && n_idx < 0) return FROST_EINVAL;
    if (c->shard_world > 1) return FROST_EINVAL;      // only frost_forces is shard-aware
    if (n == 0) return FROST_OK;
    FROST_DEVICE(c);
    return fsi_impl(c, n, ld, pos, vel, mass, idx, n_idx, dt, nullptr, nullptr);
}

int frost_fsi_steps(frost_ctx *c, int n, int ld, double *pos, double *vel, const double *mass,
                    const int32_t *idx, int n_idx, double dt, int n_steps) {
    if (!c || bad_planes(n, ld) || !pos || !vel || !mass || n_steps < 0) return FROST_EINVAL;
    if (idx && n_idx < 0) return FROST_EINVAL;
    if (c->shard_world > 1) return FROST_EINVAL;      // only frost_forces is shard-aware
    if (n == 0) return FROST_OK;
    FROST_DEVICE(c);
    return fsi_impl(c, n, ld, pos, vel, mass, idx, n_idx, dt, nullptr, nullptr, n_steps);
}

int frost_hhs_step(frost_ctx *c, int n, int ld, double *pos, double *vel, const double *mass,
                   double dt_top, frost_hhs_stats *stats) {
    if (!c || bad_planes(n, ld) || !pos || !vel || !mass || !(dt_top > 0.0)) return FROST_EINVAL;
    if (stats) *stats = frost_hhs_stats{};
    if (c->shard_world > 1) return FROST_EINVAL;      // only frost_forces is shard-aware
    if (n == 0) return FROST_OK;
    FROST_DEVICE(c);
    // every O(n) scratch buffer of the recursion is sized here, once, for the largest set it can
    // meet (all n particles), so that ensure() never has to drain the stream to grow one mid-step
    const size_t recb = (size_t)pad_rec(n) * kRecBytes;
    FROST_TRY(ensure(c, c->recA_xm, recb)); FROST_TRY(ensure(c, c->recA_v, recb));
    FROST_TRY(ensure(c, c->recB_xm, recb)); FROST_TRY(ensure(c, c->recB_v, recb));
    FROST_TRY(ensure(c, c->blockcnt, (size_t)(n / 1024 + 4) * sizeof(int)));
    FROST_TRY(ensure(c, c->acc, (size_t)3 * ld * sizeof(double)));
    FROST_TRY(ensure(c, c->grad, (size_t)3 * ld * sizeof(double)));
    FROST_TRY(ensure(c, c->tau, (size_t)ld * sizeof(double)));
    FROST_TRY(ensure(c, c->dev_stats, small_stats_bytes()));
    FROST_CUDA(c, cudaMemsetAsync(c->dev_stats.p, 0, small_stats_bytes(), c->stream));
    frost_hhs_stats local = frost_hhs_stats{};
    local.depth = -1;
    int rc = hhs_rec(c, n, ld, pos, vel, mass, nullptr, n, dt_top, 0, &local);
    if (rc != FROST_OK)      // an aborted recursion may have left forked side streams unjoined
        for (int k = 0; k < FROST_MAX_LEVELS; ++k) if (c->side[k]) cudaStreamSynchronize(c->side[k]->stream);
    // merge what the device-resident subtrees counted (also carries their status)
    struct { long long e[FROST_MAX_LEVELS], s[FROST_MAX_LEVELS], f[FROST_MAX_LEVELS], pn, pg, pt; int depth, status;
             long long nc[FROST_MAX_LEVELS]; long long nk; } d;
    static_assert(sizeof(d) >= 1, "");
    if (sizeof(d) != small_stats_bytes()) return FROST_EINVAL;
    FROST_CUDA(c, cudaMemcpyAsync(&d, c->dev_stats.p, sizeof(d), cudaMemcpyDeviceToHost, c->stream));
    FROST_CUDA(c, cudaStreamSynchronize(c->stream));
    if (rc == FROST_OK && d.status) rc = d.status;
    // the device kernel records depth = -1 when it never entered a level
    for (int k = 0; k < FROST_MAX_LEVELS; ++k) {
        local.entries[k] += d.e[k]; local.n_slow[k] += d.s[k]; local.n_fast[k] += d.f[k];
        local.n_comp[k] += d.nc[k];
    }
    local.pairs_newton += d.pn; local.pairs_gradient += d.pg; local.pairs_timestep += d.pt;
    local.n_kepler += d.nk;
    if (d.depth > local.depth) local.depth = d.depth;
    if (local.depth < 0) local.depth = 0;
    if (stats) *stats = local;
    return rc;
}

int frost_diagnostics(frost_ctx *c, int n, int ld, const double *pos, const double *vel,
                      const double *mass, double *out_phi, double *out8) {
    if (!c || bad_planes(n, ld) || !pos || !vel || !mass || !out8) return FROST_EINVAL;
    for (int k = 0; k < 8; ++k) out8[k] = 0.0;
    if (n == 0) return FROST_OK;
    FROST_DEVICE(c);
    const int pad = pad_rec(n);
    FROST_TRY(ensure(c, c->recA_xm, (size_t)pad * kRecBytes));
    FROST_TRY(ensure(c, c->tau, (size_t)(ld + 8) * sizeof(double)));
    FROST_TRY(ensure(c, c->blockcnt, 8 * sizeof(double)));
    double *xm = (double *)c->recA_xm.p;
    double *phi = out_phi ? out_phi : (double *)c->tau.p;
    double *d8 = (double *)c->blockcnt.p;
    FROST_TRY(launch_pack_xm(c, ld, pos, mass, nullptr, n, pad, xm));
    FROST_TRY(sym_potential(c, xm, n, phi));
    FROST_TRY(launch_diag(c, n, ld, pos, vel, mass, phi, d8));
    FROST_CUDA(c, cudaMemcpyAsync(out8, d8, 8 * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    FROST_CUDA(c, cudaStreamSynchronize(c->stream));
    return FROST_OK;
}

int frost_forces_masked(frost_ctx *c, int n, int ld, const double *pos, const double *mass,
                        const int32_t *idx, int n_idx, const int32_t *label, double *out_acc,
                        double *out_grad) {
    if (!c || bad_planes(n, ld) || !pos || !mass || !label || !out_acc) return FROST_EINVAL;
    if (idx && n_idx < 0) return FROST_EINVAL;
    if (c->shard_world > 1) return FROST_EINVAL;      // only frost_forces is shard-aware
    if (!idx) n_idx = n;
    if (n_idx == 0) return FROST_OK;
    FROST_DEVICE(c);
    const int pad = pad_rec(n_idx);
    FROST_TRY(ensure(c, c->recA_xm, (size_t)pad * kRecBytes));
    FROST_TRY(ensure(c, c->recA_v, (size_t)pad * kRecBytes));
    double *xm = (double *)c->recA_xm.p, *av = (double *)c->recA_v.p;
    FROST_TRY(launch_pack_xm(c, ld, pos, mass, idx, n_idx, pad, xm, 1.0, 0, av));
    FROST_TRY(launch_pack_label(c, label, n_idx, pad, av));
    // the same decision, and for the pair-symmetric kernels the same sequence, as the masked self sweep
    // of R in cross_kick: accelerations, re-pack of the total accelerations beside the labels, gradient
    if (use_sym(c, n_idx, n_idx, 0)) {
        FROST_TRY(sym_masked(c, xm, av, n_idx, idx, ld, out_acc, nullptr, 0));
        if (!out_grad) return FROST_OK;
        FROST_TRY(launch_pack_vec(c, ld, out_acc, idx, n_idx, pad, av));
        FROST_TRY(launch_pack_label(c, label, n_idx, pad, av));
        return sym_masked(c, xm, av, n_idx, idx, ld, nullptr, out_grad, 0);
    }
    return sweep_masked(c, xm, av, n_idx, idx, ld, out_acc, out_grad);
}

int frost_gather_pack(frost_ctx *c, int n, int ld, const double *pos, const double *mass,
                      const int32_t *idx, int n_idx, int n_pad, double *out_records) {
    if (!c || bad_planes(n, ld) || !pos || !mass || !out_records) return FROST_EINVAL;
    if (!idx) n_idx = n;
    if (n_idx < 0 || n_pad < n_idx) return FROST_EINVAL;
    FROST_DEVICE(c);
    return launch_pack_xm(c, ld, pos, mass, idx, n_idx, n_pad, out_records);
}

}  // extern "C"
