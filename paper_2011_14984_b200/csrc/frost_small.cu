// frost_small.cu -- SURVEY.md §8(a) row 11: the whole hhs_fsi(F, tau) subtree (Alg. 3,
// PAPER.md:572-587) of a small particle set executed by ONE CTA with the set resident in shared
// memory and an explicit level stack -- no host round trip, no launch per operator.  This is the
// B200-native stand-in for the paper's "serial CPU code ... when N <~ a few hundred particles"
// (PAPER.md:545): deep hierarchy levels hold a handful of particles and are entered 2^k times per
// top-level step, where ~20 launches plus a count read-back per entry would dominate.
//
// The arithmetic is the same pair code as the streaming sweeps (frost_pairs.cuh).  A sink is
// served by L = 1..32 adjacent lanes that split the source list and combine with warp shuffles, so
// small sink sets still use the whole CTA; the combination order is fixed (deterministic).
#include <cooperative_groups.h>

#include "frost_pairs.cuh"

namespace frost {

constexpr int kSmallMax = 1024;     // particles the subtree kernel accepts
constexpr int kSmallThreads = 512;
constexpr int kCompWarpMax = 32;    // components up to this size: one warp each, kCompWarps per CTA
constexpr int kCompWarps = 8;

struct SmallStats {                 // device-side mirror of frost_hhs_stats (+ status)
    long long entries[FROST_MAX_LEVELS], n_slow[FROST_MAX_LEVELS], n_fast[FROST_MAX_LEVELS];
    long long pairs_newton, pairs_gradient, pairs_timestep;
    int depth, status;
    long long n_comp[FROST_MAX_LEVELS];
    long long n_kepler;
};

struct SmallParams {
    const int32_t *idx;             // global indices of the set (NULL = 0..n-1)
    int n, ld;
    double *pos, *vel;
    const double *mass;
    double tau_pivot;               // pivot step of the subtree's root
    double dt_fsi;                  // mode 1: plain fsi(set, dt_fsi) instead of hhs_fsi
    int mode;                       // 0 = hhs_fsi subtree, 1 = fsi step(s)
    int n_steps;                    // mode 1: number of consecutive fsi steps
    int level0, max_depth;
    double G, eps2, eta_ff, eta_fb;
    SmallStats *stats;
    // spatial splitting of fast levels (reading 24): entries with at most split_max members
    // recurse into the connected components of their fast pairs one by one
    int split_max;
    // batched launch: CTA (or warp) b takes the set idx[desc[b].x .. desc[b].x + desc[b].y)
    const int2 *desc;
    const int *n_desc;
    int pair_path;                  // two-body frames on one thread (binary_subtree); 0: team path (tests)
    int kepler;                     // two-body COMPONENTS of a split entry follow their Kepler orbit (reading 25)
    int root_is_comp;               // the set of this launch is itself such a component
};

template <int CAP>
struct SmallSmemT {
    static constexpr int kCap = CAP, kWords = (CAP + 31) / 32;
    double4 xm[CAP];                // x, y, z, m
    double4 vv[CAP];                // vx, vy, vz, 1
    double4 aa[CAP];                // ax, ay, az, 1
    double4 gg[CAP];                // gx, gy, gz, -
    double tau[CAP];
    int perm[CAP];                  // the level sets are contiguous segments of this list
    int tmp[CAP];
    int lab[CAP];                   // component of a particle in the entry being executed (-1 = slow)
    int par[CAP];                   // union-find forest over the fast pairs of the entry's time-step sweep
    int scan[kSmallThreads / 32 + 1];
    // explicit recursion stack
    int f_start[FROST_MAX_LEVELS], f_n[FROST_MAX_LEVELS], f_ns[FROST_MAX_LEVELS], f_stage[FROST_MAX_LEVELS];
    int f_cpos[FROST_MAX_LEVELS];   // next component of F to recurse into (offset inside F)
    int f_m[FROST_MAX_LEVELS];      // number of components of F
    int f_iscomp[FROST_MAX_LEVELS]; // the frame's set is a component of a split entry
    long long f_sumsq[FROST_MAX_LEVELS];          // sum of squared component sizes
    unsigned f_bnd[FROST_MAX_LEVELS][kWords];     // bit r: a component starts at position r of F
    double f_tau[FROST_MAX_LEVELS];
    int sp, err;
};
using SmallSmem = SmallSmemT<kSmallMax>;

struct SmStats {                    // per CTA, shared by its teams (atomics)
    unsigned long long entries[FROST_MAX_LEVELS], slow[FROST_MAX_LEVELS], fast[FROST_MAX_LEVELS],
        comps[FROST_MAX_LEVELS];
    unsigned long long pn, pg, pt, kep;
    int depth;
};

// A "team" executes a subtree: the whole CTA, or -- for sets of <= 32 particles, where the cost is
// the latency of the ~40 dependent phases per hierarchy entry, not arithmetic -- a single warp
// that synchronises with __syncwarp while the other warps wait at one barrier.
struct TeamCTA {
    static constexpr bool kCluster = false;
    static constexpr int kThreads = kSmallThreads;
    __device__ static __forceinline__ void sync() { __syncthreads(); }
    __device__ static __forceinline__ int tid() { return threadIdx.x; }
};
// A cluster of CTAs, each holding a full replica of the set and of the recursion state: every CTA
// executes the same state machine (kicks, drifts, partitions and tiny sub-sets redundantly --
// bitwise identical), but a large sweep is shared out by sinks and its results are written into
// every replica through distributed shared memory, so the pair arithmetic of a 256-1024 particle
// set runs on kClusterSize SMs instead of one.
struct TeamCluster {
    static constexpr int kThreads = kSmallThreads;
    static constexpr bool kCluster = true;
    __device__ static __forceinline__ void sync() { __syncthreads(); }
    __device__ static __forceinline__ int tid() { return threadIdx.x; }
};
// Four warps of the CTA (named barrier 1): sets of 33-128 particles, where the 16-warp barrier of the
// whole CTA costs more than the phases' arithmetic.
struct TeamQuad {
    static constexpr bool kCluster = false;
    static constexpr int kThreads = 128;
    __device__ static __forceinline__ void sync() { asm volatile("bar.sync 1, 128;" ::: "memory"); }
    __device__ static __forceinline__ int tid() { return threadIdx.x; }
};
struct TeamWarp {
    static constexpr bool kCluster = false;
    static constexpr int kThreads = 32;
    __device__ static __forceinline__ void sync() { __syncwarp(); }
    __device__ static __forceinline__ int tid() { return threadIdx.x & 31; }
};
constexpr int kWarpTeamMax = 32;
constexpr int kQuadTeamMax = 128;
constexpr int kClusterSize = 16;           // non-portable size (opt-in attribute), supported on sm_100
constexpr int kClusterMinSet = 192;        // smaller sets run on one CTA
// a sweep is shared out among the cluster from this many pairs (config-5 step on B200: 8192 and
// below 14.2-14.3 s, 32768 14.8 s, 131072 16.2 s, never 17.5 s)
constexpr long long kSplitPairs = 8192;

// Sharing a sweep over nA sinks out among the CTAs of a cluster.  Protocol per shared sweep: arrive
// on the cluster barrier at the start (peers may still be reading the replica fields this sweep
// will overwrite), wait before the first remote store, cluster.sync() at the end.
struct SinkShare { int lo, hi; bool split, waited; };

template <class T>
__device__ __forceinline__ SinkShare sweep_begin(int nA, int nB, bool allow = true) {
    SinkShare sh{0, nA, false, true};
    if (T::kCluster && allow) {
        namespace cg = cooperative_groups;
        cg::cluster_group cl = cg::this_cluster();
        if ((long long)nA * nB >= kSplitPairs && cl.num_blocks() > 1) {
            const int nr = (int)cl.num_blocks(), r = (int)cl.block_rank();
            const int chunk = (nA + nr - 1) / nr;
            sh.lo = min(nA, r * chunk); sh.hi = min(nA, sh.lo + chunk);
            sh.split = true; sh.waited = false;
            cl.barrier_arrive();
        }
    }
    return sh;
}
template <class T>
__device__ __forceinline__ void sweep_wait(SinkShare &sh) {
    if (T::kCluster && !sh.waited) {
        cooperative_groups::this_cluster().barrier_wait();
        sh.waited = true;
    }
}
// store one result into the replica(s)
template <class T, class V>
__device__ __forceinline__ void publish(const SinkShare &sh, V *slot, const V &val) {
    if (T::kCluster && sh.split) {
        namespace cg = cooperative_groups;
        cg::cluster_group cl = cg::this_cluster();
        const int nr = (int)cl.num_blocks();
        for (int r = 0; r < nr; ++r) *cl.map_shared_rank(slot, r) = val;
    } else {
        *slot = val;
    }
}
template <class T>
__device__ __forceinline__ void sweep_end(const SinkShare &sh) {
    if (T::kCluster && sh.split) cooperative_groups::this_cluster().sync();
    else T::sync();
}

// lanes per sink: largest power of two <= 32 with nA * L <= blockDim
// (and no more lanes than sources: every extra doubling is one more shuffle stage of latency)
template <class T>
__device__ __forceinline__ int lanes_per_sink(int nA, int nB) {
    int L = 1;
    while (L < 32 && L < nB && nA * (L * 2) <= T::kThreads) L *= 2;
    return L;
}

__device__ __forceinline__ double shfl_sum(double v, int L) {
    for (int o = L >> 1; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ double shfl_min(double v, int L) {
    for (int o = L >> 1; o > 0; o >>= 1) v = fmin(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

// a_i = G sum_{j in B} ...  for i in segment A (Eq. 24 / 42).  Segments are [a0, a0+nA) and
// [b0, b0+nB) of sm.perm.  All threads must call (uniform control flow, shuffles).
// MASK: a source in the sink's own component (sm.lab equal; slow particles all carry -1) is skipped
// -- the kicked pair set of a split entry (reading 24).
template <class T, bool MASK, class SM>
__device__ void cta_newton(SM &sm, const SweepParams &prm, int a0, int nA, int b0, int nB) {
    SinkShare sh = sweep_begin<T>(nA, nB);
    const int L = lanes_per_sink<T>(sh.hi - sh.lo, nB);
    const int per = T::kThreads / L;
    const int sub = T::tid() & (L - 1), slot = T::tid() / L;
    for (int base = sh.lo; base < sh.hi || !sh.waited; base += per) {
        const int a = base + slot;
        const bool live = a < sh.hi;
        const int i = sm.perm[a0 + (live ? a : 0)];
        const int li = MASK ? sm.lab[i] : 0;
        NewtonPolicy::Sink s;
        const double4 r = sm.xm[i];
        s.x = r.x; s.y = r.y; s.z = r.z;
        // kIlp independent partial sums per lane: the sweep of a small set is bound by the latency
        // of the dependent FP64 chain of a pair, not by issue
        constexpr int kIlp = 4;
        NewtonPolicy::Acc accs[kIlp];
#pragma unroll
        for (int u = 0; u < kIlp; ++u) NewtonPolicy::init(accs[u]);
        int b = sub;
        for (; b + (kIlp - 1) * L < nB; b += kIlp * L) {
#pragma unroll
            for (int u = 0; u < kIlp; ++u) {
                const int j = sm.perm[b0 + b + u * L];
                double4 j0 = sm.xm[j];
                if (MASK && sm.lab[j] == li) j0.w = 0.0;
                NewtonPolicy::pair(s, accs[u], j0, j0, prm);
            }
        }
        for (; b < nB; b += L) {
            const int j = sm.perm[b0 + b];
            double4 j0 = sm.xm[j];
            if (MASK && sm.lab[j] == li) j0.w = 0.0;
            NewtonPolicy::pair(s, accs[0], j0, j0, prm);
        }
        NewtonPolicy::Acc acc;
        acc.x = (accs[0].x + accs[1].x) + (accs[2].x + accs[3].x);
        acc.y = (accs[0].y + accs[1].y) + (accs[2].y + accs[3].y);
        acc.z = (accs[0].z + accs[1].z) + (accs[2].z + accs[3].z);
        acc.x = shfl_sum(acc.x, L); acc.y = shfl_sum(acc.y, L); acc.z = shfl_sum(acc.z, L);
        sweep_wait<T>(sh);
        if (live && sub == 0)
            publish<T>(sh, &sm.aa[i], make_double4(acc.x * prm.G, acc.y * prm.G, acc.z * prm.G, 1.0));
    }
    sweep_end<T>(sh);
}

// g_i = 2G sum_{j in B} ... using sm.aa of sinks and sources (Eq. 27 / 43 / 44).
template <class T, bool MASK, class SM>
__device__ void cta_gradient(SM &sm, const SweepParams &prm, int a0, int nA, int b0, int nB) {
    SinkShare sh = sweep_begin<T>(nA, nB);
    const int L = lanes_per_sink<T>(sh.hi - sh.lo, nB);
    const int per = T::kThreads / L;
    const int sub = T::tid() & (L - 1), slot = T::tid() / L;
    for (int base = sh.lo; base < sh.hi || !sh.waited; base += per) {
        const int a = base + slot;
        const bool live = a < sh.hi;
        const int i = sm.perm[a0 + (live ? a : 0)];
        const int li = MASK ? sm.lab[i] : 0;
        GradientPolicy::Sink s;
        const double4 r = sm.xm[i], ai = sm.aa[i];
        s.x = r.x; s.y = r.y; s.z = r.z; s.ax = ai.x; s.ay = ai.y; s.az = ai.z;
        GradientPolicy::Acc acc, acc1; GradientPolicy::init(acc); GradientPolicy::init(acc1);
        int b = sub;
        for (; b + L < nB; b += 2 * L) {
            const int j = sm.perm[b0 + b], j2 = sm.perm[b0 + b + L];
            double4 x0 = sm.xm[j], x1 = sm.xm[j2];
            if (MASK && sm.lab[j] == li) x0.w = 0.0;
            if (MASK && sm.lab[j2] == li) x1.w = 0.0;
            GradientPolicy::pair(s, acc, x0, sm.aa[j], prm);
            GradientPolicy::pair(s, acc1, x1, sm.aa[j2], prm);
        }
        if (b < nB) {
            const int j = sm.perm[b0 + b];
            double4 x0 = sm.xm[j];
            if (MASK && sm.lab[j] == li) x0.w = 0.0;
            GradientPolicy::pair(s, acc, x0, sm.aa[j], prm);
        }
        acc.x += acc1.x; acc.y += acc1.y; acc.z += acc1.z;
        acc.x = shfl_sum(acc.x, L); acc.y = shfl_sum(acc.y, L); acc.z = shfl_sum(acc.z, L);
        const double k2g = 2.0 * prm.G;
        sweep_wait<T>(sh);
        if (live && sub == 0) publish<T>(sh, &sm.gg[i], make_double4(acc.x * k2g, acc.y * k2g, acc.z * k2g, 0.0));
    }
    sweep_end<T>(sh);
}

// tau_i = min over the other members of the level (Eq. 49-54); a level of one particle: +inf.
// pivot > 0: every fast pair (candidate < pivot) is also entered into the union-find forest sm.par
// (the components of the level, reading 24).  Each pair is met from both sides, and in a
// cluster every replica needs every pair, so the sweep is then not shared out.
template <class T, class SM>
__device__ void cta_timesteps(SM &sm, const SweepParams &prm, int a0, int nA, double pivot) {
    const bool edges = pivot > 0.0;
    if (edges) {
        for (int a = T::tid(); a < nA; a += T::kThreads) { const int i = sm.perm[a0 + a]; sm.par[i] = i; }
        T::sync();
    }
    SinkShare sh = sweep_begin<T>(nA, nA, !edges);
    const int L = lanes_per_sink<T>(sh.hi - sh.lo, nA);
    const int per = T::kThreads / L;
    const int sub = T::tid() & (L - 1), slot = T::tid() / L;
    for (int base = sh.lo; base < sh.hi || !sh.waited; base += per) {
        const int a = base + slot;
        const bool live = a < sh.hi;
        const int i = sm.perm[a0 + (live ? a : 0)];
        TimestepPolicy::Sink s;
        const double4 r = sm.xm[i], v = sm.vv[i];
        s.x = r.x; s.y = r.y; s.z = r.z; s.gm = r.w * prm.G; s.vx = v.x; s.vy = v.y; s.vz = v.z;
        double t0 = __longlong_as_double(0x7ff0000000000000LL), t1 = t0;
        int b = sub;
        for (; b + L < nA; b += 2 * L) {
            const int j = sm.perm[a0 + b], j2 = sm.perm[a0 + b + L];
            double4 j0 = sm.xm[j], k0 = sm.xm[j2];
            j0.w *= prm.G; k0.w *= prm.G;
            const double c0 = TimestepPolicy::candidate(s, j0, sm.vv[j], prm);
            const double c1 = TimestepPolicy::candidate(s, k0, sm.vv[j2], prm);
            t0 = fmin(t0, c0); t1 = fmin(t1, c1);
            if (edges && live) {
                if (c0 < pivot) uf_union(sm.par, i, j);
                if (c1 < pivot) uf_union(sm.par, i, j2);
            }
        }
        if (b < nA) {
            const int j = sm.perm[a0 + b];
            double4 j0 = sm.xm[j];
            j0.w *= prm.G;
            const double c0 = TimestepPolicy::candidate(s, j0, sm.vv[j], prm);
            t0 = fmin(t0, c0);
            if (edges && live && c0 < pivot) uf_union(sm.par, i, j);
        }
        t0 = fmin(t0, t1);
        t0 = shfl_min(t0, L);
        sweep_wait<T>(sh);
        if (live && sub == 0) publish<T>(sh, &sm.tau[i], t0);
    }
    sweep_end<T>(sh);
}

// v_i += c (a_i + kappa g_i) ; x_i += c v_i  on a segment (Eq. 6).
template <class T, class SM>
__device__ void cta_kick(SM &sm, int a0, int nA, double c, double kappa, bool with_g) {
    for (int a = T::tid(); a < nA; a += T::kThreads) {
        const int i = sm.perm[a0 + a];
        double4 v = sm.vv[i];
        const double4 ac = sm.aa[i];
        double ax = ac.x, ay = ac.y, az = ac.z;
        if (with_g) {
            const double4 g = sm.gg[i];
            ax = fma(kappa, g.x, ax); ay = fma(kappa, g.y, ay); az = fma(kappa, g.z, az);
        }
        v.x = fma(c, ax, v.x); v.y = fma(c, ay, v.y); v.z = fma(c, az, v.z);
        sm.vv[i] = v;
    }
    T::sync();
}

// kick then drift of the same particles in one phase (both touch only the thread's own particle):
// v_i += ck (a_i + kappa g_i) ; x_i += cd v_i.
template <class T, class SM>
__device__ void cta_kick_drift(SM &sm, int a0, int nA, double ck, double kappa, bool with_g, double cd) {
    for (int a = T::tid(); a < nA; a += T::kThreads) {
        const int i = sm.perm[a0 + a];
        double4 v = sm.vv[i];
        double4 x = sm.xm[i];
        const double4 ac = sm.aa[i];
        double ax = ac.x, ay = ac.y, az = ac.z;
        if (with_g) {
            const double4 g = sm.gg[i];
            ax = fma(kappa, g.x, ax); ay = fma(kappa, g.y, ay); az = fma(kappa, g.z, az);
        }
        v.x = fma(ck, ax, v.x); v.y = fma(ck, ay, v.y); v.z = fma(ck, az, v.z);
        x.x = fma(cd, v.x, x.x); x.y = fma(cd, v.y, x.y); x.z = fma(cd, v.z, x.z);
        sm.vv[i] = v;
        sm.xm[i] = x;
    }
    T::sync();
}

// Stable in-place partition of the segment [a0, a0+n) of sm.perm: slow (tau >= pivot) first.
// Returns |S| (Eq. 29).
template <class T, class SM>
__device__ int cta_partition(SM &sm, int a0, int n, double pivot) {
    const int lane = T::tid() & 31, w = T::tid() >> 5;
    constexpr int kWarps = T::kThreads / 32;
    if (T::kThreads == 32) {     // one warp, n <= 32: ballot
        const int i = (lane < n) ? sm.perm[a0 + lane] : 0;
        const int f = (lane < n) ? (sm.tau[i] >= pivot) : 0;
        const unsigned m = __ballot_sync(0xffffffffu, f);
        const int nS = __popc(m), before = __popc(m & ((1u << lane) - 1u));
        __syncwarp();
        if (lane < n) sm.perm[a0 + (f ? before : nS + (lane - before))] = i;
        __syncwarp();
        return nS;
    }
    int nS = 0;
    for (int base = 0; base < n; base += T::kThreads) {
        const int k = base + T::tid();
        const int f = (k < n) ? (sm.tau[sm.perm[a0 + k]] >= pivot) : 0;
        const int cw = __popc(__ballot_sync(0xffffffffu, f));     // team-wide count of f
        if (lane == 0) sm.scan[w] = cw;
        T::sync();
        for (int q = 0; q < kWarps; ++q) nS += sm.scan[q];
        T::sync();
    }
    int carry = 0;
    for (int base = 0; base < n; base += T::kThreads) {
        const int k = base + T::tid();
        const int i = (k < n) ? sm.perm[a0 + k] : 0;
        const int f = (k < n) ? (sm.tau[i] >= pivot) : 0;
        int inc = f;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += t;
        }
        if (lane == 31) sm.scan[w] = inc;
        T::sync();
        int wbase = 0, total = 0;
        for (int q = 0; q < kWarps; ++q) {
            const int v = sm.scan[q];
            if (q < w) wbase += v;
            total += v;
        }
        const int slow_before = carry + wbase + inc - f;
        if (k < n) {
            if (f) sm.tmp[slow_before] = i;
            else sm.tmp[nS + (k - slow_before)] = i;
        }
        carry += total;
        T::sync();
    }
    for (int k = T::tid(); k < n; k += T::kThreads) sm.perm[a0 + k] = sm.tmp[k];
    T::sync();
    return nS;
}

// The connected components of the fast pairs of F = segment [f0, f0+nF) (forest sm.par built by
// cta_timesteps): F is reordered so that every component is contiguous -- components by their
// smallest member, members in their previous order -- and frame `sp` records where they start.
// Returns the number of components; *sumsq = sum of their squared sizes.
template <class T, class SM>
__device__ int cta_components(SM &sm, int f0, int nF, int sp, long long *sumsq) {
    for (int p = T::tid(); p < nF; p += T::kThreads) {
        const int i = sm.perm[f0 + p];
        sm.lab[i] = uf_find(sm.par, i);
    }
    for (int w = T::tid(); w < SM::kWords; w += T::kThreads) sm.f_bnd[sp][w] = 0u;
    T::sync();
    for (int p = T::tid(); p < nF; p += T::kThreads) {          // rank = position after a stable sort by label
        const int i = sm.perm[f0 + p], li = sm.lab[i];
        int rank = 0;
        for (int q = 0; q < nF; ++q) {
            const int lq = sm.lab[sm.perm[f0 + q]];
            rank += (lq < li) || (lq == li && q < p);
        }
        sm.tmp[rank] = i;
    }
    T::sync();
    for (int p = T::tid(); p < nF; p += T::kThreads) sm.perm[f0 + p] = sm.tmp[p];
    T::sync();
    for (int p = T::tid(); p < nF; p += T::kThreads)
        if (p == 0 || sm.lab[sm.perm[f0 + p]] != sm.lab[sm.perm[f0 + p - 1]])
            atomicOr(&sm.f_bnd[sp][p >> 5], 1u << (p & 31));
    T::sync();
    int m = 0, prev = -1;
    long long ss = 0;
    for (int w = 0; w < (nF + 31) / 32; ++w) {
        unsigned bits = sm.f_bnd[sp][w];
        while (bits) {
            const int r = w * 32 + __ffs(bits) - 1;
            bits &= bits - 1;
            if (prev >= 0) ss += (long long)(r - prev) * (r - prev);
            prev = r; ++m;
        }
    }
    if (prev >= 0) ss += (long long)(nF - prev) * (nF - prev);
    *sumsq = ss;
    return m;
}

// sm.lab of the members of an entry from its recorded component boundaries: -1 for S, the component's
// ordinal for F (the recursion below this entry reuses sm.lab for its own components).
template <class T, class SM>
__device__ void cta_labels(SM &sm, int start, int nS, int nF, int sp) {
    for (int a = T::tid(); a < nS; a += T::kThreads) sm.lab[sm.perm[start + a]] = -1;
    for (int p = T::tid(); p < nF; p += T::kThreads) {
        int c = 0;
        for (int w = 0; w < (p >> 5); ++w) c += __popc(sm.f_bnd[sp][w]);
        c += __popc(sm.f_bnd[sp][p >> 5] & (0xffffffffu >> (31 - (p & 31))));
        sm.lab[sm.perm[start + nS + p]] = c;
    }
    T::sync();
}

// size of the component of F that starts at position cpos (a set bit of the frame's boundary mask)
template <class SM>
__device__ __forceinline__ int comp_size(const SM &sm, int sp, int cpos, int nF) {
    int w = (cpos + 1) >> 5;
    if (cpos + 1 >= nF) return nF - cpos;
    unsigned bits = sm.f_bnd[sp][w] & (0xffffffffu << ((cpos + 1) & 31));
    const int words = (nF + 31) / 32;
    while (!bits && ++w < words) bits = sm.f_bnd[sp][w];
    const int next = bits ? w * 32 + __ffs(bits) - 1 : nF;
    return (next < nF ? next : nF) - cpos;
}

// fsi(set, dt): Alg. 2 on the segment [a0, a0+nA).
template <class T, class SM>
__device__ void cta_fsi(SM &sm, SmStats &st, const SweepParams &pN, const SweepParams &pG, int a0, int nA,
                        double dt) {
    if (nA <= 0) return;
    cta_newton<T, false>(sm, pN, a0, nA, a0, nA);
    cta_kick_drift<T>(sm, a0, nA, dt / 6.0, 0.0, false, dt / 2.0);
    cta_newton<T, false>(sm, pN, a0, nA, a0, nA);
    cta_gradient<T, false>(sm, pG, a0, nA, a0, nA);
    cta_kick_drift<T>(sm, a0, nA, 2.0 * dt / 3.0, dt * dt / 48.0, true, dt / 2.0);
    cta_newton<T, false>(sm, pN, a0, nA, a0, nA);
    cta_kick<T>(sm, a0, nA, dt / 6.0, 0.0, false);
    if (T::tid() == 0) {
        const unsigned long long np = (unsigned long long)nA * nA;
        atomicAdd(&st.pn, 3 * np);
        atomicAdd(&st.pg, np);
    }
}

// The inter-level kick of an entry (Eq. 42-44 on its kicked pair set; Alg. 3's kick_sf): accelerations
// (and gradient accelerations if with_g) of every member, then v += c (a + kappa g).  m <= 1: the pair
// set is S x F both ways (Alg. 3 as printed); m > 1: every pair of the entry that is neither slow-slow
// nor inside one component.
template <class T, class SM>
__device__ void cta_cross_kick(SM &sm, const SweepParams &pN, const SweepParams &pG, int start, int nS,
                               int nF, int m, int sp, double c, double kappa, bool with_g) {
    const int cnt = nS + nF;
    if (m > 1) {
        cta_labels<T>(sm, start, nS, nF, sp);
        cta_newton<T, true>(sm, pN, start, cnt, start, cnt);
        if (with_g) cta_gradient<T, true>(sm, pG, start, cnt, start, cnt);
        cta_kick<T>(sm, start, cnt, c, kappa, with_g);
    } else if (nS > 0 && nF > 0) {
        cta_newton<T, false>(sm, pN, start, nS, start + nS, nF);
        cta_newton<T, false>(sm, pN, start + nS, nF, start, nS);
        if (with_g) {
            cta_gradient<T, false>(sm, pG, start, nS, start + nS, nF);
            cta_gradient<T, false>(sm, pG, start + nS, nF, start, nS);
        }
        cta_kick<T>(sm, start, cnt, c, kappa, with_g);
    }
}

// ------------------------------------------------------------------------------------------------
// A frame of exactly two particles, executed by ONE thread with both particles in registers.
// In a two-body set both members have the same time step (the one pair candidate, symmetric), so
// every entry of Alg. 3 is either a leaf -- both slow: fsi(pair, tau/2) twice, every inter-level term
// empty -- or an inner node -- both fast: hhs_fsi(pair, tau/2) twice.  The subtree is therefore a
// binary tree over the interval [0, tau0), walked here with a time index instead of a frame stack:
// a node of relative depth d spans 2^(62-d) units; after a leaf that ends at index t the next node
// starts at t with depth 62 - ctz(t) (the second child of the deepest unfinished ancestor).  Same
// pair arithmetic (frost_pairs.cuh), same operator order and same bookkeeping as the team path --
// the results are bitwise those of hhs_loop on the same frame; what changes is the latency: no
// barriers, no shuffles, no shared-memory round trips between the ~20 dependent phases of an entry.
// This is the critical path of a split level: the hardest binary's chain.
// ------------------------------------------------------------------------------------------------
struct Body { double x, y, z, vx, vy, vz, m; };

__device__ __forceinline__ void pair_newton(const Body &p, const Body &q, const SweepParams &pN, double &ax,
                                            double &ay, double &az) {
    NewtonPolicy::Sink s; s.x = p.x; s.y = p.y; s.z = p.z;
    NewtonPolicy::Acc a; NewtonPolicy::init(a);
    const double4 j0 = make_double4(q.x, q.y, q.z, q.m);
    NewtonPolicy::pair(s, a, j0, j0, pN);
    ax = a.x * pN.G; ay = a.y * pN.G; az = a.z * pN.G;
}

__device__ __forceinline__ void pair_gradient(const Body &p, const double (&ap)[3], const Body &q,
                                              const double (&aq)[3], const SweepParams &pG, double &gx,
                                              double &gy, double &gz) {
    GradientPolicy::Sink s; s.x = p.x; s.y = p.y; s.z = p.z; s.ax = ap[0]; s.ay = ap[1]; s.az = ap[2];
    GradientPolicy::Acc g; GradientPolicy::init(g);
    GradientPolicy::pair(s, g, make_double4(q.x, q.y, q.z, q.m), make_double4(aq[0], aq[1], aq[2], 1.0), pG);
    const double k2g = 2.0 * pG.G;
    gx = g.x * k2g; gy = g.y * k2g; gz = g.z * k2g;
}

__device__ __forceinline__ void body_kick(Body &p, const double (&a)[3], double c) {
    p.vx = fma(c, a[0], p.vx); p.vy = fma(c, a[1], p.vy); p.vz = fma(c, a[2], p.vz);
}
__device__ __forceinline__ void body_kick_g(Body &p, const double (&a)[3], const double (&g)[3], double c,
                                            double kappa) {
    p.vx = fma(c, fma(kappa, g[0], a[0]), p.vx);
    p.vy = fma(c, fma(kappa, g[1], a[1]), p.vy);
    p.vz = fma(c, fma(kappa, g[2], a[2]), p.vz);
}
__device__ __forceinline__ void body_drift(Body &p, double c) {
    p.x = fma(c, p.vx, p.x); p.y = fma(c, p.vy, p.y); p.z = fma(c, p.vz, p.z);
}

// fsi(pair, dt): Alg. 2 on two bodies.
__device__ __forceinline__ void pair_fsi(Body &p, Body &q, const SweepParams &pN, const SweepParams &pG,
                                         double dt) {
    double ap[3], aq[3], gp[3], gq[3];
    pair_newton(p, q, pN, ap[0], ap[1], ap[2]); pair_newton(q, p, pN, aq[0], aq[1], aq[2]);
    body_kick(p, ap, dt / 6.0); body_kick(q, aq, dt / 6.0);
    body_drift(p, dt / 2.0); body_drift(q, dt / 2.0);
    pair_newton(p, q, pN, ap[0], ap[1], ap[2]); pair_newton(q, p, pN, aq[0], aq[1], aq[2]);
    pair_gradient(p, ap, q, aq, pG, gp[0], gp[1], gp[2]); pair_gradient(q, aq, p, ap, pG, gq[0], gq[1], gq[2]);
    body_kick_g(p, ap, gp, 2.0 * dt / 3.0, dt * dt / 48.0); body_kick_g(q, aq, gq, 2.0 * dt / 3.0, dt * dt / 48.0);
    body_drift(p, dt / 2.0); body_drift(q, dt / 2.0);
    pair_newton(p, q, pN, ap[0], ap[1], ap[2]); pair_newton(q, p, pN, aq[0], aq[1], aq[2]);
    body_kick(p, ap, dt / 6.0); body_kick(q, aq, dt / 6.0);
}

// ------------------------------------------------------------------------------------------------
// Two-body propagator (reading 25; the paper lists Kepler solvers among the modules a split
// level can hand its few-body systems to): the relative vector follows the Kepler flow of
// mu = G (m_1 + m_2), advanced over dt in universal variables -- one formula for ellipses, parabolas and
// hyperbolas -- and the centre of mass moves uniformly.
//     c_k(z) = sum_n (-z)^n / (2n + k)!,  z = alpha s^2,  alpha = 2 mu / r_0 - v_0^2
//     r_0 s c_1 + (r_0.v_0) s^2 c_2 + mu s^3 c_3 = dt            (increasing in s: bracketed Newton)
//     dr = -(mu/r_0) s^2 c_2 r_0 + (dt - mu s^3 c_3) v_0
//     dv = -(mu/(r r_0)) s c_1 r_0 - (mu/r) s^2 c_2 v_0,   r = r_0 c_0 + (r_0.v_0) s c_1 + mu s^2 c_2
// The bodies are moved by DISPLACEMENTS (x_1 += V dt - (m_2/M) dr, ...), never rebuilt from the centre
// of mass, so that a binary of size 1e-5 at |x| ~ 1 keeps its relative accuracy.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void stumpff(double z, double &c0, double &c1, double &c2, double &c3) {
    int k = 0;
    while (fabs(z) > 0.1) { z *= 0.25; ++k; }
    // nested form of the two series to z^9 (|z| <= 0.1: the neglected terms are below 1e-30)
    double h2 = 1.0, h3 = 1.0;
#pragma unroll
    for (int n = 9; n >= 1; --n) {
        h2 = 1.0 - z * h2 / (double)((2 * n + 1) * (2 * n + 2));
        h3 = 1.0 - z * h3 / (double)((2 * n + 2) * (2 * n + 3));
    }
    c2 = 0.5 * h2; c3 = h3 / 6.0;
    c1 = 1.0 - z * c3; c0 = 1.0 - z * c2;
    for (; k > 0; --k) {          // c_k(4z) from c_k(z)
        c3 = 0.25 * (c2 + c0 * c3);
        c2 = 0.5 * c1 * c1;
        c1 = c0 * c1;
        c0 = 2.0 * c0 * c0 - 1.0;
    }
}

__device__ void kepler_bodies(Body &p, Body &q, double G, double dt) {
    const double rx = q.x - p.x, ry = q.y - p.y, rz = q.z - p.z;
    const double vx = q.vx - p.vx, vy = q.vy - p.vy, vz = q.vz - p.vz;
    const double mt = p.m + q.m, mu = G * mt;
    const double r0 = sqrt(rx * rx + ry * ry + rz * rz);
    const double v2 = vx * vx + vy * vy + vz * vz, u = rx * vx + ry * vy + rz * vz;
    const double alpha = 2.0 * mu / r0 - v2;
    double t = dt;
    if (alpha > 0.0) {                                  // bound: whole periods change nothing
        const double P = 6.283185307179586476925 * mu / (alpha * sqrt(alpha));
        t -= floor(t / P) * P;
    }
    double c0, c1, c2, c3, lo = 0.0, hi = t / r0, s;
    for (int it = 0; it < 1100; ++it) {                 // bracket the root
        stumpff(alpha * hi * hi, c0, c1, c2, c3);
        if (r0 * hi * c1 + u * hi * hi * c2 + mu * hi * hi * hi * c3 - t > 0.0) break;
        lo = hi; hi = 2.0 * hi + 1e-300;
    }
    s = 0.5 * (lo + hi);
    for (int it = 0; it < 100; ++it) {
        stumpff(alpha * s * s, c0, c1, c2, c3);
        const double F = r0 * s * c1 + u * s * s * c2 + mu * s * s * s * c3 - t;
        if (F == 0.0) break;
        const double dF = r0 * c0 + u * s * c1 + mu * s * s * c2;
        if (F > 0.0) hi = s; else lo = s;
        double sn = s - F / dF;
        if (!(sn >= lo && sn <= hi)) sn = 0.5 * (lo + hi);
        const bool done = fabs(sn - s) <= 2.3e-16 * fabs(s);
        s = sn;
        if (done) break;
    }
    stumpff(alpha * s * s, c0, c1, c2, c3);
    const double rr = r0 * c0 + u * s * c1 + mu * s * s * c2;
    const double fm1 = -(mu / r0) * s * s * c2, g = t - mu * s * s * s * c3;
    const double fd = -(mu / (rr * r0)) * s * c1, gdm1 = -(mu / rr) * s * s * c2;
    const double drx = fm1 * rx + g * vx, dry = fm1 * ry + g * vy, drz = fm1 * rz + g * vz;
    const double dvx = fd * rx + gdm1 * vx, dvy = fd * ry + gdm1 * vy, dvz = fd * rz + gdm1 * vz;
    const double wp = q.m / mt, wq = p.m / mt;
    const double Vx = wq * p.vx + wp * q.vx, Vy = wq * p.vy + wp * q.vy, Vz = wq * p.vz + wp * q.vz;
    p.x += fma(Vx, dt, -wp * drx); p.y += fma(Vy, dt, -wp * dry); p.z += fma(Vz, dt, -wp * drz);
    q.x += fma(Vx, dt, wq * drx); q.y += fma(Vy, dt, wq * dry); q.z += fma(Vz, dt, wq * drz);
    p.vx -= wp * dvx; p.vy -= wp * dvy; p.vz -= wp * dvz;
    q.vx += wq * dvx; q.vy += wq * dvy; q.vz += wq * dvz;
}

template <class SM>
__device__ void kepler_frame(SM &sm, SmStats &st, const SmallParams &P, int sp) {
    const int start = sm.f_start[sp];
    const int i1 = sm.perm[start], i2 = sm.perm[start + 1];
    Body p, q;
    { const double4 x = sm.xm[i1], v = sm.vv[i1]; p.x = x.x; p.y = x.y; p.z = x.z; p.m = x.w; p.vx = v.x; p.vy = v.y; p.vz = v.z; }
    { const double4 x = sm.xm[i2], v = sm.vv[i2]; q.x = x.x; q.y = x.y; q.z = x.z; q.m = x.w; q.vx = v.x; q.vy = v.y; q.vz = v.z; }
    kepler_bodies(p, q, P.G, sm.f_tau[sp]);
    sm.xm[i1] = make_double4(p.x, p.y, p.z, p.m); sm.vv[i1] = make_double4(p.vx, p.vy, p.vz, 1.0);
    sm.xm[i2] = make_double4(q.x, q.y, q.z, q.m); sm.vv[i2] = make_double4(q.vx, q.vy, q.vz, 1.0);
    atomicAdd(&st.kep, 1ull);
    sm.sp = sp - 1;
}

template <class SM>
__device__ void binary_subtree(SM &sm, SmStats &st, const SmallParams &P, const SweepParams &pN,
                               const SweepParams &pG, int sp) {
    const int start = sm.f_start[sp];
    const int i1 = sm.perm[start], i2 = sm.perm[start + 1];
    const double tau0 = sm.f_tau[sp];
    const int level0 = P.level0 + sp;
    Body p, q;
    { const double4 x = sm.xm[i1], v = sm.vv[i1]; p.x = x.x; p.y = x.y; p.z = x.z; p.m = x.w; p.vx = v.x; p.vy = v.y; p.vz = v.z; }
    { const double4 x = sm.xm[i2], v = sm.vv[i2]; q.x = x.x; q.y = x.y; q.z = x.z; q.m = x.w; q.vx = v.x; q.vy = v.y; q.vz = v.z; }
    const double inf = __longlong_as_double(0x7ff0000000000000LL);
    unsigned long long t = 0, leaves = 0, nodes = 0;
    int d = 0, dmax = 0, err = 0;
    while (true) {
        if (level0 + d >= P.max_depth || sp + d >= FROST_MAX_LEVELS - 1 || d > 61) { err = FROST_EDEPTH; break; }
        TimestepPolicy::Sink s;
        s.x = p.x; s.y = p.y; s.z = p.z; s.gm = p.m * pG.G; s.vx = p.vx; s.vy = p.vy; s.vz = p.vz;
        const double c = fmin(inf, TimestepPolicy::candidate(s, make_double4(q.x, q.y, q.z, q.m * pG.G),
                                                              make_double4(q.vx, q.vy, q.vz, 1.0), pG));
        const double tau = ldexp(tau0, -d);
        const int level = level0 + d;
        ++nodes;
        atomicAdd(&st.entries[level], 1ull);
        if (d > dmax) dmax = d;
        if (c >= tau) {                       // both slow: a leaf
            atomicAdd(&st.slow[level], 2ull);
            pair_fsi(p, q, pN, pG, 0.5 * tau);
            pair_fsi(p, q, pN, pG, 0.5 * tau);
            ++leaves;
            t += 1ull << (62 - d);
            if (t >> 62) break;               // the root's interval is done
            d = 62 - (__ffsll((long long)t) - 1);
        } else {                              // both fast: one component, recursed into twice
            atomicAdd(&st.fast[level], 2ull);
            atomicAdd(&st.comps[level], 1ull);
            ++d;
        }
    }
    atomicAdd(&st.pt, 4ull * nodes);
    atomicAdd(&st.pn, 24ull * leaves);        // two fsi per leaf, three sweeps of 4 ordered pairs each
    atomicAdd(&st.pg, 8ull * leaves);
    atomicMax(&st.depth, level0 + dmax);
    sm.xm[i1] = make_double4(p.x, p.y, p.z, p.m); sm.vv[i1] = make_double4(p.vx, p.vy, p.vz, 1.0);
    sm.xm[i2] = make_double4(q.x, q.y, q.z, q.m); sm.vv[i2] = make_double4(q.vx, q.vy, q.vz, 1.0);
    if (err) sm.err = err;
    sm.sp = sp - 1;
}

// The hhs_fsi recursion of Alg. 3 as a state machine over the explicit frame stack; runs until the
// frame at base_sp has been popped.  Stages of a frame: 0 = entry (time steps, partition, components,
// first kick, fsi(S)); 1 = first recursion pass over the components of F in progress; 2 = second pass.
template <class T, class SM>
__device__ void hhs_loop(SM &sm, SmStats &st, const SmallParams &P, const SweepParams &pN,
                         const SweepParams &pG, int base_sp) {
    while (true) {
        T::sync();
        const int sp = sm.sp;
        if (sp < base_sp || sm.err) break;
        const int start = sm.f_start[sp], cnt = sm.f_n[sp], stage = sm.f_stage[sp];
        const double tau = sm.f_tau[sp];
        const int level = P.level0 + sp;
        if (stage == 0 && cnt == 2 && P.kepler && sm.f_iscomp[sp] && P.eps2 == 0.0) {
            // a two-body component of a split entry: exact two-body motion over its span (reading 25)
            T::sync();                                    // everyone has read sm.sp before it is popped
            if (T::tid() == 0) kepler_frame(sm, st, P, sp);
            continue;
        }
        // a binary: one thread, both bodies in registers.  Not when its fast levels belong to the Kepler
        // propagator: a two-body frame that is not itself a component (the root of a two-body step, a
        // two-body F below an unsplit parent) is then split by the team path like any other entry, and
        // its one component -- the same two bodies -- takes kepler_frame above (reading 25).
        const bool kepler_owns_pairs = P.kepler && P.split_max >= 2 && P.eps2 == 0.0;
        if (stage == 0 && cnt == 2 && P.pair_path && !kepler_owns_pairs) {
            T::sync();
            if (T::tid() == 0) binary_subtree(sm, st, P, pN, pG, sp);
            continue;
        }
        if (T::kThreads > 128 && stage == 0 && cnt > kWarpTeamMax && cnt <= kQuadTeamMax) {
            // the whole subtree of this entry on warps 0-3 (see TeamQuad)
            if (threadIdx.x < 128) hhs_loop<TeamQuad>(sm, st, P, pN, pG, sp);
            continue;
        }
        if (T::kThreads > 32 && stage == 0 && cnt > 0 && cnt <= kWarpTeamMax) {
            // the whole subtree of this entry on warp 0 (latency-bound: see TeamWarp)
            if (threadIdx.x < 32) hhs_loop<TeamWarp>(sm, st, P, pN, pG, sp);
            continue;
        }
        if (stage == 0) {
            if (cnt <= 0) {
                T::sync();
                if (T::tid() == 0) sm.sp = sp - 1;
                continue;
            }
            if (level >= P.max_depth || sp >= FROST_MAX_LEVELS - 1) {
                T::sync();
                if (T::tid() == 0) sm.err = FROST_EDEPTH;
                continue;
            }
            const bool split = P.split_max > 0 && cnt <= P.split_max;
            cta_timesteps<T>(sm, pG, start, cnt, split ? tau : -1.0);
            const int nS = cta_partition<T>(sm, start, cnt, tau);
            const int nF = cnt - nS;
            int m = nF > 0 ? 1 : 0;
            long long sumsq = (long long)nF * nF;
            if (split && nF > 0) m = cta_components<T>(sm, start + nS, nF, sp, &sumsq);
            else if (T::tid() == 0) sm.f_bnd[sp][0] = 1u;
            cta_cross_kick<T>(sm, pN, pG, start, nS, nF, m, sp, tau / 6.0, 0.0, false);
            cta_fsi<T>(sm, st, pN, pG, start, nS, 0.5 * tau);
            T::sync();
            if (T::tid() == 0) {
                sm.f_ns[sp] = nS; sm.f_m[sp] = m; sm.f_sumsq[sp] = sumsq; sm.f_cpos[sp] = 0;
                atomicAdd(&st.entries[level], 1ull); atomicAdd(&st.slow[level], (unsigned long long)nS);
                atomicAdd(&st.fast[level], (unsigned long long)nF); atomicAdd(&st.comps[level], (unsigned long long)m);
                atomicAdd(&st.pt, (unsigned long long)cnt * cnt);
                atomicMax(&st.depth, level);
                sm.f_stage[sp] = 1;
            }
        } else {
            const int nS = sm.f_ns[sp], nF = cnt - nS, m = sm.f_m[sp], cpos = sm.f_cpos[sp];
            if (cpos < nF) {            // hhs_fsi(C_c, tau/2) of the next component
                const int size = (m > 1) ? comp_size(sm, sp, cpos, nF) : nF;
                T::sync();
                if (T::tid() == 0) {
                    sm.f_cpos[sp] = cpos + size;
                    sm.f_start[sp + 1] = start + nS + cpos; sm.f_n[sp + 1] = size; sm.f_ns[sp + 1] = 0;
                    sm.f_stage[sp + 1] = 0; sm.f_tau[sp + 1] = 0.5 * tau;
                    sm.f_iscomp[sp + 1] = (P.split_max > 0 && cnt <= P.split_max) ? 1 : 0;
                    sm.sp = sp + 1;
                }
            } else if (stage == 1) {
                cta_cross_kick<T>(sm, pN, pG, start, nS, nF, m, sp, 2.0 * tau / 3.0, tau * tau / 48.0, true);
                T::sync();
                if (T::tid() == 0) { sm.f_stage[sp] = 2; sm.f_cpos[sp] = 0; }
            } else {
                cta_fsi<T>(sm, st, pN, pG, start, nS, 0.5 * tau);
                cta_cross_kick<T>(sm, pN, pG, start, nS, nF, m, sp, tau / 6.0, 0.0, false);
                T::sync();
                if (T::tid() == 0) {
                    // ordered pairs of the kicked set: all but slow-slow and same-component pairs
                    const unsigned long long cr =
                        (unsigned long long)((long long)cnt * cnt - (long long)nS * nS - sm.f_sumsq[sp]);
                    atomicAdd(&st.pn, 3 * cr); atomicAdd(&st.pg, cr);
                    sm.sp = sp - 1;
                }
            }
        }
    }
}

__device__ __forceinline__ void stats_zero(SmStats &st, int tid, int nthreads) {
    for (int k = tid; k < FROST_MAX_LEVELS; k += nthreads) {
        st.entries[k] = 0; st.slow[k] = 0; st.fast[k] = 0; st.comps[k] = 0;
    }
    if (tid == 0) { st.pn = st.pg = st.pt = st.kep = 0; st.depth = -1; }
}

// atomics: an fsi(S) launch on a side stream, or other CTAs of a batch, run concurrently
__device__ __forceinline__ void stats_flush(const SmStats &st, SmallStats *out, int err, int tid, int nthreads) {
    typedef unsigned long long ull;
    for (int k = tid; k < FROST_MAX_LEVELS; k += nthreads) {
        if (st.entries[k]) {
            atomicAdd((ull *)&out->entries[k], st.entries[k]);
            atomicAdd((ull *)&out->n_slow[k], st.slow[k]);
            atomicAdd((ull *)&out->n_fast[k], st.fast[k]);
            atomicAdd((ull *)&out->n_comp[k], st.comps[k]);
        }
    }
    if (tid == 0) {
        atomicAdd((ull *)&out->pairs_newton, st.pn);
        atomicAdd((ull *)&out->pairs_gradient, st.pg);
        atomicAdd((ull *)&out->pairs_timestep, st.pt);
        if (st.kep) atomicAdd((ull *)&out->n_kepler, st.kep);
        atomicMax(&out->depth, st.depth);
        if (err) atomicCAS(&out->status, 0, err);
    }
}

template <class SM>
__device__ __forceinline__ void set_load(SM &sm, const SmallParams &P, const int32_t *idx, int n, int tid,
                                         int nthreads) {
    const int ld = P.ld;
    for (int k = tid; k < n; k += nthreads) {
        const int i = idx ? idx[k] : k;
        sm.xm[k] = make_double4(P.pos[i], P.pos[(size_t)ld + i], P.pos[2 * (size_t)ld + i], P.mass[i]);
        sm.vv[k] = make_double4(P.vel[i], P.vel[(size_t)ld + i], P.vel[2 * (size_t)ld + i], 1.0);
        sm.perm[k] = k;
    }
    if (tid == 0) {
        sm.sp = 0; sm.err = 0;
        sm.f_start[0] = 0; sm.f_n[0] = n; sm.f_ns[0] = 0; sm.f_stage[0] = 0; sm.f_tau[0] = P.tau_pivot;
        sm.f_iscomp[0] = P.root_is_comp;
    }
}

template <class SM>
__device__ __forceinline__ void set_store(const SM &sm, const SmallParams &P, const int32_t *idx, int n,
                                          int tid, int nthreads) {
    const int ld = P.ld;
    for (int k = tid; k < n; k += nthreads) {
        const int i = idx ? idx[k] : k;
        const double4 x = sm.xm[k], v = sm.vv[k];
        P.pos[i] = x.x; P.pos[(size_t)ld + i] = x.y; P.pos[2 * (size_t)ld + i] = x.z;
        P.vel[i] = v.x; P.vel[(size_t)ld + i] = v.y; P.vel[2 * (size_t)ld + i] = v.z;
    }
}

__device__ __forceinline__ void sweep_params(const SmallParams &P, SweepParams &pN, SweepParams &pG) {
    pN = SweepParams{}; pG = SweepParams{};
    pN.G = pG.G = P.G; pN.eta_ff = pG.eta_ff = P.eta_ff; pN.eta_fb = pG.eta_fb = P.eta_fb;
    pG.eps2 = P.eps2;
    pN.eps2 = P.eps2 > 0x1p-400 ? P.eps2 : 0x1p-400;     // see NewtonPolicy::pair
}

// One set per CTA (or per cluster of replica CTAs).  With P.desc the launch is a batch: CTA b takes
// the set described by desc[b] (components of 33-1024 particles of a split entry).
template <class T>
__global__ void __launch_bounds__(kSmallThreads, 1) hhs_small_kernel(const SmallParams P) {
    extern __shared__ __align__(16) unsigned char small_raw[];
    SmallSmem &sm = *reinterpret_cast<SmallSmem *>(small_raw);
    SmStats &st = *reinterpret_cast<SmStats *>(small_raw + sizeof(SmallSmem));
    const int32_t *idx = P.idx;
    int n = P.n;
    if (P.desc) {
        if ((int)blockIdx.x >= *P.n_desc) return;
        const int2 d = P.desc[blockIdx.x];
        idx = P.idx + d.x; n = d.y;
    }
    set_load(sm, P, idx, n, threadIdx.x, kSmallThreads);
    stats_zero(st, threadIdx.x, kSmallThreads);
    SweepParams pN, pG;
    sweep_params(P, pN, pG);
    __syncthreads();

    if (P.mode == 1) {
        for (int k = 0; k < P.n_steps; ++k) {
            if (n <= kWarpTeamMax) { if (threadIdx.x < 32) cta_fsi<TeamWarp>(sm, st, pN, pG, 0, n, P.dt_fsi); }
            else cta_fsi<T>(sm, st, pN, pG, 0, n, P.dt_fsi);
        }
    } else {
        hhs_loop<T>(sm, st, P, pN, pG, 0);
    }
    __syncthreads();
    if (T::kCluster) {      // replicas are identical: rank 0 writes back; nobody leaves while a peer
        namespace cg = cooperative_groups;                       // could still store into its replica
        cg::cluster_group cl = cg::this_cluster();
        cl.sync();
        if (cl.block_rank() != 0) return;
    }
    set_store(sm, P, idx, n, threadIdx.x, kSmallThreads);
    if (P.stats) stats_flush(st, P.stats, sm.err, threadIdx.x, kSmallThreads);
}

// Batch of small components (<= 32 particles each, in practice binaries and triples): one WARP per
// component, kCompWarps per CTA, each with its own 8 KB of shared memory -- the deep hierarchy of a
// hard binary is a chain of dependent phases on one warp, and all the unrelated
// binaries of a split level run their chains side by side instead of one after the other.
using CompSmem = SmallSmemT<kCompWarpMax>;

__global__ void __launch_bounds__(kCompWarps * 32) hhs_comp_kernel(const SmallParams P) {
    extern __shared__ __align__(16) unsigned char small_raw[];
    CompSmem *sms = reinterpret_cast<CompSmem *>(small_raw);
    SmStats &st = *reinterpret_cast<SmStats *>(small_raw + kCompWarps * sizeof(CompSmem));
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    stats_zero(st, threadIdx.x, kCompWarps * 32);
    __syncthreads();
    const int c = blockIdx.x * kCompWarps + warp;
    int err = 0;
    if (c < *P.n_desc) {
        CompSmem &sm = sms[warp];
        const int2 d = P.desc[c];
        const int32_t *idx = P.idx + d.x;
        set_load(sm, P, idx, d.y, lane, 32);
        SweepParams pN, pG;
        sweep_params(P, pN, pG);
        __syncwarp();
        hhs_loop<TeamWarp>(sm, st, P, pN, pG, 0);
        __syncwarp();
        set_store(sm, P, idx, d.y, lane, 32);
        err = sm.err;
    }
    err = __syncthreads_or(err);
    if (P.stats) stats_flush(st, P.stats, err ? FROST_EDEPTH : 0, threadIdx.x, kCompWarps * 32);
}

int small_max() { return kSmallMax; }
int comp_warp_max() { return kCompWarpMax; }

static SmallParams small_params(frost_ctx *c, int mode, int ld, double *pos, double *vel, const double *mass,
                                const int32_t *idx, int n, double tau_or_dt, int level0, void *dev_stats,
                                int n_steps) {
    SmallParams P{};
    P.idx = idx; P.n = n; P.ld = ld; P.pos = pos; P.vel = vel; P.mass = mass;
    P.tau_pivot = tau_or_dt; P.dt_fsi = tau_or_dt; P.mode = mode; P.level0 = level0; P.n_steps = n_steps;
    P.max_depth = c->max_depth; P.G = c->G; P.eps2 = c->eps2; P.eta_ff = c->eta_ff; P.eta_fb = c->eta_fb;
    P.stats = (SmallStats *)dev_stats;
    P.split_max = c->split_max;
    P.pair_path = c->tune_pair;
    P.kepler = c->kepler;
    return P;
}

static int small_attrs(frost_ctx *c) {
    const int bytes = (int)(sizeof(SmallSmem) + sizeof(SmStats));
    FROST_TRY(set_func_attr(c, hhs_small_kernel<TeamCTA>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
    FROST_TRY(set_func_attr(c, hhs_small_kernel<TeamCluster>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
    FROST_TRY(set_func_attr(c, hhs_small_kernel<TeamCluster>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
    FROST_TRY(set_func_attr(c, hhs_comp_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                            (int)(kCompWarps * sizeof(CompSmem) + sizeof(SmStats))));
    return FROST_OK;
}

// mode 0: hhs_fsi(set, tau) subtree rooted at hierarchy level `level0`; mode 1: fsi(set, dt).
int launch_small(frost_ctx *c, int mode, int ld, double *pos, double *vel, const double *mass,
                 const int32_t *idx, int n, double tau_or_dt, int level0, void *dev_stats, int n_steps,
                 int root_is_comp) {
    if (n <= 0) return FROST_OK;
    if (n > kSmallMax) return FROST_EINVAL;
    FROST_TRY(small_attrs(c));
    SmallParams P = small_params(c, mode, ld, pos, vel, mass, idx, n, tau_or_dt, level0, dev_stats, n_steps);
    P.root_is_comp = root_is_comp;
    const size_t bytes = sizeof(SmallSmem) + sizeof(SmStats);
    if (n >= kClusterMinSet && c->tune_cluster != 1) {   // one cluster of kClusterSize replicas
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3(kClusterSize); cfg.blockDim = dim3(kSmallThreads);
        cfg.dynamicSmemBytes = bytes; cfg.stream = c->stream;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = kClusterSize; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        FROST_CUDA(c, cudaLaunchKernelEx(&cfg, hhs_small_kernel<TeamCluster>, P));
    } else {
        hhs_small_kernel<TeamCTA><<<1, kSmallThreads, bytes, c->stream>>>(P);
    }
    return check_launch(c);
}

// hhs_fsi(C, tau) for a batch of components of one split entry (device-resident descriptors:
// desc[b] = {offset into idx, size}, *n_desc of them, at most max_desc).  warp_team: components of at
// most kCompWarpMax particles, one warp each; otherwise up to kSmallMax particles, one CTA each.
int launch_comp_batch(frost_ctx *c, int warp_team, int ld, double *pos, double *vel, const double *mass,
                      const int32_t *idx, const void *desc, const int *n_desc, int max_desc, double tau,
                      int level0, void *dev_stats) {
    if (max_desc <= 0) return FROST_OK;
    FROST_TRY(small_attrs(c));
    SmallParams P = small_params(c, 0, ld, pos, vel, mass, idx, 0, tau, level0, dev_stats, 1);
    P.desc = (const int2 *)desc; P.n_desc = n_desc; P.root_is_comp = 1;
    if (warp_team) {
        const int grid = (max_desc + kCompWarps - 1) / kCompWarps;
        hhs_comp_kernel<<<grid, kCompWarps * 32, kCompWarps * sizeof(CompSmem) + sizeof(SmStats), c->stream>>>(P);
    } else {
        hhs_small_kernel<TeamCTA><<<max_desc, kSmallThreads, sizeof(SmallSmem) + sizeof(SmStats), c->stream>>>(P);
    }
    return check_launch(c);
}

size_t small_stats_bytes() { return sizeof(SmallStats); }

}  // namespace frost
