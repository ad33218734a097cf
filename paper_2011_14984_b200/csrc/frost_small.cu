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

struct SmallStats {                 // device-side mirror of frost_hhs_stats (+ status)
    long long entries[FROST_MAX_LEVELS], n_slow[FROST_MAX_LEVELS], n_fast[FROST_MAX_LEVELS];
    long long pairs_newton, pairs_gradient, pairs_timestep;
    int depth, status;
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
};

struct SmallSmem {
    double4 xm[kSmallMax];          // x, y, z, m
    double4 vv[kSmallMax];          // vx, vy, vz, 1
    double4 aa[kSmallMax];          // ax, ay, az, 1
    double4 gg[kSmallMax];          // gx, gy, gz, -
    double tau[kSmallMax];
    int perm[kSmallMax];            // the level sets are contiguous segments of this list
    int tmp[kSmallMax];
    int scan[kSmallThreads / 32 + 1];
    // explicit recursion stack
    int f_start[FROST_MAX_LEVELS], f_n[FROST_MAX_LEVELS], f_ns[FROST_MAX_LEVELS], f_stage[FROST_MAX_LEVELS];
    double f_tau[FROST_MAX_LEVELS];
    int sp, err;
    long long st_entries[FROST_MAX_LEVELS], st_slow[FROST_MAX_LEVELS], st_fast[FROST_MAX_LEVELS];
    long long st_pn, st_pg, st_pt;
    int st_depth;
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
__device__ __forceinline__ SinkShare sweep_begin(int nA, int nB) {
    SinkShare sh{0, nA, false, true};
    if (T::kCluster) {
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
template <class T>
__device__ void cta_newton(SmallSmem &sm, const SweepParams &prm, int a0, int nA, int b0, int nB) {
    SinkShare sh = sweep_begin<T>(nA, nB);
    const int L = lanes_per_sink<T>(sh.hi - sh.lo, nB);
    const int per = T::kThreads / L;
    const int sub = T::tid() & (L - 1), slot = T::tid() / L;
    for (int base = sh.lo; base < sh.hi || !sh.waited; base += per) {
        const int a = base + slot;
        const bool live = a < sh.hi;
        const int i = sm.perm[a0 + (live ? a : 0)];
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
                const double4 j0 = sm.xm[sm.perm[b0 + b + u * L]];
                NewtonPolicy::pair(s, accs[u], j0, j0, prm);
            }
        }
        for (; b < nB; b += L) {
            const double4 j0 = sm.xm[sm.perm[b0 + b]];
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
template <class T>
__device__ void cta_gradient(SmallSmem &sm, const SweepParams &prm, int a0, int nA, int b0, int nB) {
    SinkShare sh = sweep_begin<T>(nA, nB);
    const int L = lanes_per_sink<T>(sh.hi - sh.lo, nB);
    const int per = T::kThreads / L;
    const int sub = T::tid() & (L - 1), slot = T::tid() / L;
    for (int base = sh.lo; base < sh.hi || !sh.waited; base += per) {
        const int a = base + slot;
        const bool live = a < sh.hi;
        const int i = sm.perm[a0 + (live ? a : 0)];
        GradientPolicy::Sink s;
        const double4 r = sm.xm[i], ai = sm.aa[i];
        s.x = r.x; s.y = r.y; s.z = r.z; s.ax = ai.x; s.ay = ai.y; s.az = ai.z;
        GradientPolicy::Acc acc, acc1; GradientPolicy::init(acc); GradientPolicy::init(acc1);
        int b = sub;
        for (; b + L < nB; b += 2 * L) {
            const int j = sm.perm[b0 + b], j2 = sm.perm[b0 + b + L];
            GradientPolicy::pair(s, acc, sm.xm[j], sm.aa[j], prm);
            GradientPolicy::pair(s, acc1, sm.xm[j2], sm.aa[j2], prm);
        }
        if (b < nB) {
            const int j = sm.perm[b0 + b];
            GradientPolicy::pair(s, acc, sm.xm[j], sm.aa[j], prm);
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
template <class T>
__device__ void cta_timesteps(SmallSmem &sm, const SweepParams &prm, int a0, int nA) {
    SinkShare sh = sweep_begin<T>(nA, nA);
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
        TimestepPolicy::Acc acc, acc1; TimestepPolicy::init(acc); TimestepPolicy::init(acc1);
        int b = sub;
        for (; b + L < nA; b += 2 * L) {
            const int j = sm.perm[a0 + b], j2 = sm.perm[a0 + b + L];
            double4 j0 = sm.xm[j], k0 = sm.xm[j2];
            j0.w *= prm.G; k0.w *= prm.G;
            TimestepPolicy::pair(s, acc, j0, sm.vv[j], prm);
            TimestepPolicy::pair(s, acc1, k0, sm.vv[j2], prm);
        }
        if (b < nA) {
            const int j = sm.perm[a0 + b];
            double4 j0 = sm.xm[j];
            j0.w *= prm.G;
            TimestepPolicy::pair(s, acc, j0, sm.vv[j], prm);
        }
        acc.tau = fmin(acc.tau, acc1.tau);
        acc.tau = shfl_min(acc.tau, L);
        sweep_wait<T>(sh);
        if (live && sub == 0) publish<T>(sh, &sm.tau[i], acc.tau);
    }
    sweep_end<T>(sh);
}

// v_i += c (a_i + kappa g_i) ; x_i += c v_i  on a segment (Eq. 6).
template <class T>
__device__ void cta_kick(SmallSmem &sm, int a0, int nA, double c, double kappa, bool with_g) {
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

template <class T>
__device__ void cta_drift(SmallSmem &sm, int a0, int nA, double c) {
    for (int a = T::tid(); a < nA; a += T::kThreads) {
        const int i = sm.perm[a0 + a];
        double4 x = sm.xm[i];
        const double4 v = sm.vv[i];
        x.x = fma(c, v.x, x.x); x.y = fma(c, v.y, x.y); x.z = fma(c, v.z, x.z);
        sm.xm[i] = x;
    }
    T::sync();
}

// kick then drift of the same particles in one phase (both touch only the thread's own particle):
// v_i += ck (a_i + kappa g_i) ; x_i += cd v_i.
template <class T>
__device__ void cta_kick_drift(SmallSmem &sm, int a0, int nA, double ck, double kappa, bool with_g,
                               double cd) {
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
template <class T>
__device__ int cta_partition(SmallSmem &sm, int a0, int n, double pivot) {
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

// fsi(set, dt): Alg. 2 on the segment [a0, a0+nA).
template <class T>
__device__ void cta_fsi(SmallSmem &sm, const SweepParams &pN, const SweepParams &pG, int a0, int nA,
                        double dt) {
    if (nA <= 0) return;
    cta_newton<T>(sm, pN, a0, nA, a0, nA);
    cta_kick_drift<T>(sm, a0, nA, dt / 6.0, 0.0, false, dt / 2.0);
    cta_newton<T>(sm, pN, a0, nA, a0, nA);
    cta_gradient<T>(sm, pG, a0, nA, a0, nA);
    cta_kick_drift<T>(sm, a0, nA, 2.0 * dt / 3.0, dt * dt / 48.0, true, dt / 2.0);
    cta_newton<T>(sm, pN, a0, nA, a0, nA);
    cta_kick<T>(sm, a0, nA, dt / 6.0, 0.0, false);
    if (T::tid() == 0) {
        const long long np = (long long)nA * nA;
        sm.st_pn += 3 * np;
        sm.st_pg += np;
    }
}

// The hhs_fsi recursion of Alg. 3 as a state machine over the explicit frame stack; runs until the
// frame at base_sp has been popped.
template <class T>
__device__ void hhs_loop(SmallSmem &sm, const SmallParams &P, const SweepParams &pN, const SweepParams &pG,
                         int base_sp) {
    while (true) {
        T::sync();
        const int sp = sm.sp;
        if (sp < base_sp || sm.err) break;
        const int start = sm.f_start[sp], cnt = sm.f_n[sp], stage = sm.f_stage[sp];
        const double tau = sm.f_tau[sp];
        const int level = P.level0 + sp;
        if (T::kThreads > 128 && stage == 0 && cnt > kWarpTeamMax && cnt <= kQuadTeamMax) {
            // the whole subtree of this entry on warps 0-3 (see TeamQuad)
            if (threadIdx.x < 128) hhs_loop<TeamQuad>(sm, P, pN, pG, sp);
            continue;
        }
        if (T::kThreads > 32 && stage == 0 && cnt > 0 && cnt <= kWarpTeamMax) {
            // the whole subtree of this entry on warp 0 (latency-bound: see TeamWarp)
            if (threadIdx.x < 32) hhs_loop<TeamWarp>(sm, P, pN, pG, sp);
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
            cta_timesteps<T>(sm, pG, start, cnt);
            const int nS = cta_partition<T>(sm, start, cnt, tau);
            const int nF = cnt - nS;
            if (nS > 0 && nF > 0) {
                cta_newton<T>(sm, pN, start, nS, start + nS, nF);
                cta_newton<T>(sm, pN, start + nS, nF, start, nS);
                cta_kick<T>(sm, start, cnt, tau / 6.0, 0.0, false);
            }
            cta_fsi<T>(sm, pN, pG, start, nS, 0.5 * tau);
            T::sync();
            if (T::tid() == 0) {
                sm.f_ns[sp] = nS;
                sm.st_entries[level] += 1; sm.st_slow[level] += nS; sm.st_fast[level] += nF;
                sm.st_pt += (long long)cnt * cnt;
                if (level > sm.st_depth) sm.st_depth = level;
                sm.f_stage[sp] = 1;
                if (nF > 0) {
                    sm.f_start[sp + 1] = start + nS; sm.f_n[sp + 1] = nF; sm.f_ns[sp + 1] = 0;
                    sm.f_stage[sp + 1] = 0; sm.f_tau[sp + 1] = 0.5 * tau;
                    sm.sp = sp + 1;
                }
            }
        } else if (stage == 1) {
            const int nS = sm.f_ns[sp], nF = cnt - nS;
            if (nS > 0 && nF > 0) {
                cta_newton<T>(sm, pN, start, nS, start + nS, nF);
                cta_newton<T>(sm, pN, start + nS, nF, start, nS);
                cta_gradient<T>(sm, pG, start, nS, start + nS, nF);
                cta_gradient<T>(sm, pG, start + nS, nF, start, nS);
                cta_kick<T>(sm, start, cnt, 2.0 * tau / 3.0, tau * tau / 48.0, true);
            }
            T::sync();
            if (T::tid() == 0) {
                sm.f_stage[sp] = 2;
                if (nF > 0) {
                    sm.f_start[sp + 1] = start + nS; sm.f_n[sp + 1] = nF; sm.f_ns[sp + 1] = 0;
                    sm.f_stage[sp + 1] = 0; sm.f_tau[sp + 1] = 0.5 * tau;
                    sm.sp = sp + 1;
                }
            }
        } else {
            const int nS = sm.f_ns[sp], nF = cnt - nS;
            cta_fsi<T>(sm, pN, pG, start, nS, 0.5 * tau);
            if (nS > 0 && nF > 0) {
                cta_newton<T>(sm, pN, start, nS, start + nS, nF);
                cta_newton<T>(sm, pN, start + nS, nF, start, nS);
                cta_kick<T>(sm, start, cnt, tau / 6.0, 0.0, false);
            }
            T::sync();
            if (T::tid() == 0) {
                const long long cr = 2LL * nS * nF;
                sm.st_pn += 3 * cr; sm.st_pg += cr;
                sm.sp = sp - 1;
            }
        }
    }
}

template <class T>
__global__ void __launch_bounds__(kSmallThreads, 1) hhs_small_kernel(const SmallParams P) {
    extern __shared__ __align__(16) unsigned char small_raw[];
    SmallSmem &sm = *reinterpret_cast<SmallSmem *>(small_raw);
    const int n = P.n, ld = P.ld;
    for (int k = threadIdx.x; k < n; k += kSmallThreads) {
        const int i = P.idx ? P.idx[k] : k;
        sm.xm[k] = make_double4(P.pos[i], P.pos[(size_t)ld + i], P.pos[2 * (size_t)ld + i], P.mass[i]);
        sm.vv[k] = make_double4(P.vel[i], P.vel[(size_t)ld + i], P.vel[2 * (size_t)ld + i], 1.0);
        sm.perm[k] = k;
    }
    for (int k = threadIdx.x; k < FROST_MAX_LEVELS; k += kSmallThreads) {
        sm.st_entries[k] = 0; sm.st_slow[k] = 0; sm.st_fast[k] = 0;
    }
    if (threadIdx.x == 0) {
        sm.sp = 0; sm.err = 0; sm.st_pn = sm.st_pg = sm.st_pt = 0; sm.st_depth = -1;
        sm.f_start[0] = 0; sm.f_n[0] = n; sm.f_ns[0] = 0; sm.f_stage[0] = 0; sm.f_tau[0] = P.tau_pivot;
    }
    SweepParams pN{}, pG{};
    pN.G = pG.G = P.G; pN.eta_ff = pG.eta_ff = P.eta_ff; pN.eta_fb = pG.eta_fb = P.eta_fb;
    pG.eps2 = P.eps2;
    pN.eps2 = P.eps2 > 0x1p-400 ? P.eps2 : 0x1p-400;     // see NewtonPolicy::pair
    __syncthreads();

    if (P.mode == 1) {
        for (int k = 0; k < P.n_steps; ++k) {
            if (n <= kWarpTeamMax) { if (threadIdx.x < 32) cta_fsi<TeamWarp>(sm, pN, pG, 0, n, P.dt_fsi); }
            else cta_fsi<T>(sm, pN, pG, 0, n, P.dt_fsi);
        }
    } else {
        hhs_loop<T>(sm, P, pN, pG, 0);
    }
    __syncthreads();
    if (T::kCluster) {      // replicas are identical: rank 0 writes back; nobody leaves while a peer
        namespace cg = cooperative_groups;                       // could still store into its replica
        cg::cluster_group cl = cg::this_cluster();
        cl.sync();
        if (cl.block_rank() != 0) return;
    }
    for (int k = threadIdx.x; k < n; k += kSmallThreads) {
        const int i = P.idx ? P.idx[k] : k;
        const double4 x = sm.xm[k], v = sm.vv[k];
        P.pos[i] = x.x; P.pos[(size_t)ld + i] = x.y; P.pos[2 * (size_t)ld + i] = x.z;
        P.vel[i] = v.x; P.vel[(size_t)ld + i] = v.y; P.vel[2 * (size_t)ld + i] = v.z;
    }
    if (P.stats) {      // atomics: an fsi(S) launch on a side stream may run concurrently (frost_api.cu)
        typedef unsigned long long ull;
        for (int k = threadIdx.x; k < FROST_MAX_LEVELS; k += kSmallThreads) {
            if (sm.st_entries[k]) {
                atomicAdd((ull *)&P.stats->entries[k], (ull)sm.st_entries[k]);
                atomicAdd((ull *)&P.stats->n_slow[k], (ull)sm.st_slow[k]);
                atomicAdd((ull *)&P.stats->n_fast[k], (ull)sm.st_fast[k]);
            }
        }
        if (threadIdx.x == 0) {
            atomicAdd((ull *)&P.stats->pairs_newton, (ull)sm.st_pn);
            atomicAdd((ull *)&P.stats->pairs_gradient, (ull)sm.st_pg);
            atomicAdd((ull *)&P.stats->pairs_timestep, (ull)sm.st_pt);
            atomicMax(&P.stats->depth, sm.st_depth);
            if (sm.err) atomicCAS(&P.stats->status, 0, sm.err);
        }
    }
}

int small_max() { return kSmallMax; }

// mode 0: hhs_fsi(set, tau) subtree rooted at hierarchy level `level0`; mode 1: fsi(set, dt).
int launch_small(frost_ctx *c, int mode, int ld, double *pos, double *vel, const double *mass,
                 const int32_t *idx, int n, double tau_or_dt, int level0, void *dev_stats, int n_steps) {
    if (n <= 0) return FROST_OK;
    if (n > kSmallMax) return FROST_EINVAL;
    FROST_TRY(set_func_attr(c, hhs_small_kernel<TeamCTA>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                            (int)sizeof(SmallSmem)));
    FROST_TRY(set_func_attr(c, hhs_small_kernel<TeamCluster>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                            (int)sizeof(SmallSmem)));
    FROST_TRY(set_func_attr(c, hhs_small_kernel<TeamCluster>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
    SmallParams P{};
    P.idx = idx; P.n = n; P.ld = ld; P.pos = pos; P.vel = vel; P.mass = mass;
    P.tau_pivot = tau_or_dt; P.dt_fsi = tau_or_dt; P.mode = mode; P.level0 = level0; P.n_steps = n_steps;
    P.max_depth = c->max_depth; P.G = c->G; P.eps2 = c->eps2; P.eta_ff = c->eta_ff; P.eta_fb = c->eta_fb;
    P.stats = (SmallStats *)dev_stats;
    if (n >= kClusterMinSet && c->tune_cluster != 1) {   // one cluster of kClusterSize replicas
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3(kClusterSize); cfg.blockDim = dim3(kSmallThreads);
        cfg.dynamicSmemBytes = sizeof(SmallSmem); cfg.stream = c->stream;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = kClusterSize; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        FROST_CUDA(c, cudaLaunchKernelEx(&cfg, hhs_small_kernel<TeamCluster>, P));
    } else {
        hhs_small_kernel<TeamCTA><<<1, kSmallThreads, sizeof(SmallSmem), c->stream>>>(P);
    }
    return check_launch(c);
}

size_t small_stats_bytes() { return sizeof(SmallStats); }

}  // namespace frost
