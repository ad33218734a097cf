// frost_common.cuh -- context, scratch management and PTX helpers shared by the CUDA translation
// units of libfrost_b200.so.  (Product code: shares nothing with oracle/.)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <unordered_set>

#include "../../include/frost.h"

namespace frost {

// ---- geometry of the pair sweeps -------------------------------------------------------------
constexpr int kTile = 256;        // source records per shared-memory stage
constexpr int kStages = 3;        // ring depth of the TMA bulk-copy pipeline
constexpr int kRecBytes = 32;     // one packed record: 4 doubles

struct Buf {
    void *p = nullptr;
    size_t cap = 0;
};

}  // namespace frost

struct frost_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    double G = 1.0, eps2 = 0.0, eta_ff = 0.2, eta_fb = 0.2;
    int max_depth = 64;
    int tune_k = 0, tune_slices = 0, tune_small = -1;   // -1: auto threshold for the subtree kernel
    int accumulate = 0;            // FROST_ACCUMULATE of the current frost_forces call
    int shard_rank = 0, shard_world = 1;   // frost_set_shard: this context's share of a symmetric sweep
    int tune_cluster = 0;          // subtree kernel: 0 auto (cluster of CTAs for sets >= 192), 1 one CTA
    int tune_sym = 0;              // pair-symmetric sweeps: 0 auto, 1 never, 2 whenever applicable
    int num_sms = 148;
    int last_cuda = 0;
    int64_t launches = 0;
    // scratch (grow-only)
    frost::Buf recA_xm, recB_xm;   // packed {x,y,z,m} streams of set A (sinks) and set B (sources)
    frost::Buf recA_v, recB_v;     // packed {ax,ay,az,0} or {vx,vy,vz,0}
    frost::Buf partial;            // [slices][3][n_pad] partial sums / [slices][n_pad] partial minima
    frost::Buf tau_scratch;        // Morton keys, sorted index list, bounding records, tau64 (frost_tau.cu)
    frost::Buf partialB;           // B-side partial sums of the pair-symmetric sweeps (frost_sym.cu)
    frost::Buf symtot;             // running totals across bands of a symmetric sweep
    frost::Buf symflag;            // "a sum came out non-finite" flag of the unguarded gradient pass
    frost::Buf eqflag;             // "all masses of the packed lists are equal" flag (frost_update.cu)
    const int *eq_flag_cur = nullptr;   // valid for the duration of one frost_forces call, else NULL
    int tune_eqmass = 1;           // 1: equal-mass variants of the large symmetric sweeps where the flag allows
    int tune_guard = 0;            // 1: large symmetric gradient sweeps keep the per-pair coincidence guard
    size_t sym_scratch = (size_t)4 << 30;   // cap of partialB: the B list is swept in bands
    frost::Buf acc, grad, tau;     // internal planes for fsi / hhs
    frost::Buf blockcnt;           // partition scratch
    frost::Buf dev_stats;          // SmallStats accumulated by the subtree kernel
    frost::Buf host_stage[6];      // device staging for frost_forces_host
    frost::Buf lvlS[FROST_MAX_LEVELS], lvlF[FROST_MAX_LEVELS];
    int32_t *pinned_counts = nullptr;  // host pinned int32[4]
    frost::Buf shard_idx;              // 0..n-1, for sharding the sinks of a NULL index list
    int tune_pair = 1;             // two-body frames of the subtree kernels on one thread (frost_set_pair_path)
    int kepler = 0;                // frost_set_kepler: two-body components of a split entry on their Kepler orbit
    int split_max = 0;             // frost_set_split: entries with <= split_max members split F into components
    frost::Buf uf, comp;           // union-find forest / labels, sort and descriptor scratch of a split entry
    frost::Buf lvlC[FROST_MAX_LEVELS];   // F of a split entry reordered by component
    // fsi(S) || hhs_fsi(F): one side context (own stream, own sweep scratch) per hierarchy level
    int overlap = 1;
    frost_ctx *side[FROST_MAX_LEVELS] = {};
    cudaEvent_t ev_fork[FROST_MAX_LEVELS] = {}, ev_join[FROST_MAX_LEVELS] = {};
    // function attributes (dynamic shared memory opt-in, cluster size) are per device, and a context
    // is bound to one device: remembered per context, not per process
    std::unordered_set<uint64_t> attr_done;
};

namespace frost {

#define FROST_CUDA(ctx, call)                         \
    do {                                              \
        cudaError_t e_ = (call);                      \
        if (e_ != cudaSuccess) {                      \
            (ctx)->last_cuda = (int)e_;               \
            return FROST_ECUDA;                       \
        }                                             \
    } while (0)

#define FROST_TRY(expr)                \
    do {                               \
        int rc_ = (expr);              \
        if (rc_ != FROST_OK) return rc_; \
    } while (0)

inline int ensure(frost_ctx *c, Buf &b, size_t bytes) {
    if (bytes <= b.cap) return FROST_OK;
    if (b.p) {
        // the buffer may still be in use by enqueued work: drain the stream before freeing
        cudaStreamSynchronize(c->stream);
        cudaFree(b.p);
        b.p = nullptr;
        b.cap = 0;
    }
    size_t want = bytes + bytes / 4 + 256;
    cudaError_t e = cudaMalloc(&b.p, want);
    if (e != cudaSuccess) {
        c->last_cuda = (int)e;
        b.p = nullptr;
        return FROST_ENOMEM;
    }
    b.cap = want;
    return FROST_OK;
}

// cudaFuncSetAttribute once per (context, kernel, attribute).
template <class F>
inline int set_func_attr(frost_ctx *c, F *func, cudaFuncAttribute attr, int value) {
    const uint64_t key = (uint64_t)(uintptr_t)func * 8u + (uint64_t)attr;
    if (c->attr_done.count(key)) return FROST_OK;
    FROST_CUDA(c, cudaFuncSetAttribute(func, attr, value));
    c->attr_done.insert(key);
    return FROST_OK;
}

// Entry points make the context's device current for the duration of the call and restore the
// caller's device on return.
struct DeviceGuard {
    int prev = -1;
    bool ok;
    explicit DeviceGuard(const frost_ctx *c) {
        cudaGetDevice(&prev);
        ok = (prev == c->device) || cudaSetDevice(c->device) == cudaSuccess;
        if (prev == c->device) prev = -1;
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};
#define FROST_DEVICE(ctx)                                   \
    frost::DeviceGuard guard_(ctx);                         \
    if (!guard_.ok) { (ctx)->last_cuda = (int)cudaGetLastError(); return FROST_ECUDA; }

inline int check_launch(frost_ctx *c) {
    c->launches++;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        c->last_cuda = (int)e;
        return FROST_ECUDA;
    }
    return FROST_OK;
}

inline int round_up(int v, int m) { return (v + m - 1) / m * m; }

// ---- launchers implemented in the other translation units ------------------------------------
// frost_update.cu
// wscale multiplies the mass written to .w; nan_pad = 1 pads with NaN positions instead of zeros,
// 2 with positions (1e150, 1e150, 1e150) -- mass 0 either way
// eq_flag != NULL: *eq_flag is cleared if any packed mass differs (bitwise) from the mass of the first
// particle of the list eq_ref (NULL = particle 0)
int launch_pack_xm(frost_ctx *c, int ld, const double *pos, const double *mass, const int32_t *idx,
                   int n_idx, int n_pad, double *out, double wscale = 1.0, int nan_pad = 0,
                   double *zero_tail = nullptr, int *eq_flag = nullptr, const int32_t *eq_ref = nullptr);
// w_index != 0: .w of record k carries the list position k in its low word (time-step sweeps that
// enter their fast pairs into a union-find forest); otherwise 1.0
int launch_pack_vec(frost_ctx *c, int ld, const double *planes, const int32_t *idx, int n_idx,
                    int n_pad, double *out, int w_index = 0);
// .w of record k <- component label lab[k] in its low word (records beyond n_idx: -2)
int launch_pack_label(frost_ctx *c, const int *lab, int n_idx, int n_pad, double *vec);
int launch_kick(frost_ctx *c, int ld, double *vel, const double *acc, const double *grad,
                const int32_t *idx, int n_idx, double cc, double kappa);
int launch_kick_drift(frost_ctx *c, int ld, double *pos, double *vel, const double *acc, const double *grad,
                      const int32_t *idx, int n_idx, double ck, double kappa, double cd);
int launch_drift(frost_ctx *c, int ld, double *pos, const double *vel, const int32_t *idx,
                 int n_idx, double cc);
int launch_partition(frost_ctx *c, const double *tau, const int32_t *idx, int n_idx,
                     double tau_pivot, int32_t *out_slow, int32_t *out_fast, int32_t *counts_host);
// frost_sweeps.cu
// One direction: sinks = stream A (n_snk real records, padded), sources = stream B.
int sweep_newton(frost_ctx *c, const double *snk_xm, int n_snk, const double *src_xm, int n_src,
                 const int32_t *snk_idx, int ld, double *out_acc, double *snk_a_packed);
int sweep_gradient(frost_ctx *c, const double *snk_xm, const double *snk_a, int n_snk,
                   const double *src_xm, const double *src_a, int n_src, const int32_t *snk_idx,
                   int ld, double *out_grad);
// forest != NULL: pairs with a candidate below tau_pivot are united in the forest over list positions
int sweep_timestep(frost_ctx *c, const double *xm, const double *v, int n_set,
                   const int32_t *idx, double tau_pivot, double *out_tau, int32_t *out_bin,
                   int *forest = nullptr);
// Self sweep of one list over the pairs whose component labels differ (low word of a_lab[k].w; the
// kicked pair set of a split hierarchy entry): accelerations, then (grad != NULL) gradient accelerations.
// out_acc != NULL: the Newton sweep (its sums are also written to the packed stream a_lab, labels kept);
// out_grad != NULL: the gradient sweep from the accelerations in a_lab.  accumulate: add to the planes.
int sweep_masked(frost_ctx *c, const double *xm, double *a_lab, int n_set, const int32_t *idx, int ld,
                 double *out_acc, double *out_grad, int accumulate = 0);

// frost_sym.cu: pair-symmetric sweeps (one evaluation serves i<-j and j<-i).  self: B == A.
int sym_newton(frost_ctx *c, const double *A_xm, int nA, const double *B_xm, int nB, bool self,
               const int32_t *A_idx, const int32_t *B_idx, int ld, double *out_acc,
               double *A_a_packed, double *B_a_packed);
int sym_gradient(frost_ctx *c, const double *A_xm, const double *A_a, int nA, const double *B_xm,
                 const double *B_a, int nB, bool self, const int32_t *A_idx, const int32_t *B_idx,
                 int ld, double *out_grad);
int sym_timestep(frost_ctx *c, const double *xm, const double *v, int n_set, const int32_t *idx,
                 double tau_pivot, double *out_tau, int32_t *out_bin, int *forest = nullptr);

int sym_potential(frost_ctx *c, const double *xm, int n, double *out_phi);
const char *sym_geometry();   // tile geometry of the large force sweeps (frost_version)
int sym_masked(frost_ctx *c, const double *xm, const double *a_lab, int n, const int32_t *idx, int ld,
               double *out_acc, double *out_grad, int accumulate);
// frost_update.cu: T, U, P, L (one CTA, compensated sums, fixed order) -> out8 (device)
int launch_diag(frost_ctx *c, int n, int ld, const double *pos, const double *vel, const double *mass,
                const double *phi, double *out8);
// out[k] = k0 + k ; zero the planes of the particles idx[k] (or k), k in [0, lo) and [hi, n_idx)
int launch_iota(frost_ctx *c, int32_t *out, int n, int k0);
int launch_zero_outside(frost_ctx *c, int ld, double *planes, const int32_t *idx, int n_idx, int lo, int hi);

// frost_tau.cu: time-step sweep in Morton order with exact block pruning (prune = 0: evaluate all)
int tau_pruned(frost_ctx *c, int ld, const double *pos, const double *vel, const double *mass,
               const int32_t *idx, int n, double tau_pivot, double *out_tau, int32_t *out_bin, int prune,
               int *forest = nullptr);

// frost_split.cu: the components of the fast pairs of a split hierarchy entry (reading 24)
struct SplitInfo {
    bool split = false;              // the entry is split-enabled (its components follow reading 24/25)
    int m = 0;                       // components of F
    int n_small = 0, n_med = 0, n_big = 0;   // of <= comp_warp_max(), <= small_max(), more particles
    long long sumsq = 0;             // sum of squared component sizes
    const int32_t *C = nullptr;      // F reordered: components contiguous, by smallest member (device)
    const int *labpos = nullptr;     // label of every list position of the entry's set, -1 = slow (device)
    const void *desc_small = nullptr, *desc_med = nullptr;   // int2 {offset into C, size} (device)
    const int *n_small_dev = nullptr, *n_med_dev = nullptr;
    int big_off[64], big_size[64];   // the big components (host)
    // kick decomposition: G = the largest big component (C[g_off .. g_off + g_size)), R = the rest of F
    int g_off = 0, g_size = 0, nR = 0;
    const int32_t *R = nullptr;      // R as one list (device; = C when there is no G)
    const int *labR = nullptr;       // component label of every position of R (device)
};
int split_components(frost_ctx *c, int level, int ld, const double *tau, const int32_t *set, int n_set,
                     double pivot, const int *forest, const int32_t *F, int nF, SplitInfo *out);

// frost_small.cu: one-CTA device-resident hhs_fsi subtree (mode 0) or fsi step (mode 1)
int small_max();
size_t small_stats_bytes();
int launch_small(frost_ctx *c, int mode, int ld, double *pos, double *vel, const double *mass,
                 const int32_t *idx, int n, double tau_or_dt, int level0, void *dev_stats, int n_steps = 1,
                 int root_is_comp = 0);
int comp_warp_max();
int launch_comp_batch(frost_ctx *c, int warp_team, int ld, double *pos, double *vel, const double *mass,
                      const int32_t *idx, const void *desc, const int *n_desc, int max_desc, double tau,
                      int level0, void *dev_stats);

// ---- device-side PTX helpers ------------------------------------------------------------------
#ifdef __CUDACC__
__device__ __forceinline__ uint32_t smem_u32(const void *p) {
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_fence_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)),
                 "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
// 1-D TMA bulk copy global -> shared, completion signalled on an mbarrier (SASS: UBLKCP).
__device__ __forceinline__ void bulk_g2s(void *dst_smem, const void *src_gmem, uint32_t bytes,
                                         uint64_t *bar) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::
            "r"(smem_u32(dst_smem)),
        "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
        : "memory");
}

// Lock-free union-find (global or shared memory): the root of a tree is its smallest member, so the
// final forest does not depend on the order in which the pairs arrive.
__device__ __forceinline__ int uf_find(const volatile int *par, int x) {
    while (true) {
        const int p = par[x];
        if (p == x) return x;
        x = p;
    }
}
__device__ __forceinline__ void uf_union(int *par, int a, int b) {
    while (true) {
        a = uf_find(par, a); b = uf_find(par, b);
        if (a == b) return;
        if (a < b) { const int t = a; a = b; b = t; }       // hang the larger root under the smaller
        if (atomicCAS(&par[a], a, b) == a) return;
    }
}

// fp64 reciprocal square root seed: MUFU.RSQ64H on the high word (rel. error ~2^-22), low word 0.
// Returns exactly 0 when x is zero or subnormal (exponent field 0), which is how a coincident /
// self pair is made to contribute nothing without an FP64-pipe compare.
__device__ __forceinline__ double rsqrt_seed_or_zero(double x) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const int hx = __double2hiint(x);
    const int hy = __double2hiint(y);
    return __hiloint2double(hx < 0x00100000 ? 0 : hy, 0);
}
// Unguarded seed (caller guarantees x is a positive normal number).
__device__ __forceinline__ double rsqrt_seed(double x) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    return y;
}
// The same seed with its LOW word taken from `junk` -- any value the caller no longer needs -- instead of
// zero: ptxas then lets MUFU.RSQ64H write into the high half of junk's register pair and the MOV that
// zeroes the low word (one issue slot per pair) disappears.  The seed's relative
// error grows from 2^-22 to below 2^-19.7 (32 arbitrary low mantissa bits); one cubic step still
// lands below 2^-57, the three-term series of the Newton weight below 2^-55.  Deterministic.
__device__ __forceinline__ double rsqrt_seed_lo(double x, double junk) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    return __hiloint2double(__double2hiint(y), __double2loint(junk));
}
__device__ __forceinline__ double rsqrt_full_lo(double x, double junk) {
    const double y = rsqrt_seed_lo(x, junk);
    const double t = x * y;
    const double e = fma(-t, y, 1.0);
    const double p = fma(0.375, e, 0.5);
    const double ep = e * p;
    return fma(y, ep, y);
}
// x += w*dx; y += w*dy; z += w*dz as three adjacent DFMAs with w in the same operand slot.
__device__ __forceinline__ void fma3_shared(double &x, double &y, double &z, double w, double dx,
                                            double dy, double dz) {
    asm("fma.rn.f64 %0, %3, %4, %0;\n\t"
        "fma.rn.f64 %1, %3, %5, %1;\n\t"
        "fma.rn.f64 %2, %3, %6, %2;"
        : "+d"(x), "+d"(y), "+d"(z)
        : "d"(w), "d"(dx), "d"(dy), "d"(dz));
}
// Full-precision 1/sqrt(x) from the seed by one cubic (Householder order 3) step: 5 FP64 slots.
//   e = 1 - x y^2 ;  y' = y + y (e (1/2 + 3/8 e))        (error ~ (5/16) e^3 ~ 2^-66 + rounding)
// The last FMA reads only two distinct register pairs (y twice), so it issues in 2 cycles.
__device__ __forceinline__ double rsqrt_full_or_zero(double x) {
    const double y = rsqrt_seed_or_zero(x);
    const double t = x * y;
    const double e = fma(-t, y, 1.0);
    const double p = fma(0.375, e, 0.5);
    const double ep = e * p;
    return fma(y, ep, y);
}
// Unguarded full-precision 1/sqrt(x): x = 0 gives NaN (MUFU(0) = +inf, 0*inf), NaN propagates.
__device__ __forceinline__ double rsqrt_full(double x) {
    const double y = rsqrt_seed(x);
    const double t = x * y;
    const double e = fma(-t, y, 1.0);
    const double p = fma(0.375, e, 0.5);
    const double ep = e * p;
    return fma(y, ep, y);
}
// Full-precision 1/x for x in the normal range: MUFU.RCP64H seed + one cubic step
//   e = 1 - x y ;  y' = y + y (e + e^2)                   (error ~ e^3 ~ 2^-66 + rounding)
__device__ __forceinline__ double rcp_full(double x) {
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double e = fma(-x, y, 1.0);
    const double ee = fma(e, e, e);
    return fma(y, ee, y);
}
#endif

}  // namespace frost
