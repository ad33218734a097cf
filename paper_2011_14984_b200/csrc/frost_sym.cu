// frost_sym.cu -- pair-symmetric variants of the three all-pairs sweeps: Newtonian
// accelerations (Eq. 24/42), gradient accelerations (Eq. 27/43/44), time-step criterion
// (Eq. 49-54).  Every quantity a pair (i, j) needs -- x_ji, s^-3, the tidal contraction, the
// symmetrised time-step candidate -- is either symmetric or antisymmetric under i <-> j
// ("the force-gradient term ... obeys Newton's third law"), so one evaluation
// can serve both ordered pairs (i <- j) and (j <- i): 20 instead of 2 x 16 FP64 instructions for
// the Newton pair, 32 instead of 2 x 28 for the gradient pair, one candidate instead of two for
// the time step.  The one-sided sweeps of frost_sweeps.cu cannot exploit this because their
// sources are broadcast to all lanes; here both particles of a pair live in registers:
//
//   * a CTA owns an A tile of NT*KA particles (KA per thread, resident for the CTA's life) and
//     streams B tiles of NT particles through a TMA bulk-copy ring (as frost_sweeps.cu);
//   * each warp takes one 32-particle chunk of the B tile at a time; lane l starts with B particle
//     l as its "traveller" and the travellers rotate one lane per step (accumulators by SHFL,
//     coordinates re-read from shared memory at the rotated index), so after 32 steps every A
//     particle of the warp has met every B particle of the chunk and the traveller accumulators
//     are back in their home lane;
//   * the NT/32 warps visit the chunks round-robin (warp w takes chunk (w + r) mod W in round r,
//     one __syncthreads per round), so the B-side sums of a tile are combined in shared memory in
//     a fixed order, without atomics, and leave the CTA once per (A tile, B tile);
//   * A-side sums leave once per CTA (segment of the B list), B-side sums once per tile pair; a
//     second kernel adds both kinds in a fixed order -- results are bitwise reproducible.
//
// For the self case (A list == B list) only B tiles at or beyond the A tile are visited: the
// diagonal block is evaluated one-sided (its B-side sums are dropped), everything beyond it
// two-sided.  For the bipartite case (slow/fast sets of Alg. 3) every tile pair
// is two-sided and one sweep yields both directions of acc_sf_*.
#include <cstdio>
#include <type_traits>

// Rotation steps per iteration of the main loop of sym_kernel, and whether the Newton seed takes its low
// word from a dying value (rsqrt_seed_lo).  ptxas' schedule of this loop moves the sweep time by +-1.5 %
// with such details; chosen by measurement at N = 2^20 (ms per sweep, B200):
//   Newton, equal masses:   unroll 1 / 2 / 4 = 668.5 / 670.6 / 655.6; 4 with the seed trick 665.2; 8 with it 662.4
//   Newton, general:        unroll 2 = 694.8; 4 = 692.5; 4 with the seed trick 688.2; 1 = 697.4
//                           (the seed trick is not used: both variants keep the same seed => same bits)
//   gradient, equal masses: unroll 1 / 2 / 4 = 1080.2 / 1094.8 / 1087.5
//   gradient, general:      unroll 1 / 2 / 4 = 1117.7 / 1110.3 / 1102.4

#include "frost_pairs.cuh"

namespace frost {

struct SymParams {
    const double4 *a0, *a1;   // A records {x,y,z,m} and {ax,ay,az,.} / {vx,vy,vz,.}
    const double4 *b0, *b1;   // B records
    double *partA;            // [segments][planes][na_pad]
    double *partB;            // [A tile][planes][band_len]: B-side sums of the current band
    int na_pad;
    int self;                 // A list == B list: visit only B tiles >= the A tile
    int bt0, bt1;             // the band: B tiles [bt0, bt1) of NT records (scratch is per band)
    int seg_tiles;            // B tiles per CTA
    int row0, row_stride;     // A tiles owned by this launch: row0, row0 + row_stride, ... (sharding)
    double eps2, eta_ff, eta_fb;
    double pivot;             // SymTimestepEdge: fast pairs (candidate < pivot) are united in `forest`
    int *forest;
    const int *gate;          // non-NULL: the launch does nothing unless (*gate != 0) == (gate_want != 0)
    int gate_want;            // (repair pass of the gradient sweep; equal-mass / general variants)
};

// ------------------------------------------------------------------------------------------------
// Pair policies: A particle in registers, B particle = shared-memory record + travelling sums.
// ------------------------------------------------------------------------------------------------
// EQ: every particle of both lists has the same mass (checked on the device while the streams are
// packed, frost_update.cu): then m_i s^-3 = m_j s^-3 and the second mass weight is the first one negated
// -- one DMUL less per pair, bitwise the same sums.  The two variants of a sweep are launched behind
// complementary gates on that flag.
template <bool EQ>
struct SymNewtonT {
    static constexpr int kRecs = 1, kPlanes = 3, kUnroll = 4;
    static constexpr bool kMin = false;
    struct A { double x, y, z, nm, s[3]; };
    __device__ static __forceinline__ void load(A &a, const SymParams &p, int i) {
        const double4 r = p.a0[i];
        a.x = r.x; a.y = r.y; a.z = r.z; a.nm = -r.w;
        a.s[0] = a.s[1] = a.s[2] = 0.0;
    }
    __device__ static __forceinline__ void init_b(double (&b)[3]) { b[0] = b[1] = b[2] = 0.0; }
    // 20 FP64 instructions for both ordered pairs: 12 shared (x_ji, s^2, s^-3 by the series of
    // NewtonPolicy::pair) + 2 x (mass weight + 3 accumulating FMAs).  a_i += m_j s^-3 x_ji,
    // a_j -= m_i s^-3 x_ji (Eq. 24 both ways).  eps2 is floored by the launcher.
    __device__ static __forceinline__ void pair(A &a, double (&b)[3], const double4 &j0,
                                                const double4 &, const SymParams &p) {
        const double dx = j0.x - a.x, dy = j0.y - a.y, dz = j0.z - a.z;
        const double s2 = fma(dz, dz, fma(dy, dy, fma(dx, dx, p.eps2)));
        const double y = rsqrt_seed(s2);      // (rsqrt_seed_lo: table at the top of the file; the two variants
                                              //  must use the same seed to stay bitwise equal)
        const double y2 = y * y;
        const double e = fma(-s2, y2, 1.0);
        const double w0 = y2 * y;
        const double q = fma(1.875, e, 1.5);
        const double qe = q * e;
        const double w = fma(w0, qe, w0);
        const double wa = w * j0.w;
        fma3_shared(a.s[0], a.s[1], a.s[2], wa, dx, dy, dz);
        if (EQ) {
            b[0] = fma(-wa, dx, b[0]); b[1] = fma(-wa, dy, b[1]); b[2] = fma(-wa, dz, b[2]);
        } else {
            const double wb = w * a.nm;
            fma3_shared(b[0], b[1], b[2], wb, dx, dy, dz);
        }
    }
};
using SymNewton = SymNewtonT<false>;

struct SymGradient {
    static constexpr int kRecs = 2, kPlanes = 3;
    static constexpr bool kMin = false;
    struct A { double x, y, z, nm, ax, ay, az, s[3]; };
    __device__ static __forceinline__ void load(A &a, const SymParams &p, int i) {
        const double4 r = p.a0[i];
        const double4 v = p.a1[i];
        a.x = r.x; a.y = r.y; a.z = r.z; a.nm = -r.w; a.ax = v.x; a.ay = v.y; a.az = v.z;
        a.s[0] = a.s[1] = a.s[2] = 0.0;
    }
    __device__ static __forceinline__ void init_b(double (&b)[3]) { b[0] = b[1] = b[2] = 0.0; }
    // 32 FP64 instructions for both ordered pairs: v = a_ji - 3 s^-2 (x_ji . a_ji) x_ji is odd
    // under i <-> j, s^-3 is even: g_i += m_j s^-3 v, g_j -= m_i s^-3 v  (Eq. 27 both ways).
    __device__ static __forceinline__ void pair(A &a, double (&b)[3], const double4 &j0,
                                                const double4 &j1, const SymParams &p) {
        const double dx = j0.x - a.x, dy = j0.y - a.y, dz = j0.z - a.z;
        const double ax = j1.x - a.ax, ay = j1.y - a.ay, az = j1.z - a.az;
        const double s2 = fma(dz, dz, fma(dy, dy, fma(dx, dx, p.eps2)));
        const double ri = rsqrt_full_or_zero(s2);
        const double dot = fma(dz, az, fma(dy, ay, dx * ax));
        const double q = ri * ri;
        const double w3 = ri * q;
        const double t = q * dot;
        const double u = t * -3.0;
        double vx = ax, vy = ay, vz = az;
        fma3_shared(vx, vy, vz, u, dx, dy, dz);
        const double wa = w3 * j0.w;
        const double wb = w3 * a.nm;
        fma3_shared(a.s[0], a.s[1], a.s[2], wa, vx, vy, vz);
        fma3_shared(b[0], b[1], b[2], wb, vx, vy, vz);
    }
};

// The gradient pair without the coincident-pair guard (ISETP + SEL per pair, 2.6 % of the loop).  A pair
// with s^2 = 0 -- two distinct coincident unsoftened particles; the self pair only occurs in the
// diagonal blocks, which keep the guarded routine -- then yields NaN instead of being ignored: MUFU(0)
// = +inf, 0 * inf = NaN, and NaN sticks to every sum it enters.  The reduction that scatters the
// result flags any non-finite output, and a gated second pass with the guarded kernel (a few empty
// launches when the flag is clear) recomputes the sweep: the contract of DESIGN.md reading 11 holds
// for every input, and inputs without coincident particles never pay for the guard.  Padding records
// sit at (1e150, 1e150, 1e150) with mass 0 (frost_api.cu), so that they coincide with no particle.
template <bool EQ>
struct SymGradientFastT : SymGradient {
    static constexpr bool kDiagGuard = true;
    static constexpr int kUnroll = EQ ? 1 : 4;
    __device__ static __forceinline__ void pair(A &a, double (&b)[3], const double4 &j0,
                                                const double4 &j1, const SymParams &p) {
        const double dx = j0.x - a.x, dy = j0.y - a.y, dz = j0.z - a.z;
        const double ax = j1.x - a.ax, ay = j1.y - a.ay, az = j1.z - a.az;
        const double part = fma(dy, dy, fma(dx, dx, p.eps2));
        const double s2 = fma(dz, dz, part);
        const double ri = rsqrt_full_lo(s2, part);        // (low word of the seed: see rsqrt_seed_lo)
        const double dot = fma(dz, az, fma(dy, ay, dx * ax));
        const double q = ri * ri;
        const double w3 = ri * q;
        const double t = q * dot;
        const double u = t * -3.0;
        double vx = ax, vy = ay, vz = az;
        fma3_shared(vx, vy, vz, u, dx, dy, dz);
        const double wa = w3 * j0.w;
        fma3_shared(a.s[0], a.s[1], a.s[2], wa, vx, vy, vz);
        if (EQ) {                          // equal masses: see SymNewtonT
            b[0] = fma(-wa, vx, b[0]); b[1] = fma(-wa, vy, b[1]); b[2] = fma(-wa, vz, b[2]);
        } else {
            const double wb = w3 * a.nm;
            fma3_shared(b[0], b[1], b[2], wb, vx, vy, vz);
        }
    }
    __device__ static __forceinline__ void pair_diag(A &a, double (&b)[3], const double4 &j0,
                                                     const double4 &j1, const SymParams &p) {
        SymGradient::pair(a, b, j0, j1, p);
    }
};

using SymGradientFast = SymGradientFastT<false>;

// The kick sweeps of a split hierarchy entry over the debris list R: pairs whose component
// labels are equal contribute nothing.  The label of a record travels in the low word of .w of its
// second record (as in the one-sided MaskedNewtonPolicy / MaskedGradientPolicy); the weight of a
// same-label pair is replaced by zero (ISETP + 2 SEL per pair).  Self sweeps only, guarded gradient.
struct SymNewtonMasked {
    static constexpr int kRecs = 2, kPlanes = 3;
    static constexpr bool kMin = false;
    struct A : SymNewton::A { int lab; };
    __device__ static __forceinline__ void load(A &a, const SymParams &p, int i) {
        SymNewton::load(a, p, i);
        a.lab = __double2loint(p.a1[i].w);
    }
    __device__ static __forceinline__ void init_b(double (&b)[3]) { b[0] = b[1] = b[2] = 0.0; }
    __device__ static __forceinline__ void pair(A &a, double (&b)[3], const double4 &j0,
                                                const double4 &j1, const SymParams &p) {
        const double dx = j0.x - a.x, dy = j0.y - a.y, dz = j0.z - a.z;
        const double s2 = fma(dz, dz, fma(dy, dy, fma(dx, dx, p.eps2)));
        const double y = rsqrt_seed(s2);
        const double y2 = y * y;
        const double e = fma(-s2, y2, 1.0);
        const double w0 = y2 * y;
        const double q = fma(1.875, e, 1.5);
        const double qe = q * e;
        double w = fma(w0, qe, w0);
        if (__double2loint(j1.w) == a.lab) w = 0.0;
        const double wa = w * j0.w;
        const double wb = w * a.nm;
        fma3_shared(a.s[0], a.s[1], a.s[2], wa, dx, dy, dz);
        fma3_shared(b[0], b[1], b[2], wb, dx, dy, dz);
    }
};

struct SymGradientMasked {
    static constexpr int kRecs = 2, kPlanes = 3;
    static constexpr bool kMin = false;
    struct A : SymGradient::A { int lab; };
    __device__ static __forceinline__ void load(A &a, const SymParams &p, int i) {
        SymGradient::load(a, p, i);
        a.lab = __double2loint(p.a1[i].w);
    }
    __device__ static __forceinline__ void init_b(double (&b)[3]) { b[0] = b[1] = b[2] = 0.0; }
    __device__ static __forceinline__ void pair(A &a, double (&b)[3], const double4 &j0,
                                                const double4 &j1, const SymParams &p) {
        const double dx = j0.x - a.x, dy = j0.y - a.y, dz = j0.z - a.z;
        const double ax = j1.x - a.ax, ay = j1.y - a.ay, az = j1.z - a.az;
        const double s2 = fma(dz, dz, fma(dy, dy, fma(dx, dx, p.eps2)));
        const double ri = rsqrt_full_or_zero(s2);
        const double dot = fma(dz, az, fma(dy, ay, dx * ax));
        const double q = ri * ri;
        double w3 = ri * q;
        if (__double2loint(j1.w) == a.lab) w3 = 0.0;
        const double t = q * dot;
        const double u = t * -3.0;
        double vx = ax, vy = ay, vz = az;
        fma3_shared(vx, vy, vz, u, dx, dy, dz);
        const double wa = w3 * j0.w;
        const double wb = w3 * a.nm;
        fma3_shared(a.s[0], a.s[1], a.s[2], wa, vx, vy, vz);
        fma3_shared(b[0], b[1], b[2], wb, vx, vy, vz);
    }
};

template <class P, class = void> struct UnrollOf { static constexpr int value = 2; };
template <class P> struct UnrollOf<P, std::enable_if_t<(P::kUnroll > 0)>> { static constexpr int value = P::kUnroll; };
template <class P, class = void> struct DiagGuard { static constexpr bool value = false; };
template <class P> struct DiagGuard<P, std::enable_if_t<P::kDiagGuard>> { static constexpr bool value = true; };

struct SymTimestep {
    static constexpr int kRecs = 2, kPlanes = 1;
    static constexpr bool kMin = true;
    struct A { double x, y, z, gm, vx, vy, vz, s[1]; };
    __device__ static __forceinline__ void load(A &a, const SymParams &p, int i) {
        const double4 r = p.a0[i];
        const double4 v = p.a1[i];
        a.x = r.x; a.y = r.y; a.z = r.z; a.gm = r.w; a.vx = v.x; a.vy = v.y; a.vz = v.z;
        a.s[0] = __longlong_as_double(0x7ff0000000000000LL);
    }
    __device__ static __forceinline__ void init_b(double (&b)[1]) {
        b[0] = __longlong_as_double(0x7ff0000000000000LL);
    }
    // The symmetrised candidate of Eq. 49-54 is the same number for (i <- j) and (j <- i)
    // (r.v, r^2, v^2 and m_i + m_j are even under the swap), so it is evaluated once
    // -- exactly TimestepPolicy::pair -- and min-ed into both particles.
    __device__ static __forceinline__ double candidate(const A &a, const double4 &j0, const double4 &j1,
                                                       const SymParams &p) {
        const double rx = j0.x - a.x, ry = j0.y - a.y, rz = j0.z - a.z;
        const double vx = j1.x - a.vx, vy = j1.y - a.vy, vz = j1.z - a.vz;
        const double r2 = fma(rz, rz, fma(ry, ry, rx * rx));
        const double v2 = fma(vz, vz, fma(vy, vy, vx * vx));
        const double rv = fma(rz, vz, fma(ry, vy, rx * vx));
        const double mu = a.gm + j0.w;
        const double ir = rsqrt_full(r2);
        const double iv = rsqrt_full(v2);
        const double ir2 = ir * ir;
        const double mir = mu * ir;
        const double t_ff = rsqrt_full(mir * ir2);
        const double t_fb = (r2 * ir) * iv;
        const double rvr2 = rv * ir2;
        const double q_ff = (rvr2 * t_ff) * (1.5 * p.eta_ff);
        const double f = rvr2 * t_fb;
        const double q_fb = fma(f, mir * (iv * iv), f) * p.eta_fb;
        const double c_ff = sym_factor(q_ff) * (t_ff * p.eta_ff);
        const double c_fb = sym_factor(q_fb) * (t_fb * p.eta_fb);
        return fmin(c_ff, c_fb);
    }
    __device__ static __forceinline__ void pair(A &a, double (&b)[1], const double4 &j0,
                                                const double4 &j1, const SymParams &p) {
        const double c = candidate(a, j0, j1, p);
        a.s[0] = fmin(a.s[0], c);
        b[0] = fmin(b[0], c);
    }
};

// SymTimestep for a split hierarchy entry (reading 24): every fast pair is also united in the
// union-find forest over list positions (low word of .w of the velocity records).
struct SymTimestepEdge {
    static constexpr int kRecs = 2, kPlanes = 1;
    static constexpr bool kMin = true;
    struct A : SymTimestep::A { int id; };
    __device__ static __forceinline__ void load(A &a, const SymParams &p, int i) {
        SymTimestep::load(a, p, i);
        a.id = __double2loint(p.a1[i].w);
    }
    __device__ static __forceinline__ void init_b(double (&b)[1]) { SymTimestep::init_b(b); }
    __device__ static __forceinline__ void pair(A &a, double (&b)[1], const double4 &j0,
                                                const double4 &j1, const SymParams &p) {
        const double c = SymTimestep::candidate(a, j0, j1, p);
        a.s[0] = fmin(a.s[0], c);
        b[0] = fmin(b[0], c);
        if (c < p.pivot) uf_union(p.forest, a.id, __double2loint(j1.w));
    }
};

// Specific potential phi_i = -G sum_j m_j / s_ij (Eq. 23) for the on-device
// energy diagnostic: 1/s is even under i <-> j.  12 FP64 instructions for both ordered pairs.
struct SymPotential {
    static constexpr int kRecs = 1, kPlanes = 1;
    static constexpr bool kMin = false;
    struct A { double x, y, z, m, s[1]; };
    __device__ static __forceinline__ void load(A &a, const SymParams &p, int i) {
        const double4 r = p.a0[i];
        a.x = r.x; a.y = r.y; a.z = r.z; a.m = r.w; a.s[0] = 0.0;
    }
    __device__ static __forceinline__ void init_b(double (&b)[1]) { b[0] = 0.0; }
    __device__ static __forceinline__ void pair(A &a, double (&b)[1], const double4 &j0,
                                                const double4 &, const SymParams &p) {
        const double dx = j0.x - a.x, dy = j0.y - a.y, dz = j0.z - a.z;
        const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
        // the self pair (and a pair at exactly the same point) is skipped, softened or not
        const double ri = (r2 == 0.0) ? 0.0 : rsqrt_full(r2 + p.eps2);
        a.s[0] = fma(j0.w, ri, a.s[0]);
        b[0] = fma(a.m, ri, b[0]);
    }
};

// ------------------------------------------------------------------------------------------------
// The kernel.  grid = (A tiles, segments of the B list); block = NT threads; KA A particles/thread.
// ------------------------------------------------------------------------------------------------
template <class P, int KA, int NT, int MINB>
__global__ void __launch_bounds__(NT, MINB) sym_kernel(const SymParams prm) {
    constexpr int kWarps = NT / 32;
    constexpr int TA = NT * KA;
    constexpr int PL = P::kPlanes;
    constexpr uint32_t kStageBytes = P::kRecs * 2 * NT * kRecBytes;      // chunks stored twice

    if (prm.gate && ((*prm.gate != 0) != (prm.gate_want != 0))) return;
    const int I = prm.row0 + blockIdx.x * prm.row_stride;
    const int diag_end = prm.self ? (I + 1) * KA : 0;          // tiles below this are the diagonal block
    const int row_first_tile = max(prm.self ? I * KA : 0, prm.bt0);   // first B tile of this A tile in the band
    const int tile0 = row_first_tile + blockIdx.y * prm.seg_tiles;
    if (tile0 >= prm.bt1) return;
    const int ntiles = min(prm.seg_tiles, prm.bt1 - tile0);

    extern __shared__ __align__(128) unsigned char smem_raw[];
    double4 *tiles = reinterpret_cast<double4 *>(smem_raw);                   // [kStages][kRecs][2 NT]
    double *accB = reinterpret_cast<double *>(smem_raw + kStages * kStageBytes);   // [2][PL][NT]
    uint64_t *full = reinterpret_cast<uint64_t *>(accB + 2 * PL * NT);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < kStages; ++s) mbar_init(&full[s], 1);
        mbar_fence_init();
    }
    __syncthreads();

    // Every 32-record chunk of a B tile is stored TWICE back to back, so that the rotated read of step
    // s -- record (lane - s) mod 32 -- is the plain address (chunk + 32 + lane) - s: an immediate offset
    // in the unrolled loop instead of three address instructions per step.
    auto issue = [&](int t) {
        const int s = t % kStages;
        mbar_expect_tx(&full[s], kStageBytes);
        double4 *dst = tiles + (size_t)s * P::kRecs * 2 * NT;
        const size_t off = (size_t)(tile0 + t) * NT;
#pragma unroll
        for (int c = 0; c < kWarps; ++c)
#pragma unroll
            for (int d = 0; d < 2; ++d) {
                bulk_g2s(dst + (c * 2 + d) * 32, prm.b0 + off + c * 32, 32 * kRecBytes, &full[s]);
                if (P::kRecs == 2)
                    bulk_g2s(dst + 2 * NT + (c * 2 + d) * 32, prm.b1 + off + c * 32, 32 * kRecBytes, &full[s]);
            }
    };
    if (tid == 0) {
        const int pre = min(kStages, ntiles);
        for (int t = 0; t < pre; ++t) issue(t);
    }

    typename P::A a[KA];
    const int a_first = I * TA + tid;
#pragma unroll
    for (int k = 0; k < KA; ++k) P::load(a[k], prm, a_first + k * NT);

    const int row_len = (prm.bt1 - prm.bt0) * NT;             // B particles of the band
    double *rowB = prm.partB + (size_t)blockIdx.x * PL * row_len;     // indexed by owned row
    const int row_j0 = prm.bt0 * NT;
    const int from = (lane + 31) & 31;          // travellers move to the next lane each step

    for (int t = 0; t < ntiles; ++t) {
        const int s = t % kStages;
        mbar_wait(&full[s], (uint32_t)(t / kStages) & 1u);
        const double4 *t0 = tiles + (size_t)s * P::kRecs * 2 * NT;
        const bool two_sided = (tile0 + t) >= diag_end;
        double *accT = accB + (size_t)(t & 1) * PL * NT;
        for (int r = 0; r < kWarps; ++r) {
            const int c = (warp + r) % kWarps;
            const double4 *c0 = t0 + c * 64 + 32 + lane;
            const double4 *c1 = c0 + (P::kRecs == 2 ? 2 * NT : 0);
            double b[PL];
            P::init_b(b);
            if (DiagGuard<P>::value && !two_sided) {      // diagonal block: the self pairs live here
#pragma unroll 2
                for (int step = 0; step < 32; ++step) {
                    const double4 j0 = c0[-step];
                    const double4 j1 = (P::kRecs == 2) ? c1[-step] : j0;
                    if constexpr (DiagGuard<P>::value) {
#pragma unroll
                        for (int k = 0; k < KA; ++k) P::pair_diag(a[k], b, j0, j1, prm);
                    }
#pragma unroll
                    for (int p = 0; p < PL; ++p) b[p] = __shfl_sync(0xffffffffu, b[p], from);
                }
            } else {
#pragma unroll (UnrollOf<P>::value)
                for (int step = 0; step < 32; ++step) {
                    const double4 j0 = c0[-step];
                    const double4 j1 = (P::kRecs == 2) ? c1[-step] : j0;
#pragma unroll
                    for (int k = 0; k < KA; ++k) P::pair(a[k], b, j0, j1, prm);
#pragma unroll
                    for (int p = 0; p < PL; ++p) b[p] = __shfl_sync(0xffffffffu, b[p], from);
                }
            }
            if (two_sided) {
                double *dst = accT + c * 32 + lane;
#pragma unroll
                for (int p = 0; p < PL; ++p) {
                    if (r == 0) dst[p * NT] = b[p];
                    else dst[p * NT] = P::kMin ? fmin(dst[p * NT], b[p]) : dst[p * NT] + b[p];
                }
            }
            __syncthreads();
        }
        // every warp is past the last round: the stage can be refilled, the B sums can leave
        if (tid == 0 && t + kStages < ntiles) issue(t + kStages);
        if (two_sided) {
            const int j = (tile0 + t) * NT + tid - row_j0;
#pragma unroll
            for (int p = 0; p < PL; ++p) rowB[(size_t)p * row_len + j] = accT[p * NT + tid];
        }
    }

    double *part = prm.partA + (size_t)blockIdx.y * PL * prm.na_pad;
#pragma unroll
    for (int k = 0; k < KA; ++k)
#pragma unroll
        for (int p = 0; p < PL; ++p) part[(size_t)p * prm.na_pad + a_first + k * NT] = a[k].s[p];
}

// ------------------------------------------------------------------------------------------------
// Fixed-order reduction of the partial sums of one band, carried in a running total.
//   total_i (+)= sum over the segments of i's A tile of partA    (if i is on the A side)
//              + sum over the A tiles that met i as a B particle of partB   (if i lies in the band)
// side 0: particles of the A list; side 1: particles of the B list (bipartite case only).
// first != 0: the total starts from zero (+inf for minima); last != 0: the scaled total is
// scattered to the caller's planes (and the packed stream / the bins are written).
// ------------------------------------------------------------------------------------------------
template <int PL, bool MIN>
__global__ void sym_reduce_kernel(const double *__restrict__ partA, const double *__restrict__ partB,
                                  double *__restrict__ total, int n_total, int self, int side,
                                  int TA, int NT, int na_pad, int a_tiles, int bt0, int bt1,
                                  int seg_tiles, int row0, int row_stride, int first, int last, int i0,
                                  int n_out, double scale,
                                  const int32_t *__restrict__ idx, int ld, double *__restrict__ out,
                                  double4 *__restrict__ packed, double tau_pivot,
                                  int32_t *__restrict__ out_bin, int accumulate,
                                  const int *__restrict__ gate, int *__restrict__ flag) {
    if (gate && *gate == 0) return;          // repair pass of a sweep that needed none
    const int i = i0 + blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_out) return;
    double s[PL];
#pragma unroll
    for (int p = 0; p < PL; ++p)
        s[p] = first ? (MIN ? __longlong_as_double(0x7ff0000000000000LL) : 0.0) : total[(size_t)p * n_total + i];
    auto add = [&](int p, double v) { s[p] = MIN ? fmin(s[p], v) : s[p] + v; };
    if (side == 0) {
        const int I = i / TA;
        int t_first = self ? I * (TA / NT) : 0;
        if (t_first < bt0) t_first = bt0;
        const bool mine = I >= row0 && (I - row0) % row_stride == 0;      // this shard swept i's A tile
        const int nseg = (mine && t_first < bt1) ? (bt1 - t_first + seg_tiles - 1) / seg_tiles : 0;
        for (int g = 0; g < nseg; ++g)
#pragma unroll
            for (int p = 0; p < PL; ++p) add(p, partA[((size_t)g * PL + p) * na_pad + i]);
    }
    if ((side == 1 || self) && i >= bt0 * NT && i < bt1 * NT) {
        const int rows = self ? i / TA : a_tiles;            // A tiles that met i on their B side
        const int len = (bt1 - bt0) * NT;
        const double *col = partB + (i - bt0 * NT);
        for (int I = row0, li = 0; I < rows; I += row_stride, ++li)      // owned rows, ascending
#pragma unroll
            for (int p = 0; p < PL; ++p) add(p, col[((size_t)li * PL + p) * len]);
    }
    if (!last) {
#pragma unroll
        for (int p = 0; p < PL; ++p) total[(size_t)p * n_total + i] = s[p];
        return;
    }
    const int g = idx ? idx[i] : i;
    if (MIN) {
        out[g] = s[0];
        if (out_bin) {
            int k = 0;
            if (!(s[0] > 0.0)) k = 2000;
            else {
                double pv = tau_pivot;
                while (pv > s[0] && k < 2000) { pv *= 0.5; ++k; }
            }
            out_bin[g] = k;
        }
    } else {
#pragma unroll
        for (int p = 0; p < PL; ++p) {
            s[p] *= scale;
            if (accumulate) s[p] += out[(size_t)p * ld + g];
            out[(size_t)p * ld + g] = s[p];
            // (SymGradientFast: a coincident pair leaves NaN here and asks for the guarded pass)
            if (flag && !(fabs(s[p]) <= 1.7976931348623157e308)) *flag = 1;
        }
        if (packed) packed[i] = make_double4(s[0], PL > 1 ? s[1] : 0.0, PL > 2 ? s[2] : 0.0, 1.0);
    }
}

// ------------------------------------------------------------------------------------------------
// Planning and launch.  The B list is processed in bands so that the B-side scratch
// (A tiles x planes x band length) stays below frost_ctx::sym_scratch bytes whatever N is; one band
// = one sweep launch + one reduction launch per side.
// ------------------------------------------------------------------------------------------------
struct SymJob {
    const double *A0, *A1, *B0, *B1;     // packed record streams (B* ignored when self)
    int nA, nB;
    bool self;
    const int32_t *A_idx, *B_idx;
    int ld;
    double *out;                         // planes [3][ld] (sums) or tau[n] (minima)
    double *A_packed, *B_packed;         // optional packed {s_x, s_y, s_z, 1} streams of the results
    double scale, eps2, tau_pivot;
    int32_t *out_bin;
    int *forest = nullptr;                 // time-step sweep: union-find forest of the fast pairs
    const int *gate = nullptr;             // the whole sweep runs only if *gate != 0
    const int *eq_flag = nullptr;          // run_sym<P, ..., PEQ>: *eq_flag != 0 selects the PEQ kernel
    int *flag = nullptr;                   // set to 1 if any scattered sum is not finite
    int shard_rank = 0, shard_world = 1;   // this launch sweeps A tiles rank, rank + world, ... only
    int accumulate = 0;                    // add the sums to `out` instead of overwriting it
};

template <class P, int KA, int NT, int MINB, class PEQ = P>
static int run_sym(frost_ctx *c, const SymJob &job) {
    constexpr int PL = P::kPlanes, TA = KA * NT;
    constexpr bool MIN = P::kMin;
    const bool self = job.self;
    const int na_pad = round_up(job.nA > 0 ? job.nA : 1, TA);
    const int nb_pad = self ? na_pad : round_up(job.nB > 0 ? job.nB : 1, NT);
    const int a_tiles = na_pad / TA, nb_tiles = nb_pad / NT;
    const int nB = self ? job.nA : job.nB;
    const int resident = c->num_sms * MINB;

    // bands
    const size_t row_bytes_per_tile = (size_t)a_tiles * PL * NT * sizeof(double);
    long long band_tiles = (long long)(c->sym_scratch / row_bytes_per_tile);
    if (band_tiles < 8) band_tiles = 8;
    if (band_tiles > nb_tiles) band_tiles = nb_tiles;
    const int nbands = (int)((nb_tiles + band_tiles - 1) / band_tiles);
    band_tiles = (nb_tiles + nbands - 1) / nbands;
    FROST_TRY(ensure(c, c->partialB, row_bytes_per_tile * (size_t)band_tiles + 256));
    if (nbands > 1) FROST_TRY(ensure(c, c->symtot, (size_t)PL * na_pad * sizeof(double)));

    const size_t smem = (size_t)kStages * P::kRecs * 2 * NT * kRecBytes + 2 * PL * NT * sizeof(double) +
                        kStages * sizeof(uint64_t);
    FROST_TRY(set_func_attr(c, sym_kernel<P, KA, NT, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    constexpr bool kHasEq = !std::is_same<P, PEQ>::value;
    if (kHasEq)
        FROST_TRY(set_func_attr(c, sym_kernel<PEQ, KA, NT, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));

    for (int b = 0; b < nbands; ++b) {
        const int bt0 = b * (int)band_tiles;
        const int bt1 = bt0 + (int)band_tiles < nb_tiles ? bt0 + (int)band_tiles : nb_tiles;
        const int a_rows = self ? (a_tiles < (bt1 + KA - 1) / KA ? a_tiles : (bt1 + KA - 1) / KA) : a_tiles;
        long long pairs = 0;                                  // tile pairs of this band
        const int row0 = job.shard_rank, row_stride = job.shard_world;
        const int my_rows = a_rows > row0 ? (a_rows - row0 + row_stride - 1) / row_stride : 0;
        for (int I = row0; I < a_rows; I += row_stride) {
            const int f = self && I * KA > bt0 ? I * KA : bt0;
            if (f < bt1) pairs += bt1 - f;
        }
        long long seg = pairs / (24LL * resident);            // >= 24 waves of CTAs
        if (seg < 1) seg = 1;
        if (seg > bt1 - bt0) seg = bt1 - bt0;
        if (c->tune_slices > 0) {
            seg = (bt1 - bt0 + c->tune_slices - 1) / c->tune_slices;
            if (seg < 1) seg = 1;
        }
        const int segs = (int)((bt1 - bt0 + seg - 1) / seg);
        FROST_TRY(ensure(c, c->partial, (size_t)segs * PL * na_pad * sizeof(double)));

        SymParams prm{};
        prm.a0 = (const double4 *)job.A0; prm.a1 = (const double4 *)job.A1;
        prm.b0 = (const double4 *)(self ? job.A0 : job.B0); prm.b1 = (const double4 *)(self ? job.A1 : job.B1);
        prm.partA = (double *)c->partial.p; prm.partB = (double *)c->partialB.p;
        prm.na_pad = na_pad; prm.self = self ? 1 : 0; prm.bt0 = bt0; prm.bt1 = bt1;
        prm.seg_tiles = (int)seg; prm.row0 = row0; prm.row_stride = row_stride;
        prm.eps2 = job.eps2; prm.eta_ff = c->eta_ff; prm.eta_fb = c->eta_fb;
        prm.pivot = job.tau_pivot; prm.forest = job.forest; prm.gate = job.gate; prm.gate_want = 1;
        if (my_rows > 0) {
            dim3 grid(my_rows, segs);
            if (kHasEq && job.eq_flag && !job.gate) {       // equal-mass variant | general variant
                prm.gate = job.eq_flag; prm.gate_want = 1;
                sym_kernel<PEQ, KA, NT, MINB><<<grid, NT, smem, c->stream>>>(prm);
                FROST_TRY(check_launch(c));
                prm.gate_want = 0;
            }
            sym_kernel<P, KA, NT, MINB><<<grid, NT, smem, c->stream>>>(prm);
            FROST_TRY(check_launch(c));
            prm.gate = job.gate; prm.gate_want = 1;
        }

        const int first = b == 0, last = b == nbands - 1;
        sym_reduce_kernel<PL, MIN><<<(job.nA + 255) / 256, 256, 0, c->stream>>>(
            prm.partA, prm.partB, (double *)c->symtot.p, na_pad, prm.self, 0, TA, NT, na_pad, a_tiles,
            bt0, bt1, prm.seg_tiles, row0, row_stride, first, last, 0, job.nA, job.scale, job.A_idx, job.ld, job.out,
            (double4 *)job.A_packed, job.tau_pivot, job.out_bin, job.accumulate, job.gate, job.flag);
        FROST_TRY(check_launch(c));
        if (!self) {          // a B particle only collects in its own band: no running total
            const int i0 = bt0 * NT, i1 = bt1 * NT < nB ? bt1 * NT : nB;
            if (i1 > i0) {
                sym_reduce_kernel<PL, MIN><<<(i1 - i0 + 255) / 256, 256, 0, c->stream>>>(
                    prm.partA, prm.partB, nullptr, 0, 0, 1, TA, NT, na_pad, a_tiles, bt0, bt1,
                    prm.seg_tiles, row0, row_stride, 1, 1, i0, i1, job.scale, job.B_idx, job.ld, job.out,
                    (double4 *)job.B_packed, job.tau_pivot, job.out_bin, job.accumulate, job.gate, job.flag);
                FROST_TRY(check_launch(c));
            }
        }
    }
    return FROST_OK;
}

// Geometry chosen by measurement on B200 (N = 262144; ms for Newton / gradient / time step):
//   256 threads x 2 CTAs/SM, KA = 4/2/2 (<=128 registers)   46.2 / 80.6 / 167.0
//   256 threads x 1 CTA/SM,  KA = 8/4/4                      45.2 / 76.2 / 166.5
//   128 threads x 2 CTAs/SM, KA = 8/4/4 (<=255 registers)    44.4 / 75.6 / 164.4   <- used
//   128 threads x 2 CTAs/SM, KA = 8/8/8 (255 registers)      44.3 / 79.8 / 175.9
// Round 2, N = 2^20 gradient sweep (ms): KA = 4: 1184.8; 4 with 3 CTAs/SM (166 registers): 1194.5; 3 with
// 3 CTAs/SM: 1206.5; 5: 1160.2; 6 (242 registers): 1150.4 <- used; 7 (246): 1169.8.  More warps do not help
// (the loop is not latency-bound); amortising the per-step SHFL / LDS / address instructions does: they
// cost ~27 issue cycles per rotation step.  Newton KA = 8 / 9 / 10: 702.8 / 700.6 / 699.0 (kept at 8).
// More A particles per thread amortise the per-step SHFL / LDS / address instructions; the A tile
// is 1024 (Newton) or 512 (gradient, time step) particles, the B tile 128.
constexpr int kSymNT = 128, kSymMinB = 2;
constexpr int kSymKNewton = 8, kSymKGrad = 6, kSymKTau = 4;
constexpr int kSymMinBGrad = 2, kSymNTGrad = 128;
// sets below kSymSmallN particles: A tiles of 256 so that there are enough tile pairs to fill the GPU
constexpr int kSymSmallN = 16384, kSymKSmall = 2, kSymMinBSmall = 4;

// The tile geometry of the large force sweeps, as text: part of frost_version(), so that a stored
// measurement (profiles/sym_gradient_traffic.csv) can be tied to the build it was taken on.
const char *sym_geometry() {
    static char buf[96];
    static const int n = snprintf(buf, sizeof(buf), "newton A%dxB%d; gradient A%dxB%d, %d CTAs/SM", kSymKNewton * kSymNT,
                                  kSymNT, kSymKGrad * kSymNTGrad, kSymNTGrad, kSymMinBGrad);
    (void)n;
    return buf;
}

// Newton sweep, both directions at once (Eq. 24 / 42).  self: B == A (B arguments ignored).
int sym_newton(frost_ctx *c, const double *A_xm, int nA, const double *B_xm, int nB, bool self,
               const int32_t *A_idx, const int32_t *B_idx, int ld, double *out_acc,
               double *A_a_packed, double *B_a_packed) {
    if (nA <= 0 || (!self && nB <= 0)) return FROST_OK;
    SymJob j{};
    j.A0 = A_xm; j.B0 = B_xm; j.nA = nA; j.nB = nB; j.self = self; j.A_idx = A_idx; j.B_idx = B_idx;
    j.ld = ld; j.out = out_acc; j.A_packed = A_a_packed; j.B_packed = B_a_packed;
    j.scale = c->G;
    j.eps2 = c->eps2 > 0x1p-400 ? c->eps2 : 0x1p-400;      // see NewtonPolicy::pair
    j.shard_rank = c->shard_rank; j.shard_world = c->shard_world; j.accumulate = c->accumulate;
    if (nA < kSymSmallN) return run_sym<SymNewton, kSymKSmall, kSymNT, kSymMinBSmall>(c, j);
    j.eq_flag = c->eq_flag_cur;
    return run_sym<SymNewton, kSymKNewton, kSymNT, kSymMinB, SymNewtonT<true>>(c, j);
}

// Gradient sweep, both directions at once (Eq. 27 / 43 / 44); *_a are the packed accelerations.
int sym_gradient(frost_ctx *c, const double *A_xm, const double *A_a, int nA, const double *B_xm,
                 const double *B_a, int nB, bool self, const int32_t *A_idx, const int32_t *B_idx,
                 int ld, double *out_grad) {
    if (nA <= 0 || (!self && nB <= 0)) return FROST_OK;
    SymJob j{};
    j.A0 = A_xm; j.A1 = A_a; j.B0 = B_xm; j.B1 = B_a; j.nA = nA; j.nB = nB; j.self = self;
    j.A_idx = A_idx; j.B_idx = B_idx; j.ld = ld; j.out = out_grad;
    j.scale = 2.0 * c->G; j.eps2 = c->eps2;
    j.shard_rank = c->shard_rank; j.shard_world = c->shard_world; j.accumulate = c->accumulate;
    if (nA < kSymSmallN) return run_sym<SymGradient, kSymKSmall, kSymNT, kSymMinBSmall>(c, j);
    if (c->tune_guard == 0 && !c->accumulate) {
        // unguarded pass (SymGradientFast), then the guarded pass behind a gate that only opens if a
        // scattered sum came out non-finite, i.e. if the input has distinct coincident particles
        FROST_TRY(ensure(c, c->symflag, 256));
        int *flag = (int *)c->symflag.p;
        FROST_CUDA(c, cudaMemsetAsync(flag, 0, sizeof(int), c->stream));
        j.flag = flag; j.eq_flag = c->eq_flag_cur;
        FROST_TRY((run_sym<SymGradientFast, kSymKGrad, kSymNTGrad, kSymMinBGrad, SymGradientFastT<true>>(c, j)));
        j.flag = nullptr; j.eq_flag = nullptr; j.gate = flag;
    }
    return run_sym<SymGradient, kSymKGrad, kSymNTGrad, kSymMinBGrad>(c, j);
}

// Time-step sweep over one level (Eq. 49-54); xm carries G*m in .w and NaN padding.
int sym_timestep(frost_ctx *c, const double *xm, const double *v, int n_set, const int32_t *idx,
                 double tau_pivot, double *out_tau, int32_t *out_bin, int *forest) {
    if (n_set <= 0) return FROST_OK;
    SymJob j{};
    j.A0 = xm; j.A1 = v; j.nA = n_set; j.nB = n_set; j.self = true; j.A_idx = idx;
    j.out = out_tau; j.out_bin = out_bin; j.tau_pivot = tau_pivot; j.scale = 1.0; j.forest = forest;
    if (forest) {
        if (n_set < kSymSmallN) return run_sym<SymTimestepEdge, kSymKSmall, kSymNT, kSymMinBSmall>(c, j);
        return run_sym<SymTimestepEdge, kSymKTau, kSymNT, kSymMinB>(c, j);
    }
    if (n_set < kSymSmallN) return run_sym<SymTimestep, kSymKSmall, kSymNT, kSymMinBSmall>(c, j);
    return run_sym<SymTimestep, kSymKTau, kSymNT, kSymMinB>(c, j);
}

// Masked self sweep of one list (labels in the low word of a_lab[k].w): out_acc != NULL the Newton sweep,
// out_grad != NULL the gradient sweep from the accelerations in a_lab.  accumulate: add to the planes.
int sym_masked(frost_ctx *c, const double *xm, const double *a_lab, int n, const int32_t *idx, int ld,
               double *out_acc, double *out_grad, int accumulate) {
    if (n <= 0) return FROST_OK;
    for (int pass = 0; pass < 2; ++pass) {
        if ((pass == 0 && !out_acc) || (pass == 1 && !out_grad)) continue;
        SymJob j{};
        j.A0 = xm; j.A1 = a_lab; j.nA = n; j.nB = n; j.self = true; j.A_idx = idx; j.ld = ld;
        j.accumulate = accumulate;
        if (pass == 0) {
            j.out = out_acc; j.scale = c->G; j.eps2 = c->eps2 > 0x1p-400 ? c->eps2 : 0x1p-400;
            if (n < kSymSmallN) FROST_TRY((run_sym<SymNewtonMasked, kSymKSmall, kSymNT, kSymMinBSmall>(c, j)));
            else FROST_TRY((run_sym<SymNewtonMasked, kSymKNewton, kSymNT, kSymMinB>(c, j)));
        } else {
            j.out = out_grad; j.scale = 2.0 * c->G; j.eps2 = c->eps2;
            if (n < kSymSmallN) FROST_TRY((run_sym<SymGradientMasked, kSymKSmall, kSymNT, kSymMinBSmall>(c, j)));
            else FROST_TRY((run_sym<SymGradientMasked, kSymKGrad, kSymNTGrad, kSymMinBGrad>(c, j)));
        }
    }
    return FROST_OK;
}

// phi_i = -G sum_{j != i} m_j / s_ij for all particles of the packed stream (always symmetric).
int sym_potential(frost_ctx *c, const double *xm, int n, double *out_phi) {
    if (n <= 0) return FROST_OK;
    SymJob j{};
    j.A0 = xm; j.nA = n; j.nB = n; j.self = true; j.ld = n; j.out = out_phi;
    j.scale = -c->G; j.eps2 = c->eps2;
    return run_sym<SymPotential, kSymKGrad, kSymNT, kSymMinB>(c, j);
}

}  // namespace frost
