// frost_pairs.cuh -- what one ordered pair (sink i <- source j) contributes in each of the three
// sweeps: Newtonian acceleration (Eq. 24/42), gradient acceleration (Eq. 27/43/44), symmetrised
// time-step candidates (Eq. 49-54).  Shared by the streaming sweeps (frost_sweeps.cu) and the
// device-resident small-set subtree (frost_small.cu).
#pragma once
#include "frost_common.cuh"

namespace frost {

// ------------------------------------------------------------------------------------------------
// Policies: what one sink carries, what one ordered pair adds.
// ------------------------------------------------------------------------------------------------
struct SweepParams {
    const double4 *snk0;   // sink records {x,y,z,m}
    const double4 *snk1;   // sink records {ax,ay,az,0} or {vx,vy,vz,0} (policies with 2 records)
    const double4 *src0;   // source records {x,y,z,m}
    const double4 *src1;   // second source record stream
    double *partial;       // [slices][planes][n_pad]
    int n_pad;             // padded sink count (plane stride of `partial`)
    int n_tiles;           // source tiles in total
    int tiles_per_slice;
    double eps2;
    double G, eta_ff, eta_fb;
    double pivot;          // TimestepEdgePolicy: pairs with a candidate below it are united in `forest`
    int *forest;
};

struct NewtonPolicy {
    static constexpr int kRecs = 1;
    static constexpr int kPlanes = 3;
    struct Sink { double x, y, z; };
    struct Acc { double x, y, z; };
    __device__ static __forceinline__ void load(Sink &s, const SweepParams &p, int i) {
        const double4 r = p.snk0[i];
        s.x = r.x; s.y = r.y; s.z = r.z;
    }
    __device__ static __forceinline__ void init(Acc &a) { a.x = a.y = a.z = 0.0; }
    // Eq. (24): a_i += m_j x_ji / s^3.  16 FP64-pipe instructions + 1 MUFU, nothing else.
    // w = m y^3 (1-e)^(-3/2) with e = 1 - s2 y^2 ~ 2^-22: series to e^2 (next term 35/16 e^3).
    // p.eps2 is floored at 2^-400 by the launcher, so s2 > 0 and the MUFU seed is finite without
    // any guard: the self pair then has dx = dy = dz = 0 exactly and a finite w, and adds 0.
    // The three accumulating FMAs share w in the same operand slot and are kept adjacent so that
    // the operand-reuse cache serves it (a DFMA reading three distinct register pairs costs 3
    // issue cycles instead of 2 on sm_100a -- DESIGN.md "FP64 issue model").
    __device__ static __forceinline__ void pair(const Sink &s, Acc &a, const double4 &j0,
                                                const double4 &, const SweepParams &p) {
        const double dx = j0.x - s.x, dy = j0.y - s.y, dz = j0.z - s.z;
        const double s2 = fma(dz, dz, fma(dy, dy, fma(dx, dx, p.eps2)));
        const double y = rsqrt_seed(s2);
        const double y2 = y * y;
        const double e = fma(-s2, y2, 1.0);
        const double ym = y * j0.w;
        const double w0 = y2 * ym;
        const double q = fma(1.875, e, 1.5);
        const double qe = q * e;
        const double w = fma(w0, qe, w0);
        fma3_shared(a.x, a.y, a.z, w, dx, dy, dz);
    }
    __device__ static __forceinline__ void store(const Acc &a, double *part, int n_pad, int i) {
        part[i] = a.x; part[n_pad + i] = a.y; part[2 * n_pad + i] = a.z;
    }
};

struct GradientPolicy {
    static constexpr int kRecs = 2;
    static constexpr int kPlanes = 3;
    struct Sink { double x, y, z, ax, ay, az; };
    struct Acc { double x, y, z; };
    __device__ static __forceinline__ void load(Sink &s, const SweepParams &p, int i) {
        const double4 r = p.snk0[i];
        const double4 a = p.snk1[i];
        s.x = r.x; s.y = r.y; s.z = r.z; s.ax = a.x; s.ay = a.y; s.az = a.z;
    }
    __device__ static __forceinline__ void init(Acc &a) { a.x = a.y = a.z = 0.0; }
    // Eq. (27): g_i += m_j s^-3 ( a_ji - 3 s^-2 (x_ji . a_ji) x_ji ).  28 FP64-pipe instructions.
    __device__ static __forceinline__ void pair(const Sink &s, Acc &g, const double4 &j0,
                                                const double4 &j1, const SweepParams &p) {
        const double dx = j0.x - s.x, dy = j0.y - s.y, dz = j0.z - s.z;
        const double ax = j1.x - s.ax, ay = j1.y - s.ay, az = j1.z - s.az;
        const double s2 = fma(dz, dz, fma(dy, dy, fma(dx, dx, p.eps2)));
        const double ri = rsqrt_full_or_zero(s2);
        const double dot = fma(dz, az, fma(dy, ay, dx * ax));
        const double q = ri * ri;
        const double mr = j0.w * ri;
        const double w3 = mr * q;
        const double t = q * dot;
        const double u = t * -3.0;
        double vx = ax, vy = ay, vz = az;
        fma3_shared(vx, vy, vz, u, dx, dy, dz);
        fma3_shared(g.x, g.y, g.z, w3, vx, vy, vz);
    }
    __device__ static __forceinline__ void store(const Acc &a, double *part, int n_pad, int i) {
        part[i] = a.x; part[n_pad + i] = a.y; part[2 * n_pad + i] = a.z;
    }
};

// Harmonic symmetrisation factor of Eq. (49) in the cancellation-free form 1 + q/(1+sqrt(1+q^2))
// (reading 10), without IEEE sqrt/div sequences: with u = 1/sqrt(1+q^2) in (0,1],
//   q/(1+sqrt(1+q^2)) = q u / (1 + u);  1/(1+u) by MUFU.RCP64H + one cubic step.  13 FP64 instr.
// s(q) > 0 for every q, but for q < -1e15 the sum below cancels to within its rounding error and
// can come out as -0 or a tiny negative number; the |.| (a free source modifier of the consuming
// DMUL) keeps every candidate >= 0 in all three time-step routines alike, which the bit-pattern
// atomicMin of frost_tau.cu relies on.  NaN (self pair, padding) stays NaN.
__device__ __forceinline__ double sym_factor(double q) {
    const double h = fma(q, q, 1.0);
    const double u = rsqrt_full(h);
    const double qu = q * u;
    const double d = u + 1.0;
    const double rd = rcp_full(d);
    return fabs(fma(qu, rd, 1.0));
}

struct TimestepPolicy {
    static constexpr int kRecs = 2;
    static constexpr int kPlanes = 1;
    struct Sink { double x, y, z, gm, vx, vy, vz; };
    struct Acc { double tau; };
    __device__ static __forceinline__ void load(Sink &s, const SweepParams &p, int i) {
        const double4 r = p.snk0[i];
        const double4 v = p.snk1[i];
        s.x = r.x; s.y = r.y; s.z = r.z; s.gm = r.w; s.vx = v.x; s.vy = v.y; s.vz = v.z;
    }
    __device__ static __forceinline__ void init(Acc &a) { a.tau = __longlong_as_double(0x7ff0000000000000LL); }
    // Eq. (50)-(54) + Eq. (49) per ordered pair, min over the candidates.
    // The position record carries G*m in .w.  No branch and no compare: the self pair (r2 = 0), a
    // padding record (NaN position) and a pair at rest (v2 = 0, fly-by only) turn into NaN through
    // MUFU(0) = +inf and 0*inf, and fmin() returns its non-NaN operand, so such candidates drop out
    // exactly as DESIGN.md reading 11 requires.  ~77 FP64 instructions + 7 MUFU per pair.
    __device__ static __forceinline__ double candidate(const Sink &s, const double4 &j0, const double4 &j1,
                                                       const SweepParams &p) {
        const double rx = j0.x - s.x, ry = j0.y - s.y, rz = j0.z - s.z;
        const double vx = j1.x - s.vx, vy = j1.y - s.vy, vz = j1.z - s.vz;
        const double r2 = fma(rz, rz, fma(ry, ry, rx * rx));
        const double v2 = fma(vz, vz, fma(vy, vy, vx * vx));
        const double rv = fma(rz, vz, fma(ry, vy, rx * vx));
        const double mu = s.gm + j0.w;                 // G (m_i + m_j)
        const double ir = rsqrt_full(r2);              // 1/r       (NaN for r2 = 0)
        const double iv = rsqrt_full(v2);              // 1/v       (NaN for v2 = 0)
        const double ir2 = ir * ir;
        const double mir = mu * ir;
        const double t_ff = rsqrt_full(mir * ir2);     // Eq. 50: (r^3/mu)^(1/2) = (mu/r^3)^(-1/2)
        const double t_fb = (r2 * ir) * iv;            // Eq. 51: r / v
        const double rvr2 = rv * ir2;                  // (r.v)/r^2
        const double q_ff = (rvr2 * t_ff) * (1.5 * p.eta_ff);                 // eta * Eq. 53
        const double f = rvr2 * t_fb;
        const double q_fb = fma(f, mir * (iv * iv), f) * p.eta_fb;            // eta * Eq. 54
        const double c_ff = sym_factor(q_ff) * (t_ff * p.eta_ff);
        const double c_fb = sym_factor(q_fb) * (t_fb * p.eta_fb);
        return fmin(c_ff, c_fb);
    }
    __device__ static __forceinline__ void pair(const Sink &s, Acc &a, const double4 &j0,
                                                const double4 &j1, const SweepParams &p) {
        a.tau = fmin(a.tau, candidate(s, j0, j1, p));
    }
    __device__ static __forceinline__ void store(const Acc &a, double *part, int n_pad, int i) {
        part[i] = a.tau;
    }
};

// The time-step sweep of a split hierarchy entry (reading 24): as TimestepPolicy, and every
// fast pair (candidate < pivot) is united in the union-find forest over list positions.  The list
// position of a record travels in the low word of .w of its velocity record.
struct TimestepEdgePolicy {
    static constexpr int kRecs = 2;
    static constexpr int kPlanes = 1;
    struct Sink : TimestepPolicy::Sink { int id; };
    using Acc = TimestepPolicy::Acc;
    __device__ static __forceinline__ void load(Sink &s, const SweepParams &p, int i) {
        TimestepPolicy::load(s, p, i);
        s.id = __double2loint(p.snk1[i].w);
    }
    __device__ static __forceinline__ void init(Acc &a) { TimestepPolicy::init(a); }
    __device__ static __forceinline__ void pair(const Sink &s, Acc &a, const double4 &j0,
                                                const double4 &j1, const SweepParams &p) {
        const double c = TimestepPolicy::candidate(s, j0, j1, p);
        a.tau = fmin(a.tau, c);
        if (c < p.pivot) uf_union(p.forest, s.id, __double2loint(j1.w));
    }
    __device__ static __forceinline__ void store(const Acc &a, double *part, int n_pad, int i) {
        part[i] = a.tau;
    }
};

// Eq. 42 / 43-44 on the kicked pair set of a split entry: a source whose component label (low word of
// .w of the second record) equals the sink's contributes nothing.  Slow particles all carry -1.
struct MaskedNewtonPolicy {
    static constexpr int kRecs = 2;
    static constexpr int kPlanes = 3;
    struct Sink : NewtonPolicy::Sink { int lab; };
    using Acc = NewtonPolicy::Acc;
    __device__ static __forceinline__ void load(Sink &s, const SweepParams &p, int i) {
        NewtonPolicy::load(s, p, i);
        s.lab = __double2loint(p.snk1[i].w);
    }
    __device__ static __forceinline__ void init(Acc &a) { NewtonPolicy::init(a); }
    __device__ static __forceinline__ void pair(const Sink &s, Acc &a, const double4 &j0,
                                                const double4 &j1, const SweepParams &p) {
        double4 jm = j0;
        if (__double2loint(j1.w) == s.lab) jm.w = 0.0;
        NewtonPolicy::pair(s, a, jm, jm, p);
    }
    __device__ static __forceinline__ void store(const Acc &a, double *part, int n_pad, int i) {
        NewtonPolicy::store(a, part, n_pad, i);
    }
};

struct MaskedGradientPolicy {
    static constexpr int kRecs = 2;
    static constexpr int kPlanes = 3;
    struct Sink : GradientPolicy::Sink { int lab; };
    using Acc = GradientPolicy::Acc;
    __device__ static __forceinline__ void load(Sink &s, const SweepParams &p, int i) {
        GradientPolicy::load(s, p, i);
        s.lab = __double2loint(p.snk1[i].w);
    }
    __device__ static __forceinline__ void init(Acc &a) { GradientPolicy::init(a); }
    __device__ static __forceinline__ void pair(const Sink &s, Acc &g, const double4 &j0,
                                                const double4 &j1, const SweepParams &p) {
        double4 jm = j0;
        if (__double2loint(j1.w) == s.lab) jm.w = 0.0;
        GradientPolicy::pair(s, g, jm, j1, p);
    }
    __device__ static __forceinline__ void store(const Acc &a, double *part, int n_pad, int i) {
        GradientPolicy::store(a, part, n_pad, i);
    }
};

}  // namespace frost
