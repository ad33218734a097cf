/*
 * frost_oracle.c -- the CPU ORACLE for the HHS-FSI hot path.  TEST INFRASTRUCTURE ONLY.
 *
 * This file is a plain, slow, obviously-correct restatement of what the paper
 * (Rantala, Naab & Springel, "FROST", arXiv 2011.14984; /root/reference/PAPER.md) says the hot
 * path computes.  It exists so that the CUDA library can be checked element by element, and so
 * that bench.py can time "the oracle as it stands" as the cpu_baseline.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may call it.  It
 * shares NO code, header, table or constant with paper_2011_14984_b200/csrc/ and neither side
 * includes the other.
 *
 * Style: one loop nest per definition, in the paper's order and notation; no blocking, fusion
 * or reordering.  Sums over pairs are accumulated in `long double` (x87 80-bit on x86-64) with
 * j ascending and rounded to double once at the end, so that the oracle's own rounding error
 * (~1e-19 relative per term) is far below the 1e-12 / 1e-10 parity tolerances.  The time-step
 * criterion, kick and drift are computed in plain double, because the method itself is an fp64
 * method and the slow/fast decision tau_i >= tau_pivot must be taken in that precision on both
 * sides.  Compile with -ffp-contract=off (oracle/build.py does) so no FMA contraction happens.
 * OpenMP parallelises over sinks only: each sink's sum is sequential, so results do not depend
 * on the number of threads.
 *
 * Pins (tests/test_oracle_pins.py; every function below is pinned unless it says otherwise):
 *   O1 oracle_forces ACC   : autograd / finite differences of U (Eq. 23), two-body closed form,
 *                            sum m a = 0, Plummer mean field (Eq. A2).
 *   O2 oracle_forces GRAD  : autograd / finite differences of G_P = -sum m |a|^2 (Eq. 17, 39),
 *                            two-body closed form g = 4 G (m1+m2) r^-3 a (Eq. 25-26), sum m g = 0.
 *   O3 oracle_timesteps    : circular binary tau = eta P / 2 pi (Eq. 52), s(q) values and
 *                            symmetries (Eq. 49, Fig. 2), brute-force scalar re-evaluation.
 *                            The choice "eta inside q" (reading 9) is PARITY UNPINNED:
 *                            nothing the paper prints separates it from "q without eta".
 *                            Softened time-steps (reading 14) are PARITY UNPINNED.
 *   O5 oracle_fsi_step     : 4th-order convergence against the Kepler closed form, time reversal.
 *   O6 oracle_hhs_step     : 4th-order convergence with a frozen partition on a star+planets
 *                            system, momentum at roundoff, five-body Solar system (Tables A1/A2).
 *   O6s split fast levels  : (PAPER.md:759 names the idea only; the definition is DESIGN.md reading
 *                            24) bit-for-bit Alg. 3 when F is one component; components against an
 *                            independent graph routine; 4th-order convergence with a frozen
 *                            partition into components; momentum at roundoff; energy error of the
 *                            size of Alg. 3's on a cluster with binaries.
 *   O6k two-body propagator: (PAPER.md:759 lists Kepler solvers as plug-ins; reading 25) the
 *                            classical-elements solution through the eccentric anomaly for
 *                            e = 0 ... 0.99 and up to 123 periods; energy, angular momentum, the
 *                            group property and time reversal on unbound orbits; a fine FSI run.
 *   O7 oracle_diagnostics  : textbook definitions (Eq. 23); used by the pins.
 *
 * Array convention (same as include/frost.h, restated independently): positions, velocities,
 * accelerations are three SoA planes, component c of particle i at p[c*ld + i]; index arrays
 * are int32, NULL means "all particles 0..n-1".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_ACC 1
#define ORACLE_GRAD 2
#define ORACLE_MUTUAL 4

#define ORACLE_OK 0
#define ORACLE_EINVAL (-1)
#define ORACLE_ENOMEM (-3)
#define ORACLE_EDEPTH (-4)

#define ORACLE_MAX_LEVELS 64

typedef long double ld_t;

typedef struct {
    int32_t depth;                          /* deepest level entered with a non-empty set */
    int32_t reserved;
    int64_t entries[ORACLE_MAX_LEVELS];     /* non-empty entries of hhs_fsi at level k */
    int64_t n_slow[ORACLE_MAX_LEVELS];      /* sum of |S| over those entries */
    int64_t n_fast[ORACLE_MAX_LEVELS];      /* sum of |F| over those entries */
    int64_t pairs_newton;                   /* ordered pairs swept by Eq. 24 / 42 */
    int64_t pairs_gradient;                 /* ordered pairs swept by Eq. 27 / 43 / 44 */
    int64_t pairs_timestep;                 /* ordered pairs swept by Eq. 49-54 */
    int64_t n_comp[ORACLE_MAX_LEVELS];      /* sum over those entries of the number of fast components
                                               recursed into (Alg. 3 itself: 1 per entry with |F| > 0) */
    int64_t n_kepler;                       /* two-body components advanced by the Kepler propagator (O6k) */
} oracle_hhs_stats;

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_set_num_threads(int t) {
#ifdef _OPENMP
    if (t > 0) omp_set_num_threads(t);
#else
    (void)t;
#endif
}

static inline int pick(const int32_t *idx, int k) { return idx ? idx[k] : k; }

/* ---------------------------------------------------------------------------------------------
 * O1.  Newtonian acceleration, Eq. (24) PAPER.md:216-219 (self) and Eq. (42)
 * (inter-level), with the Plummer-softening substitution r -> (r^2+eps_p^2)^(1/2) of PAPER.md:250:
 *     a_i = G * sum_{j in J, s_ij^2 > 0} m_j x_ji / s_ij^3,   x_ji = x_j - x_i,
 *     s_ij^2 = |x_ji|^2 + eps2.
 * "j != i" is expressed as s_ij^2 > 0 (reading 11).
 * ------------------------------------------------------------------------------------------- */
static void newton_one_direction(int ld, const double *pos, const double *mass,
                                 const int32_t *I, int nI, const int32_t *J, int nJ,
                                 double G, double eps2, double *acc) {
#pragma omp parallel for schedule(dynamic, 16)
    for (int a = 0; a < nI; ++a) {
        const int i = pick(I, a);
        const ld_t xi = pos[i], yi = pos[ld + i], zi = pos[2 * ld + i];
        ld_t ax = 0, ay = 0, az = 0;
        for (int b = 0; b < nJ; ++b) {
            const int j = pick(J, b);
            const ld_t dx = (ld_t)pos[j] - xi;
            const ld_t dy = (ld_t)pos[ld + j] - yi;
            const ld_t dz = (ld_t)pos[2 * ld + j] - zi;
            const ld_t s2 = dx * dx + dy * dy + dz * dz + (ld_t)eps2;
            if (s2 > 0) {
                const ld_t s = sqrtl(s2);
                const ld_t w = (ld_t)mass[j] / (s2 * s);
                ax += w * dx;
                ay += w * dy;
                az += w * dz;
            }
        }
        acc[i] = (double)((ld_t)G * ax);
        acc[ld + i] = (double)((ld_t)G * ay);
        acc[2 * ld + i] = (double)((ld_t)G * az);
    }
}

/* ---------------------------------------------------------------------------------------------
 * O2.  Gradient acceleration, Eq. (27) PAPER.md:234-239 (self) and Eq. (43)-(44)
 * PAPER.md:373-387 (inter-level):
 *     g_i = 2 G * sum_{j in J, s>0} m_j / s^5 * ( s^2 a_ji - 3 (x_ji . a_ji) x_ji ),
 *     a_ji = a_j - a_i,  x_ji = x_j - x_i.
 * `acc` must hold, for every i in I and j in J, the acceleration generated by the same pair set
 * (reading O2).  The prefactor 2 is the one printed in Eq. (27); Eq. (28)'s G eps^2/24
 * is 2/48.
 * ------------------------------------------------------------------------------------------- */
static void gradient_one_direction(int ld, const double *pos, const double *mass,
                                   const int32_t *I, int nI, const int32_t *J, int nJ,
                                   double G, double eps2, const double *acc, double *grad) {
#pragma omp parallel for schedule(dynamic, 16)
    for (int a = 0; a < nI; ++a) {
        const int i = pick(I, a);
        const ld_t xi = pos[i], yi = pos[ld + i], zi = pos[2 * ld + i];
        const ld_t axi = acc[i], ayi = acc[ld + i], azi = acc[2 * ld + i];
        ld_t gx = 0, gy = 0, gz = 0;
        for (int b = 0; b < nJ; ++b) {
            const int j = pick(J, b);
            const ld_t dx = (ld_t)pos[j] - xi;
            const ld_t dy = (ld_t)pos[ld + j] - yi;
            const ld_t dz = (ld_t)pos[2 * ld + j] - zi;
            const ld_t s2 = dx * dx + dy * dy + dz * dz + (ld_t)eps2;
            if (s2 > 0) {
                const ld_t dax = (ld_t)acc[j] - axi;
                const ld_t day = (ld_t)acc[ld + j] - ayi;
                const ld_t daz = (ld_t)acc[2 * ld + j] - azi;
                const ld_t s = sqrtl(s2);
                const ld_t s5 = s2 * s2 * s;
                const ld_t xa = dx * dax + dy * day + dz * daz;
                const ld_t w = (ld_t)mass[j] / s5;
                gx += w * (s2 * dax - 3 * xa * dx);
                gy += w * (s2 * day - 3 * xa * dy);
                gz += w * (s2 * daz - 3 * xa * dz);
            }
        }
        grad[i] = (double)(2 * (ld_t)G * gx);
        grad[ld + i] = (double)(2 * (ld_t)G * gy);
        grad[2 * ld + i] = (double)(2 * (ld_t)G * gz);
    }
}

/* ---------------------------------------------------------------------------------------------
 * O2b.  Magnitude sum of the terms of Eq. (27) / (43)-(44), PAPER.md:234-239, 373-387:
 *     T_i = 2 G * sum_{j in J, s>0} | m_j / s^5 * ( s^2 a_ji - 3 (x_ji . a_ji) x_ji ) |_2
 * -- the same terms gradient_one_direction adds, with the Euclidean norm taken before the sum.
 * T_i / |g_i| is the condition number of the gradient sum: any evaluation of Eq. (27) from fp64
 * accelerations carries an error of order 2^-53 T_i (reading 22), which is what the
 * parity tests gate on where hard binaries make T_i >> |g_i|.  Not a step of the method.
 * Pins (tests/test_oracle_pins.py): equals |g_i| for two bodies (closed form of Eq. 25-26),
 * collinear closed form, triangle inequality |g_i| <= T_i, homogeneity.
 * ------------------------------------------------------------------------------------------- */
int oracle_gradient_termsum(int n, int ld, const double *pos, const double *mass,
                            const int32_t *I, int nI, const int32_t *J, int nJ, double G,
                            double eps2, const double *acc, double *out_T) {
    if (n < 0 || ld < n || !pos || !mass || !acc || !out_T) return ORACLE_EINVAL;
    if (!I) nI = n;
    if (!J) nJ = n;
#pragma omp parallel for schedule(dynamic, 16)
    for (int a = 0; a < nI; ++a) {
        const int i = pick(I, a);
        const ld_t xi = pos[i], yi = pos[ld + i], zi = pos[2 * ld + i];
        const ld_t axi = acc[i], ayi = acc[ld + i], azi = acc[2 * ld + i];
        ld_t T = 0;
        for (int b = 0; b < nJ; ++b) {
            const int j = pick(J, b);
            const ld_t dx = (ld_t)pos[j] - xi;
            const ld_t dy = (ld_t)pos[ld + j] - yi;
            const ld_t dz = (ld_t)pos[2 * ld + j] - zi;
            const ld_t s2 = dx * dx + dy * dy + dz * dz + (ld_t)eps2;
            if (s2 > 0) {
                const ld_t dax = (ld_t)acc[j] - axi;
                const ld_t day = (ld_t)acc[ld + j] - ayi;
                const ld_t daz = (ld_t)acc[2 * ld + j] - azi;
                const ld_t s = sqrtl(s2);
                const ld_t s5 = s2 * s2 * s;
                const ld_t xa = dx * dax + dy * day + dz * daz;
                const ld_t w = (ld_t)mass[j] / s5;
                const ld_t tx = w * (s2 * dax - 3 * xa * dx);
                const ld_t ty = w * (s2 * day - 3 * xa * dy);
                const ld_t tz = w * (s2 * daz - 3 * xa * dz);
                T += sqrtl(tx * tx + ty * ty + tz * tz);
            }
        }
        out_T[i] = (double)(2 * (ld_t)G * T);
    }
    return ORACLE_OK;
}

/* compute_acc_newton / compute_acc_gradient (Alg. 2) when I == J; one direction of
 * acc_sf_newton / acc_sf_gradient (Alg. 3) when I != J; both directions under
 * ORACLE_MUTUAL.  Entries of acc/grad outside I (and J under MUTUAL) are not touched. */
int oracle_forces(int n, int ld, const double *pos, const double *mass,
                  const int32_t *sink_idx, int n_sink, const int32_t *source_idx, int n_source,
                  double G, double eps2, double *acc, double *grad, int flags) {
    if (n < 0 || ld < n || !pos || !mass || !acc) return ORACLE_EINVAL;
    if (!sink_idx) n_sink = n;
    if (!source_idx) n_source = n;
    if ((flags & ORACLE_GRAD) && !grad) return ORACLE_EINVAL;
    if (flags & ORACLE_ACC) {
        newton_one_direction(ld, pos, mass, sink_idx, n_sink, source_idx, n_source, G, eps2, acc);
        if (flags & ORACLE_MUTUAL)
            newton_one_direction(ld, pos, mass, source_idx, n_source, sink_idx, n_sink, G, eps2, acc);
    }
    if (flags & ORACLE_GRAD) {
        gradient_one_direction(ld, pos, mass, sink_idx, n_sink, source_idx, n_source, G, eps2, acc, grad);
        if (flags & ORACLE_MUTUAL)
            gradient_one_direction(ld, pos, mass, source_idx, n_source, sink_idx, n_sink, G, eps2, acc, grad);
    }
    return ORACLE_OK;
}

/* ---------------------------------------------------------------------------------------------
 * O3.  Symmetrised free-fall / fly-by time-steps, Eq. (49)-(54) PAPER.md:429-474, over the
 * particles of ONE hierarchy level: sinks = sources = idx.
 * ------------------------------------------------------------------------------------------- */

/* Harmonic symmetrisation factor of Eq. (49), PAPER.md:431:
 *     s(q) = [ q + sqrt(1+q^2) - 1 ] / q ,   q = d tau / dt,
 * written in the algebraically identical form 1 + q / (1 + sqrt(1+q^2)) which has no 0/0 at q=0
 * and no cancellation (reading 10). */
double oracle_sym_factor(double q) { return 1.0 + q / (1.0 + sqrt(1.0 + q * q)); }

/* The symmetrised step candidates of one ordered pair (i <- j).  out[0] = free-fall candidate,
 * out[1] = fly-by candidate (+inf if the pair gives none).  r = x_j - x_i, v = v_j - v_i. */
void oracle_pair_timestep(const double xi[3], const double vi[3], double mi,
                          const double xj[3], const double vj[3], double mj,
                          double G, double eta_ff, double eta_fb, int eta_in_q, double out[2]) {
    const double rx = xj[0] - xi[0], ry = xj[1] - xi[1], rz = xj[2] - xi[2];
    const double vx = vj[0] - vi[0], vy = vj[1] - vi[1], vz = vj[2] - vi[2];
    const double r2 = rx * rx + ry * ry + rz * rz;
    const double v2 = vx * vx + vy * vy + vz * vz;
    out[0] = INFINITY;
    out[1] = INFINITY;
    if (!(r2 > 0.0)) return;                    /* coincident pair / self: ignored (reading 11) */
    const double r = sqrt(r2);
    const double mu = G * (mi + mj);
    const double rv = rx * vx + ry * vy + rz * vz;
    /* Eq. (50): t_ff = ( r^3 / (G (m_i+m_j)) )^(1/2) */
    const double t_ff = sqrt(r2 * r / mu);
    /* Eq. (53): d t_ff/dt = (3/2) (r.v)/r^2 t_ff */
    const double dt_ff = 1.5 * (rv / r2) * t_ff;
    const double q_ff = eta_in_q ? eta_ff * dt_ff : dt_ff;
    out[0] = oracle_sym_factor(q_ff) * (eta_ff * t_ff);
    if (v2 > 0.0) {                             /* v = 0: no fly-by candidate (reading 11) */
        /* Eq. (51): t_fb = r / v */
        const double t_fb = r / sqrt(v2);
        /* Eq. (54), two-body approximation: d t_fb/dt = (r.v)/r^2 [ 1 + G(m_i+m_j)/(v^2 r) ] t_fb */
        const double dt_fb = (rv / r2) * (1.0 + mu / (v2 * r)) * t_fb;
        const double q_fb = eta_in_q ? eta_fb * dt_fb : dt_fb;
        out[1] = oracle_sym_factor(q_fb) * (eta_fb * t_fb);
    }
}

/* bin = smallest k >= 0 with tau_pivot * 2^-k <= tau (include/frost.h restates this). */
static int32_t bin_of(double tau, double tau_pivot) {
    int32_t k = 0;
    double p = tau_pivot;
    if (!(tau > 0.0)) return 2000;
    while (p > tau && k < 2000) {
        p *= 0.5;
        ++k;
    }
    return k;
}

/* assign_timesteps: tau_i = min_j min( tau_ff_sym, tau_fb_sym ).
 * A level with a single particle gets tau = +inf. */
int oracle_timesteps(int n, int ld, const double *pos, const double *vel, const double *mass,
                     const int32_t *idx, int n_idx, double G, double eta_ff, double eta_fb,
                     int eta_in_q, double tau_pivot, double *out_tau, int32_t *out_bin) {
    if (n < 0 || ld < n || !pos || !vel || !mass || !out_tau) return ORACLE_EINVAL;
    if (!idx) n_idx = n;
#pragma omp parallel for schedule(dynamic, 16)
    for (int a = 0; a < n_idx; ++a) {
        const int i = pick(idx, a);
        const double xi[3] = {pos[i], pos[ld + i], pos[2 * ld + i]};
        const double vi[3] = {vel[i], vel[ld + i], vel[2 * ld + i]};
        double tau = INFINITY;
        for (int b = 0; b < n_idx; ++b) {
            const int j = pick(idx, b);
            if (j == i) continue;
            const double xj[3] = {pos[j], pos[ld + j], pos[2 * ld + j]};
            const double vj[3] = {vel[j], vel[ld + j], vel[2 * ld + j]};
            double c[2];
            oracle_pair_timestep(xi, vi, mass[i], xj, vj, mass[j], G, eta_ff, eta_fb, eta_in_q, c);
            if (c[0] < tau) tau = c[0];
            if (c[1] < tau) tau = c[1];
        }
        out_tau[i] = tau;
        if (out_bin) out_bin[i] = bin_of(tau, tau_pivot);
    }
    return ORACLE_OK;
}

/* Same definition, evaluated only for the sinks listed in `sel` (a subset of the level `idx`):
 * tau_i = min over ALL other members j of the level.  Lets the tests check sampled outputs of a
 * level too large for a full O(n^2) oracle pass. */
int oracle_timesteps_sampled(int n, int ld, const double *pos, const double *vel,
                             const double *mass, const int32_t *idx, int n_idx,
                             const int32_t *sel, int n_sel, double G, double eta_ff,
                             double eta_fb, int eta_in_q, double tau_pivot, double *out_tau,
                             int32_t *out_bin) {
    if (n < 0 || ld < n || !pos || !vel || !mass || !out_tau || !sel) return ORACLE_EINVAL;
    if (!idx) n_idx = n;
#pragma omp parallel for schedule(dynamic, 1)
    for (int a = 0; a < n_sel; ++a) {
        const int i = sel[a];
        const double xi[3] = {pos[i], pos[ld + i], pos[2 * ld + i]};
        const double vi[3] = {vel[i], vel[ld + i], vel[2 * ld + i]};
        double tau = INFINITY;
        for (int b = 0; b < n_idx; ++b) {
            const int j = pick(idx, b);
            if (j == i) continue;
            const double xj[3] = {pos[j], pos[ld + j], pos[2 * ld + j]};
            const double vj[3] = {vel[j], vel[ld + j], vel[2 * ld + j]};
            double c[2];
            oracle_pair_timestep(xi, vi, mass[i], xj, vj, mass[j], G, eta_ff, eta_fb, eta_in_q, c);
            if (c[0] < tau) tau = c[0];
            if (c[1] < tau) tau = c[1];
        }
        out_tau[i] = tau;
        if (out_bin) out_bin[i] = bin_of(tau, tau_pivot);
    }
    return ORACLE_OK;
}

/* ---------------------------------------------------------------------------------------------
 * O4.  kick and drift, Eq. (6); Alg. 2; kick_sf PAPER.md:596-597.
 *     kick : v_i <- v_i + c (a_i + kappa g_i)      (kappa = eps^2/48 forms a~ of Eq. 28, or 0)
 *     drift: x_i <- x_i + c v_i
 * ------------------------------------------------------------------------------------------- */
int oracle_kick(int n, int ld, double *vel, const double *acc, const double *grad,
                const int32_t *idx, int n_idx, double c, double kappa) {
    if (n < 0 || ld < n || !vel || !acc) return ORACLE_EINVAL;
    if (!idx) n_idx = n;
    for (int a = 0; a < n_idx; ++a) {
        const int i = pick(idx, a);
        for (int k = 0; k < 3; ++k) {
            double at = acc[k * ld + i];
            if (grad && kappa != 0.0) at = at + kappa * grad[k * ld + i];
            vel[k * ld + i] = vel[k * ld + i] + c * at;
        }
    }
    return ORACLE_OK;
}

int oracle_drift(int n, int ld, double *pos, const double *vel, const int32_t *idx, int n_idx,
                 double c) {
    if (n < 0 || ld < n || !pos || !vel) return ORACLE_EINVAL;
    if (!idx) n_idx = n;
    for (int a = 0; a < n_idx; ++a) {
        const int i = pick(idx, a);
        for (int k = 0; k < 3; ++k) pos[k * ld + i] = pos[k * ld + i] + c * vel[k * ld + i];
    }
    return ORACLE_OK;
}

/* ---------------------------------------------------------------------------------------------
 * O5.  FSI, Eq. (21); Alg. 2 PAPER.md:554:
 *   a <- newton; kick dt/6; drift dt/2; (a, g) <- newton + gradient; kick 2dt/3 with
 *   a~ = a + dt^2 g / 48 (Eq. 28; eps = this operator's own step, reading 7);
 *   drift dt/2; a <- newton; kick dt/6.   Empty set: no-op.
 * `acc`, `grad` are caller-provided scratch planes [3][ld].
 * ------------------------------------------------------------------------------------------- */
static int fsi_on_set(int n, int ld, double *pos, double *vel, const double *mass,
                      const int32_t *idx, int n_idx, double dt, double G, double eps2,
                      double *acc, double *grad, oracle_hhs_stats *st) {
    if (!idx) n_idx = n;
    if (n_idx == 0) return ORACLE_OK;
    const int64_t np = (int64_t)n_idx * n_idx;
    oracle_forces(n, ld, pos, mass, idx, n_idx, idx, n_idx, G, eps2, acc, NULL, ORACLE_ACC);
    oracle_kick(n, ld, vel, acc, NULL, idx, n_idx, dt / 6.0, 0.0);
    oracle_drift(n, ld, pos, vel, idx, n_idx, dt / 2.0);
    oracle_forces(n, ld, pos, mass, idx, n_idx, idx, n_idx, G, eps2, acc, grad, ORACLE_ACC | ORACLE_GRAD);
    oracle_kick(n, ld, vel, acc, grad, idx, n_idx, 2.0 * dt / 3.0, dt * dt / 48.0);
    oracle_drift(n, ld, pos, vel, idx, n_idx, dt / 2.0);
    oracle_forces(n, ld, pos, mass, idx, n_idx, idx, n_idx, G, eps2, acc, NULL, ORACLE_ACC);
    oracle_kick(n, ld, vel, acc, NULL, idx, n_idx, dt / 6.0, 0.0);
    if (st) {
        st->pairs_newton += 3 * np;
        st->pairs_gradient += np;
    }
    return ORACLE_OK;
}

int oracle_fsi_step(int n, int ld, double *pos, double *vel, const double *mass,
                    const int32_t *idx, int n_idx, double dt, double G, double eps2) {
    if (n < 0 || ld < n || !pos || !vel || !mass) return ORACLE_EINVAL;
    double *acc = (double *)calloc((size_t)3 * ld + 1, sizeof(double));
    double *grad = (double *)calloc((size_t)3 * ld + 1, sizeof(double));
    if (!acc || !grad) {
        free(acc);
        free(grad);
        return ORACLE_ENOMEM;
    }
    const int rc = fsi_on_set(n, ld, pos, vel, mass, idx, n_idx, dt, G, eps2, acc, grad, NULL);
    free(acc);
    free(grad);
    return rc;
}

/* ---------------------------------------------------------------------------------------------
 * O6s.  Spatial splitting of a fast level.  The paper only names it: "the further
 * spatial Hamiltonian splitting of the individual hierarchy levels into field stars, binaries and
 * multiple star systems" (primordial binaries are left to future work).
 * The definition used here (reading 24) applies the rule the paper already uses for
 * particles -- "whatever evolves slower than tau_pivot is integrated with tau_pivot" (Eq. 29,
 * PAPER.md:260-266) -- to PAIRS:
 *   * the symmetrised pair step of Eq. (49)-(54) is c_ij = min(tau_ff_sym, tau_fb_sym), and
 *     tau_i = min_j c_ij.  The pair (i, j) of one level's set is FAST iff
 *     c_ij < tau_pivot.  Slow particles (tau_i >= tau_pivot) are exactly those without a fast pair;
 *   * the fast pairs are the edges of a graph on F; its connected components C_1..C_m are mutually
 *     coupled by slow pairs only, so H_F = sum_c H_{C_c} + sum_{c<c'} U_{cc'} and the second sum is
 *     moved out of the recursion into the inter-level kick of Eq. (41): the kicked pair set becomes
 *         P = { (i, j) in set^2 : not both slow, not in the same component }
 *     (for m = 1 this is Alg. 3's S x F both ways), with the gradient force of Eq. (43)-(44)
 *     evaluated on P with the accelerations of P ("the interaction potential");
 *   * every component is then advanced on its own by hhs_fsi(C_c, tau/2), where the rule applies
 *     again.
 * ------------------------------------------------------------------------------------------- */

/* Component label of every member of `set`: the smallest member index of its component in the
 * graph whose edges are the fast pairs c_ij < tau_pivot; -1 for a member without a fast pair.
 * Plain relabelling to a fixed point over the explicit edge list.  label is indexed globally. */
int oracle_components(int n, int ld, const double *pos, const double *vel, const double *mass,
                      const int32_t *set, int n_set, double G, double eta_ff, double eta_fb,
                      int eta_in_q, double tau_pivot, int32_t *label) {
    if (n < 0 || ld < n || !pos || !vel || !mass || !label) return ORACLE_EINVAL;
    if (!set) n_set = n;
    size_t cap = 1024, ne = 0;
    int32_t *ei = (int32_t *)malloc(cap * sizeof(int32_t)), *ej = (int32_t *)malloc(cap * sizeof(int32_t));
    if (!ei || !ej) { free(ei); free(ej); return ORACLE_ENOMEM; }
    for (int a = 0; a < n_set; ++a) label[pick(set, a)] = -1;
    for (int a = 0; a < n_set; ++a) {
        const int i = pick(set, a);
        const double xi[3] = {pos[i], pos[ld + i], pos[2 * ld + i]};
        const double vi[3] = {vel[i], vel[ld + i], vel[2 * ld + i]};
        for (int b = a + 1; b < n_set; ++b) {
            const int j = pick(set, b);
            const double xj[3] = {pos[j], pos[ld + j], pos[2 * ld + j]};
            const double vj[3] = {vel[j], vel[ld + j], vel[2 * ld + j]};
            double c[2];
            oracle_pair_timestep(xi, vi, mass[i], xj, vj, mass[j], G, eta_ff, eta_fb, eta_in_q, c);
            if (c[0] < tau_pivot || c[1] < tau_pivot) {
                if (ne == cap) {
                    cap *= 2;
                    int32_t *ni = (int32_t *)realloc(ei, cap * sizeof(int32_t));
                    int32_t *nj = ni ? (int32_t *)realloc(ej, cap * sizeof(int32_t)) : NULL;
                    if (!ni || !nj) { free(ni ? ni : ei); free(nj ? nj : ej); return ORACLE_ENOMEM; }
                    ei = ni; ej = nj;
                }
                ei[ne] = i; ej[ne] = j; ++ne;
                if (label[i] < 0) label[i] = i;
                if (label[j] < 0) label[j] = j;
            }
        }
    }
    for (int changed = 1; changed;) {
        changed = 0;
        for (size_t k = 0; k < ne; ++k) {
            const int32_t li = label[ei[k]], lj = label[ej[k]];
            if (li < lj) { label[ej[k]] = li; changed = 1; }
            else if (lj < li) { label[ei[k]] = lj; changed = 1; }
        }
    }
    free(ei); free(ej);
    return ORACLE_OK;
}

/* Eq. (42) on the pair set P of O6s: a_i = G sum_{j in set, label_j != label_i} m_j x_ji / s^3.
 * (label is -1 for every slow particle, so slow-slow pairs and i = j drop out with the same test.) */
static void newton_masked(int ld, const double *pos, const double *mass, const int32_t *set,
                          int n_set, const int32_t *label, double G, double eps2, double *acc) {
#pragma omp parallel for schedule(dynamic, 16)
    for (int a = 0; a < n_set; ++a) {
        const int i = set[a];
        const ld_t xi = pos[i], yi = pos[ld + i], zi = pos[2 * ld + i];
        ld_t ax = 0, ay = 0, az = 0;
        for (int b = 0; b < n_set; ++b) {
            const int j = set[b];
            if (label[j] == label[i]) continue;
            const ld_t dx = (ld_t)pos[j] - xi;
            const ld_t dy = (ld_t)pos[ld + j] - yi;
            const ld_t dz = (ld_t)pos[2 * ld + j] - zi;
            const ld_t s2 = dx * dx + dy * dy + dz * dz + (ld_t)eps2;
            if (s2 > 0) {
                const ld_t s = sqrtl(s2);
                const ld_t w = (ld_t)mass[j] / (s2 * s);
                ax += w * dx;
                ay += w * dy;
                az += w * dz;
            }
        }
        acc[i] = (double)((ld_t)G * ax);
        acc[ld + i] = (double)((ld_t)G * ay);
        acc[2 * ld + i] = (double)((ld_t)G * az);
    }
}

/* Eq. (43)-(44) on the pair set P of O6s, with the accelerations of P. */
static void gradient_masked(int ld, const double *pos, const double *mass, const int32_t *set,
                            int n_set, const int32_t *label, double G, double eps2,
                            const double *acc, double *grad) {
#pragma omp parallel for schedule(dynamic, 16)
    for (int a = 0; a < n_set; ++a) {
        const int i = set[a];
        const ld_t xi = pos[i], yi = pos[ld + i], zi = pos[2 * ld + i];
        const ld_t axi = acc[i], ayi = acc[ld + i], azi = acc[2 * ld + i];
        ld_t gx = 0, gy = 0, gz = 0;
        for (int b = 0; b < n_set; ++b) {
            const int j = set[b];
            if (label[j] == label[i]) continue;
            const ld_t dx = (ld_t)pos[j] - xi;
            const ld_t dy = (ld_t)pos[ld + j] - yi;
            const ld_t dz = (ld_t)pos[2 * ld + j] - zi;
            const ld_t s2 = dx * dx + dy * dy + dz * dz + (ld_t)eps2;
            if (s2 > 0) {
                const ld_t dax = (ld_t)acc[j] - axi;
                const ld_t day = (ld_t)acc[ld + j] - ayi;
                const ld_t daz = (ld_t)acc[2 * ld + j] - azi;
                const ld_t s = sqrtl(s2);
                const ld_t s5 = s2 * s2 * s;
                const ld_t xa = dx * dax + dy * day + dz * daz;
                const ld_t w = (ld_t)mass[j] / s5;
                gx += w * (s2 * dax - 3 * xa * dx);
                gy += w * (s2 * day - 3 * xa * dy);
                gz += w * (s2 * daz - 3 * xa * dz);
            }
        }
        grad[i] = (double)(2 * (ld_t)G * gx);
        grad[ld + i] = (double)(2 * (ld_t)G * gy);
        grad[2 * ld + i] = (double)(2 * (ld_t)G * gz);
    }
}

/* The masked sweeps as a callable (for the pins): label indexed globally, -1 = slow. */
int oracle_forces_masked(int n, int ld, const double *pos, const double *mass, const int32_t *set,
                         int n_set, const int32_t *label, double G, double eps2, double *acc,
                         double *grad, int flags) {
    if (n < 0 || ld < n || !pos || !mass || !acc || !label || !set) return ORACLE_EINVAL;
    if ((flags & ORACLE_GRAD) && !grad) return ORACLE_EINVAL;
    if (flags & ORACLE_ACC) newton_masked(ld, pos, mass, set, n_set, label, G, eps2, acc);
    if (flags & ORACLE_GRAD) gradient_masked(ld, pos, mass, set, n_set, label, G, eps2, acc, grad);
    return ORACLE_OK;
}

/* ---------------------------------------------------------------------------------------------
 * O6k.  Two-body propagator for a component of exactly two particles (second half: the
 * paper lists "regularised integrators ..., Wisdom-Holman integrators and Kepler solvers" as the
 * modules a spatially split level can hand its few-body systems to; it defines none.
 * DESIGN.md reading 25).  A two-body component's Hamiltonian H_C is integrable: the centre of mass
 * moves uniformly and the relative vector r = x_2 - x_1, v = v_2 - v_1 follows the Kepler flow with
 * mu = G (m_1 + m_2), advanced here over dt by the universal-variable form of Kepler's equation
 * (valid for ellipses, parabolas and hyperbolas alike), with the Stumpff functions
 *     c_k(z) = sum_{n>=0} (-z)^n / (2n + k)!,   z = alpha s^2,   alpha = 2 mu / r_0 - v_0^2 :
 *     r_0 s c_1 + (r_0.v_0) s^2 c_2 + mu s^3 c_3 = dt                       (solved for s)
 *     f = 1 - (mu/r_0) s^2 c_2,   g = dt - mu s^3 c_3,
 *     r = r_0 c_0 + (r_0.v_0) s c_1 + mu s^2 c_2,
 *     f' = -(mu / (r r_0)) s c_1,   g' = 1 - (mu / r) s^2 c_2,
 *     r(dt) = f r_0 + g v_0,   v(dt) = f' r_0 + g' v_0.
 * The left-hand side is increasing in s (its derivative is the separation r > 0): the root is found
 * by Newton's method kept inside a bracket.  For a bound orbit whole periods are removed from dt first.
 * long double throughout (the oracle's accuracy margin); unsoftened only.
 * ------------------------------------------------------------------------------------------- */
static void stumpff(ld_t z, ld_t c[4]) {
    /* quarter the argument until the series converges fast, then the duplication formulas
     * c_0(4z) = 2 c_0(z)^2 - 1, c_1(4z) = c_0 c_1, c_2(4z) = c_1^2 / 2, c_3(4z) = (c_2 + c_0 c_3) / 4 */
    int k = 0;
    while (fabsl(z) > 0.1L) { z *= 0.25L; ++k; }
    ld_t c2 = 0, c3 = 0, t2 = 0.5L, t3 = 1.0L / 6.0L;
    for (int n = 0; n < 16; ++n) {            /* (-z)^n / (2n+2)!  and  (-z)^n / (2n+3)! */
        c2 += t2; c3 += t3;
        t2 *= -z / (ld_t)((2 * n + 3) * (2 * n + 4));
        t3 *= -z / (ld_t)((2 * n + 4) * (2 * n + 5));
    }
    ld_t c1 = 1.0L - z * c3, c0 = 1.0L - z * c2;
    for (; k > 0; --k) {
        c3 = 0.25L * (c2 + c0 * c3);
        c2 = 0.5L * c1 * c1;
        c1 = c0 * c1;
        c0 = 2.0L * c0 * c0 - 1.0L;
    }
    c[0] = c0; c[1] = c1; c[2] = c2; c[3] = c3;
}

/* relative position r and velocity v (in place) advanced by dt > 0 along the Kepler flow of mu */
int oracle_kepler_relative(double mu, double dt, double r[3], double v[3]) {
    if (!(mu > 0.0) || !(dt >= 0.0)) return ORACLE_EINVAL;
    const ld_t rx = r[0], ry = r[1], rz = r[2], vx = v[0], vy = v[1], vz = v[2];
    const ld_t r0 = sqrtl(rx * rx + ry * ry + rz * rz);
    if (!(r0 > 0)) return ORACLE_EINVAL;
    const ld_t v2 = vx * vx + vy * vy + vz * vz, u = rx * vx + ry * vy + rz * vz;
    const ld_t M = mu, alpha = 2 * M / r0 - v2;
    ld_t t = dt;
    if (alpha > 0) {                                   /* bound: remove whole periods */
        const ld_t P = 2 * 3.14159265358979323846264338327950288L * M / (alpha * sqrtl(alpha));
        t -= floorl(t / P) * P;
    }
    ld_t c[4], lo = 0, hi = t / r0, s;
    for (;;) {                                         /* bracket the root: F(lo) <= 0 < F(hi) */
        stumpff(alpha * hi * hi, c);
        if (r0 * hi * c[1] + u * hi * hi * c[2] + M * hi * hi * hi * c[3] - t > 0) break;
        lo = hi; hi = 2 * hi + 1e-300L;
    }
    s = 0.5L * (lo + hi);
    for (int it = 0; it < 200; ++it) {
        stumpff(alpha * s * s, c);
        const ld_t F = r0 * s * c[1] + u * s * s * c[2] + M * s * s * s * c[3] - t;
        const ld_t dF = r0 * c[0] + u * s * c[1] + M * s * s * c[2];
        if (F == 0) break;
        if (F > 0) hi = s; else lo = s;
        ld_t sn = s - F / dF;
        if (!(sn >= lo && sn <= hi)) sn = 0.5L * (lo + hi);
        if (fabsl(sn - s) <= 1e-19L * fabsl(s)) { s = sn; break; }
        s = sn;
    }
    stumpff(alpha * s * s, c);
    const ld_t rr = r0 * c[0] + u * s * c[1] + M * s * s * c[2];
    const ld_t f = 1 - (M / r0) * s * s * c[2], g = t - M * s * s * s * c[3];
    const ld_t fd = -(M / (rr * r0)) * s * c[1], gd = 1 - (M / rr) * s * s * c[2];
    r[0] = (double)(f * rx + g * vx); r[1] = (double)(f * ry + g * vy); r[2] = (double)(f * rz + g * vz);
    v[0] = (double)(fd * rx + gd * vx); v[1] = (double)(fd * ry + gd * vy); v[2] = (double)(fd * rz + gd * vz);
    return ORACLE_OK;
}

/* particles i and j advanced by dt along their exact two-body motion (centre of mass uniform) */
static int kepler_pair(int ld, double *pos, double *vel, const double *mass, int i, int j, double G, double dt) {
    const ld_t mi = mass[i], mj = mass[j], mt = mi + mj;
    ld_t X[3], V[3];
    double r[3], v[3];
    for (int k = 0; k < 3; ++k) {
        X[k] = (mi * pos[k * ld + i] + mj * pos[k * ld + j]) / mt;
        V[k] = (mi * vel[k * ld + i] + mj * vel[k * ld + j]) / mt;
        r[k] = pos[k * ld + j] - pos[k * ld + i];
        v[k] = vel[k * ld + j] - vel[k * ld + i];
    }
    const int rc = oracle_kepler_relative(G * (mass[i] + mass[j]), dt, r, v);
    if (rc != ORACLE_OK) return rc;
    for (int k = 0; k < 3; ++k) {
        const ld_t Xk = X[k] + V[k] * (ld_t)dt;
        pos[k * ld + i] = (double)(Xk - (mj / mt) * r[k]); pos[k * ld + j] = (double)(Xk + (mi / mt) * r[k]);
        vel[k * ld + i] = (double)(V[k] - (mj / mt) * v[k]); vel[k * ld + j] = (double)(V[k] + (mi / mt) * v[k]);
    }
    return ORACLE_OK;
}

/* ---------------------------------------------------------------------------------------------
 * O6.  HHS-FSI, Eq. (41); Alg. 3, line by line.
 * `frozen_level` (may be NULL): if given, particle i is slow at the first level k with
 * k >= frozen_level[i] instead of by its time-step -- the "frozen partition" used only by the
 * convergence-order pin (with adaptive steps the partition changes with tau and the error is no
 * longer a smooth function of the step).
 * ------------------------------------------------------------------------------------------- */
typedef struct {
    int n, ld;
    double *pos, *vel;
    const double *mass;
    double G, eps2, eta_ff, eta_fb;
    int eta_in_q, max_depth;
    const int32_t *frozen_level;
    int split_max;                     /* O6s: entries with |set| <= split_max split F into components */
    int kepler;                        /* O6k: two-body components of a split entry follow their Kepler orbit */
    const int32_t *frozen_comp;        /* with frozen_level: the component of particle i (any labels) */
    double *acc, *grad, *tau;
    int32_t *label;
    oracle_hhs_stats *st;
} hhs_env;

static int cmp_label_then_index(const void *pa, const void *pb) {
    const int32_t *a = (const int32_t *)pa, *b = (const int32_t *)pb;      /* {label, index} */
    if (a[0] != b[0]) return a[0] < b[0] ? -1 : 1;
    return a[1] < b[1] ? -1 : (a[1] > b[1] ? 1 : 0);
}

static int hhs_recursive(hhs_env *e, const int32_t *set, int n_set, double tau_pivot, int level) {
    if (n_set == 0) return ORACLE_OK;                          /* "if set != empty" */
    if (level >= e->max_depth || level >= ORACLE_MAX_LEVELS) return ORACLE_EDEPTH;
    const int n = e->n, ld = e->ld;
    /* {tau_i} <- assign_timesteps(set): only this level's members */
    oracle_timesteps(n, ld, e->pos, e->vel, e->mass, set, n_set, e->G, e->eta_ff, e->eta_fb,
                     e->eta_in_q, tau_pivot, e->tau, NULL);
    /* partition (Eq. 29): slow iff tau_i >= tau_pivot; stable order */
    int32_t *S = (int32_t *)malloc(sizeof(int32_t) * (size_t)(n_set + 1));
    int32_t *F = (int32_t *)malloc(sizeof(int32_t) * (size_t)(n_set + 1));
    int32_t *key = (int32_t *)malloc(sizeof(int32_t) * 2 * (size_t)(n_set + 1));
    int32_t *cstart = (int32_t *)malloc(sizeof(int32_t) * (size_t)(n_set + 2));
    if (!S || !F || !key || !cstart) {
        free(S); free(F); free(key); free(cstart);
        return ORACLE_ENOMEM;
    }
    int nS = 0, nF = 0;
    for (int a = 0; a < n_set; ++a) {
        const int i = set[a];
        int slow;
        if (e->frozen_level) slow = (level >= e->frozen_level[i]);
        else slow = (e->tau[i] >= tau_pivot);
        if (slow) S[nS++] = i;
        else F[nF++] = i;
    }
    /* O6s: the components of F (members ascending inside a component, components by their smallest
     * member); one component = F itself when the entry is not split */
    int m = nF > 0 ? 1 : 0;
    cstart[0] = 0; cstart[1] = nF;
    if (e->split_max > 0 && n_set <= e->split_max && nF > 0) {
        if (e->frozen_level) {
            for (int a = 0; a < nS; ++a) e->label[S[a]] = -1;
            for (int a = 0; a < nF; ++a) e->label[F[a]] = e->frozen_comp ? e->frozen_comp[F[a]] : 0;
        } else {
            oracle_components(n, ld, e->pos, e->vel, e->mass, set, n_set, e->G, e->eta_ff, e->eta_fb,
                              e->eta_in_q, tau_pivot, e->label);
        }
        for (int a = 0; a < nF; ++a) { key[2 * a] = e->label[F[a]]; key[2 * a + 1] = F[a]; }
        qsort(key, (size_t)nF, 2 * sizeof(int32_t), cmp_label_then_index);
        m = 0;
        for (int a = 0; a < nF; ++a) {
            F[a] = key[2 * a + 1];
            if (a == 0 || key[2 * a] != key[2 * a - 2]) cstart[m++] = a;
        }
        cstart[m] = nF;
    }
    oracle_hhs_stats *st = e->st;
    if (st) {
        if (level > st->depth) st->depth = level;
        st->entries[level] += 1;
        st->n_slow[level] += nS;
        st->n_fast[level] += nF;
        st->n_comp[level] += m;
        st->pairs_timestep += (int64_t)n_set * n_set;
    }
    /* ordered pairs of P: everything but slow-slow and same-component pairs (m <= 1: 2 |S| |F|) */
    int64_t cross = (int64_t)n_set * n_set - (int64_t)nS * nS;
    for (int c = 0; c < m; ++c) cross -= (int64_t)(cstart[c + 1] - cstart[c]) * (cstart[c + 1] - cstart[c]);
    int rc = ORACLE_OK;
    const double h = 0.5 * tau_pivot;
    const double kap = tau_pivot * tau_pivot / 48.0;
    /* acc_sf_newton (Eq. 42) on P; kick_sf by tau/6 */
    if (m <= 1) oracle_forces(n, ld, e->pos, e->mass, S, nS, F, nF, e->G, e->eps2, e->acc, NULL, ORACLE_ACC | ORACLE_MUTUAL);
    else newton_masked(ld, e->pos, e->mass, set, n_set, e->label, e->G, e->eps2, e->acc);
    oracle_kick(n, ld, e->vel, e->acc, NULL, S, nS, tau_pivot / 6.0, 0.0);
    oracle_kick(n, ld, e->vel, e->acc, NULL, F, nF, tau_pivot / 6.0, 0.0);
    /* fsi(S, tau/2); hhs_fsi(C_c, tau/2) for every component (Alg. 3: hhs_fsi(F, tau/2)) */
    rc = fsi_on_set(n, ld, e->pos, e->vel, e->mass, S, nS, h, e->G, e->eps2, e->acc, e->grad, st);
    const int kep = e->kepler && e->split_max > 0 && n_set <= e->split_max && e->eps2 == 0.0;
    for (int c = 0; c < m && rc == ORACLE_OK; ++c) {
        if (kep && cstart[c + 1] - cstart[c] == 2) {
            rc = kepler_pair(ld, e->pos, e->vel, e->mass, F[cstart[c]], F[cstart[c] + 1], e->G, h);
            if (st) st->n_kepler += 1;
        } else rc = hhs_recursive(e, F + cstart[c], cstart[c + 1] - cstart[c], h, level + 1);
    }
    if (rc == ORACLE_OK) {
        /* acc_sf_gradient (Eq. 43-44) with the inter-level a of Eq. 42; kick_sf by 2 tau/3 with
         * a~ = a + tau_pivot^2 g / 48 (eps = this level's step, reading 7).  The recursion
         * overwrote the labels of F's members: restore this entry's before the masked sweeps. */
        if (m > 1) {
            for (int c = 0; c < m; ++c)
                for (int a = cstart[c]; a < cstart[c + 1]; ++a) e->label[F[a]] = c;
            for (int a = 0; a < nS; ++a) e->label[S[a]] = -1;
            newton_masked(ld, e->pos, e->mass, set, n_set, e->label, e->G, e->eps2, e->acc);
            gradient_masked(ld, e->pos, e->mass, set, n_set, e->label, e->G, e->eps2, e->acc, e->grad);
        } else {
            oracle_forces(n, ld, e->pos, e->mass, S, nS, F, nF, e->G, e->eps2, e->acc, e->grad,
                          ORACLE_ACC | ORACLE_GRAD | ORACLE_MUTUAL);
        }
        oracle_kick(n, ld, e->vel, e->acc, e->grad, S, nS, 2.0 * tau_pivot / 3.0, kap);
        oracle_kick(n, ld, e->vel, e->acc, e->grad, F, nF, 2.0 * tau_pivot / 3.0, kap);
        /* hhs_fsi(C_c, tau/2); fsi(S, tau/2) */
        for (int c = 0; c < m && rc == ORACLE_OK; ++c) {
            if (kep && cstart[c + 1] - cstart[c] == 2) {
                rc = kepler_pair(ld, e->pos, e->vel, e->mass, F[cstart[c]], F[cstart[c] + 1], e->G, h);
                if (st) st->n_kepler += 1;
            } else rc = hhs_recursive(e, F + cstart[c], cstart[c + 1] - cstart[c], h, level + 1);
        }
    }
    if (rc == ORACLE_OK)
        rc = fsi_on_set(n, ld, e->pos, e->vel, e->mass, S, nS, h, e->G, e->eps2, e->acc, e->grad, st);
    if (rc == ORACLE_OK) {
        /* acc_sf_newton on P; kick_sf by tau/6 */
        if (m > 1) {
            for (int c = 0; c < m; ++c)
                for (int a = cstart[c]; a < cstart[c + 1]; ++a) e->label[F[a]] = c;
            for (int a = 0; a < nS; ++a) e->label[S[a]] = -1;
            newton_masked(ld, e->pos, e->mass, set, n_set, e->label, e->G, e->eps2, e->acc);
        } else {
            oracle_forces(n, ld, e->pos, e->mass, S, nS, F, nF, e->G, e->eps2, e->acc, NULL, ORACLE_ACC | ORACLE_MUTUAL);
        }
        oracle_kick(n, ld, e->vel, e->acc, NULL, S, nS, tau_pivot / 6.0, 0.0);
        oracle_kick(n, ld, e->vel, e->acc, NULL, F, nF, tau_pivot / 6.0, 0.0);
        if (st) {
            st->pairs_newton += 3 * cross;
            st->pairs_gradient += cross;
        }
    }
    free(S); free(F); free(key); free(cstart);
    return rc;
}

/* split_max = 0: Alg. 3 as printed.  split_max > 0: O6s on every entry with |set| <= split_max. */
int oracle_hhs_split_step(int n, int ld, double *pos, double *vel, const double *mass, double dt_top,
                          double G, double eps2, double eta_ff, double eta_fb, int eta_in_q,
                          int max_depth, const int32_t *frozen_level, int split_max,
                          const int32_t *frozen_comp, int kepler, oracle_hhs_stats *stats) {
    if (n < 0 || ld < n || !pos || !vel || !mass || !(dt_top > 0.0) || split_max < 0) return ORACLE_EINVAL;
    hhs_env e;
    e.n = n; e.ld = ld; e.pos = pos; e.vel = vel; e.mass = mass;
    e.G = G; e.eps2 = eps2; e.eta_ff = eta_ff; e.eta_fb = eta_fb;
    e.eta_in_q = eta_in_q; e.max_depth = max_depth; e.frozen_level = frozen_level;
    e.split_max = split_max; e.frozen_comp = frozen_comp; e.kepler = kepler;
    e.acc = (double *)calloc((size_t)3 * ld + 1, sizeof(double));
    e.grad = (double *)calloc((size_t)3 * ld + 1, sizeof(double));
    e.tau = (double *)calloc((size_t)ld + 1, sizeof(double));
    e.label = (int32_t *)calloc((size_t)ld + 1, sizeof(int32_t));
    int32_t *all = (int32_t *)malloc(sizeof(int32_t) * (size_t)(n + 1));
    if (stats) memset(stats, 0, sizeof(*stats));
    e.st = stats;
    int rc = ORACLE_ENOMEM;
    if (e.acc && e.grad && e.tau && e.label && all) {
        for (int i = 0; i < n; ++i) all[i] = i;
        rc = hhs_recursive(&e, all, n, dt_top, 0);
    }
    free(e.acc); free(e.grad); free(e.tau); free(e.label); free(all);
    return rc;
}

int oracle_hhs_step(int n, int ld, double *pos, double *vel, const double *mass, double dt_top,
                    double G, double eps2, double eta_ff, double eta_fb, int eta_in_q,
                    int max_depth, const int32_t *frozen_level, oracle_hhs_stats *stats) {
    return oracle_hhs_split_step(n, ld, pos, vel, mass, dt_top, G, eps2, eta_ff, eta_fb, eta_in_q,
                                 max_depth, frozen_level, 0, NULL, 0, stats);
}

/* ---------------------------------------------------------------------------------------------
 * O7.  Diagnostics (Eq. 23):
 *   out[0] = T = 1/2 sum m v^2,  out[1] = U = -G sum_{i<j} m_i m_j / s_ij,
 *   out[2..4] = P = sum m v,  out[5..7] = L = sum m x cross v.
 * ------------------------------------------------------------------------------------------- */
int oracle_diagnostics(int n, int ld, const double *pos, const double *vel, const double *mass,
                       double G, double eps2, double *out) {
    if (n < 0 || ld < n || !pos || !vel || !mass || !out) return ORACLE_EINVAL;
    ld_t T = 0, U = 0, P[3] = {0, 0, 0}, L[3] = {0, 0, 0};
    for (int i = 0; i < n; ++i) {
        const ld_t m = mass[i];
        const ld_t x = pos[i], y = pos[ld + i], z = pos[2 * ld + i];
        const ld_t vx = vel[i], vy = vel[ld + i], vz = vel[2 * ld + i];
        T += 0.5L * m * (vx * vx + vy * vy + vz * vz);
        P[0] += m * vx; P[1] += m * vy; P[2] += m * vz;
        L[0] += m * (y * vz - z * vy);
        L[1] += m * (z * vx - x * vz);
        L[2] += m * (x * vy - y * vx);
    }
#pragma omp parallel for schedule(dynamic, 16) reduction(+ : U)
    for (int i = 0; i < n; ++i) {
        ld_t u = 0;
        for (int j = i + 1; j < n; ++j) {
            const ld_t dx = (ld_t)pos[j] - pos[i];
            const ld_t dy = (ld_t)pos[ld + j] - pos[ld + i];
            const ld_t dz = (ld_t)pos[2 * ld + j] - pos[2 * ld + i];
            const ld_t s2 = dx * dx + dy * dy + dz * dz + (ld_t)eps2;
            if (s2 > 0) u += (ld_t)mass[j] / sqrtl(s2);
        }
        U += -(ld_t)G * (ld_t)mass[i] * u;
    }
    out[0] = (double)T; out[1] = (double)U;
    for (int k = 0; k < 3; ++k) { out[2 + k] = (double)P[k]; out[5 + k] = (double)L[k]; }
    return ORACLE_OK;
}
