/*
 * frost.h -- C-ABI of the B200-native HHS-FSI hot path (libfrost_b200.so).
 *
 * What is behind it: the fp64 O(N_sink x N_source) direct-summation sweeps of the hierarchical
 * fourth-order forward symplectic integrator of Rantala, Naab & Springel (FROST, arXiv 2011.14984;
 * citations below are /root/reference/PAPER.md line numbers) written as CUDA kernels for sm_100a.
 * There is no CPU fallback: every entry point fails with FROST_ECUDA if no device is usable.
 *
 * Conventions for every call
 *   - Returns 0 (FROST_OK) or a negative FROST_E* code; frost_strerror() names it.  No exceptions,
 *     no aborts, nothing is printed.
 *   - Unless a parameter is marked HOST, pointers are DEVICE pointers owned by the caller (e.g.
 *     torch tensors).  The library never frees or reallocates caller memory; it owns only scratch
 *     inside the context.  Work is enqueued on the context's stream and the call returns without
 *     synchronising, except where a HOST result is returned (noted per call).
 *   - Particle vectors (pos, vel, acc, grad) are three fp64 SoA planes: component c of particle i
 *     is p[c*ld + i], 0 <= i < n <= ld.  mass, tau are fp64[n]; bins and index arrays are int32.
 *   - Every call makes the context's device current while it runs and restores the caller's current
 *     device before it returns.
 *   - Index arrays list distinct particle indices in [0,n); NULL means "all particles 0..n-1"
 *     (the count argument is then ignored).  Partial sums are formed per source slice / tile pair and
 *     added in a fixed order (no floating-point atomics), so results are bitwise reproducible run
 *     to run for a fixed tuning.
 *   - A pair with |x_j-x_i|^2 + eps2 == 0 (the self pair, or two coincident unsoftened particles)
 *     contributes nothing anywhere (reading 11).
 */
#ifndef FROST_H
#define FROST_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define FROST_OK 0
#define FROST_EINVAL (-1)     /* bad argument (NULL where data is required, n > ld, bad flags) */
#define FROST_ECUDA (-2)      /* a CUDA call failed; frost_last_cuda_error() has the cudaError_t */
#define FROST_ENOMEM (-3)     /* scratch allocation failed */
#define FROST_EDEPTH (-4)     /* frost_hhs_step recursed beyond max_depth */
#define FROST_ENONFINITE (-5) /* reserved: non-finite input detected (debug scans) */
#define FROST_ETOOBIG (-6)    /* frost_acc_noalloc: n exceeds FROST_NOALLOC_MAX_N (its scratch is a fixed array) */
#define FROST_ELIMIT (-7)     /* frost_hhs_step with frost_set_split: one entry has more than 64 components of
                                 more than 1024 particles (a fixed list; no allocation failed) */

/* flags of frost_forces */
#define FROST_ACC 1    /* compute Newtonian accelerations of the sinks */
#define FROST_GRAD 2   /* compute gradient accelerations of the sinks */
#define FROST_MUTUAL 4 /* also the reverse direction (sources as sinks): acc_sf_* of Alg. 3 */
#define FROST_ACCUMULATE 8 /* add the sums to out_acc / out_grad instead of overwriting them */

#define FROST_MAX_LEVELS 64

typedef struct frost_ctx frost_ctx;

/* HOST struct filled by frost_hhs_step (Alg. 3 bookkeeping). */
typedef struct {
    int32_t depth;                      /* deepest hierarchy level entered with a non-empty set */
    int32_t reserved;
    int64_t entries[FROST_MAX_LEVELS];  /* non-empty hhs_fsi entries at level k */
    int64_t n_slow[FROST_MAX_LEVELS];   /* sum of |S| over those entries */
    int64_t n_fast[FROST_MAX_LEVELS];   /* sum of |F| over those entries */
    int64_t pairs_newton;               /* ordered pairs swept by the Newton kernel */
    int64_t pairs_gradient;             /* ordered pairs swept by the gradient kernel */
    int64_t pairs_timestep;             /* ordered pairs swept by the time-step kernel */
    int64_t n_comp[FROST_MAX_LEVELS];   /* sum over those entries of the fast components recursed into
                                           (Alg. 3 as printed: 1 per entry with |F| > 0; frost_set_split) */
    int64_t n_kepler;                   /* two-body components advanced by the Kepler propagator (frost_set_kepler) */
} frost_hhs_stats;

/* allocate_memory / free_memory of Alg. 4: creates a context bound to CUDA
 * device `device` and to `stream` (a cudaStream_t passed as void*; NULL = the legacy default
 * stream).  Scratch grows on demand and is released by frost_destroy.  *out is HOST. */
int frost_create(frost_ctx **out, int device, void *stream);
int frost_destroy(frost_ctx *ctx);

/* Parameter file of Alg. 4: Newton's constant G (Eq. 23), squared Plummer softening
 * eps2 = eps_p^2, accuracy parameters eta_ff, eta_fb (Eq. 50-51) and
 * the recursion limit of frost_hhs_step.  Defaults: G=1, eps2=0, eta_ff=eta_fb=0.2
 * (PAPER.md:682), max_depth=64. */
int frost_set_params(frost_ctx *ctx, double G, double eps2, double eta_ff, double eta_fb,
                     int max_depth);

/* compute_acc_newton / compute_acc_gradient (Alg. 1-2) when sinks ==
 * sources; one direction of acc_sf_newton / acc_sf_gradient (Alg. 3) otherwise.
 *   FROST_ACC : out_acc[i] <- G sum_{j in J} m_j x_ji / s_ij^3 for each sink i        (Eq. 24, 42)
 *   FROST_GRAD: out_grad[i] <- 2G sum_{j in J} m_j s^-5 (s^2 a_ji - 3 (x_ji.a_ji) x_ji),
 *               a_ji = out_acc[j] - out_acc[i]                                  (Eq. 27, 43, 44)
 *               so out_acc must hold, for every sink and source, the acceleration generated by
 *               the same pair set -- which FROST_ACC of the same call provides for the sinks
 *               (and, under FROST_MUTUAL, for the sources).
 *   FROST_MUTUAL: sweep both directions I<-J and J<-I (all accelerations first, then all
 *               gradients); both index arrays must then be non-NULL or both NULL.
 *   FROST_ACCUMULATE: the sums of this call are ADDED to out_acc (FROST_ACC) or out_grad
 *               (FROST_GRAD) of the swept sinks, so that a pair set can be swept in pieces -- e.g.
 *               "active subset A against everything" as self(A) + mutual(A, rest),
 *               both of which the pair-symmetric kernels serve; FROST_ACC | FROST_GRAD in one
 *               accumulating call is FROST_EINVAL (the gradient needs the total accelerations).
 *   s_ij^2 = |x_j - x_i|^2 + eps2.  `vel` is not read (reserved; may be NULL).  Entries of out_*
 *   outside the swept sink sets are untouched.  out_grad may be NULL without FROST_GRAD.
 *   The self case is recognised by POINTER: sink_idx == source_idx (both NULL, or the same array)
 *   with equal counts.  Two different arrays with equal contents give the same sums through the
 *   one-sided kernels (each ordered pair evaluated on its own: ~1.6x the arithmetic of the
 *   pair-symmetric self sweep).
 *   Accuracy: a_i to ~1e-15 |a_i|; g_i to ~2^-53 x the magnitude sum of Eq. 27's terms, which for
 *   a particle that sees a hard binary from afar can exceed 1e-10 |g_i| (the definition itself is
 *   that sensitive to the last bit of out_acc; reading 22).
 *   Asynchronous. */
int frost_forces(frost_ctx *ctx, int n, int ld, const double *pos, const double *vel,
                 const double *mass, const int32_t *sink_idx, int n_sink,
                 const int32_t *source_idx, int n_source, double *out_acc, double *out_grad,
                 int flags);

/* Same operation on HOST buffers (pageable or pinned): copies pos and mass to device scratch --
 * and out_acc / out_grad too, unless every particle is a sink of an overwriting sweep (sink_idx
 * NULL, ld == n, no FROST_ACCUMULATE; out_acc additionally only if FROST_ACC is set), in which
 * case they are pure outputs --, sweeps, copies out_acc / out_grad back, and synchronises the
 * stream.  This is the end-to-end path bench.py's "e2e" times; the
 * host-device copy per call is exactly what Alg. 1 does.  Index arrays are
 * HOST too. */
int frost_forces_host(frost_ctx *ctx, int n, int ld, const double *pos, const double *mass,
                      const int32_t *sink_idx, int n_sink, const int32_t *source_idx,
                      int n_source, double *out_acc, double *out_grad, int flags);

/* assign_timesteps (Alg. 3) over ONE hierarchy level (sinks = sources = idx,
 * PAPER.md:448):  out_tau[i] = min_{j != i} min( s(q_ff) eta_ff t_ff , s(q_fb) eta_fb t_fb ) with
 * t_ff, t_fb of Eq. 50-51, their derivatives Eq. 53-54, q = eta * dt/dt (reading 9) and
 * the harmonic factor s(q) of Eq. 49.  A level of one particle gets +inf.  The time-step criterion
 * is never softened (reading 14).  out_bin (nullable): smallest k >= 0 with
 * tau_pivot * 2^-k <= out_tau[i].  Asynchronous. */
int frost_timesteps(frost_ctx *ctx, int n, int ld, const double *pos, const double *vel,
                    const double *mass, const int32_t *idx, int n_idx, double tau_pivot,
                    double *out_tau, int32_t *out_bin);

/* partition (Eq. 29): stable split of idx (NULL = 0..n-1) into
 * out_slow (tau[i] >= tau_pivot) followed by out_fast (tau[i] < tau_pivot), both int32 arrays of
 * capacity n_idx.  counts is HOST int32[2] = {|S|, |F|}; the call synchronises the stream. */
int frost_partition(frost_ctx *ctx, int n, const double *tau, const int32_t *idx, int n_idx,
                    double tau_pivot, int32_t *out_slow, int32_t *out_fast, int32_t *counts);

/* kick / kick_sf (Eq. 6): v_i += c * (a_i + kappa * g_i) for i in idx.
 * kappa = eps^2/48 forms the modified acceleration of Eq. 28; grad may be NULL iff kappa == 0.
 * Asynchronous. */
int frost_kick(frost_ctx *ctx, int n, int ld, double *vel, const double *acc, const double *grad,
               const int32_t *idx, int n_idx, double c, double kappa);

/* drift (Eq. 6): x_i += c * v_i for i in idx.  Asynchronous. */
int frost_drift(frost_ctx *ctx, int n, int ld, double *pos, const double *vel,
                const int32_t *idx, int n_idx, double c);

/* fsi (Eq. 21; Alg. 2) on the particles of idx: newton, kick dt/6, drift dt/2,
 * newton+gradient, kick 2dt/3 with kappa = dt^2/48, drift dt/2, newton, kick dt/6.
 * Asynchronous. */
int frost_fsi_step(frost_ctx *ctx, int n, int ld, double *pos, double *vel, const double *mass,
                   const int32_t *idx, int n_idx, double dt);

/* n_steps consecutive fsi steps with the same dt on the same set ("FSI on a single level", the
 * comparison runs of PAPER.md:658-674).  Bitwise the same result as n_steps calls of
 * frost_fsi_step, but the trailing Newton sweep of a step doubles as the leading sweep of the next
 * (same positions): 3 all-pairs sweeps per step instead of 4; sets of <= 1024 particles take all
 * steps inside one launch of the device-resident kernel.  Asynchronous. */
int frost_fsi_steps(frost_ctx *ctx, int n, int ld, double *pos, double *vel, const double *mass,
                    const int32_t *idx, int n_idx, double dt, int n_steps);

/* hhs_fsi (Eq. 41; Alg. 3) on all n particles with first pivot step dt_top
 * (Alg. 4).  Level sets of more than 1024 particles are recursed from the host (one
 * count read-back per entry); a set of <= 1024 particles is handed, with its whole subtree, to the
 * device-resident subtree kernel (a thread-block cluster, a CTA, four warps or one warp by set size;
 * see frost_set_tuning).  Synchronises; stats (HOST, nullable) receives the bookkeeping. */
int frost_hhs_step(frost_ctx *ctx, int n, int ld, double *pos, double *vel, const double *mass,
                   double dt_top, frost_hhs_stats *stats);

/* Gather / pack (step 1 of the path): out[k] = {x, y, z, m} of particle idx[k] as 32-byte records,
 * k < n_idx; records n_idx..n_pad-1 are zero.  Exposed so the HBM-bound staging kernel can be timed
 * and tested on its own; the sweeps call the same kernel internally.  Asynchronous. */
int frost_gather_pack(frost_ctx *ctx, int n, int ld, const double *pos, const double *mass,
                      const int32_t *idx, int n_idx, int n_pad, double *out_records);

/* Conserved quantities (Eq. 23; the on-the-fly diagnostics of PAPER.md:632-636,
 * 644) of all n particles, computed on the device:
 *   out8 (HOST double[8]) = { T = sum m v^2/2, U = -G sum_{i<j} m_i m_j / s_ij, P_x, P_y, P_z,
 *                             L_x, L_y, L_z },  s_ij^2 = |x_j - x_i|^2 + eps2; a pair at exactly one point is skipped.
 * U comes from a pair-symmetric all-pairs sweep of the specific potential phi_i = -G sum_j m_j/s_ij
 * (U = sum m_i phi_i / 2); out_phi (DEVICE double[n], nullable) receives phi.  The O(N) sums are
 * compensated and added in a fixed order.  Synchronises the stream. */
int frost_diagnostics(frost_ctx *ctx, int n, int ld, const double *pos, const double *vel,
                      const double *mass, double *out_phi, double *out8);

/* Bookkeeping (HOST results, no device work). */
int64_t frost_launch_count(const frost_ctx *ctx); /* kernels launched through this context (side streams included) */
int frost_last_cuda_error(const frost_ctx *ctx);  /* last cudaError_t seen, 0 if none */
const char *frost_strerror(int status);
const char *frost_version(void);

/* Tuning knob used by tests and bench.py to force a kernel variant: sinks per thread (1, 2 or 4;
 * 0 = auto), the number of source slices (0 = auto), and the largest set handed to the
 * device-resident subtree kernel by frost_hhs_step / frost_fsi_step (-1 = auto = 1024, 0 = never).
 * subtree_one_cta: 0 = sets of >= 192 particles run on a thread-block cluster of 16 CTAs that hold
 * replicas of the set and share the large sweeps out by sinks over distributed shared memory,
 * 1 = always a single CTA.  Results are deterministic for a fixed setting. */
int frost_set_tuning(frost_ctx *ctx, int sinks_per_thread, int source_slices, int small_set_max,
                     int subtree_one_cta);

/* Pair-symmetric sweeps.  Every per-pair quantity of Eq. 24, 27 and 49-54 is even or odd under
 * i <-> j (the gradient force obeys Newton's third law as the Newtonian one
 * does), so for a self sweep (sinks == sources) and for a FROST_MUTUAL sweep one evaluation of a
 * pair can update both of its particles.  mode 0 (default): used when the sets are large enough to
 * fill the GPU with tile pairs (self force sweeps from ~6000 particles, time-step sweeps from 4096,
 * mutual sweeps from ~1000 x 1000); time-step sweeps of >= 32768 particles additionally run in
 * Morton order with exact block pruning (csrc/frost_tau.cu: pairs that provably cannot lower a
 * minimum are discarded; bitwise the same minima).  mode 1: never (always the one-sided sweeps);
 * 2: symmetric whenever applicable (tests); 3 / 4 / 5 (tests): as 2 with the time-step sweep
 * unpruned / through the pruning machinery with pruning off / pruned at any size.
 * The sums a particle collects as the streamed ("B") partner of a pair leave the CTA once per tile
 * pair; the B list is therefore swept in bands so that this scratch stays below scratch_mib MiB
 * whatever N is (0 = default 4096; one band = one sweep launch + one reduction).  Either way sums
 * are added in a fixed order: results are bitwise reproducible for a fixed setting, and the two
 * kinds of sweep agree to rounding. */
int frost_set_symmetric(frost_ctx *ctx, int mode, int scratch_mib);

/* Multi-GPU share of the pair-symmetric sweeps (one process and one context per GPU).  After
 * frost_set_shard(ctx, rank, world) a symmetric self or mutual sweep of frost_forces evaluates only
 * the tile pairs whose register-resident ("A") tile index is congruent to rank modulo world -- a
 * balanced 1/world of the pairs -- and writes PARTIAL sums for every particle of the swept sets:
 * the caller adds out_acc (then, in a second call, out_grad) over the ranks (one all-reduce of
 * 24 B per particle).  Because the gradient needs the complete accelerations,
 * FROST_ACC | FROST_GRAD in one call is FROST_EINVAL while world > 1.
 * A sweep that the one-sided kernels serve (subset <- all, small sets, frost_set_symmetric mode 1)
 * honours the same contract: each direction sweeps this rank's contiguous block of its sink list
 * and writes zeros for the other sinks of the list, so the sum over ranks is complete whichever
 * kernels ran (and each sink's sum is then bitwise the unsharded one).  While world > 1,
 * FROST_ACCUMULATE is FROST_EINVAL too (the old content would be added once per rank), and
 * frost_fsi_step(s) / frost_hhs_step return FROST_EINVAL before touching anything: only
 * frost_forces is shard-aware; time steps and diagnostics are not sharded.  Default: rank 0 of 1. */
int frost_set_shard(frost_ctx *ctx, int rank, int world);

/* fsi(S, tau/2) and hhs_fsi(F, tau/2) of one hierarchy entry commute and touch disjoint particles
 * (PAPER.md:357).  on = 1 (default): frost_hhs_step runs every host-driven entry's fsi(S) on a side
 * stream of the context (one per hierarchy level, with its own sweep scratch) concurrently with the
 * recursion into F, and joins it before the next inter-level sweep -- same kernels, same inputs:
 * bitwise the result of on = 0, where the two run back to back on the context's stream. */
int frost_set_overlap(frost_ctx *ctx, int on);

/* Spatial splitting of fast hierarchy levels -- the paper's own outlook ("the further spatial
 * Hamiltonian splitting of the individual hierarchy levels into field stars, binaries and multiple
 * star systems"; binaries are left to future work).  The paper gives no
 * algorithm; the one built here applies Eq. 29's rule to pairs (reading 24):
 *   - a pair of one entry's set is FAST iff its symmetrised step of Eq. 49-54 is below tau_pivot
 *     (a particle is slow iff it has no fast pair -- Eq. 29 unchanged);
 *   - the fast pairs are the edges of a graph on F; hhs_fsi(F, tau/2) of Alg. 3 becomes one
 *     hhs_fsi(C, tau/2) per connected component C, and the pairs between different components join
 *     the inter-level kicks of Eq. 41-44 (kicked set: every pair of the entry that is neither
 *     slow-slow nor inside one component; for a single component this is Alg. 3 bit for bit).
 * split_max > 0 applies this to every entry with at most split_max members (larger entries run Alg. 3
 * as printed); 0 (default) switches it off.  A level that still percolates -- one giant component G plus
 * debris R -- gains too: the next level then holds G alone, and the kick is swept as S x F + G x R
 * (pair-symmetric) plus the pairs of R in different components.  Components of at most 32 particles --
 * binaries, triples -- are advanced side by side, one warp each, by one batched launch per recursion
 * pass; components of up to 1024 particles one CTA each; larger ones by the host recursion.  Result: deterministic; not the numbers of
 * split_max = 0 (a different, equally fourth-order splitting of the same Hamiltonian).
 * Limits: the components of a split entry are classified by these fixed sizes (32 / 1024), NOT by
 * frost_set_tuning's small_set_max -- that knob moves the hand-over of whole ENTRIES to the subtree kernel
 * only, so small_set_max = 0 still advances components of <= 1024 particles in the batched kernels.  An
 * entry may have at most 64 components above 1024 particles (a system of many sub-clusters can exceed
 * this); beyond that frost_hhs_step returns FROST_ELIMIT with the particles partly advanced. */
int frost_set_split(frost_ctx *ctx, int split_max);

/* Two-body propagator for the binaries of a split level -- PAPER.md:759 lists "regularised integrators,
 * Wisdom-Holman integrators and Kepler solvers" as the modules a spatially split level can hand its
 * few-body systems to, and defines none (reading 25).  on = 1 (needs frost_set_split, eps2 = 0):
 * hhs_fsi(C, tau/2) of a component C of exactly two particles is replaced by the exact two-body flow
 * over tau/2 -- the relative vector along its Kepler orbit (universal variables: ellipse, parabola and
 * hyperbola alike), the centre of mass uniformly -- instead of 2^k sub-steps.  H_C is then integrated
 * exactly, the order of the splitting is unchanged; frost_hhs_stats.n_kepler counts the calls.
 * Default 0. */
int frost_set_kepler(frost_ctx *ctx, int on);

/* Inside the device-resident subtree kernels a hierarchy entry of exactly two particles -- a binary,
 * the deepest and most often entered sets of a cluster with hard binaries -- is advanced by ONE thread
 * with both bodies in registers (a two-body set is either all slow or all fast at every entry, so its
 * subtree is a binary tree over the step interval).  Same arithmetic, operator order and bookkeeping
 * as the team path: bitwise the same result, ~4x less latency per entry.  on = 1 (default); 0 keeps
 * such entries on the warp team (tests). */
int frost_set_pair_path(frost_ctx *ctx, int on);

/* Pair-symmetric gradient sweeps of 16384 particles or more run WITHOUT the per-pair test for
 * coincident particles (|x_j - x_i|^2 + eps2 == 0, which the contract above ignores): such a pair then
 * yields NaN, the reduction that scatters the result notices any non-finite sum, and a gated second
 * pass with the guarded kernel recomputes the sweep -- a handful of empty launches for every input
 * without distinct coincident particles, a sweep at 2.5 x the cost for one that has them; the result
 * honours the contract either way.  on = 1 keeps the guard in the loop instead (one pass, 2.6 % slower
 * at N = 2^20).  Default 0. */
int frost_set_gradient_guard(frost_ctx *ctx, int on);

/* Pair-symmetric force sweeps of 16384 particles or more have an equal-mass variant: if every particle
 * of the sink and source lists has bitwise the same mass -- checked on the device while the streams
 * are packed; Plummer models, configs 1-4 -- the weight of the reverse direction is the forward weight
 * negated, one FP64 multiplication less per pair and bitwise the same sums.  Both variants of a sweep
 * are enqueued behind complementary device-side gates, so no host decision or read-back is involved.
 * on = 1 (default); 0 always runs the general kernels. */
int frost_set_equal_mass_path(frost_ctx *ctx, int on);

/* The kick sweeps of a split entry on their own (Eq. 42-44 on the pair set "labels differ"):
 *   out_acc[i]  <- G sum_{j in idx, label_j != label_i} m_j x_ji / s_ij^3,
 *   out_grad[i] <- 2G sum over the same j of m_j s^-5 (s^2 a_ji - 3 (x_ji.a_ji) x_ji) with the a of this call
 * for every i of the list idx (DEVICE int32[n_idx], NULL = all).  label (DEVICE int32[n_idx]) is
 * indexed by LIST POSITION; equal labels = same component, so the pair is skipped (frost_hhs_step
 * gives every slow particle -1).  out_grad nullable.  Served by the kernels frost_hhs_step uses for the
 * debris list of a split entry: pair-symmetric masked sweeps from ~6000 list members (or whenever
 * frost_set_symmetric mode >= 2), one-sided masked sweeps below.  Asynchronous. */
int frost_forces_masked(frost_ctx *ctx, int n, int ld, const double *pos, const double *mass,
                        const int32_t *idx, int n_idx, const int32_t *label, double *out_acc,
                        double *out_grad);

/* ---- The entry point that allocates nothing -------------------------------------------------------
 * Every call above may grow the context's scratch with cudaMalloc (and frost_create itself allocates).
 * Some callers cannot have that: a host application whose memory pool owns the whole device, a
 * latency-critical loop that cannot take the device-wide synchronisation a cudaFree implies, a program
 * that runs under a memory budget fixed at start-up.  For them:
 *
 *   out_acc[c*ld + i] <- G sum_{j != i} m_j (x_j - x_i)_c / (|x_j - x_i|^2 + eps2)^(3/2),  0 <= i < n
 *
 * (Eq. 24: the Newtonian accelerations of all n particles from all n particles, the
 * FROST_ACC self sweep of frost_forces) with no context and no allocation of any kind: the call issues
 * no cudaMalloc, cudaFree or allocating library routine, on the host or on the device.  Its scratch --
 * the packed source records and the per-slice partial sums of the one-sided Newton sweep it is a
 * variant of -- is a static __device__ array of 6.5 MiB compiled into the library, which every GPU
 * that loads the library's module keeps until the process exits.  Hence the limit:
 * n <= FROST_NOALLOC_MAX_N, otherwise FROST_ETOOBIG and nothing is launched (frost_noalloc_max_n()
 * returns the limit of the loaded build).
 *   device, stream : the CUDA device the pointers live on and the stream (cudaStream_t as void*, NULL =
 *                    legacy default stream) the three kernels are enqueued on; the device is made
 *                    current for the call and the caller's current device restored.  Asynchronous.
 *   pos, mass      : DEVICE inputs, layout as everywhere in this header; out_acc: DEVICE output, three
 *                    planes of stride ld, entries i >= n untouched.  Caller-owned; nothing is retained.
 *   cuda_error     : HOST, nullable: receives the cudaError_t when the status is FROST_ECUDA, else 0.
 * Sharing: all calls on a device use the one array and it keeps the previous call's contents.  A call
 * rewrites everything it later reads, so consecutive calls of any sizes on ordered streams are
 * independent -- but two calls that OVERLAP on the GPU (different streams without an event between
 * them, or two host threads) race on it and both results are garbage.  Serialise them.
 * First call: the first call on each device looks up the array's device address (cudaGetSymbolAddress,
 * which may load the module).  Make that call before starting any stream capture.
 * Same pair arithmetic as frost_forces (results agree to rounding, ~1e-15 |a_i|; the slice count, and
 * so the summation order, differs); coincident pairs contribute nothing, as above. */
#define FROST_NOALLOC_MAX_N 16384
int frost_acc_noalloc(int device, void *stream, int n, int ld, const double *pos, const double *mass,
                      double G, double eps2, double *out_acc, int *cuda_error);
int frost_noalloc_max_n(void);

#ifdef __cplusplus
}
#endif
#endif /* FROST_H */
