"""Parity of the pair-symmetric sweeps (csrc/frost_sym.cu; one evaluation of a pair updates both of
its particles) against the CPU oracle, element by element, forced on at sizes the oracle finishes
in seconds: ragged A tiles (1024 / 512 particles) and B tiles (128), several bands of the B list
(scratch cap of 1-3 MiB), self, mutual (slow/fast) and time-step sweeps, softening, coincident
particles, the central-mass-at-the-origin case that meets the zero padding, determinism.
Tolerances as in test_gpu_parity.py (north_star; reading 19)."""
import os

import numpy as np
import pytest
import torch

import frost_inputs as fi
from test_gpu_parity import (TOL_TAU, check_forces, dev, envelope_ratio, momentum_change,
                             oracle_hhs_with_envelope)

pytestmark = pytest.mark.gpu


@pytest.fixture()
def frs():
    import paper_2011_14984_b200 as frost
    f = frost.Frost()
    f.set_symmetric(2, 0)
    yield f
    f.close()


@pytest.mark.parametrize("n,mib", [(2, 0), (127, 0), (129, 0), (1025, 1), (3000, 1), (5000, 3), (9000, 1)])
def test_self_forces_symmetric(frs, oracle, n, mib):
    frs.set_symmetric(2, mib)
    pos, vel, mass = fi.plummer(n, 11)
    a, g, _, _ = check_forces(frs, oracle, pos, mass)
    # Newton's third law holds pair by pair in these sweeps: momentum change at rounding level
    assert np.abs((mass * a).sum(1)).max() <= 1e-14 * (mass * np.abs(a)).sum(1).max()
    assert np.abs((mass * g).sum(1)).max() <= 1e-12 * (mass * np.abs(g)).sum(1).max()


def test_self_forces_symmetric_unequal_masses_softened_scaled_G(frs, oracle):
    # config 5's recipe at its default hardness: g through the forward-error gate of reading 22
    pos, vel, mass, _ = fi.star_cluster(4096, 4)
    check_forces(frs, oracle, pos, mass, forward_gate=True)    # central mass at the origin meets the padding
    check_forces(frs, oracle, pos, mass, G=6.674e-3, eps2=1e-4, forward_gate=True)


def test_gradient_only_on_given_accelerations(frs, oracle):
    pos, vel, mass = fi.plummer(3000, 12)
    rng = np.random.default_rng(3)
    acc0 = np.ascontiguousarray(rng.normal(size=(3, 3000)))
    check_forces(frs, oracle, pos, mass, flags=2, acc0=acc0)


@pytest.mark.parametrize("nS,nF,mib", [(700, 1800, 0), (1800, 700, 0), (2500, 300, 1), (1, 2000, 0), (1500, 1, 0)])
def test_mutual_sets_symmetric(frs, oracle, nS, nF, mib):
    frs.set_symmetric(2, mib)
    n = 3000
    pos, vel, mass = fi.plummer(n, 5)
    perm = np.random.default_rng(1).permutation(n).astype(np.int32)
    S, F = np.sort(perm[:nS]), np.sort(perm[nS:nS + nF])
    a, g, _, _ = check_forces(frs, oracle, pos, mass, I=S, J=F, flags=7)
    out = np.sort(perm[nS + nF:])
    assert (a[:, out] == 0).all() and (g[:, out] == 5.0).all()       # untouched outside S u F
    both = np.concatenate([S, F])
    assert np.abs((mass[both] * a[:, both]).sum(1)).max() <= 1e-14 * (mass[both] * np.abs(a[:, both])).sum(1).max()


def test_coincident_particles_and_determinism(frs, oracle):
    pos, vel, mass = fi.plummer(2500, 2)
    pos[:, 5] = pos[:, 9]                # two coincident unsoftened particles: the pair is ignored
    pos[:, 700] = pos[:, 2400]
    check_forces(frs, oracle, pos, mass)
    p, m = dev(pos), dev(mass)
    a1, g1 = frs.forces(p, m)
    a2, g2 = frs.forces(p, m)
    torch.cuda.synchronize()
    assert torch.equal(a1, a2) and torch.equal(g1, g2)


@pytest.mark.parametrize("n,mib", [(2, 0), (100, 0), (513, 0), (4097, 1)])
def test_timesteps_symmetric(frs, oracle, n, mib):
    frs.set_symmetric(2, mib)
    pos, vel, mass = fi.plummer(n, 4)
    pivot = 1.0 / 64
    tau_ref, bin_ref = oracle.timesteps(pos, vel, mass, tau_pivot=pivot)
    tau, bins = frs.timesteps(dev(pos), dev(vel), dev(mass), tau_pivot=pivot)
    np.testing.assert_allclose(tau.cpu().numpy(), tau_ref, rtol=TOL_TAU)
    assert np.array_equal(bins.cpu().numpy(), bin_ref)


def test_timesteps_symmetric_on_subset(frs, oracle):
    n = 5000
    pos, vel, mass, _ = fi.star_cluster(n, 6)
    idx = fi.active_subset(n, 0.3, 6)
    frs.set_params(eta_ff=0.1, eta_fb=0.3)
    tau_ref, _ = oracle.timesteps(pos, vel, mass, idx=idx, eta_ff=0.1, eta_fb=0.3)
    tau, _ = frs.timesteps(dev(pos), dev(vel), dev(mass), idx=dev(idx), want_bins=False)
    t = tau.cpu().numpy()
    np.testing.assert_allclose(t[idx], tau_ref[idx], rtol=TOL_TAU)
    assert np.isinf(np.delete(t, idx)).all()
    frs.set_params()


@pytest.mark.parametrize("small", [0, 100])
def test_hhs_step_symmetric_matches_oracle(frs, oracle, small):
    """A whole HHS-FSI step (reduced-N replica of config 5 at full hardness, e <= 0.1; top step
    2^-11 so that the host-driven recursion stays at ~1e4 entries) with every streamed sweep --
    self, mutual slow/fast and time step -- forced through the symmetric kernels."""
    n = 3000
    pos, vel, mass, pairs = fi.star_cluster(n, 4, e_max=0.1)
    dt = 2.0 ** -11
    frs.set_params(eta_ff=0.2, eta_fb=0.2)
    frs.set_tuning(0, 0, small)
    pr, vr, st_ref, env_p, env_v, sts = oracle_hhs_with_envelope(oracle, pos, vel, mass, dt)
    assert all(s == st_ref for s in sts)
    p, v = dev(pos), dev(vel)
    try:
        st = frs.hhs_step(p, v, dev(mass), dt)
    finally:
        frs.set_tuning(0, 0, -1)
    assert st == st_ref and st["depth"] >= 10
    pg, vg = p.cpu().numpy(), v.cpu().numpy()
    rp, rv = envelope_ratio(pg, vg, pr, vr, env_p, env_v)
    assert rp <= 1.0 and rv <= 1.0, (rp, rv)
    assert momentum_change(mass, vel, vg, vr) <= 1.0


@pytest.mark.parametrize("world", [2, 3])
def test_pair_sharded_shares_add_up(frs, oracle, world):
    """frost_set_shard: the partial sums of the `world` shares (computed one after the other on this
    one GPU) add up to the unsharded result and match the oracle; FROST_ACC | FROST_GRAD in one
    sharded call is refused."""
    import paper_2011_14984_b200 as frost
    n = 6000
    pos, vel, mass = fi.plummer(n, 21)
    p, m = dev(pos), dev(mass)
    a_ref, g_ref = oracle.forces(pos, mass)
    acc = torch.zeros_like(p)
    for r in range(world):
        frs.set_shard(r, world)
        part = torch.zeros_like(p)
        frs.forces(p, m, out_acc=part, flags=frost.ACC)
        acc += part
    a = acc.cpu().numpy()
    assert (np.abs(a - a_ref).max(0) / np.linalg.norm(a_ref, axis=0)).max() < 1e-12
    grad = torch.zeros_like(p)
    for r in range(world):
        frs.set_shard(r, world)
        part = torch.zeros_like(p)
        frs.forces(p, m, out_acc=acc, out_grad=part, flags=frost.GRAD)
        grad += part
    g = grad.cpu().numpy()
    assert (np.abs(g - g_ref).max(0) / np.linalg.norm(g_ref, axis=0)).max() < 1e-10
    with pytest.raises(frost.FrostError):
        frs.forces(p, m, flags=frost.ACC | frost.GRAD)
    frs.set_shard(0, 1)


@pytest.mark.parametrize("n,mode,world", [(3000, 0, 2), (3000, 1, 3), (9000, 1, 2), (9000, 0, 4)])
def test_sharded_contract_is_path_independent(frs, oracle, n, mode, world):
    """frost_set_shard on sweeps the ONE-SIDED kernels serve (n below the symmetric threshold in auto
    mode 0, or mode 1 = never symmetric): every rank sweeps its block of the sink list and zeroes the
    rest, so adding the ranks' outputs gives the complete sums exactly as on the symmetric path --
    self, subset <- all, and mutual sweeps; ACC|GRAD in one call and ACCUMULATE are refused, and
    frost_fsi_step / frost_hhs_step refuse to run on a sharded context before touching anything."""
    import paper_2011_14984_b200 as frost
    pos, vel, mass = fi.plummer(n, 21)
    p, v, m = dev(pos), dev(vel), dev(mass)
    frs.set_symmetric(mode, 0)
    rng = np.random.default_rng(5)
    perm = rng.permutation(n).astype(np.int32)
    A, B = np.sort(perm[: n // 5]), np.sort(perm[n // 5: n // 5 + 700])
    cases = [(None, None, 0), (A, None, 0), (A, B, frost.MUTUAL)]
    try:
        for I, J, extra in cases:
            dI = None if I is None else dev(I); dJ = None if J is None else dev(J)
            frs.set_shard(0, 1)
            a_one = torch.full_like(p, 3.0); g_one = torch.full_like(p, 5.0)
            frs.forces(p, m, dI, dJ, out_acc=a_one, flags=frost.ACC | extra)
            frs.forces(p, m, dI, dJ, out_acc=a_one, out_grad=g_one, flags=frost.GRAD | extra)
            acc = torch.zeros_like(p); grad = torch.zeros_like(p)
            for r in range(world):
                frs.set_shard(r, world)
                part = torch.full_like(p, 3.0)
                frs.forces(p, m, dI, dJ, out_acc=part, flags=frost.ACC | extra)
                acc += part
            swept = np.arange(n) if I is None else (I if not extra else np.concatenate([I, J]))
            sw = dev(swept).long()
            rest = torch.ones(n, dtype=torch.bool, device="cuda"); rest[sw] = False
            assert (acc[:, rest] == 3.0 * world).all()                 # untouched outside the swept sets
            full = a_one.clone(); full[:, sw] = acc[:, sw]
            for r in range(world):
                frs.set_shard(r, world)
                part = torch.full_like(p, 5.0)
                frs.forces(p, m, dI, dJ, out_acc=full, out_grad=part, flags=frost.GRAD | extra)
                grad += part
            na = a_one[:, sw].norm(dim=0); ng = g_one[:, sw].norm(dim=0)
            assert ((acc - a_one)[:, sw].abs().max(0).values / na).max() < 1e-13
            assert ((grad - g_one)[:, sw].abs().max(0).values / ng).max() < 1e-10
            if mode == 1 or n < 6000:       # one-sided: each sink's sum comes from one rank, same bits
                assert torch.equal(acc[:, sw], a_one[:, sw])
        frs.set_shard(1, world)
        with pytest.raises(frost.FrostError):
            frs.forces(p, m, flags=frost.ACC | frost.GRAD)
        with pytest.raises(frost.FrostError):
            frs.forces(p, m, flags=frost.ACC | frost.ACCUMULATE)
        p0, v0 = p.clone(), v.clone()
        for call in (lambda: frs.fsi_step(p, v, m, 1e-3), lambda: frs.fsi_steps(p, v, m, 1e-3, 2),
                     lambda: frs.hhs_step(p, v, m, 1e-3)):
            with pytest.raises(frost.FrostError):
                call()
        torch.cuda.synchronize()
        assert torch.equal(p, p0) and torch.equal(v, v0)
    finally:
        frs.set_shard(0, 1)
        frs.set_symmetric(2, 0)


def test_symmetric_and_one_sided_sweeps_agree_on_random_shapes(frs):
    """Tile-edge fuzz (no oracle): 24 random set sizes, mutual splits, scratch caps (bands) and
    shard counts; the symmetric and the one-sided kernels must agree to rounding everywhere and
    leave everything outside the swept sets untouched."""
    import paper_2011_14984_b200 as frost
    rng = np.random.default_rng(2024)
    for case in range(24):
        n = int(rng.choice([rng.integers(1, 300), rng.integers(300, 5000), rng.integers(5000, 30000)]))
        pos, vel, mass = fi.plummer(max(n, 2), 100 + case)
        pos, vel, mass = np.ascontiguousarray(pos[:, :n]), np.ascontiguousarray(vel[:, :n]), mass[:n].copy()
        mass *= rng.uniform(0.2, 5.0, size=n)
        p, v, m = dev(pos), dev(vel), dev(mass)
        mib = int(rng.choice([0, 1, 2, 7]))
        mutual = n >= 4 and rng.random() < 0.5
        if mutual:
            perm = rng.permutation(n).astype(np.int32)
            k1 = int(rng.integers(1, n - 1)); k2 = int(rng.integers(k1 + 1, n + 1))
            I, J = dev(np.sort(perm[:k1])), dev(np.sort(perm[k1:k2]))
            flags = frost.ACC | frost.GRAD | frost.MUTUAL
        else:
            I = J = None
            flags = frost.ACC | frost.GRAD
        res = []
        for mode in (1, 2):
            frs.set_symmetric(mode, mib)
            a = torch.full_like(p, 3.0); g = torch.full_like(p, 5.0)
            frs.forces(p, m, I, J, out_acc=a, out_grad=g, flags=flags)
            t, b = frs.timesteps(p, v, m, tau_pivot=1.0 / 64)
            res.append((a, g, t[:n], b[:n]))
        (a1, g1, t1, b1), (a2, g2, t2, b2) = res
        sel = torch.cat([I, J]).long() if mutual else torch.arange(n, device="cuda")
        na, ng = a1[:, sel].norm(dim=0), g1[:, sel].norm(dim=0)
        ok = na > 0
        if ok.any():
            assert (((a1 - a2)[:, sel].abs().max(0).values)[ok] / na[ok]).max() < 1e-12, (case, n)
            assert (((g1 - g2)[:, sel].abs().max(0).values)[ok] / ng[ok]).max() < 1e-9, (case, n)
        if mutual:
            rest = torch.ones(n, dtype=torch.bool, device="cuda"); rest[sel] = False
            assert (a2[:, rest] == 3.0).all() and (g2[:, rest] == 5.0).all(), (case, n)
        fin = torch.isfinite(t1)
        assert torch.equal(fin, torch.isfinite(t2)) and torch.equal(b1, b2), (case, n)
        if fin.any():
            assert ((t1 - t2)[fin].abs() / t1[fin]).max() < 1e-13, (case, n)
    frs.set_symmetric(2, 0)


@pytest.mark.parametrize("mode", [0, 2])
def test_active_subset_against_all_as_self_plus_mutual(frs, oracle, mode):
    """Config 4's pair set {(i, j): i in A or j in A} swept in two pieces with FROST_ACCUMULATE --
    self(A) + mutual(A, rest), both served by the pair-symmetric kernels -- equals the oracle's
    A <- all and rest <- A sums, for a and (on the total a) for g; the resulting kick conserves
    momentum to roundoff."""
    import paper_2011_14984_b200 as frost
    n = 20000
    pos, vel, mass = fi.plummer(n, 3)
    frs.set_symmetric(mode, 0)
    p, m = dev(pos), dev(mass)
    for frac in (0.01, 0.3):
        A = fi.active_subset(n, frac, 3)
        rest = np.setdiff1d(np.arange(n, dtype=np.int32), A).astype(np.int32)
        a_ref = np.zeros((3, n)); g_ref = np.zeros((3, n))
        oracle.forces(pos, mass, sink_idx=A, source_idx=None, flags=oracle.ACC, acc=a_ref, grad=g_ref)
        oracle.forces(pos, mass, sink_idx=rest, source_idx=A, flags=oracle.ACC, acc=a_ref, grad=g_ref)
        oracle.forces(pos, mass, sink_idx=A, source_idx=None, flags=oracle.GRAD, acc=a_ref, grad=g_ref)
        oracle.forces(pos, mass, sink_idx=rest, source_idx=A, flags=oracle.GRAD, acc=a_ref, grad=g_ref)
        dA, dR = dev(A), dev(rest)
        acc = torch.zeros_like(p); grad = torch.zeros_like(p)
        frs.forces(p, m, dA, dA, out_acc=acc, out_grad=grad, flags=frost.ACC)
        frs.forces(p, m, dA, dR, out_acc=acc, out_grad=grad, flags=frost.ACC | frost.MUTUAL | frost.ACCUMULATE)
        frs.forces(p, m, dA, dA, out_acc=acc, out_grad=grad, flags=frost.GRAD)
        frs.forces(p, m, dA, dR, out_acc=acc, out_grad=grad, flags=frost.GRAD | frost.MUTUAL | frost.ACCUMULATE)
        a, g = acc.cpu().numpy(), grad.cpu().numpy()
        assert (np.abs(a - a_ref).max(0) / np.linalg.norm(a_ref, axis=0)).max() < 1e-12
        assert (np.abs(g - g_ref).max(0) / np.linalg.norm(g_ref, axis=0)).max() < 1e-10
        assert np.abs((mass * a).sum(1)).max() < 1e-14 * (mass * np.abs(a)).sum(1).max()
        with pytest.raises(frost.FrostError):
            frs.forces(p, m, dA, dR, out_acc=acc, out_grad=grad,
                       flags=frost.ACC | frost.GRAD | frost.MUTUAL | frost.ACCUMULATE)
    frs.set_symmetric(2, 0)


@pytest.mark.parametrize("kind,n", [("plummer", 1000), ("plummer", 60000), ("cluster", 50000)])
def test_pruned_timestep_sweep_is_bitwise_the_unpruned_minimum(frs, oracle, kind, n):
    """csrc/frost_tau.cu: Morton order + block-level discard of pairs that cannot lower a minimum.
    The result must be bitwise that of the plain symmetric sweep and of the pruning machinery with
    pruning off, and match the oracle on sampled particles (hard binaries, central mass included)."""
    if kind == "plummer":
        pos, vel, mass = fi.plummer(n, 31)
        sample = fi.active_subset(n, min(1.0, 300 / n), 5)
    else:
        pos, vel, mass, pairs = fi.star_cluster(n, 4)
        sample = np.concatenate([[0], pairs[:40].ravel(), fi.active_subset(n, 200 / n, 5)]).astype(np.int32)
    p, v, m = dev(pos), dev(vel), dev(mass)
    pivot = 2.0 ** -7
    out = {}
    for mode in (3, 4, 5):
        frs.set_symmetric(mode, 0)
        t, b = frs.timesteps(p, v, m, tau_pivot=pivot)
        out[mode] = (t.clone(), b.clone())
    frs.set_symmetric(2, 0)
    assert torch.equal(out[3][0], out[4][0]) and torch.equal(out[3][0], out[5][0])
    assert torch.equal(out[3][1], out[5][1])
    tau_ref, bin_ref = oracle.timesteps_sampled(pos, vel, mass, sample, tau_pivot=pivot)
    th, bh = out[5][0].cpu().numpy(), out[5][1].cpu().numpy()
    np.testing.assert_allclose(th[sample], tau_ref[sample], rtol=TOL_TAU)
    assert np.array_equal(bh[sample], bin_ref[sample])


def test_pruned_timestep_sweep_on_index_subset(frs):
    """The pruned sweep on a level given as an index list (as frost_hhs_step passes it): bitwise the
    plain symmetric sweep's result, everything outside the list untouched."""
    n = 70000
    pos, vel, mass, _ = fi.star_cluster(n, 9)
    idx = fi.active_subset(n, 0.8, 9)
    p, v, m, di = dev(pos), dev(vel), dev(mass), dev(idx)
    res = []
    for mode in (3, 5):
        frs.set_symmetric(mode, 0)
        t, b = frs.timesteps(p, v, m, idx=di, tau_pivot=2.0 ** -6)
        res.append((t.clone(), b.clone()))
    frs.set_symmetric(2, 0)
    assert torch.equal(res[0][0], res[1][0]) and torch.equal(res[0][1], res[1][1])
    out = np.setdiff1d(np.arange(n), idx)
    assert torch.isinf(res[1][0][dev(out).long()]).all()


@pytest.mark.skipif(torch.cuda.device_count() < 2, reason="needs two CUDA devices")
def test_two_devices_pair_sharded_and_sink_sharded(oracle):
    """SURVEY 8(f).3 on real peers (skipped on a one-GPU box): rank r = a context on device r with the
    state replicated.  Pair sharding (the default N > 1 arm of bench.py): the two ranks' partial sums,
    added the way the all-reduce adds them, equal the unsharded result to 1e-12 / 1e-10 and the oracle.
    Sink sharding (bench.py --one-sided, the paper's scatter-compute-gather): each rank's
    block of sinks is bitwise the one-GPU result."""
    import paper_2011_14984_b200 as frost
    from paper_2011_14984_b200 import sharding
    n = 20000
    pos, vel, mass = fi.plummer(n, 23)
    a_ref, g_ref = oracle.forces(pos, mass)
    ctx = [frost.Frost(d) for d in (0, 1)]
    P = [torch.as_tensor(pos).to(f"cuda:{d}") for d in (0, 1)]
    M = [torch.as_tensor(mass).to(f"cuda:{d}") for d in (0, 1)]
    try:
        one_a, one_g = ctx[0].forces(P[0], M[0])
        # pair sharding
        parts = []
        for r in (0, 1):
            ctx[r].set_shard(r, 2)
            part = torch.zeros_like(P[r])
            ctx[r].forces(P[r], M[r], out_acc=part, flags=frost.ACC)
            parts.append(part)
        acc = parts[0] + parts[1].to("cuda:0")
        gparts = []
        for r in (0, 1):
            part = torch.zeros_like(P[r])
            ctx[r].forces(P[r], M[r], out_acc=acc.to(f"cuda:{r}"), out_grad=part, flags=frost.GRAD)
            gparts.append(part)
        grad = gparts[0] + gparts[1].to("cuda:0")
        a, g = acc.cpu().numpy(), grad.cpu().numpy()
        assert (np.abs(a - a_ref).max(0) / np.linalg.norm(a_ref, axis=0)).max() < 1e-12
        assert (np.abs(g - g_ref).max(0) / np.linalg.norm(g_ref, axis=0)).max() < 1e-10
        assert (np.abs(a - one_a.cpu().numpy()).max(0) / np.linalg.norm(a_ref, axis=0)).max() < 1e-12
        # sink sharding with the one-sided kernels: bitwise per block
        for r in (0, 1):
            ctx[r].set_shard(0, 1)
            ctx[r].set_symmetric(1)
        ref_a = torch.zeros_like(P[0]); ref_g = torch.zeros_like(P[0])
        ctx[0].forces(P[0], M[0], out_acc=ref_a, out_grad=ref_g)
        full_a = torch.zeros_like(P[0])
        blocks = []
        for r in (0, 1):
            lo, hi = sharding.shard_range(n, r, 2)
            idx = torch.arange(lo, hi, dtype=torch.int32, device=f"cuda:{r}")
            part = torch.zeros_like(P[r])
            ctx[r].forces(P[r], M[r], sink_idx=idx, out_acc=part, flags=frost.ACC)
            full_a[:, lo:hi] = part[:, lo:hi].to("cuda:0")
            blocks.append((lo, hi, idx))
        assert torch.equal(full_a, ref_a)
        for r, (lo, hi, idx) in enumerate(blocks):
            part = torch.zeros_like(P[r])
            ctx[r].forces(P[r], M[r], sink_idx=idx, out_acc=full_a.to(f"cuda:{r}"), out_grad=part, flags=frost.GRAD)
            assert torch.equal(part[:, lo:hi].to("cuda:0"), ref_g[:, lo:hi])
    finally:
        for f in ctx:
            f.close()


@pytest.mark.parametrize("guard", [0, 1])
def test_unguarded_gradient_pass_and_its_repair(frs, oracle, guard):
    """frost_set_gradient_guard: pair-symmetric gradient sweeps of >= 16384 particles run without the
    per-pair coincidence test; an input with two DISTINCT coincident unsoftened particles (ignored
    pairwise, reading 11) then turns up as NaN in the first pass and is recomputed by the
    gated guarded pass -- same contract, same tolerances, self and mutual sweeps; a particle at the
    exact origin must not meet the padding records; guard = 1 keeps the test in the loop."""
    import paper_2011_14984_b200 as frost
    n = 20000
    pos, vel, mass = fi.plummer(n, 31)
    frs.set_gradient_guard(guard)
    try:
        for coincident in (False, True):
            x = pos.copy()
            x[:, 7] = 0.0                                  # exactly at the origin
            if coincident:
                x[:, 5] = x[:, 9]                          # inside one set
                x[:, 17000] = x[:, 100]                    # across the two sets of the mutual sweep
            a_ref, g_ref = oracle.forces(x, mass)
            a, g = frs.forces(dev(x), dev(mass))
            a, g = a.cpu().numpy(), g.cpu().numpy()
            assert np.isfinite(g).all()
            assert (np.abs(a - a_ref).max(0) / np.linalg.norm(a_ref, axis=0)).max() < 1e-12
            assert (np.abs(g - g_ref).max(0) / np.linalg.norm(g_ref, axis=0)).max() < 1e-10
            I = np.arange(0, 16500, dtype=np.int32); J = np.arange(16500, n, dtype=np.int32)
            a_ref, g_ref = oracle.forces(x, mass, sink_idx=I, source_idx=J, flags=oracle.ACC | oracle.GRAD | oracle.MUTUAL)
            am, gm = frs.forces(dev(x), dev(mass), dev(I), dev(J), flags=frost.ACC | frost.GRAD | frost.MUTUAL)
            am, gm = am.cpu().numpy(), gm.cpu().numpy()
            assert np.isfinite(gm).all()
            assert (np.abs(am - a_ref).max(0) / np.linalg.norm(a_ref, axis=0)).max() < 1e-12
            assert (np.abs(gm - g_ref).max(0) / np.linalg.norm(g_ref, axis=0)).max() < 1e-10
    finally:
        frs.set_gradient_guard(0)


def test_equal_mass_variant_is_bitwise_the_general_kernels(frs, oracle):
    """frost_set_equal_mass_path: on an equal-mass Plummer sphere the large pair-symmetric sweeps take
    the variant with one multiplication less per pair (flag computed on the device by the pack kernels,
    both variants enqueued behind complementary gates) -- bitwise the general kernels' sums, self and
    mutual; one different mass anywhere in the swept lists switches the sweep back to the general
    kernels (parity with the oracle either way)."""
    import paper_2011_14984_b200 as frost
    n = 20000
    pos, vel, mass = fi.plummer(n, 33)
    I = np.arange(0, 16500, dtype=np.int32); J = np.arange(16500, n, dtype=np.int32)
    for tweak in (False, True):
        m = mass.copy()
        if tweak:
            m[17777] *= 1.5
        res = []
        for on in (1, 0):
            frs.set_equal_mass_path(on)
            a, g = frs.forces(dev(pos), dev(m))
            am, gm = frs.forces(dev(pos), dev(m), dev(I), dev(J), flags=frost.ACC | frost.GRAD | frost.MUTUAL)
            res.append((a, g, am, gm))
        frs.set_equal_mass_path(1)
        for x, y in zip(res[0], res[1]):
            assert torch.equal(x, y)
        a_ref, g_ref = oracle.forces(pos, m)
        a, g = res[0][0].cpu().numpy(), res[0][1].cpu().numpy()
        assert (np.abs(a - a_ref).max(0) / np.linalg.norm(a_ref, axis=0)).max() < 1e-12
        assert (np.abs(g - g_ref).max(0) / np.linalg.norm(g_ref, axis=0)).max() < 1e-10


@pytest.mark.parametrize("world,extra", [(2, []), (3, []), (2, ["--one-sided"])])
def test_multi_rank_bench_path_on_one_device(oracle, tmp_path, world, extra):
    """The N > 1 path of bench.py EXECUTED on the one GPU of the box: `world`
    ranks under torch.distributed.run, all on cuda:0, process group gloo (NCCL refuses two ranks on a
    device; the exchanges are staged through the host).  Every rank runs bench.py's own step -- its
    share of the tile pairs (frost_set_shard) + all-reduce of a and of g, or with --one-sided its block
    of sinks + all-gather of a -- and saves the sharded pass at the initial positions.  Checked: one JSON
    line with n_gpus = world and an end-to-end number; every rank holds the same complete a (bitwise);
    a and g equal the unsharded call to 1e-12 / 1e-10 and the oracle (scatter, compute,
    gather)."""
    import json
    import subprocess
    import sys
    import paper_2011_14984_b200 as frost
    n = 20000
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    cmd = [sys.executable, os.path.join(root, "bench.py"), "--gpus", str(world), "--backend", "gloo",
           "--same-device", "--n", str(n), "--steps", "1", "--warmup", "1", "--e2e-steps", "1", "--no-rows",
           "--cpu-sinks", "256", "--dump-dir", str(tmp_path)] + extra
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=900)
    assert r.returncode == 0, r.stderr[-3000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, r.stdout[-2000:]
    out = json.loads(lines[0])
    assert out["n_gpus"] == world and out["value"] > 0 and out["e2e"]["value"] > 0
    assert out["e2e"]["h2d_bytes_per_step"] == world * 32 * n and out["e2e"]["d2h_bytes_per_step"] == 48 * n
    par = out["cpu_baseline"]["parity_of_the_sharded_pass"]
    assert par["acc_rel_err"] < 1e-12 and par["grad_rel_err"] < 1e-10

    pos, vel, mass = fi.plummer(n, 2)                     # bench.py's input: seed 2
    a_ref, g_ref = oracle.forces(pos, mass)
    fr = frost.Frost()
    try:
        if extra:
            fr.set_symmetric(1)
        one_a, one_g = fr.forces(dev(pos), dev(mass))
        torch.cuda.synchronize()
        one_a, one_g = one_a.cpu().numpy(), one_g.cpu().numpy()
    finally:
        fr.close()
    na, ng = np.linalg.norm(a_ref, axis=0), np.linalg.norm(g_ref, axis=0)
    dumps = [np.load(os.path.join(tmp_path, f"rank{k}.npz")) for k in range(world)]
    for d in dumps:
        assert np.array_equal(d["acc"], dumps[0]["acc"])            # the exchange leaves every rank with the same a
        assert (np.abs(d["acc"] - a_ref).max(0) / na).max() < 1e-12
        assert (np.abs(d["acc"] - one_a).max(0) / na).max() < 1e-12
        lo, hi = (0, n) if not extra else (int(d["lo"]), int(d["hi"]))   # sink sharding: g of the own block only
        assert (np.abs(d["grad"] - g_ref)[:, lo:hi].max(0) / ng[lo:hi]).max() < 1e-10
        assert (np.abs(d["grad"] - one_g)[:, lo:hi].max(0) / ng[lo:hi]).max() < 1e-10
        if extra:                                                       # one-sided kernels: same bits per sink
            assert np.array_equal(d["acc"], one_a) and np.array_equal(d["grad"][:, lo:hi], one_g[:, lo:hi])
    if not extra:
        for d in dumps:
            assert np.array_equal(d["grad"], dumps[0]["grad"])
