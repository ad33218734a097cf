"""Spatial splitting of fast hierarchy levels (frost_set_split) against the oracle's
definition of it (oracle/frost_oracle.c O6s, reading 24): the masked kick sweeps element by
element, the bookkeeping of a split step IDENTICAL (level sets, components per level, pair counts), the
trajectory inside the oracle's own +-1-ulp envelope, momentum at rounding level -- on the host-driven
levels, in the batched one-warp-per-component kernel and inside the device-resident subtree kernel."""
import numpy as np
import pytest
import torch

import frost_inputs as fi
from test_gpu_parity import (C_FWD, TOL_A, TOL_G, dev, envelope_ratio, momentum_change, oracle_hhs_with_envelope,
                             vec_err)

pytestmark = pytest.mark.gpu
BIG = 1 << 20


@pytest.fixture(scope="module")
def fr():
    import paper_2011_14984_b200 as frost
    f = frost.Frost()
    yield f
    f.close()


def masked_termsum(pos, mass, acc, idx, label_g, G, eps2, sinks):
    """T_i of DESIGN.md reading 22 (the magnitude sum of Eq. 27's terms, as oracle_gradient_termsum forms
    it) over the MASKED pair set, for the listed sinks.  A bound for the forward-error gate, not an
    expected value: plain fp64 numpy."""
    xj, mj, aj, lj = pos[:, idx], mass[idx], acc[:, idx], label_g[idx]
    T = np.zeros(len(sinks))
    for c0 in range(0, len(sinks), 256):
        ii = sinks[c0:c0 + 256]
        dx = xj[:, None, :] - pos[:, ii, None]
        da = aj[:, None, :] - acc[:, ii, None]
        s2 = (dx * dx).sum(0) + eps2
        xa = (dx * da).sum(0)
        ok = (s2 > 0) & (lj[None, :] != label_g[ii, None])
        s2 = np.where(ok, s2, 1.0)
        t = s2[None] * da - 3.0 * xa[None] * dx
        T[c0:c0 + 256] = 2.0 * G * np.where(ok, mj[None, :] * np.sqrt((t * t).sum(0)) / (s2 * s2 * np.sqrt(s2)), 0.0).sum(1)
    return T


def check_masked(fr, oracle, pos, mass, idx, label_g, G, eps2):
    """frost_forces_masked against oracle_forces_masked, every sink of the list: a to 1e-12 |a_i|; g to
    1e-10 |g_i|, and where a hard binary inside the swept pair set makes Eq. 27 itself ill-conditioned
    (reading 22) to 1e-10 |g_i| + C_FWD 2^-53 T_i with T_i over the masked pairs."""
    n = mass.size
    fr.set_params(G=G, eps2=eps2)
    a_ref, g_ref = oracle.forces_masked(pos, mass, idx, label_g, G=G, eps2=eps2)
    out_a = torch.full((3, n), 5.0, dtype=torch.float64, device="cuda")
    out_g = torch.full((3, n), 6.0, dtype=torch.float64, device="cuda")
    a, g = fr.forces_masked(dev(pos), dev(mass), torch.as_tensor(label_g[idx]).cuda(),
                            idx=torch.as_tensor(idx).cuda(), out_acc=out_a, out_grad=out_g)
    torch.cuda.synchronize()
    fr.set_params()
    a, g = a.cpu().numpy(), g.cpu().numpy()
    out = np.setdiff1d(np.arange(n), idx)
    assert (a[:, out] == 5.0).all() and (g[:, out] == 6.0).all()         # untouched outside the list
    assert np.isfinite(a).all() and np.isfinite(g).all()
    ea = vec_err(a[:, idx], a_ref[:, idx])
    assert ea <= TOL_A, ea
    d = np.abs(g - g_ref).max(0)[idx]
    nrm = np.linalg.norm(g_ref, axis=0)[idx]
    bad = np.nonzero(d > TOL_G * nrm)[0]
    assert bad.size <= 4096, bad.size             # the ill-conditioned sinks are the few next to a hard binary
    ratio = 0.0
    if bad.size:
        T = masked_termsum(pos, mass, a_ref, idx, label_g, G, eps2, idx[bad])
        ratio = float((d[bad] / (TOL_G * nrm[bad] + C_FWD * 2.0 ** -53 * T)).max())
        assert ratio <= 1.0, ratio
    return ea, bad.size, ratio


@pytest.mark.parametrize("n,eps2", [(700, 0.0), (5000, 0.0), (5000, 1e-6)])
def test_masked_kick_sweeps_match_oracle(fr, oracle, n, eps2):
    """frost_forces_masked (the kick sweeps of a split entry, Eq. 42-44 on "labels differ") against
    oracle_forces_masked on a sub-list with slow particles (-1), two-body and larger components; the
    one-sided kernels (lists below ~6000), config 5's recipe at its default hardness."""
    pos, vel, mass, pairs = fi.star_cluster(n, 4)
    rng = np.random.default_rng(n)
    idx = np.sort(rng.choice(n, size=n - n // 7, replace=False)).astype(np.int32)
    lab_pos = rng.integers(0, idx.size // 3, size=idx.size).astype(np.int32)       # ~3 members per label
    lab_pos[rng.random(idx.size) < 0.4] = -1
    label_g = np.full(n, -7, dtype=np.int32)
    label_g[idx] = lab_pos
    fr.set_symmetric(1)
    try:
        check_masked(fr, oracle, pos, mass, idx, label_g, 0.9, eps2)
    finally:
        fr.set_symmetric(0)


@pytest.mark.parametrize("n,eps2,labels,mib", [(129, 0.0, "random", 0), (3000, 0.0, "random", 1), (3000, 1e-6, "binaries", 0),
                                                (9000, 0.0, "binaries", 1), (9000, 1e-6, "random", 0),
                                                (20000, 0.0, "binaries", 1), (20000, 0.0, "random", 0),
                                                (20000, 1e-6, "random", 1)])
def test_masked_pair_symmetric_sweeps_match_oracle(fr, oracle, n, eps2, labels, mib, capsys):
    """The pair-symmetric masked kernels (SymNewtonMasked / SymGradientMasked: the debris list of every
    large split entry of frost_hhs_step) element by element against oracle_forces_masked, Eq. 42-44
    (PAPER.md:365-387): the small-tile geometry (n < 16384) and the large one, the B list in one band and
    in several (scratch cap 1 MiB), labels -1, two-body and large components, two coincident particles in
    different components, with and without softening, on config 5's recipe at its default hardness.
    labels = "binaries": every binary is one component (what a split entry produces: the hard pairs are
    masked out); "random": labels drawn at random, so hard binaries sit INSIDE the swept pair set and the
    sinks around them take the forward-error gate of reading 22."""
    pos, vel, mass, pairs = fi.star_cluster(n, 4)
    rng = np.random.default_rng(n + 1)
    idx = np.sort(rng.choice(n, size=n - n // 9, replace=False)).astype(np.int32)
    k = idx.size
    lab_pos = rng.integers(0, max(k // 3, 2), size=k).astype(np.int32)             # ~3 members per label
    lab_pos[rng.random(k) < 0.3] = -1                                              # "slow" members
    big = rng.random(k) < 0.25
    lab_pos[big] = k + 1                                                           # one component of ~k/4
    label_g = np.full(n, -7, dtype=np.int32)
    label_g[idx] = lab_pos
    if labels == "binaries":
        for b, (i1, i2) in enumerate(pairs):
            label_g[i1] = label_g[i2] = 2 * k + b
    # two coincident particles of the list in different components (reading 11: the pair adds nothing)
    free = idx[np.isin(idx, pairs.ravel(), invert=True) & (idx > 0)]
    i, j = free[3], free[11]
    pos = pos.copy()
    pos[:, j] = pos[:, i]
    label_g[i], label_g[j] = 3 * k + 1, 3 * k + 2
    fr.set_symmetric(2, mib)
    l0 = fr.launch_count()
    try:
        ea, nbad, ratio = check_masked(fr, oracle, pos, mass, idx, label_g, 0.9, eps2)
    finally:
        fr.set_symmetric(0)
    with capsys.disabled():
        print(f"\n[masked sym n={n} eps2={eps2} {labels} cap={mib}] launches {fr.launch_count() - l0}, "
              f"a err {ea:.1e}, sinks beyond 1e-10|g| {nbad}, worst gate ratio {ratio:.2f}")


def _split_case(fr, oracle, pos, vel, mass, dt, small, one_cta=0, **kw):
    pr, vr, st_ref, env_p, env_v, sts = oracle_hhs_with_envelope(oracle, pos, vel, mass, dt, split_max=BIG, **kw)
    assert all(s == st_ref for s in sts)
    fr.set_tuning(0, 0, small, one_cta)
    fr.set_split(BIG)
    p, v = dev(pos), dev(vel)
    try:
        st = fr.hhs_step(p, v, dev(mass), dt)
    finally:
        fr.set_split(0)
        fr.set_tuning(0, 0, -1, 0)
    return st, st_ref, p.cpu().numpy(), v.cpu().numpy(), pr, vr, env_p, env_v


@pytest.mark.parametrize("n,small,one_cta,log2dt", [(256, -1, 0, 7), (256, -1, 1, 7), (256, 48, 0, 7), (256, 0, 0, 9),
                                                    (1024, -1, 0, 8), (3000, -1, 0, 8), (3000, 100, 0, 8),
                                                    (2000, 0, 0, 9)])
def test_split_step_matches_split_oracle(fr, oracle, n, small, one_cta, log2dt, capsys):
    """One split HHS-FSI step of config 5's recipe (binaries a = 1e-5..1e-3, e <= 0.1 so that no pair
    step oscillates across a pivot): n <= 1024 with small = -1 runs entirely inside the subtree kernel
    (cluster or one CTA at the top, components handed to the quad / warp teams); small = 48 / 100 /
    0 drive the top levels from the host, with the masked kick sweeps, and advance the components by
    the batched one-warp-per-component launches."""
    pos, vel, mass, pairs = fi.star_cluster(n, 4, e_max=0.1)
    fr.set_params(eta_ff=0.2, eta_fb=0.2)
    st, st_ref, pg, vg, pr, vr, env_p, env_v = _split_case(fr, oracle, pos, vel, mass, 2.0 ** -log2dt, small, one_cta)
    assert st == st_ref
    assert st["depth"] >= 12 and st["n_comp"][0] > 1
    rp, rv = envelope_ratio(pg, vg, pr, vr, env_p, env_v)
    with capsys.disabled():
        print(f"\n[split n={n} small={small} one_cta={one_cta}] depth {st['depth']}, components per level "
              f"{st['n_comp'][:6]}..., entries {sum(st['entries'])}; envelope ratio x {rp:.3f}, v {rv:.3f}")
    assert rp <= 1.0 and rv <= 1.0, (rp, rv)
    assert momentum_change(mass, vel, vg, vr) <= 1.0


def test_split_with_one_component_is_the_unsplit_step_bitwise(fr):
    """A hard binary among distant slow stars: F is the binary (one component) at every level, so the
    split step must be Alg. 3's bits -- with every entry driven from the host (small = 0; the components
    themselves still run in the batched kernels: frost.h, frost_set_split) and inside the subtree kernel
    alike."""
    b_pos, b_vel, b_mass, P = fi.kepler_binary(1.0, 0.7, 1e-3, 0.3)
    rng = np.random.default_rng(3)
    pos = np.ascontiguousarray(np.concatenate([b_pos, rng.normal(size=(3, 6)) * 3.0], axis=1))
    vel = np.ascontiguousarray(np.concatenate([b_vel, rng.normal(size=(3, 6)) * 0.1], axis=1))
    mass = np.concatenate([b_mass, np.full(6, 0.5)])
    fr.set_params()
    for small in (-1, 0):
        out = []
        for split in (0, BIG):
            fr.set_tuning(0, 0, small)
            fr.set_split(split)
            p, v = dev(pos), dev(vel)
            try:
                st = fr.hhs_step(p, v, dev(mass), 2.0 ** -6)
            finally:
                fr.set_split(0)
                fr.set_tuning(0, 0, -1)
            out.append((st, p, v))
        assert out[0][0] == out[1][0] and out[0][0]["depth"] >= 2
        assert torch.equal(out[0][1], out[1][1]) and torch.equal(out[0][2], out[1][2])


def test_split_max_limits_the_split_to_small_entries(fr, oracle):
    """split_max = 500 on a 2000-star cluster: the entries above 500 members run Alg. 3 as printed, the
    ones below split -- bookkeeping identical to the oracle's with the same parameter."""
    pos, vel, mass, pairs = fi.star_cluster(2000, 4, e_max=0.1)
    fr.set_params(eta_ff=0.2, eta_fb=0.2)
    pr, vr = pos.copy(), vel.copy()
    st_ref = oracle.hhs_step(pr, vr, mass, 2.0 ** -8, split_max=500)
    fr.set_split(500)
    p, v = dev(pos), dev(vel)
    try:
        st = fr.hhs_step(p, v, dev(mass), 2.0 ** -8)
    finally:
        fr.set_split(0)
    assert st == st_ref
    assert st["n_comp"][0] == 1 and any(c > e for c, e in zip(st["n_comp"], st["entries"]))
    assert np.abs((mass * (v.cpu().numpy() - vel)).sum(1)).max() < 1e-15


@pytest.mark.parametrize("n,split", [(256, 0), (256, BIG), (3000, BIG)])
def test_pair_path_is_bitwise_the_team_path(fr, n, split):
    """frost_set_pair_path: two-body hierarchy entries on one thread (both bodies in registers, the
    subtree walked as a binary tree over the step interval) against the same entries on the warp
    team -- same pair arithmetic, operator order and bookkeeping, so the same bits: with Alg. 3 as
    printed (binaries that end up alone at depth) and with split levels (every binary its own tree)."""
    pos, vel, mass, pairs = fi.star_cluster(n, 4)
    fr.set_params(eta_ff=0.2, eta_fb=0.2)
    out = []
    try:
        for on in (0, 1):
            fr.set_pair_path(on)
            fr.set_split(split)
            p, v = dev(pos), dev(vel)
            st = fr.hhs_step(p, v, dev(mass), 2.0 ** -8)
            out.append((st, p, v))
    finally:
        fr.set_pair_path(1)
        fr.set_split(0)
    assert out[0][0] == out[1][0] and out[0][0]["depth"] >= 14
    assert torch.equal(out[0][1], out[1][1]) and torch.equal(out[0][2], out[1][2])


def test_split_tiny_and_degenerate_systems(fr, oracle):
    """Edge cases of the split step against the oracle: one, two, three and five bodies (no fast pair,
    one fast pair, a chain), softening, the Kepler propagator on and off, the five-body Solar system (F = {Sun, Jupiter}: one component,
    several levels), an empty fast set at the top (everything slow)."""
    rng = np.random.default_rng(11)
    cases = []
    for n in (1, 2, 3, 5):
        pos = np.ascontiguousarray(rng.normal(size=(3, n)))
        vel = np.ascontiguousarray(rng.normal(size=(3, n)) * 0.3)
        mass = rng.uniform(0.5, 2.0, n)
        if n >= 3:                                  # a close pair on a circular orbit inside
            r = np.array([1e-3, 2e-3, 0.0])
            pos[:, 1] = pos[:, 0] + r
            vc = np.sqrt((mass[0] + mass[1]) / np.linalg.norm(r))
            vel[:, 1] = vel[:, 0] + vc * np.array([-r[1], r[0], 0.0]) / np.linalg.norm(r)
        cases.append((pos, vel, mass, 2.0 ** -5, dict(G=1.0, eps2=0.0)))
        cases.append((pos, vel, mass, 2.0 ** -5, dict(G=1.0, eps2=1e-6)))
        cases.append((pos, vel, mass, 2.0 ** -20, dict(G=1.0, eps2=0.0)))       # all slow at the top
    sp, sv, sm, sG = fi.solar_system()
    cases.append((sp, sv, sm, 512.0, dict(G=sG, eps2=0.0)))
    for pos, vel, mass, dt, kw in cases:
        for small, kepler in ((-1, 0), (0, 0), (-1, 1), (0, 1)):
            fr.set_params(G=kw["G"], eps2=kw["eps2"], eta_ff=0.1, eta_fb=0.1)
            fr.set_tuning(0, 0, small)
            fr.set_split(BIG)
            fr.set_kepler(kepler)                 # (ignored with softening, by both sides)
            pr, vr = pos.copy(), vel.copy()
            st_ref = oracle.hhs_step(pr, vr, mass, dt, eta_ff=0.1, eta_fb=0.1, split_max=BIG, kepler=bool(kepler), **kw)
            p, v = dev(pos), dev(vel)
            try:
                st = fr.hhs_step(p, v, dev(mass), dt)
            finally:
                fr.set_split(0)
                fr.set_kepler(0)
                fr.set_tuning(0, 0, -1)
                fr.set_params()
            assert st == st_ref, (mass.size, dt, small, kepler)
            scale = max(1.0, np.abs(pr).max())
            # (a tight pair turns a rounding difference into an orbital phase difference: |dv| ~ v dphi)
            assert np.abs(p.cpu().numpy() - pr).max() < 1e-10 * scale
            assert np.abs(v.cpu().numpy() - vr).max() < 1e-7 * max(1.0, np.abs(vr).max())


def test_fast_two_body_frames_take_the_kepler_propagator_on_every_path(fr, oracle):
    """A two-body frame that is fast but not itself a component -- the root of a two-body step, or a
    two-body F below a parent too large to be split (split_max = 2) -- is split like any entry: its one
    component is the pair, which the Kepler propagator advances over tau/2 twice (reading 25).  The
    one-thread binary path must not swallow such a frame: bookkeeping (n_kepler included) equal to the
    oracle's with the pair path on and off, on the device-resident and on the host recursion."""
    rng = np.random.default_rng(23)
    cases = []
    for n, split_max in ((2, BIG), (2, 2), (5, 2)):
        pos = np.ascontiguousarray(rng.normal(size=(3, n)))
        vel = np.ascontiguousarray(rng.normal(size=(3, n)) * 0.3)
        mass = rng.uniform(0.5, 2.0, n)
        r = np.array([1e-3, 2e-3, 0.0])                 # a close pair on a circular orbit
        pos[:, 1] = pos[:, 0] + r
        vc = np.sqrt((mass[0] + mass[1]) / np.linalg.norm(r))
        vel[:, 1] = vel[:, 0] + vc * np.array([-r[1], r[0], 0.0]) / np.linalg.norm(r)
        cases.append((pos, vel, mass, split_max))
    dt = 2.0 ** -5
    for pos, vel, mass, split_max in cases:
        pr, vr = pos.copy(), vel.copy()
        st_ref = oracle.hhs_step(pr, vr, mass, dt, eta_ff=0.1, eta_fb=0.1, split_max=split_max, kepler=True)
        assert st_ref["n_kepler"] >= 2, st_ref
        for small, pair in ((-1, 1), (-1, 0), (0, 1), (0, 0)):
            fr.set_params(eta_ff=0.1, eta_fb=0.1)
            fr.set_tuning(0, 0, small)
            fr.set_split(split_max)
            fr.set_kepler(1)
            fr.set_pair_path(pair)
            p, v = dev(pos), dev(vel)
            try:
                st = fr.hhs_step(p, v, dev(mass), dt)
            finally:
                fr.set_split(0); fr.set_kepler(0); fr.set_pair_path(1)
                fr.set_tuning(0, 0, -1); fr.set_params()
            assert st == st_ref, (mass.size, split_max, small, pair)
            assert np.abs(p.cpu().numpy() - pr).max() < 1e-10 * max(1.0, np.abs(pr).max())
            assert np.abs(v.cpu().numpy() - vr).max() < 1e-7 * max(1.0, np.abs(vr).max())


def test_split_multi_step_run_conserves_like_alg3(fr, capsys):
    """Sixteen steps of a 6000-star cluster with a central mass and binaries down to a = 1e-4, with the
    fast levels split and with Alg. 3 as printed, from the same start: linear momentum at rounding
    level and angular momentum at 1e-13 in both, no secular energy drift
    (the energy error stays at the size of the first step's), the split run's energy error within a
    factor of a few of Alg. 3's, and the two end states apart only by the truncation error."""
    n = 6000
    pos, vel, mass, pairs = fi.star_cluster(n, 7, a_lo=1e-4, a_hi=1e-2)
    fr.set_params(eta_ff=0.2, eta_fb=0.2)
    out = {}
    try:
        for split in (0, BIG):
            fr.set_split(split)
            p, v, m = dev(pos), dev(vel), dev(mass)
            d0 = fr.diagnostics(p, v, m)
            de = []
            for _ in range(16):
                st = fr.hhs_step(p, v, m, 2.0 ** -8)
                de.append(fr.diagnostics(p, v, m)["E"] / d0["E"] - 1)
            d1 = fr.diagnostics(p, v, m)
            assert st["depth"] >= 10 and bool(torch.isfinite(p).all())
            assert np.abs(np.array(d1["P"]) - np.array(d0["P"])).max() < 1e-15
            assert np.linalg.norm(np.array(d1["L"]) - np.array(d0["L"])) < 1e-13 * np.linalg.norm(d0["L"])
            out[split] = (np.array(de), p.cpu().numpy())
    finally:
        fr.set_split(0)
    de0, de1 = out[0][0], out[BIG][0]
    with capsys.disabled():
        print(f"\n[16 steps, n = {n}] max |dE/E|: Alg. 3 {np.abs(de0).max():.2e} (last {de0[-1]:.2e}), "
              f"split {np.abs(de1).max():.2e} (last {de1[-1]:.2e}); max |dx| between the runs "
              f"{np.abs(out[0][1] - out[BIG][1]).max():.2e}")
    assert np.abs(de0).max() < 1e-6 and np.abs(de1).max() < 1e-6
    assert np.abs(de1).max() < 10 * np.abs(de0).max() + 1e-9
    assert np.abs(out[0][1] - out[BIG][1]).max() < 1e-4


@pytest.mark.parametrize("n,small,log2dt", [(256, -1, 7), (256, 0, 9), (3000, -1, 8), (3000, 100, 8), (2000, 0, 9), (3000, -1, 4)])
def test_split_step_with_kepler_components_matches_oracle(fr, oracle, n, small, log2dt, capsys):
    """frost_set_kepler on top of the split step: every two-body component follows its exact Kepler orbit
    (reading 25; oracle O6k) -- bookkeeping identical to the oracle's (fewer and shallower entries, the
    same number of propagator calls), trajectory inside the oracle's 1-ulp envelope, momentum at
    rounding level: inside the subtree kernel (small = -1, n = 256), through the batched component
    launches, and with every entry driven from the host (small = 0; components of <= 1024 particles still
    run in the batched kernels).  dt_top = 2^-4 at n = 3000 makes level 0
    percolate (one component of ~2800 particles beside a few small ones): the S x F + G x R + masked-R
    kick and the host recursion into the giant component, against the oracle."""
    pos, vel, mass, pairs = fi.star_cluster(n, 4, e_max=0.1)
    dt = 2.0 ** -log2dt
    fr.set_params(eta_ff=0.2, eta_fb=0.2)
    pr, vr, st_ref, env_p, env_v, sts = oracle_hhs_with_envelope(oracle, pos, vel, mass, dt, split_max=BIG, kepler=True)
    assert all(s == st_ref for s in sts)
    fr.set_tuning(0, 0, small)
    fr.set_split(BIG)
    fr.set_kepler(1)
    p, v = dev(pos), dev(vel)
    try:
        st = fr.hhs_step(p, v, dev(mass), dt)
    finally:
        fr.set_kepler(0)
        fr.set_split(0)
        fr.set_tuning(0, 0, -1)
    assert st == st_ref and st["n_kepler"] > 0
    pg, vg = p.cpu().numpy(), v.cpu().numpy()
    rp, rv = envelope_ratio(pg, vg, pr, vr, env_p, env_v)
    with capsys.disabled():
        print(f"\n[split + kepler n={n} small={small}] depth {st['depth']}, {st['n_kepler']} propagator calls, "
              f"{sum(st['entries'])} entries; max |dx| {np.abs(pg - pr).max():.2e} (envelope {env_p.max():.2e}); "
              f"ratio x {rp:.3f}, v {rv:.3f}")
    assert rp <= 1.0 and rv <= 1.0, (rp, rv)
    assert momentum_change(mass, vel, vg, vr) <= 1.0


def test_pruned_time_step_sweep_finds_every_fast_pair(fr):
    """Levels of >= 32768 particles take the pruned time-step sweep, which in a split entry must still
    meet every pair below the pivot (it discards against max(running minimum, tau_pivot)).  The same
    split step with the pruning machinery off (frost_set_symmetric mode 3: the plain pair-symmetric
    sweep evaluates all pairs) must give the same components and bookkeeping, and the same state up to
    the last bit of a few sums (mode 3 also sends the small force sweeps through the symmetric kernels,
    which add in another order: 81 velocity components differ by one ulp)."""
    n = 40000
    pos, vel, mass, pairs = fi.star_cluster(n, 4, a_lo=1e-4, a_hi=1e-2)
    fr.set_params(eta_ff=0.2, eta_fb=0.2)
    out = []
    try:
        for mode in (0, 3):
            fr.set_symmetric(mode)
            fr.set_split(BIG)
            p, v = dev(pos), dev(vel)
            st = fr.hhs_step(p, v, dev(mass), 2.0 ** -8)
            out.append((st, p, v))
    finally:
        fr.set_symmetric(0)
        fr.set_split(0)
    assert out[0][0] == out[1][0]
    assert out[0][0]["n_comp"][0] > 100 and out[0][0]["depth"] >= 8
    assert (out[0][1] - out[1][1]).abs().max() < 1e-14 and (out[0][2] - out[1][2]).abs().max() < 1e-13
