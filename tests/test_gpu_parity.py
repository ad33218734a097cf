"""Parity of the CUDA path (through the C-ABI binding) against the CPU oracle, element by element
on the same seeded inputs.  Tolerances are north_star's, read per particle against the vector norm
(reading 19): |da_k| <= 1e-12 |a_i|, |dg_k| <= 1e-10 |g_i|; bins identical; index work
bit-exact."""
import numpy as np
import pytest
import torch

import frost_inputs as fi

pytestmark = pytest.mark.gpu

TOL_A, TOL_G, TOL_TAU = 1e-12, 1e-10, 1e-13


@pytest.fixture(scope="module")
def fr():
    import paper_2011_14984_b200 as frost
    f = frost.Frost()
    yield f
    f.close()


def dev(a, dtype=None):
    return torch.as_tensor(np.ascontiguousarray(a), dtype=dtype).cuda()


def vec_err(x, ref):
    """max over particles of max_k |dx_k| / |ref_i|_2 (particles with ref == 0 must match exactly)."""
    nrm = np.linalg.norm(ref, axis=0)
    d = np.abs(x - ref).max(axis=0)
    ok0 = (nrm == 0)
    assert (d[ok0] == 0).all()
    return float((d[~ok0] / nrm[~ok0]).max()) if (~ok0).any() else 0.0


def check_forces(fr, oracle, pos, mass, I=None, J=None, flags=3, G=1.0, eps2=0.0, acc0=None):
    fr.set_params(G=G, eps2=eps2)
    n = mass.size
    a0 = np.zeros((3, n)) if acc0 is None else acc0.copy()
    a_ref, g_ref = oracle.forces(pos, mass, sink_idx=I, source_idx=J, G=G, eps2=eps2, flags=flags,
                                 acc=a0.copy(), grad=np.full((3, n), 5.0))
    a_gpu = dev(a0)
    g_gpu = torch.full((3, n), 5.0, dtype=torch.float64, device="cuda")
    fr.forces(dev(pos), dev(mass), None if I is None else dev(I), None if J is None else dev(J),
              out_acc=a_gpu, out_grad=g_gpu, flags=flags)
    torch.cuda.synchronize()
    a, g = a_gpu.cpu().numpy(), g_gpu.cpu().numpy()
    ea = vec_err(a, a_ref)
    eg = vec_err(g, g_ref) if flags & 2 else 0.0
    assert ea <= TOL_A, ea
    assert eg <= TOL_G, eg
    return a, g, a_ref, g_ref


@pytest.mark.parametrize("n", [1, 2, 3, 255, 256, 257, 1024, 3000])
def test_self_forces_small_and_ragged(fr, oracle, n):
    pos, vel, mass = fi.plummer(max(n, 2), 0)
    pos, mass = np.ascontiguousarray(pos[:, :n]), mass[:n].copy()
    check_forces(fr, oracle, pos, mass)


@pytest.mark.parametrize("k,slices", [(1, 1), (1, 5), (2, 1), (2, 3), (4, 2), (0, 0)])
def test_every_kernel_variant_and_slice_count(fr, oracle, k, slices):
    pos, vel, mass = fi.plummer(5000, 7)
    fr.set_tuning(k, slices, -1)
    try:
        check_forces(fr, oracle, pos, mass, eps2=1e-6)
    finally:
        fr.set_tuning(0, 0, -1)


def test_softened_and_scaled_G(fr, oracle):
    pos, vel, mass = fi.plummer(2048, 3)
    check_forces(fr, oracle, pos, mass, G=6.674e-3, eps2=1e-4)


def test_config1_plummer_1024_acc_grad(fr, oracle):
    pos, vel, mass = fi.plummer(1024, 0)
    a, g, _, _ = check_forces(fr, oracle, pos, mass)
    assert np.abs((mass * a).sum(1)).max() < 1e-15 * (mass * np.abs(a)).sum(1).max()
    assert np.abs((mass * g).sum(1)).max() < 1e-13 * (mass * np.abs(g)).sum(1).max()


def test_sink_subset_vs_all_and_reverse_config4_shape(fr, oracle):
    """Config 4's structure at N = 20000: A<-all, (all\\A)<-A, then both gradients; momentum of
    the resulting kick vanishes to roundoff."""
    n = 20000
    pos, vel, mass = fi.plummer(n, 3)
    for frac in (0.001, 0.01, 0.1):
        A = fi.active_subset(n, frac, 3)
        rest = np.setdiff1d(np.arange(n, dtype=np.int32), A).astype(np.int32)
        a, _, a_ref, _ = check_forces(fr, oracle, pos, mass, I=A, J=None, flags=1)
        a2, _, a_ref2, _ = check_forces(fr, oracle, pos, mass, I=rest, J=A, flags=1, acc0=a_ref)
        _, g, _, g_ref = check_forces(fr, oracle, pos, mass, I=A, J=None, flags=2, acc0=a_ref2)
        _, g2, _, _ = check_forces(fr, oracle, pos, mass, I=rest, J=A, flags=2, acc0=a_ref2)
        gt = g.copy(); gt[:, rest] = g2[:, rest]
        assert np.abs((mass * a2).sum(1)).max() < 1e-14 * (mass * np.abs(a2)).sum(1).max()
        assert np.abs((mass * gt).sum(1)).max() < 1e-12 * (mass * np.abs(gt)).sum(1).max()


def test_mutual_slow_fast_sets(fr, oracle):
    n = 3000
    pos, vel, mass = fi.plummer(n, 5)
    rng = np.random.default_rng(1)
    perm = rng.permutation(n).astype(np.int32)
    S, F = np.sort(perm[:700]), np.sort(perm[700:2500])      # 500 particles in neither set
    a, g, a_ref, g_ref = check_forces(fr, oracle, pos, mass, I=S, J=F, flags=7)
    out = np.sort(perm[2500:])
    assert (a[:, out] == 0).all() and (g[:, out] == 5.0).all()   # untouched outside S u F


def test_empty_and_degenerate_sets(fr, oracle):
    pos, vel, mass = fi.plummer(300, 2)
    e = np.zeros(0, dtype=np.int32)
    one = np.array([17], dtype=np.int32)
    check_forces(fr, oracle, pos, mass, I=e, J=None, flags=3)
    check_forces(fr, oracle, pos, mass, I=one, J=one, flags=3)
    check_forces(fr, oracle, pos, mass, I=one, J=e, flags=1)
    # two coincident unsoftened particles are ignored pairwise (reading 11)
    p2 = pos.copy(); p2[:, 5] = p2[:, 9]
    check_forces(fr, oracle, p2, mass)


def test_run_to_run_bitwise_determinism(fr):
    pos, vel, mass = fi.plummer(40000, 9)
    p, m = dev(pos), dev(mass)
    a1, g1 = fr.forces(p, m)
    a2, g2 = fr.forces(p, m)
    torch.cuda.synchronize()
    assert torch.equal(a1, a2) and torch.equal(g1, g2)


@pytest.mark.parametrize("n", [2, 100, 1000, 4097])
def test_timesteps_and_bins(fr, oracle, n):
    pos, vel, mass = fi.plummer(n, 4)
    fr.set_params(G=1.0, eta_ff=0.2, eta_fb=0.2)
    pivot = 1.0 / 64
    tau_ref, bin_ref = oracle.timesteps(pos, vel, mass, tau_pivot=pivot)
    tau, bins = fr.timesteps(dev(pos), dev(vel), dev(mass), tau_pivot=pivot)
    tau, bins = tau.cpu().numpy(), bins.cpu().numpy()
    np.testing.assert_allclose(tau, tau_ref, rtol=TOL_TAU)
    bad = np.nonzero(bins != bin_ref)[0]
    for i in bad:      # accepted only within 1e-13 of a bin edge (reading 20); expected count 0
        edge = pivot * 2.0 ** -min(bins[i], bin_ref[i])
        assert abs(tau_ref[i] / edge - 1) < 1e-13
    assert bad.size == 0


def test_timesteps_on_level_subset_and_partition(fr, oracle):
    n = 5000
    pos, vel, mass = fi.plummer(n, 6)
    idx = fi.active_subset(n, 0.3, 6)
    fr.set_params(eta_ff=0.1, eta_fb=0.3)
    tau_ref, _ = oracle.timesteps(pos, vel, mass, idx=idx, eta_ff=0.1, eta_fb=0.3)
    tau, _ = fr.timesteps(dev(pos), dev(vel), dev(mass), idx=dev(idx), want_bins=False)
    t = tau.cpu().numpy()
    np.testing.assert_allclose(t[idx], tau_ref[idx], rtol=TOL_TAU)
    assert np.isinf(np.delete(t, idx)).all()
    fr.set_params()
    pivot = float(np.median(tau_ref[idx]))
    slow, fast = fr.partition(dev(tau_ref), pivot, idx=dev(idx))
    s_ref = idx[tau_ref[idx] >= pivot]; f_ref = idx[tau_ref[idx] < pivot]
    assert np.array_equal(slow.cpu().numpy(), s_ref) and np.array_equal(fast.cpu().numpy(), f_ref)
    slow, fast = fr.partition(dev(tau_ref), 0.0)                 # all slow, idx = None
    assert slow.numel() == n and fast.numel() == 0
    assert np.array_equal(slow.cpu().numpy(), np.arange(n))


def test_kick_drift_gather(fr, oracle):
    n = 3333
    rng = np.random.default_rng(0)
    pos, vel, mass = fi.plummer(n, 8)
    acc = np.ascontiguousarray(rng.normal(size=(3, n))); grad = np.ascontiguousarray(rng.normal(size=(3, n)))
    idx = fi.active_subset(n, 0.5, 8)
    for ii in (None, idx):
        v_ref, p_ref = vel.copy(), pos.copy()
        oracle.kick(v_ref, acc, grad, idx=ii, c=0.37, kappa=0.011)
        oracle.drift(p_ref, v_ref, idx=ii, c=0.21)
        v, p = dev(vel), dev(pos)
        fr.kick(v, dev(acc), dev(grad), idx=None if ii is None else dev(ii), c=0.37, kappa=0.011)
        fr.drift(p, v, idx=None if ii is None else dev(ii), c=0.21)
        np.testing.assert_allclose(v.cpu().numpy(), v_ref, rtol=0, atol=4e-16 * np.abs(v_ref).max())
        np.testing.assert_allclose(p.cpu().numpy(), p_ref, rtol=0, atol=4e-16 * np.abs(p_ref).max())
    rec = fr.gather_pack(dev(pos), dev(mass), idx=dev(idx), n_pad=idx.size + 7).cpu().numpy()
    assert np.array_equal(rec[: idx.size, :3], pos[:, idx].T) and np.array_equal(rec[: idx.size, 3], mass[idx])
    assert (rec[idx.size:] == 0).all()


@pytest.mark.parametrize("n,eps2", [(1, 0.0), (2, 0.0), (1000, 0.0), (5000, 1e-4), (20000, 0.0)])
def test_diagnostics_match_oracle(fr, oracle, n, eps2):
    """frost_diagnostics (on-device E, P, L with an O(N^2) potential sweep) against
    the oracle's long-double textbook sums (Eq. 23)."""
    pos, vel, mass, _ = fi.star_cluster(max(n, 64), 4, a_lo=1e-3, a_hi=1e-2)
    pos, vel, mass = np.ascontiguousarray(pos[:, :n]), np.ascontiguousarray(vel[:, :n]), mass[:n].copy()
    fr.set_params(G=0.7, eps2=eps2)
    phi = torch.zeros(n, dtype=torch.float64, device="cuda")
    d = fr.diagnostics(dev(pos), dev(vel), dev(mass), out_phi=phi)
    ref = oracle.diagnostics(pos, vel, mass, G=0.7, eps2=eps2)
    fr.set_params()
    assert abs(d["T"] - ref["T"]) <= 1e-14 * abs(ref["T"])
    assert abs(d["U"] - ref["U"]) <= 1e-13 * abs(ref["U"]) + 0.0
    scale_p = (mass * np.abs(vel)).sum()
    assert np.abs(np.array(d["P"]) - ref["P"]).max() <= 1e-15 * scale_p
    scale_l = (mass * np.linalg.norm(pos, axis=0) * np.linalg.norm(vel, axis=0)).sum()
    assert np.abs(np.array(d["L"]) - ref["L"]).max() <= 1e-15 * scale_l
    # U = sum m phi / 2
    assert abs(0.5 * float((dev(mass) * phi).sum()) - ref["U"]) <= 1e-12 * abs(ref["U"]) + 0.0


def test_energy_conservation_measured_on_device(fr, oracle):
    """Config 1 with the energy read from the device: |dE/E| after 10 FSI steps at dt = 1/1024 is
    the oracle's to rounding (the trajectories agree to 1e-11) and small."""
    pos, vel, mass = fi.plummer(1024, 0)
    p, v, m = dev(pos), dev(vel), dev(mass)
    fr.set_params()
    e0 = fr.diagnostics(p, v, m)
    pr, vr = pos.copy(), vel.copy()
    for _ in range(10):
        fr.fsi_step(p, v, m, 1.0 / 1024)
        oracle.fsi_step(pr, vr, mass, 1.0 / 1024)
    e1 = fr.diagnostics(p, v, m)
    r0, r1 = oracle.diagnostics(pos, vel, mass), oracle.diagnostics(pr, vr, mass)
    de_gpu, de_ref = (e1["E"] - e0["E"]) / e0["E"], (r1["E"] - r0["E"]) / r0["E"]
    assert abs(de_gpu - de_ref) < 1e-11
    assert abs(de_gpu) < 1e-3


@pytest.mark.parametrize("small", [-1, 0])
def test_config1_ten_fsi_steps(fr, oracle, small):
    """Config 1: N = 1024, 10 fixed-step FSI steps with dt = 1/1024 -- through the one-CTA
    device-resident kernel (small = -1) and through the streaming sweeps (small = 0)."""
    pos, vel, mass = fi.plummer(1024, 0)
    p, v, m = dev(pos), dev(vel), dev(mass)
    fr.set_params()
    fr.set_tuning(0, 0, small)
    pr, vr = pos.copy(), vel.copy()
    d0 = oracle.diagnostics(pos, vel, mass)
    try:
        for _ in range(10):
            fr.fsi_step(p, v, m, 1.0 / 1024)
            oracle.fsi_step(pr, vr, mass, 1.0 / 1024)
    finally:
        fr.set_tuning(0, 0, -1)
    pg, vg = p.cpu().numpy(), v.cpu().numpy()
    assert np.abs(pg - pr).max() < 1e-11 and np.abs(vg - vr).max() < 1e-10
    d1 = oracle.diagnostics(pg, vg, mass)
    assert np.abs(d1["P"] - d0["P"]).max() < 1e-15
    assert np.linalg.norm(d1["L"] - d0["L"]) < 1e-13


@pytest.mark.parametrize("n", [700, 3000, 9000])
def test_fsi_steps_equal_repeated_fsi_step_bitwise(fr, n):
    """frost_fsi_steps reuses the trailing Newton sweep of a step as the leading one of the next:
    same bits as repeated frost_fsi_step (device-resident kernel, one-sided and symmetric sweeps)."""
    pos, vel, mass = fi.plummer(n, 13)
    fr.set_params()
    p1, v1, m = dev(pos), dev(vel), dev(mass)
    p2, v2 = dev(pos), dev(vel)
    for _ in range(4):
        fr.fsi_step(p1, v1, m, 1.0 / 2048)
    fr.fsi_steps(p2, v2, m, 1.0 / 2048, 4)
    torch.cuda.synchronize()
    assert torch.equal(p1, p2) and torch.equal(v1, v2)


@pytest.mark.parametrize("n,small", [(1024, -1), (1024, 0), (1024, 48), (3000, -1), (3000, 100)])
def test_hhs_step_small_cluster(fr, oracle, n, small):
    """Reduced-N replica of config 5: level sets, bookkeeping and the trajectory must match the
    oracle whether the recursion runs on the host (small = 0), in the device-resident subtree
    kernel (whole problem for n <= 1024) or in a mix of both."""
    pos, vel, mass, pairs = fi.star_cluster(n, 4, a_lo=1e-3, a_hi=1e-2)
    fr.set_params(eta_ff=0.2, eta_fb=0.2)
    fr.set_tuning(0, 0, small)
    pr, vr = pos.copy(), vel.copy()
    st_ref = oracle.hhs_step(pr, vr, mass, 1.0 / 256)
    p, v = dev(pos), dev(vel)
    try:
        st = fr.hhs_step(p, v, dev(mass), 1.0 / 256)
    finally:
        fr.set_tuning(0, 0, -1)
    assert st == st_ref
    assert st["depth"] >= 3
    pg, vg = p.cpu().numpy(), v.cpu().numpy()
    assert np.abs(pg - pr).max() < 1e-10 and np.abs(vg - vr).max() < 1e-8 * np.abs(vr).max()
    assert np.abs((mass * vg).sum(1) - (mass * vel).sum(1)).max() < 1e-16


@pytest.mark.parametrize("n", [150, 700, 1024])
def test_subtree_kernel_one_cta_and_cluster_agree_bitwise(fr, n):
    """The device-resident subtree kernel on one CTA and on a thread-block cluster of replicas
    (large sweeps shared out by sinks) must give the same bits: a sink's sum is formed by the same
    lanes in the same order either way... as long as the lane split is the same, so compare to
    rounding, and the bookkeeping exactly."""
    pos, vel, mass, pairs = fi.star_cluster(n, 4, a_lo=1e-3, a_hi=1e-2)
    fr.set_params(eta_ff=0.2, eta_fb=0.2)
    out = []
    for one_cta in (1, 0):
        fr.set_tuning(0, 0, -1, one_cta)
        p, v = dev(pos), dev(vel)
        st = fr.hhs_step(p, v, dev(mass), 1.0 / 256)
        out.append((st, p.cpu().numpy(), v.cpu().numpy()))
    fr.set_tuning(0, 0, -1, 0)
    assert out[0][0] == out[1][0]
    assert np.abs(out[0][1] - out[1][1]).max() < 1e-12 and np.abs(out[0][2] - out[1][2]).max() < 1e-10


def test_hhs_tiny_systems_and_depth_limit(fr, oracle):
    """Five-body Solar system (Tables A1/A2) entirely inside the subtree kernel; a hard binary with
    a far too long top step must stop with FROST_EDEPTH instead of recursing forever."""
    import paper_2011_14984_b200 as frost
    pos, vel, mass, G = fi.solar_system()
    vel = vel - (vel * mass).sum(1, keepdims=True) / mass.sum()
    fr.set_params(G=G, eta_ff=0.05, eta_fb=0.05)
    pr, vr = pos.copy(), np.ascontiguousarray(vel.copy())
    p, v = dev(pos), dev(vel)
    for _ in range(3):
        st_ref = oracle.hhs_step(pr, vr, mass, 512.0, G=G, eta_ff=0.05, eta_fb=0.05)
        st = fr.hhs_step(p, v, dev(mass), 512.0)
        assert st == st_ref
    assert np.abs(p.cpu().numpy() - pr).max() < 1e-11 * 30 and st["depth"] >= 2
    b_pos, b_vel, b_mass, P = fi.kepler_binary(1.0, 1.0, 1e-6, 0.0)
    fr.set_params(G=1.0, max_depth=12)
    with pytest.raises(frost.FrostError, match="deeper"):
        fr.hhs_step(dev(b_pos), dev(b_vel), dev(b_mass), 1.0)
    fr.set_params()


def test_solar_system_run_on_device(fr, oracle):
    """the paper's only printed multi-level input (Sun + 4 giant planets, Tables
    A1/A2) integrated for 40 top steps of 512 days by frost_hhs_step with the
    conserved quantities read by frost_diagnostics -- nothing but the initial conditions crosses the
    host.  |dE/E| falls steeply with eta (~eta^4), |dP| stays at roundoff
    (PAPER.md:674), the hierarchy has several populated levels, and the end state equals the
    oracle's."""
    errs = []
    for eta in (0.2, 0.05):
        pos, vel, mass, G = fi.solar_system()
        vel = np.ascontiguousarray(vel - (vel * mass).sum(1, keepdims=True) / mass.sum())
        fr.set_params(G=G, eta_ff=eta, eta_fb=eta)
        p, v, m = dev(pos), dev(vel), dev(mass)
        pr, vr = pos.copy(), vel.copy()
        d0 = fr.diagnostics(p, v, m)
        depth = 0
        for _ in range(40):
            st = fr.hhs_step(p, v, m, 512.0)
            oracle.hhs_step(pr, vr, mass, 512.0, G=G, eta_ff=eta, eta_fb=eta)
            depth = max(depth, st["depth"])
        d1 = fr.diagnostics(p, v, m)
        ref = oracle.diagnostics(pr, vr, mass, G=G)
        errs.append(abs(d1["E"] / d0["E"] - 1))
        assert np.abs(np.array(d1["P"]) - np.array(d0["P"])).max() < 1e-17
        assert np.linalg.norm(np.array(d1["L"]) - np.array(d0["L"])) < 1e-12 * np.linalg.norm(d0["L"])
        assert depth >= 2
        assert abs(d1["E"] - ref["E"]) < 1e-12 * abs(ref["E"])
        assert np.abs(p.cpu().numpy() - pr).max() < 1e-9 * 30
    fr.set_params()
    assert errs[0] < 1e-6 and errs[1] < errs[0] / 20


def test_hhs_multi_step_run_conserves_momentum_to_roundoff(fr):
    """The paper's headline property on the device: eight HHS-FSI
    steps of a 6000-star cluster with a central mass and binaries down to a = 1e-4 (depth >= 10);
    linear momentum stays at rounding level, angular momentum at 1e-13 relative, energy at the
    truncation level of eta = 0.2."""
    n = 6000
    pos, vel, mass, pairs = fi.star_cluster(n, 7, a_lo=1e-4, a_hi=1e-2)
    fr.set_params(eta_ff=0.2, eta_fb=0.2)
    p, v, m = dev(pos), dev(vel), dev(mass)
    d0 = fr.diagnostics(p, v, m)
    depth = 0
    for _ in range(8):
        depth = max(depth, fr.hhs_step(p, v, m, 2.0 ** -8)["depth"])
    d1 = fr.diagnostics(p, v, m)
    assert depth >= 10 and bool(torch.isfinite(p).all())
    assert np.abs(np.array(d1["P"]) - np.array(d0["P"])).max() < 1e-15
    assert np.linalg.norm(np.array(d1["L"]) - np.array(d0["L"])) < 1e-13 * np.linalg.norm(d0["L"])
    assert abs(d1["E"] / d0["E"] - 1) < 1e-6
