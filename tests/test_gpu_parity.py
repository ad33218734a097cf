"""Parity of the CUDA path (through the C-ABI binding) against the CPU oracle, element by element
on the same seeded inputs.  Tolerances are north_star's, read per particle against the vector norm
(reading 19): |da_k| <= 1e-12 |a_i|, |dg_k| <= 1e-10 |g_i|; bins identical; index work
bit-exact.  Inputs with config 5's hard binaries use the forward-error gate of DESIGN.md reading 22
for g: |dg_k| <= 1e-10 |g_i| + C_FWD 2^-53 T_i, T_i = the oracle's magnitude sum of Eq. 27's terms
(the definition itself moves by up to 2.4 x 2^-53 T_i > 1e-10 |g_i| under +-1 ulp of the fp64
accelerations it is evaluated from: tests/test_oracle_pins.py)."""
import os

import numpy as np
import pytest
import torch

import frost_inputs as fi

pytestmark = pytest.mark.gpu

TOL_A, TOL_G, TOL_TAU = 1e-12, 1e-10, 1e-13
C_FWD = 8.0          # forward-error constant of reading 22 (<= 8; the definition's own floor is 2.4)


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


def grad_gate_ratio(oracle, pos, mass, a_ref, g, g_ref, I=None, J=None, flags=3, G=1.0, eps2=0.0):
    """max over the swept sinks of |dg_k| / (1e-10 |g_i| + C_FWD 2^-53 T_i)  (reading 22)."""
    n = mass.size
    T = oracle.gradient_termsum(pos, mass, a_ref, sink_idx=I, source_idx=J, G=G, eps2=eps2)
    sel = np.arange(n) if I is None else np.asarray(I)
    if flags & 4:
        T += oracle.gradient_termsum(pos, mass, a_ref, sink_idx=J, source_idx=I, G=G, eps2=eps2)
        sel = np.concatenate([sel, np.arange(n) if J is None else np.asarray(J)])
    d = np.abs(g - g_ref).max(0)[sel]
    bound = TOL_G * np.linalg.norm(g_ref, axis=0)[sel] + C_FWD * 2.0 ** -53 * T[sel]
    assert (d[bound == 0] == 0).all()
    return float((d[bound > 0] / bound[bound > 0]).max()) if (bound > 0).any() else 0.0


def check_forces(fr, oracle, pos, mass, I=None, J=None, flags=3, G=1.0, eps2=0.0, acc0=None,
                 forward_gate=False):
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
    assert ea <= TOL_A, ea
    if (flags & 2) and forward_gate:
        ratio = grad_gate_ratio(oracle, pos, mass, a_ref, g, g_ref, I, J, flags, G, eps2)
        assert ratio <= 1.0, ratio
    elif flags & 2:
        eg = vec_err(g, g_ref)
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


@pytest.mark.parametrize("sym", [1, 2])
def test_self_forces_at_config5_hardness_forward_error_gate(fr, oracle, sym, capsys):
    """Self sweep ACC|GRAD on config 5's recipe at its DEFAULT hardness (binaries a = 1e-5..1e-3),
    one-sided (sym = 1) and pair-symmetric (sym = 2) kernels.  a holds 1e-12; g is gated by the
    forward-error bound of reading 22.  Also the gradient alone from the ORACLE's accelerations
    (identical fp64 inputs on both sides: what remains is the kernel's own arithmetic)."""
    pos, vel, mass, _ = fi.star_cluster(4096, 4)
    fr.set_symmetric(sym, 0)
    try:
        a, g, a_ref, g_ref = check_forces(fr, oracle, pos, mass, forward_gate=True)
        r1 = grad_gate_ratio(oracle, pos, mass, a_ref, g, g_ref)
        _, g2, _, g_ref2 = check_forces(fr, oracle, pos, mass, flags=2, acc0=a_ref, forward_gate=True)
        r2 = grad_gate_ratio(oracle, pos, mass, a_ref, g2, g_ref2, flags=2)
        check_forces(fr, oracle, pos, mass, G=6.674e-3, eps2=1e-12, forward_gate=True)
    finally:
        fr.set_symmetric(0, 0)
    plain = vec_err(g, g_ref)
    with capsys.disabled():
        print(f"\n[g gate] sym={sym}: plain max |dg|/|g| = {plain:.2e}; gate ratio end-to-end {r1:.3f}, "
              f"gradient-only on the oracle's a {r2:.3f} (C_FWD = {C_FWD})")
    assert np.abs((mass * g).sum(1)).max() < 1e-12 * (mass * np.abs(g)).sum(1).max()


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


@pytest.mark.parametrize("n,ld", [(65536, 65536), (70001, 70002), (70001, 70001), (200003, 200010)])
def test_dense_update_kernels_are_bitwise_the_indexed_ones(fr, oracle, n, ld):
    """Dense lists (idx = None) of >= 65536 particles take the four-particles-per-thread kernels with
    16-byte accesses (even plane stride; an odd stride keeps the one-particle kernels): kick with and
    without the gradient term, drift and gather/pack must give the bits of the one-particle kernels --
    reached through the explicit index list 0..n-1 -- and the oracle's values, for even and odd n,
    leaving the entries n..ld-1 untouched."""
    rng = np.random.default_rng(n)
    mk = lambda: np.ascontiguousarray(rng.normal(size=(3, ld)))
    pos, vel, acc, grad = mk(), mk(), mk(), mk()
    mass = rng.uniform(0.5, 2.0, n)
    iota = torch.arange(n, dtype=torch.int32, device="cuda")
    m = dev(mass)
    out = {}
    for name, ii in (("dense", None), ("indexed", iota)):
        v, p, a, g = dev(vel), dev(pos), dev(acc), dev(grad)
        lib = fr.lib
        import ctypes as C
        P = lambda t: None if t is None else C.c_void_p(t.data_ptr())
        # (through the C-ABI directly: the binding passes ld for n)
        assert lib.frost_kick(fr.h, n, ld, P(v), P(a), P(g), P(ii), n, 0.37, 0.011) == 0
        assert lib.frost_kick(fr.h, n, ld, P(v), P(a), None, P(ii), n, -0.2, 0.0) == 0
        assert lib.frost_drift(fr.h, n, ld, P(p), P(v), P(ii), n, 0.21) == 0
        rec = torch.full((n + 5, 4), 7.0, dtype=torch.float64, device="cuda")
        assert lib.frost_gather_pack(fr.h, n, ld, P(p), P(m), None if ii is None else P(ii), n, n + 5, P(rec)) == 0
        torch.cuda.synchronize()
        out[name] = (v, p, rec)
    for a, b in zip(out["dense"], out["indexed"]):
        assert torch.equal(a, b)
    v, p, rec = (t.cpu().numpy() for t in out["dense"])
    v_ref, p_ref = vel.copy(), pos.copy()
    sub = lambda x: np.ascontiguousarray(x[:, :n])
    vr, pr = sub(v_ref), sub(p_ref)
    oracle.kick(vr, sub(acc), sub(grad), c=0.37, kappa=0.011)
    oracle.kick(vr, sub(acc), None, c=-0.2, kappa=0.0)
    oracle.drift(pr, vr, c=0.21)
    np.testing.assert_allclose(v[:, :n], vr, rtol=0, atol=4e-16 * np.abs(vr).max())
    np.testing.assert_allclose(p[:, :n], pr, rtol=0, atol=4e-16 * np.abs(pr).max())
    assert np.array_equal(v[:, n:], vel[:, n:]) and np.array_equal(p[:, n:], pos[:, n:])
    assert np.array_equal(rec[:n, :3], p[:, :n].T) and np.array_equal(rec[:n, 3], mass) and (rec[n:] == 0).all()


@pytest.mark.parametrize("n,eps2", [(1, 0.0), (2, 0.0), (1000, 0.0), (5000, 1e-4), (20000, 0.0)])
def test_diagnostics_match_oracle(fr, oracle, n, eps2):
    """frost_diagnostics (on-device E, P, L with an O(N^2) potential sweep) against
    the oracle's long-double textbook sums (Eq. 23)."""
    pos, vel, mass, _ = fi.star_cluster(max(n, 64), 4)
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


ENV_K = 8.0          # GPU-vs-oracle deviation allowed, in units of the oracle's own +-1-ulp envelope


def oracle_hhs_with_envelope(oracle, pos, vel, mass, dt, trials=3, seed=0, keep_states=False, **kw):
    """The oracle's HHS-FSI step plus its own sensitivity to the last bit of its inputs: the step is
    repeated from positions and velocities moved by +-1 ulp per component (random signs, seeded).
    Returns (pos_ref, vel_ref, stats_ref, env_pos[n], env_vel[n], stats_of_every_trial).

    Why this is the yardstick (reading 23): a hard binary at |x| ~ 1 resolves its own
    separation only to ulp(x)/a ~ 1e-11; any two correct fp64 evaluations of Alg. 3 (different
    summation order, FMA contraction) part by an ulp of x or v somewhere along the 2^depth
    sub-steps, after which they differ the way the oracle differs from itself under a 1-ulp input
    change (the earliest, hence largest, such change).  Several independent partings add in
    quadrature, so the GPU is held to ENV_K = 8 times the envelope, per particle."""
    n = mass.size
    if n <= 512:
        oracle.set_num_threads(1)             # tiny level sets: OpenMP fork/join would dominate
    try:
        pr, vr = pos.copy(), vel.copy()
        st = oracle.hhs_step(pr, vr, mass, dt, **kw)
        rng = np.random.default_rng(seed)
        env_p, env_v, sts, states = np.zeros(n), np.zeros(n), [], []
        for _ in range(trials):
            pp = np.ascontiguousarray(np.nextafter(pos, rng.choice([-1.0, 1.0], size=pos.shape) * np.inf))
            vv = np.ascontiguousarray(np.nextafter(vel, rng.choice([-1.0, 1.0], size=vel.shape) * np.inf))
            sts.append(oracle.hhs_step(pp, vv, mass, dt, **kw))
            env_p = np.maximum(env_p, np.abs(pp - pr).max(0))
            env_v = np.maximum(env_v, np.abs(vv - vr).max(0))
            if keep_states:
                states.append((pp, vv))
    finally:
        oracle.set_num_threads(os.cpu_count() or 1)
    if keep_states:
        return pr, vr, st, env_p, env_v, sts, states
    return pr, vr, st, env_p, env_v, sts


def momentum_change(mass, v0, v1, v_ref=None):
    """|sum m dv|_max of a step in units of what "roundoff" is for it: every kick is pairwise
    antisymmetric but individually rounded, so the sum random-walks with the number of kicks (a hard
    binary, |v| ~ 10-100, is kicked ~2^depth times per top step).  The unit is 4 x the oracle's own
    |sum m dv| over the same step (v_ref) where given, and never less than 8 x 2^-53 x sum m |v|."""
    unit = 8 * 2.0 ** -53 * (mass * np.linalg.norm(v1, axis=0)).sum()
    if v_ref is not None:
        unit = max(unit, 4 * np.abs((mass * (v_ref - v0)).sum(1)).max())
    return float(np.abs((mass * (v1 - v0)).sum(1)).max() / unit)


def envelope_ratio(pg, vg, pr, vr, env_p, env_v):
    """max over particles of |dx| / (ENV_K env_x + 8 ulp) and the same for v."""
    fl_p = 8 * np.spacing(np.abs(pr).max(0) + 1e-300)
    fl_v = 8 * np.spacing(np.abs(vr).max(0) + 1e-300)
    rp = np.abs(pg - pr).max(0) / (ENV_K * env_p + fl_p)
    rv = np.abs(vg - vr).max(0) / (ENV_K * env_v + fl_v)
    return float(rp.max()), float(rv.max())


@pytest.mark.parametrize("n,small,log2dt", [(1024, -1, 8), (1024, 0, 11), (1024, 48, 8), (3000, -1, 8),
                                            (3000, 100, 8)])
def test_hhs_step_small_cluster(fr, oracle, n, small, log2dt):
    """Reduced-N replica of config 5 at its full hardness (binaries a = 1e-5..1e-3; eccentricities
    capped at 0.1 so that no time-step oscillates across a pivot and the level sets are a
    reproducible function of the input -- the oracle's own +-1-ulp trials confirm it): level sets
    and bookkeeping IDENTICAL to the oracle's and the trajectory inside the oracle's 1-ulp envelope,
    whether the recursion runs on the host (small = 0; shorter top step, ~45 launches per entry), in
    the device-resident subtree kernel (whole problem for n <= 1024) or in a mix of both."""
    pos, vel, mass, pairs = fi.star_cluster(n, 4, e_max=0.1)
    dt = 2.0 ** -log2dt
    fr.set_params(eta_ff=0.2, eta_fb=0.2)
    fr.set_tuning(0, 0, small)
    pr, vr, st_ref, env_p, env_v, sts = oracle_hhs_with_envelope(oracle, pos, vel, mass, dt)
    assert all(s == st_ref for s in sts)
    p, v = dev(pos), dev(vel)
    try:
        st = fr.hhs_step(p, v, dev(mass), dt)
    finally:
        fr.set_tuning(0, 0, -1)
    assert st == st_ref
    assert st["depth"] >= (12 if small == 0 else 14)
    rp, rv = envelope_ratio(p.cpu().numpy(), v.cpu().numpy(), pr, vr, env_p, env_v)
    assert rp <= 1.0 and rv <= 1.0, (rp, rv)
    assert momentum_change(mass, vel, v.cpu().numpy(), vr) <= 1.0


@pytest.mark.parametrize("small,one_cta,log2dt", [(-1, 0, 7), (-1, 1, 7), (48, 0, 7), (0, 0, 10)])
def test_hhs_step_matches_oracle_at_config5_depth(fr, oracle, small, one_cta, log2dt, capsys):
    """Alg. 3 at config 5's depth, element by element: 256 stars of config 5's
    recipe (binaries down to a = 1e-5, e <= 0.1), dt_top = 2^-7 => depth 17 with every level
    populated (2^18 - 1 hierarchy entries).  small = -1: one launch of the subtree kernel -- the
    16-CTA cluster team (one_cta = 0) or the CTA team (one_cta = 1) at the top, the quad team for
    sub-sets of 33-128 and the warp team for sub-sets of <= 32 at depth; small = 48: host recursion
    down to sets of <= 48, then quad / warp teams; small = 0: host recursion only (2^-10: depth 14).
    Bookkeeping identical to the oracle's; trajectory inside ENV_K x the oracle's 1-ulp envelope;
    momentum change at rounding level."""
    n = 256
    pos, vel, mass, pairs = fi.star_cluster(n, 4, e_max=0.1)
    dt = 2.0 ** -log2dt
    fr.set_params(eta_ff=0.2, eta_fb=0.2)
    pr, vr, st_ref, env_p, env_v, sts = oracle_hhs_with_envelope(oracle, pos, vel, mass, dt)
    assert all(s == st_ref for s in sts)
    fr.set_tuning(0, 0, small, one_cta)
    p, v = dev(pos), dev(vel)
    try:
        st = fr.hhs_step(p, v, dev(mass), dt)
    finally:
        fr.set_tuning(0, 0, -1, 0)
    assert st == st_ref
    assert st["depth"] >= (14 if small == 0 else 15)
    pg, vg = p.cpu().numpy(), v.cpu().numpy()
    rp, rv = envelope_ratio(pg, vg, pr, vr, env_p, env_v)
    with capsys.disabled():
        print(f"\n[hhs depth {st['depth']}] small={small} one_cta={one_cta}: max |dx| {np.abs(pg - pr).max():.2e} "
              f"(envelope {env_p.max():.2e}), max |dv| {np.abs(vg - vr).max():.2e} (envelope {env_v.max():.2e}); "
              f"ratio to {ENV_K:.0f} x envelope: x {rp:.3f}, v {rv:.3f}")
    assert rp <= 1.0 and rv <= 1.0, (rp, rv)
    assert momentum_change(mass, vel, vg, vr) <= 1.0


@pytest.mark.parametrize("n,small", [(20000, -1), (6000, 200)])
def test_hhs_overlap_of_fsi_S_with_hhs_F_is_bitwise_the_serial_step(fr, n, small):
    """frost_set_overlap: fsi(S, tau/2) on a side stream concurrently with the recursion into F
    (the two commute and touch disjoint particles) must give the bits of the serial
    order, with the same bookkeeping, step after step."""
    pos, vel, mass, pairs = fi.star_cluster(n, 4, a_lo=1e-4, a_hi=1e-2)
    fr.set_params(eta_ff=0.2, eta_fb=0.2)
    fr.set_tuning(0, 0, small)
    out = []
    try:
        for on in (0, 1):
            fr.set_overlap(on)
            p, v, m = dev(pos), dev(vel), dev(mass)
            sts = [fr.hhs_step(p, v, m, 2.0 ** -9) for _ in range(2)]
            out.append((sts, p.clone(), v.clone()))
    finally:
        fr.set_overlap(1)
        fr.set_tuning(0, 0, -1)
    assert out[0][0] == out[1][0] and out[0][0][0]["depth"] >= 5
    assert torch.equal(out[0][1], out[1][1]) and torch.equal(out[0][2], out[1][2])


def hhs_stats_invariants(st):
    """What every correct execution of Alg. 3 satisfies whatever its rounding: a level is entered at
    most twice per entry of its parent, and the members of level k+1 are the fast members of level k
    entered twice."""
    e, s, f = st["entries"], st["n_slow"], st["n_fast"]
    assert e[0] == 1
    for k in range(st["depth"]):
        assert e[k + 1] <= 2 * e[k] and e[k + 1] % 2 == 0
        assert s[k + 1] + f[k + 1] == 2 * f[k]
    assert f[st["depth"]] == 0


@pytest.mark.parametrize("n,small", [(256, -1), (1024, -1), (3000, -1)])
def test_hhs_step_thermal_binaries_unique_part_and_validity(fr, oracle, n, small, capsys):
    """Config 5's recipe unchanged (thermal eccentricities up to 0.99): an eccentric hard binary
    sweeps its time-step across several pivots every orbit, thousands of times per top step, and the
    oracle's own +-1-ulp trials then disagree with each other about the deepest levels' entry counts
    (reading 23).  Compared here: what is unique -- the bookkeeping of every level down to the first
    one on which the oracle's trials disagree must be IDENTICAL, and every particle must lie inside
    ENV_K x the oracle's envelope (which is ~1e-16 for everything but the hard binaries) -- and that
    the rest is valid: the structural invariants of Alg. 3's bookkeeping, momentum at rounding
    level, energy error of the oracle's size -- the oracle's own dE/E moves by up to 10x between its
    +-1-ulp trials here (2.3e-5 .. 2.1e-4 at n = 256: the truncation error of the e ~ 0.99 binaries
    depends on where along the orbit a pivot is crossed), so "the oracle's size" is the largest
    |dE/E| over the oracle's trials, and the GPU is held to twice that."""
    pos, vel, mass, pairs = fi.star_cluster(n, 4)
    dt = 2.0 ** -8
    fr.set_params(eta_ff=0.2, eta_fb=0.2)
    fr.set_tuning(0, 0, small)
    pr, vr, st_ref, env_p, env_v, sts, states = oracle_hhs_with_envelope(oracle, pos, vel, mass, dt,
                                                                         keep_states=True)
    p, v = dev(pos), dev(vel)
    try:
        st = fr.hhs_step(p, v, dev(mass), dt)
    finally:
        fr.set_tuning(0, 0, -1)
    hhs_stats_invariants(st)
    hhs_stats_invariants(st_ref)
    agree = 0                                   # levels on which all oracle trials agree
    keys = ("entries", "n_slow", "n_fast")
    while agree <= min(s["depth"] for s in sts + [st_ref]) and all(
            s[k][agree] == st_ref[k][agree] for s in sts for k in keys):
        agree += 1
    for k in keys:
        assert st[k][:agree] == st_ref[k][:agree], (k, agree)
    assert agree >= 6 and abs(st["depth"] - st_ref["depth"]) <= 2
    pg, vg = p.cpu().numpy(), v.cpu().numpy()
    rp, rv = envelope_ratio(pg, vg, pr, vr, env_p, env_v)
    e0 = oracle.diagnostics(pos, vel, mass)["E"]
    de_gpu = oracle.diagnostics(pg, vg, mass)["E"] / e0 - 1
    de_ref = oracle.diagnostics(pr, vr, mass)["E"] / e0 - 1
    de_size = max([abs(de_ref)] + [abs(oracle.diagnostics(pp, vv, mass)["E"] / e0 - 1) for pp, vv in states])
    with capsys.disabled():
        print(f"\n[hhs thermal n={n}] levels identical down to {agree - 1} of {st_ref['depth']} "
              f"(gpu depth {st['depth']}); envelope ratio x {rp:.3f}, v {rv:.3f}; dE/E gpu {de_gpu:.2e} oracle {de_ref:.2e} "
              f"(largest over its +-1-ulp trials {de_size:.2e})")
    assert rp <= 1.0 and rv <= 1.0, (rp, rv)
    assert momentum_change(mass, vel, vg, vr) <= 1.0
    assert abs(de_gpu) <= 2 * de_size + 1e-12


@pytest.mark.parametrize("n", [150, 700, 1024])
def test_subtree_kernel_one_cta_and_cluster_agree_bitwise(fr, n):
    """The device-resident subtree kernel on one CTA and on a thread-block cluster of replicas
    (large sweeps shared out by sinks) form a sink's sum with a different lane split, so the two
    agree to rounding, not bitwise; the bookkeeping must be identical (config 5's hardness, e <= 0.1
    so that the level sets do not depend on the last bit)."""
    pos, vel, mass, pairs = fi.star_cluster(n, 4, e_max=0.1)
    fr.set_params(eta_ff=0.2, eta_fb=0.2)
    out = []
    for one_cta in (1, 0):
        fr.set_tuning(0, 0, -1, one_cta)
        p, v = dev(pos), dev(vel)
        st = fr.hhs_step(p, v, dev(mass), 1.0 / 256)
        out.append((st, p.cpu().numpy(), v.cpu().numpy()))
    fr.set_tuning(0, 0, -1, 0)
    assert out[0][0] == out[1][0]
    assert out[0][0]["depth"] >= 12
    assert np.abs(out[0][1] - out[1][1]).max() < 1e-8 and np.abs(out[0][2] - out[1][2]).max() < 1e-3


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


FIG5_ETAS = (0.032, 0.064, 0.128, 0.256, 0.512, 1.024)


def test_solar_system_fig5_eta_sweep_order_four_and_fsi_gap(fr, oracle, capsys):
    """SURVEY 8(f).2 / Fig. 5 (Tables A1/A2): Sun + 4 giant planets
    for 45 top steps of 8192 days (1009 yr; the paper runs 1000 yr) at six accuracy parameters
    eta = 0.032 ... 1.024 (the truncation-dominated range: the paper sees round-off below 0.004).
      * HHS-FSI (frost_hhs_step, individual steps): max |dE/E| over the run follows eta^4
        (PAPER.md:664, 672): every doubling of eta multiplies it by 10..50 (16 = fourth order; the
        oracle gives 14.5-16.7 at both ends of the range and 30-38 between eta = 0.064 and 0.256,
        whatever the top step: DESIGN.md section 10), least-squares slope 4 +- 0.5 (oracle: 4.4);
      * the same span with all five bodies forced to the fastest level -- frost_fsi_steps at the
        smallest sub-step the hierarchy reached -- has a smaller error at every eta (the paper:
        "approximately an order of magnitude");
      * |dP| < 1e-15 and |dL/L| < 1e-13 in both arms;
      * the device run's final energy equals the oracle's run of the same steps to 1e-11 relative.
    The energy is read by frost_diagnostics after every top step; nothing else crosses the host."""
    dt_top, n_top = 8192.0, 45
    rows = []
    for eta in FIG5_ETAS:
        pos, vel, mass, G = fi.solar_system()
        vel = np.ascontiguousarray(vel - (vel * mass).sum(1, keepdims=True) / mass.sum())
        fr.set_params(G=G, eta_ff=eta, eta_fb=eta)
        p, v, m = dev(pos), dev(vel), dev(mass)
        pr, vr = pos.copy(), vel.copy()
        d0 = fr.diagnostics(p, v, m)
        L0 = np.array(d0["L"])
        de_hhs, depth = 0.0, 0
        for _ in range(n_top):
            st = fr.hhs_step(p, v, m, dt_top)
            oracle.hhs_step(pr, vr, mass, dt_top, G=G, eta_ff=eta, eta_fb=eta)
            depth = max(depth, st["depth"])
            de_hhs = max(de_hhs, abs(fr.diagnostics(p, v, m)["E"] / d0["E"] - 1))
        d1 = fr.diagnostics(p, v, m)
        e_ref = oracle.diagnostics(pr, vr, mass, G=G)["E"]
        assert abs(d1["E"] - e_ref) <= 1e-11 * abs(e_ref), (eta, d1["E"], e_ref)
        dp_hhs = np.abs(np.array(d1["P"]) - np.array(d0["P"])).max()
        dl_hhs = np.linalg.norm(np.array(d1["L"]) - L0) / np.linalg.norm(L0)
        # all five bodies on the fastest level: fsi with the step of the deepest level's fsi(S, tau/2)
        dt_min = dt_top * 2.0 ** -(depth + 1)
        per_top = int(round(dt_top / dt_min))
        p, v = dev(pos), dev(vel)
        de_fsi = 0.0
        for _ in range(n_top):
            fr.fsi_steps(p, v, m, dt_min, per_top)
            de_fsi = max(de_fsi, abs(fr.diagnostics(p, v, m)["E"] / d0["E"] - 1))
        d2 = fr.diagnostics(p, v, m)
        dp_fsi = np.abs(np.array(d2["P"]) - np.array(d0["P"])).max()
        dl_fsi = np.linalg.norm(np.array(d2["L"]) - L0) / np.linalg.norm(L0)
        rows.append((eta, depth, de_hhs, de_fsi, dp_hhs, dl_hhs, dp_fsi, dl_fsi))
    fr.set_params()
    slope = np.polyfit(np.log([r[0] for r in rows]), np.log([r[2] for r in rows]), 1)[0]
    with capsys.disabled():
        print("\n[Fig. 5] eta  depth  max|dE/E| HHS-FSI   FSI(fastest level)  ratio   |dP| HHS  |dL/L| HHS")
        for r in rows:
            print(f"[Fig. 5] {r[0]:5.3f} {r[1]:3d}   {r[2]:.3e}        {r[3]:.3e}         {r[2] / r[3]:6.1f}  "
                  f"{r[4]:.1e}  {r[5]:.1e}")
        print(f"[Fig. 5] log-log slope of the HHS-FSI energy error: {slope:.2f}")
    slope_fsi = np.polyfit(np.log([r[0] for r in rows]), np.log([r[3] for r in rows]), 1)[0]
    ratios = [rows[k + 1][2] / rows[k][2] for k in range(len(rows) - 1)]
    with capsys.disabled():
        print(f"[Fig. 5] error growth per doubling of eta: {' '.join(f'{x:.1f}' for x in ratios)}; "
              f"slope of the FSI arm {slope_fsi:.2f}")
    assert abs(slope - 4.0) <= 0.5, slope
    assert abs(slope_fsi - 4.0) <= 0.1, slope_fsi
    assert all(10.0 <= x <= 50.0 for x in ratios), ratios
    for eta, depth, de_hhs, de_fsi, dp_hhs, dl_hhs, dp_fsi, dl_fsi in rows:
        assert depth >= 2
        assert de_fsi < de_hhs, (eta, de_fsi, de_hhs)
        assert dp_hhs < 1e-15 and dp_fsi < 1e-15, (eta, dp_hhs, dp_fsi)
        assert dl_hhs < 1e-13 and dl_fsi < 1e-13, (eta, dl_hhs, dl_fsi)


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
