"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (planner on
auto).  Where the oracle cannot finish a full pass in seconds, sampled sinks are compared one by one
(each sink's sum is a pure function of the inputs, so a sample is exact evidence for those
outputs) and size-independent properties (momentum, bitwise determinism) cover the rest."""
import numpy as np
import pytest
import torch

import json
import os

import frost_inputs as fi
from test_gpu_parity import C_FWD, hhs_stats_invariants

pytestmark = pytest.mark.gpu
TOL_A, TOL_G, TOL_TAU = 1e-12, 1e-10, 1e-13
GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "config5_gate.json")


@pytest.fixture(scope="module")
def fr():
    import paper_2011_14984_b200 as frost
    f = frost.Frost()
    yield f
    f.close()


def dev(a):
    return torch.as_tensor(np.ascontiguousarray(a)).cuda()


def rel(x, ref):
    return float((np.abs(x - ref).max(0) / np.linalg.norm(ref, axis=0)).max())


def test_config2_full_pass_n65536(fr, oracle):
    """Config 2: N = 65536, full self acc+gradient pass plus the pairwise time-step pass, every
    output compared."""
    n = 65536
    pos, vel, mass = fi.plummer(n, 1)
    fr.set_params()
    a, g = fr.forces(dev(pos), dev(mass))
    tau, bins = fr.timesteps(dev(pos), dev(vel), dev(mass), tau_pivot=1.0 / 128)
    torch.cuda.synchronize()
    a_ref, g_ref = oracle.forces(pos, mass)
    tau_ref, bin_ref = oracle.timesteps(pos, vel, mass, tau_pivot=1.0 / 128)
    a, g = a.cpu().numpy(), g.cpu().numpy()
    assert rel(a, a_ref) <= TOL_A and rel(g, g_ref) <= TOL_G
    np.testing.assert_allclose(tau.cpu().numpy(), tau_ref, rtol=TOL_TAU)
    assert np.array_equal(bins.cpu().numpy(), bin_ref)
    assert np.abs((mass * a).sum(1)).max() < 1e-15 * (mass * np.abs(a)).sum(1).max()
    assert np.abs((mass * g).sum(1)).max() < 1e-13 * (mass * np.abs(g)).sum(1).max()


def test_config3_headline_pass_n2pow20_sampled(fr, oracle):
    """Config 3: N = 2^20 full pass; 384 random sinks compared one by one.  The oracle's gradient
    sum is fed the GPU's full acceleration array (step 3 is a pure function of (x, m, a)), the
    acceleration sample itself is checked end to end."""
    n = 1 << 20
    pos, vel, mass = fi.plummer(n, 2)
    fr.set_params()
    p, m = dev(pos), dev(mass)
    a, g = fr.forces(p, m)
    a2, g2 = fr.forces(p, m)
    torch.cuda.synchronize()
    assert torch.equal(a, a2) and torch.equal(g, g2)                  # bitwise reproducible
    a, g = a.cpu().numpy(), g.cpu().numpy()
    s = fi.active_subset(n, 384 / n, 77)
    a_ref = np.zeros((3, n)); g_ref = np.zeros((3, n))
    oracle.forces(pos, mass, sink_idx=s, flags=oracle.ACC, acc=a_ref, grad=g_ref)
    assert rel(a[:, s], a_ref[:, s]) <= TOL_A
    a_in = a.copy()
    oracle.forces(pos, mass, sink_idx=s, flags=oracle.GRAD, acc=a_in, grad=g_ref)
    assert rel(g[:, s], g_ref[:, s]) <= TOL_G
    assert np.abs((mass * a).sum(1)).max() < 1e-14 * (mass * np.abs(a)).sum(1).max()
    assert np.abs((mass * g).sum(1)).max() < 1e-12 * (mass * np.abs(g)).sum(1).max()


@pytest.mark.parametrize("frac", [0.001, 0.01, 0.1])
def test_config4_active_subsets_n2pow20(fr, oracle, frac):
    """Config 4: active set A (0.1 %, 1 %, 10 % of N = 2^20) against all sources, the reverse
    (all \\ A) <- A, both gradients, then the momentum-conserving kick of every particle."""
    n = 1 << 20
    pos, vel, mass = fi.plummer(n, 3)
    A = fi.active_subset(n, frac, 3)
    rest = np.setdiff1d(np.arange(n, dtype=np.int32), A).astype(np.int32)
    fr.set_params()
    p, m, v = dev(pos), dev(mass), dev(vel)
    dA, dR = dev(A), dev(rest)
    acc = torch.zeros_like(p); grad = torch.zeros_like(p)
    import paper_2011_14984_b200 as frost
    fr.forces(p, m, sink_idx=dA, source_idx=None, out_acc=acc, out_grad=grad, flags=frost.ACC)
    fr.forces(p, m, sink_idx=dR, source_idx=dA, out_acc=acc, out_grad=grad, flags=frost.ACC)
    fr.forces(p, m, sink_idx=dA, source_idx=None, out_acc=acc, out_grad=grad, flags=frost.GRAD)
    fr.forces(p, m, sink_idx=dR, source_idx=dA, out_acc=acc, out_grad=grad, flags=frost.GRAD)
    dt = 1.0 / 1024
    fr.kick(v, acc, grad, idx=None, c=2 * dt / 3, kappa=dt * dt / 48)
    torch.cuda.synchronize()
    a, g, vk = acc.cpu().numpy(), grad.cpu().numpy(), v.cpu().numpy()
    # sampled parity: 128 sinks of A (sources: all) and 128 of the rest (sources: A)
    sA, sR = A[:: max(1, A.size // 128)][:128], rest[:: rest.size // 128][:128]
    a_ref = np.zeros((3, n)); g_ref = np.zeros((3, n))
    oracle.forces(pos, mass, sink_idx=sA, source_idx=None, flags=oracle.ACC, acc=a_ref, grad=g_ref)
    oracle.forces(pos, mass, sink_idx=sR, source_idx=A, flags=oracle.ACC, acc=a_ref, grad=g_ref)
    assert rel(a[:, sA], a_ref[:, sA]) <= TOL_A and rel(a[:, sR], a_ref[:, sR]) <= TOL_A
    a_in = a.copy()
    oracle.forces(pos, mass, sink_idx=sA, source_idx=None, flags=oracle.GRAD, acc=a_in, grad=g_ref)
    oracle.forces(pos, mass, sink_idx=sR, source_idx=A, flags=oracle.GRAD, acc=a_in, grad=g_ref)
    assert rel(g[:, sA], g_ref[:, sA]) <= TOL_G and rel(g[:, sR], g_ref[:, sR]) <= TOL_G
    # pairwise (momentum-conserving) kick: sum m dv = 0 to roundoff
    dP = (mass * (vk - vel)).sum(1)
    scale = (mass * np.abs(vk - vel)).sum(1).max()
    assert np.abs(dP).max() < 1e-13 * scale


def test_config5_first_level_n262144(fr, oracle):
    """Config 5 at full size: the first hierarchy entry -- time-steps of all N = 262144 particles
    (sampled sinks), their bins, and the slow/fast partition at dt_top = 2^-7 (bit-exact given
    tau) -- plus the first inter-level sweep S<->F (sampled)."""
    n = 262144
    pos, vel, mass, pairs = fi.star_cluster(n, 4)
    pivot = 2.0 ** -7
    fr.set_params(eta_ff=0.2, eta_fb=0.2)
    p, v, m = dev(pos), dev(vel), dev(mass)
    tau, bins = fr.timesteps(p, v, m, tau_pivot=pivot)
    slow, fast = fr.partition(tau, pivot)
    torch.cuda.synchronize()
    tau_h, bins_h = tau.cpu().numpy(), bins.cpu().numpy()
    s = np.concatenate([[0], pairs[:64].ravel(), fi.active_subset(n, 256 / n, 9)]).astype(np.int32)
    # sampled sinks (central mass, binary members, random stars), each against the whole level
    tau_ref, bin_ref = oracle.timesteps_sampled(pos, vel, mass, s, tau_pivot=pivot)
    np.testing.assert_allclose(tau_h[s], tau_ref[s], rtol=TOL_TAU)
    assert np.array_equal(bins_h[s], bin_ref[s])
    k = bins_h.astype(np.float64)
    ok = np.isfinite(tau_h)
    assert (pivot * 2.0 ** -k[ok] <= tau_h[ok]).all()
    assert ((k[ok] == 0) | (tau_h[ok] < pivot * 2.0 ** -(k[ok] - 1))).all()
    idx = np.arange(n, dtype=np.int32)
    assert np.array_equal(slow.cpu().numpy(), idx[tau_h >= pivot])
    assert np.array_equal(fast.cpu().numpy(), idx[tau_h < pivot])
    assert fast.numel() >= 2 * pairs.shape[0] * 0.9 and bins_h.max() >= 10
    # first inter-level sweep, both directions, sampled
    import paper_2011_14984_b200 as frost
    S, F = slow.cpu().numpy(), fast.cpu().numpy()
    acc = torch.zeros_like(p); grad = torch.zeros_like(p)
    fr.forces(p, m, sink_idx=slow, source_idx=fast, out_acc=acc, out_grad=grad,
              flags=frost.ACC | frost.GRAD | frost.MUTUAL)
    torch.cuda.synchronize()
    a, g = acc.cpu().numpy(), grad.cpu().numpy()
    sS, sF = S[:: S.size // 64][:64], F[:: F.size // 64][:64]
    a_ref = np.zeros((3, n)); g_ref = np.zeros((3, n))
    oracle.forces(pos, mass, sink_idx=sS, source_idx=F, flags=oracle.ACC, acc=a_ref, grad=g_ref)
    oracle.forces(pos, mass, sink_idx=sF, source_idx=S, flags=oracle.ACC, acc=a_ref, grad=g_ref)
    assert rel(a[:, sS], a_ref[:, sS]) <= TOL_A and rel(a[:, sF], a_ref[:, sF]) <= TOL_A
    a_in = a.copy()
    oracle.forces(pos, mass, sink_idx=sS, source_idx=F, flags=oracle.GRAD, acc=a_in, grad=g_ref)
    oracle.forces(pos, mass, sink_idx=sF, source_idx=S, flags=oracle.GRAD, acc=a_in, grad=g_ref)
    assert rel(g[:, sS], g_ref[:, sS]) <= TOL_G and rel(g[:, sF], g_ref[:, sF]) <= TOL_G
    assert np.abs((mass * a).sum(1)).max() < 1e-13 * (mass * np.abs(a)).sum(1).max()
    # full self sweep ACC|GRAD over all 262144 particles at config 5's hardness, sampled sinks
    # (central mass, binary members, random stars): a to 1e-12; g through the forward-error gate of
    # DESIGN.md reading 22, the oracle's sums fed the GPU's full acceleration array
    acc, grad = fr.forces(p, m)
    torch.cuda.synchronize()
    a, g = acc.cpu().numpy(), grad.cpu().numpy()
    a_ref = np.zeros((3, n)); g_ref = np.zeros((3, n))
    oracle.forces(pos, mass, sink_idx=s, flags=oracle.ACC, acc=a_ref, grad=g_ref)
    assert rel(a[:, s], a_ref[:, s]) <= TOL_A
    a_in = a.copy()
    oracle.forces(pos, mass, sink_idx=s, flags=oracle.GRAD, acc=a_in, grad=g_ref)
    T = oracle.gradient_termsum(pos, mass, a_in, sink_idx=s)
    d = np.abs(g[:, s] - g_ref[:, s]).max(0)
    bound = TOL_G * np.linalg.norm(g_ref[:, s], axis=0) + C_FWD * 2.0 ** -53 * T[s]
    assert (d <= bound).all(), float((d / bound).max())


def test_config5_first_level_histogram_matches_golden_n262144(fr):
    """SURVEY 8(c) last pin row, first part: the time-step bins of the first hierarchy entry of
    config 5 at full size against the histogram the oracle wrote (tests/golden/config5_gate.json,
    made by tests/golden/make_config5_gate.py from oracle/ alone) -- identical, bin by bin."""
    gold = json.load(open(GOLDEN))["first_level"]
    n = gold["n"]
    pos, vel, mass, pairs = fi.star_cluster(n, gold["seed"])
    fr.set_params(eta_ff=gold["eta"], eta_fb=gold["eta"])
    tau, bins = fr.timesteps(dev(pos), dev(vel), dev(mass), tau_pivot=gold["dt_top"])
    torch.cuda.synchronize()
    hist = np.bincount(bins.cpu().numpy()[:n]).tolist()
    assert hist == gold["bin_histogram"]
    t = tau.cpu().numpy()[:n]
    assert int((t >= gold["dt_top"]).sum()) == gold["n_slow"] and int((t < gold["dt_top"]).sum()) == gold["n_fast"]
    assert abs(t.min() / gold["tau_min"] - 1) < TOL_TAU


def _conserved(fr, p, v, m):
    d = fr.diagnostics(p, v, m)
    return d["E"], np.array(d["P"]), np.array(d["L"])


def test_config5_full_step_gate_n262144(fr):
    """SURVEY 8(c) last pin row at full size: one whole HHS-FSI step of config 5 (N = 262144,
    dt_top = 2^-7; the launch configuration bench.py times).  What is a unique function of the input
    is compared exactly with the oracle's golden values -- |S|, |F| of the first entry --; the rest
    must be valid: the structural invariants of Alg. 3's bookkeeping, sum m dv at roundoff
    (PAPER.md:656, 698), |dL|/|L| < 1e-12, and an energy error no larger than
    the oracle's own on the N = 32768 replica (its two runs from inputs 1 ulp apart give 4.9e-7 and
    -2.0e-7: the energy error of one step is set by the few hardest binaries and is not reproducible
    beyond its size; reading 23)."""
    gold = json.load(open(GOLDEN))
    g0 = gold["first_level"]
    n = g0["n"]
    pos, vel, mass, pairs = fi.star_cluster(n, g0["seed"])
    fr.set_params(eta_ff=g0["eta"], eta_fb=g0["eta"])
    p, v, m = dev(pos), dev(vel), dev(mass)
    e0, p0, l0 = _conserved(fr, p, v, m)
    st = fr.hhs_step(p, v, m, g0["dt_top"])
    e1, p1, l1 = _conserved(fr, p, v, m)
    assert st["n_slow"][0] == g0["n_slow"] and st["n_fast"][0] == g0["n_fast"] and st["entries"][0] == 1
    hhs_stats_invariants(st)
    assert st["depth"] >= 20 and bool(torch.isfinite(p).all()) and bool(torch.isfinite(v).all())
    assert np.abs(p1 - p0).max() < 1e-15
    assert np.linalg.norm(l1 - l0) < 1e-12 * np.linalg.norm(l0)
    rep = gold["replica"]
    assert abs(e1 / e0 - 1) <= 2 * max(abs(rep["base"]["dE_rel"]), abs(rep["ulp_perturbed"]["dE_rel"]))


@pytest.mark.parametrize("split_max,kepler", [(32768, 0), (1 << 20, 0), (1 << 20, 1)])
def test_config5_full_step_with_split_levels_n262144(fr, split_max, kepler):
    """The same step with the fast levels split into components (frost_set_split; 2^20 = every level,
    the launch configuration bench.py times as `hhs_step_config5_split`, with frost_set_kepler as
    `hhs_step_config5_split_kepler`).  The slow / fast partition of level 0 is the one
    of Alg. 3: |S|, |F| equal the oracle's golden values.  The split levels
    cannot be run by the oracle at this size (its element-by-element parity is tests/test_gpu_split.py,
    n <= 3000); here: every level entered by as many components as its parent recursed into (twice
    each), sum m dv at roundoff, |dL|/|L| < 1e-12, energy error below the replica gate of the
    unsplit step, far fewer launches than hierarchy entries."""
    gold = json.load(open(GOLDEN))
    g0 = gold["first_level"]
    n = g0["n"]
    pos, vel, mass, pairs = fi.star_cluster(n, g0["seed"])
    fr.set_params(eta_ff=g0["eta"], eta_fb=g0["eta"])
    p, v, m = dev(pos), dev(vel), dev(mass)
    e0, p0, l0 = _conserved(fr, p, v, m)
    fr.set_split(split_max)
    fr.set_kepler(kepler)
    l_before = fr.launch_count()
    try:
        st = fr.hhs_step(p, v, m, g0["dt_top"])
    finally:
        fr.set_split(0)
        fr.set_kepler(0)
    launches = fr.launch_count() - l_before
    e1, p1, l1 = _conserved(fr, p, v, m)
    assert st["n_slow"][0] == g0["n_slow"] and st["n_fast"][0] == g0["n_fast"] and st["entries"][0] == 1
    e, c, s, f = st["entries"], st["n_comp"], st["n_slow"], st["n_fast"]
    for k in range(st["depth"]):
        # (two-body components on their Kepler orbits enter no level)
        assert e[k + 1] <= 2 * c[k], k
        assert (s[k + 1] + f[k + 1] <= 2 * f[k]) if kepler else (s[k + 1] + f[k + 1] == 2 * f[k]), k
    assert max(ck / ek for ck, ek in zip(c, e)) > 100          # thousands of binaries side by side
    assert st["depth"] >= (5 if kepler else 20) and bool(torch.isfinite(p).all()) and bool(torch.isfinite(v).all())
    assert (st["n_kepler"] > 100000) == bool(kepler)
    assert launches < 10000 and (kepler or sum(e) > 10000)
    assert np.abs(p1 - p0).max() < 1e-15
    assert np.linalg.norm(l1 - l0) < 1e-12 * np.linalg.norm(l0)
    rep = gold["replica"]
    assert abs(e1 / e0 - 1) <= 2 * max(abs(rep["base"]["dE_rel"]), abs(rep["ulp_perturbed"]["dE_rel"]))


def test_config5_replica_step_against_golden_n32768(fr):
    """The same gate with the oracle's WHOLE step beside it, on the N = 32768 replica of config 5
    (same recipe, seed and dt_top; a full-size oracle step would take ~12 h).  Level 0 is a unique
    function of the input: identical.  From level 1 on the oracle itself is not reproducible under
    a 1-ulp change of its input (golden: `levels_reproducible_under_1ulp` = 1 -- the second entry of
    level 1 already sees binaries whose phase depends on the last bit), so the deeper levels'
    populations must agree with the oracle's within 8 x the oracle's own 1-ulp difference plus 0.5 %,
    the pair counts within 0.1 %, and the conserved quantities must behave as the oracle's do."""
    rep = json.load(open(GOLDEN))["replica"]
    base, pert = rep["base"]["stats"], rep["ulp_perturbed"]["stats"]
    n = rep["n"]
    pos, vel, mass, pairs = fi.star_cluster(n, rep["seed"])
    fr.set_params(eta_ff=rep["eta"], eta_fb=rep["eta"])
    p, v, m = dev(pos), dev(vel), dev(mass)
    e0, p0, l0 = _conserved(fr, p, v, m)
    st = fr.hhs_step(p, v, m, rep["dt_top"])
    e1, p1, l1 = _conserved(fr, p, v, m)
    hhs_stats_invariants(st)
    for k in ("entries", "n_slow", "n_fast"):
        assert st[k][0] == base[k][0]
    assert abs(st["depth"] - base["depth"]) <= 1
    for lvl in range(1, min(st["depth"], base["depth"], pert["depth"]) + 1):
        for k in ("entries", "n_slow", "n_fast"):
            tol = 8 * abs(base[k][lvl] - pert[k][lvl]) + 0.005 * base[k][lvl] + 8
            assert abs(st[k][lvl] - base[k][lvl]) <= tol, (k, lvl, st[k][lvl], base[k][lvl], tol)
    for k in ("pairs_newton", "pairs_gradient", "pairs_timestep"):
        assert abs(st[k] / base[k] - 1) < 1e-3, k
    assert np.abs(p1 - p0).max() <= max(4 * rep["base"]["dP_max"], 1e-15)
    assert np.linalg.norm(l1 - l0) < 1e-12 * np.linalg.norm(l0)
    assert abs(e1 / e0 - 1) <= 4 * max(abs(rep["base"]["dE_rel"]), abs(rep["ulp_perturbed"]["dE_rel"]))


def test_config5_replica_split_kepler_step_against_golden_n32768(fr):
    """The N = 32768 replica with every level split into the components of its fast pairs and the
    two-body components on their Kepler orbits (frost_set_split(2^20) + frost_set_kepler)
    against the oracle's WHOLE step of the same definition (golden `replica_split`, written by
    tests/golden/make_config5_gate.py from oracle/ alone).  Without the deep binary recursion the
    oracle's bookkeeping is reproducible under a 1-ulp change of its input on every level, so the
    device's must be IDENTICAL: entries, |S|, |F|, components and propagator calls per level, pair
    counts -- through the pruned time-step sweep with edge output (level 0 has 32768 members), the
    S x F + G x R + masked-R kick decomposition and the batched component kernels.  Energy error equal
    to the oracle's to 1 %, momentum at roundoff."""
    rep = json.load(open(GOLDEN))["replica_split"]
    base, pert = rep["base"]["stats"], rep["ulp_perturbed"]["stats"]
    assert base == pert and rep["levels_reproducible_under_1ulp"] == base["depth"] + 1
    n = rep["n"]
    pos, vel, mass, pairs = fi.star_cluster(n, rep["seed"])
    fr.set_params(eta_ff=rep["eta"], eta_fb=rep["eta"])
    p, v, m = dev(pos), dev(vel), dev(mass)
    e0, p0, l0 = _conserved(fr, p, v, m)
    fr.set_split(rep["split_max"])
    fr.set_kepler(1 if rep["kepler"] else 0)
    try:
        st = fr.hhs_step(p, v, m, rep["dt_top"])
    finally:
        fr.set_split(0)
        fr.set_kepler(0)
    e1, p1, l1 = _conserved(fr, p, v, m)
    assert st == base
    assert abs((e1 / e0 - 1) / rep["base"]["dE_rel"] - 1) < 1e-2
    assert np.abs(p1 - p0).max() <= max(4 * rep["base"]["dP_max"], 1e-16)
    assert np.linalg.norm(l1 - l0) < 1e-13 * np.linalg.norm(l0)
