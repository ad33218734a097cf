#!/usr/bin/env python
"""bench.py -- headline measurement of the HHS-FSI hot path on B200.

Metric (BASELINE.json): ordered pair interactions per second of the fp64 Newton + gradient double
sweep on a Plummer sphere with N = 2^20 (config 3), plus the fraction of the B200 FP64 roofline.
One "step" = the middle stage of an FSI step on all particles, through the C-ABI:
    gather/pack -> Newton sweep -> slice reduction -> gradient sweep -> slice reduction
    -> kick with a~ = a + dt^2 g/48 -> drift            (Alg. 2 lines 5-7)
One "pair interaction" = one ordered pair visited once by each of the two sweeps.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--n 1048576] [--impl reference]

Prints ONE JSON line (rank 0).  See DESIGN.md "Measurement" for every field.  With --gpus N > 1 and
no torchrun environment the script re-launches itself under torch.distributed.run with N ranks
(one per GPU, NCCL).  Side modes used by the commands in profiles/*.md (no JSON line):
    --probe          print the FP64 issue-model table of this GPU (libfrost_probe.so, CUDA events)
    --rows-only      launch every O(N) kernel and the three time-step sweeps once or twice (for ncu)
    --subtree K      the device-resident subtree kernel on K/2 hard binaries (for ncu)
    --hhs-only       one HHS-FSI step of config 5 (N = 262144) with its validity numbers
    --hhs-plummer N  one HHS-FSI step of an equal-mass Plummer sphere of N particles (Alg. 3 / split + Kepler)
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import frost_inputs as fi  # noqa: E402

FLOPS_NEWTON, FLOPS_GRAD = 18, 34          # per ordered pair (FMA = 2, add/mul = 1, rsqrt = 1)
# FP64-pipe instructions per ORDERED pair as compiled: the pair-symmetric sweeps (frost_sym.cu) spend
# 20 (Newton) and 32 (gradient) per unordered pair; the one-sided sweeps 16 and 28 per ordered pair
SLOTS_NEWTON, SLOTS_GRAD = 10, 16
# ... and one DMUL less per unordered pair in their equal-mass variant (frost_set_equal_mass_path; config 3)
SLOTS_NEWTON_EQ, SLOTS_GRAD_EQ = 9.5, 15.5
SLOTS_NEWTON_1S, SLOTS_GRAD_1S = 16, 28
SM_COUNT, FP64_LANES_PER_SM = 148, 64      # B200: 64 FP64 FMA lanes per SM
SPLIT_MAX_CONFIG5 = 1 << 20                # frost_set_split for the split arms of the config-5 step: every level
METRIC = "pair interactions/s (acc+gradient, fp64) at N=2^20"
UNIT = "pair interactions/s"


def _sweep_traffic(variant, n, version):
    """dram__bytes_read.sum + dram__bytes_write.sum of one whole gradient sweep (all its band launches
    and reductions) from a committed ncu capture -- only if that capture was taken on the same size, the
    same kernel variant (eqmass | general | one_sided) and the same tile geometry as the running build
    (the geometry is part of frost_version()); else None with the reason.
    profiles/sym_gradient_traffic.csv: n,variant,geometry,dram_bytes,source."""
    path = os.path.join(ROOT, "profiles", "sym_gradient_traffic.csv")
    if os.path.exists(path):
        for ln in open(path):
            f = [x.strip() for x in ln.split(",", 4)]
            if len(f) >= 5 and f[0].isdigit() and int(f[0]) == n and f[1] == variant \
                    and f[2].replace(",", "") in version.replace(",", ""):
                return float(f[3]), f[4]
    return None, f"no ncu capture committed for n={n}, variant={variant}, build '{version}' (see profiles/)"


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        d = json.load(open(path))
        return d.get("hbm_gbs", 6650.0), d.get("sm_max_mhz", 1965.0), "measured"
    return 6650.0, 1965.0, "fallback"


_probe_lib = None


def fp64_probe(device, stream, mode, iters, blocks_per_sm, scratch):
    """frost_fp64_probe of libfrost_probe.so (paper_2011_14984_b200/probe/: measurement code, its own
    library, not part of the product ABI); returns the thread-level FP64 instructions it executes."""
    global _probe_lib
    import ctypes as C
    if _probe_lib is None:
        from paper_2011_14984_b200 import build as b
        _probe_lib = C.CDLL(b.build_probe())
        _probe_lib.frost_fp64_probe.argtypes = [C.c_int, C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_void_p,
                                                C.POINTER(C.c_int64)]
    n = C.c_int64()
    rc = _probe_lib.frost_fp64_probe(device, C.c_void_p(stream.cuda_stream), mode, iters, blocks_per_sm,
                                     C.c_void_p(scratch.data_ptr()), C.byref(n))
    if rc != 0:
        raise RuntimeError(f"frost_fp64_probe: status {rc}")
    return int(n.value)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                 "--format=csv,noheader,nounits", "-lms", "200"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.rows.append([x.strip() for x in ln.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
                for k, nm in enumerate(names):
                    if r[3 + k].lower().startswith("active"):
                        reasons.add(nm)
            except Exception:
                pass
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        busy = [s for s, p in zip(sm, pw) if p > 0.5 * max(pw)] or sm
        return {"sm_mhz": float(np.median(busy)), "sm_max_mhz": float(max(mx)),
                "power_w_max": float(max(pw)), "samples": len(sm), "reasons": sorted(reasons)}


def cpu_oracle_rate(n, seed, sample_sinks, acc_full=None):
    """The oracle as it stands, timed on the host cores on a bounded sample of the same workload:
    `sample_sinks` random sinks against all n sources, Newton sweep then gradient sweep."""
    import oracle
    pos, vel, mass = fi.plummer(n, seed)
    sinks = fi.active_subset(n, sample_sinks / n, seed + 100)
    acc = np.zeros((3, n)) if acc_full is None else acc_full.copy()
    grad = np.zeros((3, n))
    t0 = time.perf_counter()
    oracle.forces(pos, mass, sink_idx=sinks, source_idx=None, flags=oracle.ACC, acc=acc, grad=grad)
    t1 = time.perf_counter()
    oracle.forces(pos, mass, sink_idx=sinks, source_idx=None, flags=oracle.GRAD, acc=acc, grad=grad)
    t2 = time.perf_counter()
    pairs = float(sinks.size) * n
    return {"value": pairs / (t2 - t0), "unit": UNIT, "cores": oracle.num_threads(),
            "kind": "oracle", "newton_pairs_per_s": pairs / (t1 - t0),
            "gradient_pairs_per_s": pairs / (t2 - t1), "seconds": t2 - t0,
            "sample": f"{sinks.size} random sinks x all {n} sources, Newton then gradient sweep "
                      f"(long-double accumulation, OpenMP over sinks)"}, sinks, acc, grad


def run_reference(args):
    """--impl reference: the oracle on the host cores, same metric/config, bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    n, seed = args.n, 2
    sample = max(64, min(args.ref_sinks, n))
    vals = []
    for s in range(args.warmup + args.steps):
        r, *_ = cpu_oracle_rate(n, seed, sample)
        if s >= args.warmup:
            vals.append(r)
    val = float(np.mean([v["value"] for v in vals]))
    secs = float(np.mean([v["seconds"] for v in vals]))
    cb = dict(vals[-1]); cb["value"] = val
    out = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
           "steps": args.steps, "warmup": args.warmup, "ms_per_step": secs * 1e3,
           "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f64",
           "data": "synthetic",
           "config": {"workload": f"Plummer sphere N={n}, equal masses, G=1, seed 2 (config 3); "
                                  f"each step = {sample}-sink sample x all sources"},
           "cpu_baseline": cb,
           "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(out))



def measure_rows(fr, frost, torch, dev, flush, hbm_peak, hhs=True):
    """Side measurements of the other SURVEY.md 8(a) rows (not part of `value`): the time-step sweep
    on config 2, the HBM-bound O(N) kernels at N = 2^20 (algorithmic bytes per particle as in DESIGN.md),
    and a timed row with its oracle error for each of BASELINE.json's configs 1, 2, 4 and 5."""
    def ev():
        return torch.cuda.Event(enable_timing=True)

    def best(f, reps=5, do_flush=True):
        f(); torch.cuda.synchronize()
        ts = []
        for _ in range(reps):
            if do_flush:
                flush.fill_(1.0)
            a, b = ev(), ev()
            a.record(); f(); b.record(); torch.cuda.synchronize()
            ts.append(a.elapsed_time(b))
        return min(ts)

    out = {}
    n2 = 65536
    pos, vel, mass = fi.plummer(n2, 1)
    p, v, m = (torch.as_tensor(x).to(dev) for x in (pos, vel, mass))
    tau = torch.empty(n2, dtype=torch.float64, device=dev)
    bins = torch.empty(n2, dtype=torch.int32, device=dev)
    ms = best(lambda: fr.timesteps(p, v, m, tau_pivot=1.0 / 128, out_tau=tau, out_bin=bins), 3, False)
    out["timestep_sweep_config2"] = {"n": n2, "ms": ms, "pairs_per_s": float(n2) * n2 / (ms * 1e-3)}
    # O(N) kernels at N = 2^20: kReps launches back to back inside ONE event pair, each on its own set of
    # buffers (kSets x 24-32 MB per operand >> 126 MB of L2 in total, so every launch streams from HBM);
    # the launch gaps are inside the timed region, as they are in a step
    n = 1 << 20
    kSets, kReps = 8, 24
    mk = lambda: [torch.randn((3, n), dtype=torch.float64, device=dev) for _ in range(kSets)]
    xs, ws, as_, gs = mk(), mk(), mk(), mk()
    mms = [torch.rand(n, dtype=torch.float64, device=dev) for _ in range(kSets)]
    recs = [torch.empty((n, 4), dtype=torch.float64, device=dev) for _ in range(kSets)]
    lib, h = fr.lib, fr.h
    import ctypes as C
    P = lambda t: C.c_void_p(t.data_ptr())
    cases = {
        "kick_with_gradient": (96, lambda k: fr.kick(ws[k], as_[k], gs[k], c=1e-9, kappa=1e-9)),
        "kick": (72, lambda k: fr.kick(ws[k], as_[k], None, c=1e-9, kappa=0.0)),
        "drift": (72, lambda k: fr.drift(xs[k], ws[k], c=1e-12)),
        "gather_pack": (64, lambda k: lib.frost_gather_pack(h, n, n, P(xs[k]), P(mms[k]), None, 0, n, P(recs[k]))),
    }
    for name, (bpp, f) in cases.items():
        def many():
            for r in range(kReps):
                f(r % kSets)
        ms = best(many, 3) / kReps
        gbs = n * bpp / (ms * 1e-3) / 1e9
        out[name] = {"n": n, "us": ms * 1e3, "bytes_per_particle": bpp, "GB_per_s": gbs,
                     "frac_of_hbm_peak": gbs / hbm_peak,
                     "timing": f"{kReps} back-to-back launches over {kSets} rotating buffer sets, one event pair"}
    del xs, ws, as_, gs, mms, recs
    out.update(config_rows(fr, frost, torch, dev, flush))
    if hhs:
        out["hhs_step_config5"] = hhs_config5(fr, torch, dev)
        out["hhs_step_config5_split"] = hhs_config5(fr, torch, dev, split_max=SPLIT_MAX_CONFIG5)
        out["hhs_step_config5_split_kepler"] = hhs_config5(fr, torch, dev, split_max=SPLIT_MAX_CONFIG5, kepler=1)
    return out


def _rel_err(x, ref):
    return float((np.abs(x - ref).max(0) / np.linalg.norm(ref, axis=0)).max())


def config_rows(fr, frost, torch, dev, flush):
    """Driver-timed rows for BASELINE.json's configs 1, 2 and 4 (config 3 is the headline, config 5 the
    hhs_step_* rows), each with its error against the oracle on a sample so that the number carries its
    validity.  CUDA events on the context's stream; best of 3 after a warm-up call."""
    import oracle
    SLOT_PEAK = SM_COUNT * FP64_LANES_PER_SM * _peaks()[1] * 1e6

    def ev():
        return torch.cuda.Event(enable_timing=True)

    def timed(f, reps=3, do_flush=False):
        f(); torch.cuda.synchronize()
        ts = []
        for _ in range(reps):
            if do_flush:
                flush.fill_(1.0)
            a, b = ev(), ev()
            l0 = fr.launch_count()
            a.record(); f(); b.record(); torch.cuda.synchronize()
            ts.append((a.elapsed_time(b), fr.launch_count() - l0))
        return min(ts)

    T = lambda x: torch.as_tensor(np.ascontiguousarray(x)).to(dev)
    out = {}
    fr.set_params(G=1.0, eps2=0.0)

    # ---- config 1: N = 1024, seed 0: one acc+gradient evaluation; 10 FSI steps, dt = 1/1024 ----------
    n1, dt1 = 1024, 1.0 / 1024
    pos, vel, mass = fi.plummer(n1, 0)
    p, v, m = T(pos), T(vel), T(mass)
    acc = torch.zeros_like(p); grad = torch.zeros_like(p)
    ms, nl = timed(lambda: fr.forces(p, m, out_acc=acc, out_grad=grad), 5)
    a_ref, g_ref = oracle.forces(pos, mass)
    row = {"n": n1, "acc_grad_us": ms * 1e3, "acc_grad_launches": int(nl),
           "acc_rel_err": _rel_err(acc.cpu().numpy(), a_ref), "grad_rel_err": _rel_err(grad.cpu().numpy(), g_ref)}
    pr, vr = pos.copy(), vel.copy()
    for _ in range(10):
        oracle.fsi_step(pr, vr, mass, dt1)
    for name, small in (("resident", -1), ("streaming", 0)):
        fr.set_tuning(0, 0, small)
        state = {}

        def ten():
            state["p"], state["v"] = p.clone(), v.clone()
            fr.fsi_steps(state["p"], state["v"], m, dt1, 10)
        ms, nl = timed(ten, 3)          # (two 24 KB clones inside the timed region: < 1 % of either path)
        row[f"fsi10_{name}_us_per_step"] = ms * 1e2
        row[f"fsi10_{name}_launches"] = int(nl)
        row[f"fsi10_{name}_max_abs_dx_vs_oracle"] = float(np.abs(state["p"].cpu().numpy() - pr).max())
    fr.set_tuning(0, 0, -1)
    out["config1_n1024"] = row

    # ---- config 2: N = 65536, seed 1: full self acc+gradient pass (the time-step pass is its own row) --
    n2 = 65536
    pos, vel, mass = fi.plummer(n2, 1)
    p, m = T(pos), T(mass)
    acc = torch.zeros_like(p); grad = torch.zeros_like(p)
    ms, nl = timed(lambda: fr.forces(p, m, out_acc=acc, out_grad=grad), 3, True)
    s = fi.active_subset(n2, 256 / n2, 101)
    a_r = np.zeros((3, n2)); g_r = np.zeros((3, n2))
    oracle.forces(pos, mass, sink_idx=s, flags=oracle.ACC, acc=a_r, grad=g_r)
    a_in = acc.cpu().numpy().copy()
    oracle.forces(pos, mass, sink_idx=s, flags=oracle.GRAD, acc=a_in, grad=g_r)
    pairs = float(n2) * n2
    out["config2_acc_grad_n65536"] = {
        "n": n2, "ms": ms, "launches": int(nl), "pairs_per_s": pairs / (ms * 1e-3),
        "fp64_pipe_frac_at_max_clock": pairs * (SLOTS_NEWTON_EQ + SLOTS_GRAD_EQ) / (ms * 1e-3) / SLOT_PEAK,
        "acc_rel_err_256_sinks": _rel_err(acc.cpu().numpy()[:, s], a_r[:, s]),
        "grad_rel_err_256_sinks": _rel_err(grad.cpu().numpy()[:, s], g_r[:, s])}

    # ---- config 4: N = 2^20, seed 3: active subset A (0.1 / 1 / 10 %), pair set {i in A or j in A} ------
    n4, dt4 = 1 << 20, 1.0 / 1024
    pos, vel, mass = fi.plummer(n4, 3)
    p, m, v0 = T(pos), T(mass), T(vel)
    rows4 = {}
    for frac in (0.001, 0.01, 0.1):
        A = fi.active_subset(n4, frac, 3)
        rest = np.setdiff1d(np.arange(n4, dtype=np.int32), A).astype(np.int32)
        dA, dR = T(A), T(rest)
        acc = torch.zeros_like(p); grad = torch.zeros_like(p)

        def one_directional():      # A <- all, rest <- A (one-sided kernels with source slices)
            fr.forces(p, m, sink_idx=dA, source_idx=None, out_acc=acc, out_grad=grad, flags=frost.ACC)
            fr.forces(p, m, sink_idx=dR, source_idx=dA, out_acc=acc, out_grad=grad, flags=frost.ACC)
            fr.forces(p, m, sink_idx=dA, source_idx=None, out_acc=acc, out_grad=grad, flags=frost.GRAD)
            fr.forces(p, m, sink_idx=dR, source_idx=dA, out_acc=acc, out_grad=grad, flags=frost.GRAD)

        def self_plus_mutual():     # self(A) + mutual(A, rest) with FROST_ACCUMULATE (pair-symmetric kernels)
            acc.zero_(); grad.zero_()   # (the accumulating piece adds to whatever the rest holds)
            fr.forces(p, m, dA, dA, out_acc=acc, out_grad=grad, flags=frost.ACC)
            fr.forces(p, m, dA, dR, out_acc=acc, out_grad=grad, flags=frost.ACC | frost.MUTUAL | frost.ACCUMULATE)
            fr.forces(p, m, dA, dA, out_acc=acc, out_grad=grad, flags=frost.GRAD)
            fr.forces(p, m, dA, dR, out_acc=acc, out_grad=grad, flags=frost.GRAD | frost.MUTUAL | frost.ACCUMULATE)

        # ordered pairs of the set: A x all (minus self) + rest x A
        pairs = float(A.size) * n4 + float(rest.size) * A.size
        sA, sR = A[:: max(1, A.size // 64)][:64], rest[:: rest.size // 64][:64]
        a_ref = np.zeros((3, n4)); g_ref = np.zeros((3, n4))
        oracle.forces(pos, mass, sink_idx=sA, source_idx=None, flags=oracle.ACC, acc=a_ref, grad=g_ref)
        oracle.forces(pos, mass, sink_idx=sR, source_idx=A, flags=oracle.ACC, acc=a_ref, grad=g_ref)
        ss = np.concatenate([sA, sR])
        r = {"n_active": int(A.size), "ordered_pairs": pairs}
        for name, f in (("one_directional", one_directional), ("self_plus_mutual", self_plus_mutual)):
            ms, nl = timed(f, 2, True)
            a = acc.cpu().numpy()
            a_in = a.copy()
            oracle.forces(pos, mass, sink_idx=sA, source_idx=None, flags=oracle.GRAD, acc=a_in, grad=g_ref)
            oracle.forces(pos, mass, sink_idx=sR, source_idx=A, flags=oracle.GRAD, acc=a_in, grad=g_ref)
            vk = v0.clone()
            fr.kick(vk, acc, grad, idx=None, c=2 * dt4 / 3, kappa=dt4 * dt4 / 48)
            dv = vk.cpu().numpy() - vel
            r[name] = {"ms": ms, "launches": int(nl), "pairs_per_s": pairs / (ms * 1e-3),
                       "acc_rel_err_128_sinks": _rel_err(a[:, ss], a_ref[:, ss]),
                       "grad_rel_err_128_sinks": _rel_err(grad.cpu().numpy()[:, ss], g_ref[:, ss]),
                       "sum_m_dv_over_sum_m_abs_dv": float(np.abs((mass * dv).sum(1)).max() /
                                                           (mass * np.abs(dv)).sum(1).max())}
        rows4[f"active_{frac:g}"] = r
    out["config4_active_subsets_n2pow20"] = rows4
    fr.set_params()
    return out


def hhs_config5(fr, torch, dev, n5=262144, split_max=0, kepler=0):
    """Config 5: one whole HHS-FSI step over all time-step levels (latency-bound: DESIGN.md 7), with
    the numbers that make the timing valid: momentum, angular momentum and energy change read by
    frost_diagnostics before and after (SURVEY 8(c) last pin row; expected floors PAPER.md:646-656,
    696-698), and the level bookkeeping that tests/test_gpu_fullsize.py checks against the golden file."""
    pos5, vel5, mass5, _ = fi.star_cluster(n5, 4)
    p5, v5, m5 = (torch.as_tensor(x).to(dev) for x in (pos5, vel5, mass5))
    fr.set_params(G=1.0, eps2=0.0, eta_ff=0.2, eta_fb=0.2)
    d0 = fr.diagnostics(p5, v5, m5)
    fr.set_split(split_max)
    fr.set_kepler(kepler)
    l0 = fr.launch_count()
    torch.cuda.synchronize(); t0 = time.perf_counter()
    try:
        st = fr.hhs_step(p5, v5, m5, 2.0 ** -7)
    finally:
        fr.set_split(0)
        fr.set_kepler(0)
    torch.cuda.synchronize(); t1 = time.perf_counter()
    launches = int(fr.launch_count() - l0)
    d1 = fr.diagnostics(p5, v5, m5)
    L0, L1 = np.array(d0["L"]), np.array(d1["L"])
    return {"n": n5, "dt_top": 2.0 ** -7, "split_max": split_max, "kepler": kepler, "kepler_calls": int(st["n_kepler"]),
            "seconds": t1 - t0, "depth": st["depth"],
            "hierarchy_entries": int(sum(st["entries"])), "launches": launches,
            "pairs_newton": int(st["pairs_newton"]), "pairs_gradient": int(st["pairs_gradient"]),
            "pairs_timestep": int(st["pairs_timestep"]),
            "dP": float(np.abs(np.array(d1["P"]) - np.array(d0["P"])).max()),
            "dL_rel": float(np.linalg.norm(L1 - L0) / np.linalg.norm(L0)),
            "dE_rel": float(d1["E"] / d0["E"] - 1.0),
            "level0": {"n_slow": int(st["n_slow"][0]), "n_fast": int(st["n_fast"][0])},
            "entries_per_level": [int(x) for x in st["entries"]],
            "components_per_level": [int(x) for x in st["n_comp"]]}


def run_probe():
    """--probe: the FP64 issue-model table of this GPU: issue cycles per FP64 warp
    instruction per SM sub-partition at the max SM clock (2.0 = the nominal rate of a 16-lane pipe)."""
    import torch
    import paper_2011_14984_b200 as frost
    modes = [(1, "DADD, 2 distinct register pairs", 0),
             (2, "DMUL, 2 distinct register pairs", 0),
             (6, "DFMA, 2 register pairs + immediate", 0),
             (0, "DFMA, 1 register pair + 2 loop-invariant pairs (.reuse)", 0),
             (4, "DFMA, 3 distinct register pairs", 0),
             (5, "DFMA triples sharing one operand, adjacent (.reuse) [48 of 64] + 16 DADD", 0),
             (3, "mix: DFMA(2 pairs) / DADD / DMUL", 0),
             (7, "DADD + 12 integer-ALU instr per 16 FP64 instr", 12),
             (8, "DADD + 2 MUFU.RSQ64H per 16 FP64 instr", 2),
             (9, "DADD + 4 LDS.128 per 16 FP64 instr", 4)]
    _, mhz, _ = _peaks()
    fr = frost.Frost(0)
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    scratch = torch.zeros(sms * 8 * 256, dtype=torch.float64, device="cuda")
    ev = lambda: torch.cuda.Event(enable_timing=True)
    print(f"# {torch.cuda.get_device_name(0)}, {sms} SMs, cycles at {mhz:.0f} MHz; 4 CTAs x 256 threads per SM")
    print(f"# {'probe':78s} cyc/FP64-inst  extra cyc per extra instr")
    base = None
    for mode, name, extras in modes:
        fp64_probe(fr.device, fr.stream, mode, 2000, 4, scratch); torch.cuda.synchronize()
        a, b = ev(), ev()
        a.record(); ninst = fp64_probe(fr.device, fr.stream, mode, 40000, 4, scratch); b.record(); torch.cuda.synchronize()
        cyc = a.elapsed_time(b) * 1e-3 * mhz * 1e6 / (ninst / 32 / (sms * 4))
        if mode == 1:
            base = cyc
        extra = "" if not extras else f"{(cyc - base) * 16 / extras:6.2f}"
        print(f"  {name:78s} {cyc:6.3f}        {extra}")
    for mode, name in ((10, "DFMA"), (11, "DADD")):      # latency: 1 CTA of 8 warps per SM, one chain per thread
        fp64_probe(fr.device, fr.stream, mode, 2000, 1, scratch); torch.cuda.synchronize()
        a, b = ev(), ev()
        a.record(); fp64_probe(fr.device, fr.stream, mode, 40000, 1, scratch); b.record(); torch.cuda.synchronize()
        cyc = a.elapsed_time(b) * 1e-3 * mhz * 1e6 / (40000 * 64)
        print(f"  dependent {name} chain, 2 warps per sub-partition: {cyc:6.2f} cycles per instruction (latency)")
    fr.close()


def run_rows_only(n):
    """--rows-only: every kernel family of the path once or twice at a fixed size, for ncu: the O(N)
    kernels (gather/pack, kick, drift, partition) on n particles after an L2 flush, the time-step
    sweeps (plain symmetric, one-sided, pruned) on min(n, 65536) particles."""
    import torch
    import paper_2011_14984_b200 as frost
    pos, vel, mass = fi.plummer(n, 2)
    dev = torch.device("cuda", 0)
    p, v, m = (torch.as_tensor(x).to(dev) for x in (pos, vel, mass))
    a = torch.randn_like(p); g = torch.randn_like(p)
    tau = torch.rand(n, dtype=torch.float64, device=dev)
    flush = torch.empty(256 * 1024 * 1024 // 8, dtype=torch.float64, device=dev)
    fr = frost.Frost(0)
    for _ in range(2):
        flush.fill_(1.0); fr.gather_pack(p, m)
        flush.fill_(1.0); fr.kick(v, a, g, c=1e-9, kappa=1e-9)
        flush.fill_(1.0); fr.kick(v, a, None, c=1e-9, kappa=0.0)
        flush.fill_(1.0); fr.drift(p, v, c=1e-12)
        flush.fill_(1.0); fr.partition(tau, 0.5)
    n2 = min(n, 65536)
    p2, v2, m2 = p[:, :n2].contiguous(), v[:, :n2].contiguous(), m[:n2].contiguous()
    for mode in (3, 1, 0):      # plain symmetric sweep, one-sided sweep, default (pruned from 32768 particles)
        fr.set_symmetric(mode)
        fr.timesteps(p2, v2, m2, tau_pivot=1.0 / 128)
    torch.cuda.synchronize()
    fr.close()


def run_subtree(k):
    """--subtree K: the device-resident subtree kernel on a set of K/2 hard binaries (latency-bound)."""
    import torch
    import paper_2011_14984_b200 as frost
    pos, vel, mass, pairs = fi.star_cluster(4096, 4, binary_fraction=0.6)
    sel = pairs[: k // 2].ravel()
    dev = torch.device("cuda", 0)
    p = torch.as_tensor(np.ascontiguousarray(pos[:, sel])).to(dev)
    v = torch.as_tensor(np.ascontiguousarray(vel[:, sel])).to(dev)
    m = torch.as_tensor(mass[sel].copy()).to(dev)
    fr = frost.Frost(0)
    for _ in range(2):
        pp, vv = p.clone(), v.clone()
        torch.cuda.synchronize(); t0 = time.perf_counter()
        st = fr.hhs_step(pp, vv, m, 2.0 ** -12)
        torch.cuda.synchronize(); t1 = time.perf_counter()
    ent = sum(st["entries"])
    print(f"hierarchy entries: {ent} depth: {st['depth']} seconds: {t1 - t0:.4f} us/entry: {(t1 - t0) / ent * 1e6:.2f}")
    fr.close()


def run_hhs_only(arm):
    import torch
    import paper_2011_14984_b200 as frost
    fr = frost.Frost(0)
    dev = torch.device("cuda", 0)
    out = {}
    if arm in ("both", "alg3"):
        out["hhs_step_config5"] = hhs_config5(fr, torch, dev)
    if arm in ("both", "split"):
        out["hhs_step_config5_split"] = hhs_config5(fr, torch, dev, split_max=SPLIT_MAX_CONFIG5)
        out["hhs_step_config5_split_kepler"] = hhs_config5(fr, torch, dev, split_max=SPLIT_MAX_CONFIG5, kepler=1)
    print(json.dumps(out))
    fr.close()


def run_hhs_plummer(n):
    """--hhs-plummer N: one whole HHS-FSI step (dt_top = 2^-7, eta = 0.2) of an equal-mass Plummer sphere of
    N particles -- the paper's million-body setting in synthetic form -- with Alg. 3 as
    printed and with every level split + Kepler components; conserved quantities by frost_diagnostics."""
    import torch
    import paper_2011_14984_b200 as frost
    fr = frost.Frost(0)
    dev = torch.device("cuda", 0)
    pos, vel, mass = fi.plummer(n, 2)
    out = {}
    for name, split, kep in (("alg3", 0, 0), ("split_kepler", 1 << 20, 1)):
        p, v, m = (torch.as_tensor(x).to(dev) for x in (pos, vel, mass))
        fr.set_params(G=1.0, eps2=0.0, eta_ff=0.2, eta_fb=0.2)
        d0 = fr.diagnostics(p, v, m)
        fr.set_split(split); fr.set_kepler(kep)
        l0 = fr.launch_count()
        torch.cuda.synchronize(); t0 = time.perf_counter()
        st = fr.hhs_step(p, v, m, 2.0 ** -7)
        torch.cuda.synchronize(); t1 = time.perf_counter()
        fr.set_split(0); fr.set_kepler(0)
        d1 = fr.diagnostics(p, v, m)
        L0, L1 = np.array(d0["L"]), np.array(d1["L"])
        out[name] = {"n": n, "seconds": t1 - t0, "launches": int(fr.launch_count() - l0), "depth": st["depth"],
                     "hierarchy_entries": int(sum(st["entries"])), "kepler_calls": int(st["n_kepler"]),
                     "pairs_newton": int(st["pairs_newton"]), "pairs_gradient": int(st["pairs_gradient"]),
                     "pairs_timestep": int(st["pairs_timestep"]),
                     "dE_rel": float(d1["E"] / d0["E"] - 1.0),
                     "dP": float(np.abs(np.array(d1["P"]) - np.array(d0["P"])).max()),
                     "dL_rel": float(np.linalg.norm(L1 - L0) / np.linalg.norm(L0))}
    print(json.dumps({"hhs_step_plummer": out}))
    fr.close()


def run_frost(args):
    import torch
    import torch.distributed as dist
    import paper_2011_14984_b200 as frost
    from paper_2011_14984_b200 import sharding

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.same_device:
        local = 0            # every rank on cuda:0 (one-GPU execution of the N > 1 path; needs --backend gloo)
    torch.cuda.set_device(local)
    if world > 1:
        if args.backend == "nccl":
            dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        else:
            dist.init_process_group("gloo")      # exchanges staged through the host (sharding.py)
    n, seed, dt = args.n, 2, 1.0 / 1024
    hbm_peak, sm_max_mhz, peak_src = _peaks()

    pos_h, vel_h, mass_h = fi.plummer(n, seed)
    dev = torch.device("cuda", local)
    pos0 = torch.as_tensor(pos_h).to(dev)
    vel0 = torch.as_tensor(vel_h).to(dev)
    mass = torch.as_tensor(mass_h).to(dev)
    pos, vel = pos0.clone(), vel0.clone()
    acc = torch.zeros_like(pos); grad = torch.zeros_like(pos)
    fr = frost.Frost(local)
    fr.set_params(G=1.0, eps2=0.0)
    if args.one_sided:
        fr.set_symmetric(1)
    if args.no_eqmass:
        fr.set_equal_mass_path(0)
    # N > 1: the PAIRS are sharded (frost_set_shard: every rank sweeps 1/world of the tile pairs of
    # the symmetric kernels and holds partial sums for all particles; one all-reduce per sweep)
    lo, hi = 0, n
    sink_idx = None
    pair_sharded = world > 1 and not args.one_sided
    if pair_sharded:
        fr.set_shard(rank, world)
    elif world > 1:          # --one-sided: sinks sharded, all-gather of a between the sweeps
        lo, hi = sharding.shard_range(n, rank, world)
        sink_idx = torch.arange(lo, hi, dtype=torch.int32, device=dev)
    flush = torch.empty(256 * 1024 * 1024 // 8, dtype=torch.float64, device=dev)   # > 126 MB L2

    def ev():
        return torch.cuda.Event(enable_timing=True)

    def force_pass(pos, acc, grad, e=None):
        """Newton sweep, exchange of a, gradient sweep, exchange of g: this rank's share of the pairs
        (or of the sinks) and the one real exchange step of the path after each sweep."""
        fr.forces(pos, mass, sink_idx=sink_idx, source_idx=None, out_acc=acc, out_grad=grad,
                  flags=frost.ACC)
        if pair_sharded:
            sharding.all_reduce_planes(acc, world)
        elif world > 1:
            sharding.all_gather_planes(acc[:, lo:hi].contiguous(), n, rank, world, acc)
        if e: e[1].record()
        fr.forces(pos, mass, sink_idx=sink_idx, source_idx=None, out_acc=acc, out_grad=grad,
                  flags=frost.GRAD)
        if pair_sharded:
            sharding.all_reduce_planes(grad, world)

    def step(record=None):
        """One pass of the path; returns nothing, records events if asked."""
        e = [ev() for _ in range(4)] if record is not None else None
        if e: e[0].record()
        force_pass(pos, acc, grad, e)
        if e: e[2].record()
        fr.kick(vel, acc, grad, idx=sink_idx, c=2.0 * dt / 3.0, kappa=dt * dt / 48.0)
        fr.drift(pos, vel, idx=sink_idx, c=dt / 2.0)
        if e:
            e[3].record()
            record.append(e)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    launches0 = fr.launch_count()
    recs = []
    barrier()
    for _ in range(args.steps):
        flush.fill_(1.0)                         # L2 flush between timed iterations (not timed)
        torch.cuda.synchronize()
        step(recs)
        barrier()
    launches = fr.launch_count() - launches0
    clocks = sampler.stop() if rank == 0 else None
    t_step = [e[0].elapsed_time(e[3]) for e in recs]
    t_newton = [e[0].elapsed_time(e[1]) for e in recs]
    t_grad = [e[1].elapsed_time(e[2]) for e in recs]
    t_upd = [e[2].elapsed_time(e[3]) for e in recs]
    def max_over_ranks(x):
        t = torch.tensor([x], dtype=torch.float64, device=dev if args.backend == "nccl" else "cpu")
        if world > 1:
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    total_ms = max_over_ranks(sum(t_step))
    pairs_step = float(n) * float(n)
    value = pairs_step * args.steps / (total_ms * 1e-3)

    # ---- end to end through the host-buffer C-ABI entry (pinned host memory, copies timed) -------
    e2e = None
    if world == 1:
        hp = torch.as_tensor(pos_h).pin_memory(); hm = torch.as_tensor(mass_h).pin_memory()
        ha = torch.zeros((3, n), dtype=torch.float64).pin_memory()
        hg = torch.zeros((3, n), dtype=torch.float64).pin_memory()
        fr.forces_host(hp, hm, out_acc=ha, out_grad=hg)            # warm-up (allocates staging)
        ts = []
        for _ in range(max(1, args.e2e_steps)):
            flush.fill_(1.0); torch.cuda.synchronize()
            t0 = time.perf_counter()
            fr.forces_host(hp, hm, out_acc=ha, out_grad=hg)        # synchronises internally
            ts.append(time.perf_counter() - t0)
        e2e = {"value": pairs_step / float(np.mean(ts)), "unit": UNIT,
               "h2d_bytes_per_step": int(hp.numel() * 8 + hm.numel() * 8),   # acc / grad are pure outputs here
               "d2h_bytes_per_step": int(ha.numel() * 8 + hg.numel() * 8),
               "steps": len(ts), "ms_per_step": float(np.mean(ts)) * 1e3}

    if world > 1:
        # N > 1: the state is replicated, so every rank copies pos and mass from its pinned host buffers,
        # sweeps its share, takes part in the two exchanges, and rank 0 reads a and g back; wall clock
        # between barriers, max over ranks
        hp = torch.as_tensor(pos_h).pin_memory(); hm = torch.as_tensor(mass_h).pin_memory()
        ha = torch.zeros((3, n), dtype=torch.float64).pin_memory()
        hg = torch.zeros((3, n), dtype=torch.float64).pin_memory()
        dp = torch.empty_like(pos0)
        da, dg = torch.zeros_like(pos0), torch.zeros_like(pos0)
        ts = []
        for it in range(1 + max(1, args.e2e_steps)):
            flush.fill_(1.0); barrier()
            t0 = time.perf_counter()
            dp.copy_(hp, non_blocking=True); mass.copy_(hm, non_blocking=True)
            force_pass(dp, da, dg)
            if rank == 0:
                ha.copy_(da, non_blocking=True); hg.copy_(dg, non_blocking=True)
            barrier()
            if it > 0:
                ts.append(max_over_ranks(time.perf_counter() - t0))
        e2e = {"value": pairs_step / float(np.mean(ts)), "unit": UNIT,
               "h2d_bytes_per_step": int(world * (hp.numel() + hm.numel()) * 8),
               "d2h_bytes_per_step": int((ha.numel() + hg.numel()) * 8),
               "steps": len(ts), "ms_per_step": float(np.mean(ts)) * 1e3,
               "note": "per-rank H2D of the replicated state + sharded sweeps + exchanges + D2H on rank 0"}
        # every rank: the sharded pass at the ORIGINAL positions (rank 0 compares it with the oracle and
        # with the unsharded pass below; --dump-dir keeps every rank's copy for tests/)
        a_sh, g_sh = torch.zeros_like(pos0), torch.zeros_like(pos0)
        force_pass(pos0, a_sh, g_sh)
        torch.cuda.synchronize()
        if args.dump_dir:
            os.makedirs(args.dump_dir, exist_ok=True)
            np.savez(os.path.join(args.dump_dir, f"rank{rank}.npz"), acc=a_sh.cpu().numpy(), grad=g_sh.cpu().numpy(),
                     lo=lo, hi=hi)

    if rank != 0:
        if world > 1:
            dist.barrier()                       # stay until rank 0 has printed its line
            dist.destroy_process_group()
        return

    # ---- FP64 issue-rate probe: measured sustained pipe rate (MEASURED_PEAKS.json has none) ------
    probe = {}
    scratch = torch.zeros(torch.cuda.get_device_properties(local).multi_processor_count * 8 * 256,
                          dtype=torch.float64, device=dev)
    for mode, nm in ((0, "dfma"), (3, "mixed")):
        fp64_probe(fr.device, fr.stream, mode, 2000, 4, scratch); torch.cuda.synchronize()
        a, b = ev(), ev()
        a.record(); ninst = fp64_probe(fr.device, fr.stream, mode, 60000, 4, scratch); b.record(); torch.cuda.synchronize()
        probe[nm + "_thread_inst_per_s"] = ninst / (a.elapsed_time(b) * 1e-3)

    sm_mhz = (clocks or {}).get("sm_mhz") or sm_max_mhz
    peak_tflops = SM_COUNT * FP64_LANES_PER_SM * 2 * sm_max_mhz * 1e6 / 1e12
    slot_peak = SM_COUNT * FP64_LANES_PER_SM * sm_max_mhz * 1e6          # thread-level FP64 inst / s
    g_ms = float(np.mean(t_grad)); n_ms = float(np.mean(t_newton))
    sinks_here = hi - lo
    pairs_rank = float(n) * n / world if pair_sharded else float(sinks_here) * n
    variant = "general"
    if args.one_sided:      # forced: the one-sided sweeps run
        variant = "one_sided"
        slots_n, slots_g, kname = SLOTS_NEWTON_1S, SLOTS_GRAD_1S, "sweep_kernel<GradientPolicy> (one-sided gradient sweep, Eq. 27)"
    elif bool((mass_h == mass_h[0]).all()) and not args.no_eqmass:
        variant = "eqmass"
        slots_n, slots_g = SLOTS_NEWTON_EQ, SLOTS_GRAD_EQ
        kname = "sym_kernel<SymGradientFastT<true>> (pair-symmetric gradient sweep, Eq. 27; equal-mass variant, no coincidence guard)"
    else:
        slots_n, slots_g, kname = SLOTS_NEWTON, SLOTS_GRAD, "sym_kernel<SymGradientFastT<false>> (pair-symmetric gradient sweep, Eq. 27)"
    traffic, traffic_src = _sweep_traffic(variant, n, fr.lib.frost_version().decode())
    # measured FP64 rate of this run's probe (MEASURED_PEAKS.json carries no fp64 entry): a DFMA with two
    # loop-invariant operands issues every 2 cycles, i.e. thread instructions/s x 2 flop
    peak_measured = probe.get("dfma_thread_inst_per_s", 0.0) * 2 / 1e12
    roof = {"bound": "alu", "kernel": kname,
            "achieved": pairs_rank * FLOPS_GRAD / (g_ms * 1e-3) / 1e12, "peak": peak_tflops,
            "unit": "TFLOP/s",
            "traffic": traffic, "traffic_scope": traffic_src,
            "peak_source": f"derived: {SM_COUNT} SMs x {FP64_LANES_PER_SM} FP64 lanes x 2 x "
                           f"{sm_max_mhz:.0f} MHz ({peak_src} sm_max_mhz); HBM peak n/a",
            "peak_measured": peak_measured,
            "peak_measured_source": "frost_fp64_probe mode 0 (DFMA, register-only chains) timed in this run",
            "flops_per_pair": FLOPS_GRAD, "fp64_slots_per_pair": slots_g,
            "ms_per_launch": g_ms,
            "fp64_pipe_frac_at_max_clock": pairs_rank * slots_g / (g_ms * 1e-3) / slot_peak,
            "fp64_pipe_frac_at_sampled_clock":
                pairs_rank * slots_g / (g_ms * 1e-3) / (slot_peak * sm_mhz / sm_max_mhz),
            "newton": {"ms_per_launch": n_ms,
                       "achieved": pairs_rank * FLOPS_NEWTON / (n_ms * 1e-3) / 1e12,
                       "fp64_pipe_frac_at_max_clock": pairs_rank * slots_n / (n_ms * 1e-3) / slot_peak},
            "probe": probe,
            "probe_dfma_frac_of_nominal": probe.get("dfma_thread_inst_per_s", 0.0) / slot_peak}
    if peak_measured > 0:
        roof["frac_of_peak_measured"] = roof["achieved"] / peak_measured
    roof["frac"] = roof["achieved"] / roof["peak"]
    roof["step_tflops"] = value * (FLOPS_NEWTON + FLOPS_GRAD) / 1e12
    roof["step_frac"] = roof["step_tflops"] / peak_tflops

    # ---- the oracle as it stands on the host cores, bounded sample; doubles as a full-size check -
    cpu = None
    if not args.no_cpu:
        acc_np = acc.cpu().numpy()
        cpu, sinks, acc_ref, grad_ref = cpu_oracle_rate(n, seed, args.cpu_sinks, acc_full=acc_np)
        # positions drifted after the last step: recompute the GPU result at the ORIGINAL positions
        a_chk = torch.zeros_like(pos0); g_chk = torch.zeros_like(pos0)
        fr.set_shard(0, 1)                       # the check is a whole (unsharded) pass on rank 0
        fr.forces(pos0, mass, out_acc=a_chk, out_grad=g_chk)
        torch.cuda.synchronize()
        a_g = a_chk.cpu().numpy()
        import oracle
        a_r = np.zeros((3, n)); g_r = np.zeros((3, n))
        oracle.forces(pos_h, mass_h, sink_idx=sinks[:256], flags=oracle.ACC, acc=a_r, grad=g_r)
        a_mix = a_g.copy()
        oracle.forces(pos_h, mass_h, sink_idx=sinks[:256], flags=oracle.GRAD, acc=a_mix, grad=g_r)
        s = sinks[:256]
        ea = (np.abs(a_g[:, s] - a_r[:, s]).max(0) / np.linalg.norm(a_r[:, s], axis=0)).max()
        eg = (np.abs(g_chk.cpu().numpy()[:, s] - g_r[:, s]).max(0) / np.linalg.norm(g_r[:, s], axis=0)).max()
        cpu["parity_on_256_sampled_sinks"] = {"acc_rel_err": float(ea), "grad_rel_err": float(eg)}
        if world > 1:      # the sharded + exchanged pass of this rank against the same oracle sample
            own = s if pair_sharded else s[(s >= lo) & (s < hi)]
            cpu["parity_of_the_sharded_pass"] = {
                "acc_rel_err": float((np.abs(a_sh.cpu().numpy()[:, s] - a_r[:, s]).max(0) / np.linalg.norm(a_r[:, s], axis=0)).max()),
                "grad_rel_err": float((np.abs(g_sh.cpu().numpy()[:, own] - g_r[:, own]).max(0) /
                                       np.linalg.norm(g_r[:, own], axis=0)).max()) if own.size else None}

    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True,
           "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": f"Plummer sphere N={n}, equal masses, G=1, seed 2 (config 3): full "
                                  "self acc+gradient pass + kick + drift per step",
                      "l2": "flushed between timed iterations (256 MB fill)",
                      "parallelism": "1 GPU" if world == 1 else (
                          f"tile pairs of the symmetric sweeps sharded over {world} ranks, all-reduce of a "
                          "and of g" if pair_sharded else
                          f"sinks sharded over {world} ranks, all-gather of a between the sweeps"),
                      "backend": None if world == 1 else args.backend + (", all ranks on cuda:0" if args.same_device else "")},
           "gflops": value * (FLOPS_NEWTON + FLOPS_GRAD) / 1e9,
           "flops_convention": "Newton 18 + gradient 34 = 52 flops per ordered pair (FMA=2, add/mul=1, rsqrt=1)",
           "breakdown_ms": {"newton+pack+reduce": n_ms, "gradient+pack+reduce": g_ms,
                            "kick+drift": float(np.mean(t_upd))},
           "gpu_launches": int(launches), "clocks": clocks, "roofline": roof,
           "cpu_baseline": cpu, "e2e": e2e}
    if world == 1 and not args.no_rows:
        out["other_rows"] = measure_rows(fr, frost, torch, dev, flush, hbm_peak, hhs=not args.no_hhs)
    print(json.dumps(out), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--n", "--particles", dest="n", type=int, default=1 << 20)
    ap.add_argument("--impl", default="frost", choices=["frost", "reference"])
    ap.add_argument("--cpu-sinks", type=int, default=6144)
    ap.add_argument("--one-sided", action="store_true", help="force the one-sided sweeps (no pair symmetry)")
    ap.add_argument("--ref-sinks", type=int, default=1024)
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--backend", default="nccl", choices=["nccl", "gloo"],
                    help="process-group backend for --gpus N > 1 (gloo: exchanges staged through the host)")
    ap.add_argument("--same-device", action="store_true",
                    help="all ranks on cuda:0 (executes the N > 1 path on a one-GPU box; needs --backend gloo)")
    ap.add_argument("--dump-dir", default="", help="N > 1: every rank saves its sharded acc / grad at the initial positions here")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-rows", action="store_true", help="skip the side measurements of the O(N) rows")
    ap.add_argument("--no-hhs", action="store_true", help="skip the config-5 HHS-FSI step (about 15 s)")
    ap.add_argument("--probe", action="store_true", help="print the FP64 issue-model table and exit")
    ap.add_argument("--rows-only", action="store_true", help="launch the O(N) kernels and time-step sweeps (for ncu)")
    ap.add_argument("--subtree", type=int, default=0, help="run the subtree kernel on K/2 hard binaries (for ncu)")
    ap.add_argument("--hhs-only", action="store_true", help="one HHS-FSI step of config 5 with its validity numbers")
    ap.add_argument("--hhs-plummer", type=int, default=0, help="one HHS-FSI step of a Plummer sphere of N particles")
    ap.add_argument("--no-eqmass", action="store_true", help="general kernels even on equal masses (frost_set_equal_mass_path(0))")
    ap.add_argument("--hhs-arm", default="both", choices=["both", "alg3", "split"],
                    help="--hhs-only: Alg. 3 as printed, the split fast levels (frost_set_split), or both")
    args = ap.parse_args()
    if args.same_device and args.backend != "gloo":
        ap.error("--same-device needs --backend gloo (NCCL refuses two ranks on one device)")
    if args.probe:
        return run_probe()
    if args.rows_only:
        return run_rows_only(args.n)
    if args.subtree:
        return run_subtree(args.subtree)
    if args.hhs_only:
        return run_hhs_only(args.hhs_arm)
    if args.hhs_plummer:
        return run_hhs_plummer(args.hhs_plummer)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # not under torchrun: launch one rank per GPU ourselves (rank 0 prints the JSON line)
        import socket
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)]
        # (torch.distributed.run's own parser rejects "--n" even behind the script name: it is an ambiguous
        #  prefix of --nnodes / --nproc-per-node / ...; the long spelling is not)
        cmd += ["--particles" if a == "--n" else a.replace("--n=", "--particles=", 1) if a.startswith("--n=") else a
                for a in sys.argv[1:]]
        env = dict(os.environ)
        env.setdefault("NCCL_DEBUG", "INFO")              # the communicator log shows the N ranks ...
        env.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
        env.setdefault("NCCL_DEBUG_FILE", "/dev/stderr")  # ... and stays off stdout (one JSON line)
        sys.exit(subprocess.call(cmd, env=env))
    if args.impl == "reference":
        run_reference(args)
    else:
        world = int(os.environ.get("WORLD_SIZE", "1"))
        if world != args.gpus:
            sys.stderr.write(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}; using WORLD_SIZE\n")
        run_frost(args)


if __name__ == "__main__":
    main()
