#!/usr/bin/env python
"""bench.py -- headline measurement of the HHS-FSI hot path on B200.

Metric (BASELINE.json): ordered pair interactions per second of the fp64 Newton + gradient double
sweep on a Plummer sphere with N = 2^20 (config 3), plus the fraction of the B200 FP64 roofline.
One "step" = the middle stage of an FSI step on all particles, through the C-ABI:
    gather/pack -> Newton sweep -> slice reduction -> gradient sweep -> slice reduction
    -> kick with a~ = a + dt^2 g/48 -> drift            (Alg. 2 lines 5-7)
One "pair interaction" = one ordered pair visited once by each of the two sweeps.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--n 1048576] [--impl reference]

Prints ONE JSON line (rank 0).  See DESIGN.md "Measurement" for every field.
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
SLOTS_NEWTON_1S, SLOTS_GRAD_1S = 16, 28
SM_COUNT, FP64_LANES_PER_SM = 148, 64      # B200: 64 FP64 FMA lanes per SM
METRIC = "pair interactions/s (acc+gradient, fp64) at N=2^20"
UNIT = "pair interactions/s"


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        d = json.load(open(path))
        return d.get("hbm_gbs", 6650.0), d.get("sm_max_mhz", 1965.0), "measured"
    return 6650.0, 1965.0, "fallback"


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
    for s in range(args.warmup_ref + args.steps):
        r, *_ = cpu_oracle_rate(n, seed, sample)
        if s >= args.warmup_ref:
            vals.append(r)
    val = float(np.mean([v["value"] for v in vals]))
    secs = float(np.mean([v["seconds"] for v in vals]))
    cb = dict(vals[-1]); cb["value"] = val
    out = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
           "steps": args.steps, "warmup": args.warmup_ref, "ms_per_step": secs * 1e3,
           "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f64",
           "data": "synthetic",
           "config": {"workload": f"Plummer sphere N={n}, equal masses, G=1, seed 2 (config 3); "
                                  f"each step = {sample}-sink sample x all sources"},
           "cpu_baseline": cb,
           "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(out))



def measure_rows(fr, frost, torch, dev, flush, hbm_peak, hhs=True):
    """Side measurements of the other SURVEY.md 8(a) rows (not part of `value`): the time-step sweep
    on config 2 and the HBM-bound O(N) kernels at N = 2^20 (L2 flushed before every timed launch;
    algorithmic bytes per particle as in DESIGN.md)."""
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
    n = 1 << 20
    x = torch.randn((3, n), dtype=torch.float64, device=dev)
    w = torch.randn((3, n), dtype=torch.float64, device=dev)
    a = torch.randn((3, n), dtype=torch.float64, device=dev)
    g = torch.randn((3, n), dtype=torch.float64, device=dev)
    mm = torch.rand(n, dtype=torch.float64, device=dev)
    rec = torch.empty((n, 4), dtype=torch.float64, device=dev)
    lib, h = fr.lib, fr.h
    import ctypes as C
    P = lambda t: C.c_void_p(t.data_ptr())
    cases = {
        "kick_with_gradient": (96, lambda: fr.kick(w, a, g, c=1e-9, kappa=1e-9)),
        "kick": (72, lambda: fr.kick(w, a, None, c=1e-9, kappa=0.0)),
        "drift": (72, lambda: fr.drift(x, w, c=1e-12)),
        "gather_pack": (64, lambda: lib.frost_gather_pack(h, n, n, P(x), P(mm), None, 0, n, P(rec))),
    }
    for name, (bpp, f) in cases.items():
        ms = best(f)
        gbs = n * bpp / (ms * 1e-3) / 1e9
        out[name] = {"n": n, "us": ms * 1e3, "bytes_per_particle": bpp, "GB_per_s": gbs,
                     "frac_of_hbm_peak": gbs / hbm_peak}
    if hhs:
        # config 5: one whole HHS-FSI step over all time-step levels (latency-bound: DESIGN.md 7)
        n5 = 262144
        pos5, vel5, mass5, _ = fi.star_cluster(n5, 4)
        p5, v5, m5 = (torch.as_tensor(x).to(dev) for x in (pos5, vel5, mass5))
        fr.set_params(G=1.0, eps2=0.0, eta_ff=0.2, eta_fb=0.2)
        l0 = fr.launch_count()
        torch.cuda.synchronize(); t0 = time.perf_counter()
        st = fr.hhs_step(p5, v5, m5, 2.0 ** -7)
        torch.cuda.synchronize(); t1 = time.perf_counter()
        out["hhs_step_config5"] = {"n": n5, "dt_top": 2.0 ** -7, "seconds": t1 - t0, "depth": st["depth"],
                                   "hierarchy_entries": int(sum(st["entries"])),
                                   "launches": int(fr.launch_count() - l0),
                                   "pairs_newton": int(st["pairs_newton"]),
                                   "pairs_gradient": int(st["pairs_gradient"]),
                                   "pairs_timestep": int(st["pairs_timestep"])}
    return out


def run_frost(args):
    import torch
    import torch.distributed as dist
    import paper_2011_14984_b200 as frost
    from paper_2011_14984_b200 import sharding

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
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

    def step(record=None):
        """One pass of the path; returns nothing, records events if asked."""
        e = [ev() for _ in range(4)] if record is not None else None
        if e: e[0].record()
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
    total_ms = torch.tensor([sum(t_step)], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(total_ms, op=dist.ReduceOp.MAX)
    total_ms = float(total_ms.item())
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
               "h2d_bytes_per_step": int(hp.numel() * 8 + hm.numel() * 8 + ha.numel() * 8 + hg.numel() * 8),
               "d2h_bytes_per_step": int(ha.numel() * 8 + hg.numel() * 8),
               "steps": len(ts), "ms_per_step": float(np.mean(ts)) * 1e3}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- FP64 issue-rate probe: measured sustained pipe rate (MEASURED_PEAKS.json has none) ------
    probe = {}
    scratch = torch.zeros(148 * 8 * 256 * 2, dtype=torch.float64, device=dev)
    for mode, nm in ((0, "dfma"), (3, "mixed")):
        fr.fp64_probe(mode, 2000, 4, scratch); torch.cuda.synchronize()
        a, b = ev(), ev()
        a.record(); ninst = fr.fp64_probe(mode, 60000, 4, scratch); b.record(); torch.cuda.synchronize()
        probe[nm + "_thread_inst_per_s"] = ninst / (a.elapsed_time(b) * 1e-3)

    sm_mhz = (clocks or {}).get("sm_mhz") or sm_max_mhz
    peak_tflops = SM_COUNT * FP64_LANES_PER_SM * 2 * sm_max_mhz * 1e6 / 1e12
    slot_peak = SM_COUNT * FP64_LANES_PER_SM * sm_max_mhz * 1e6          # thread-level FP64 inst / s
    g_ms = float(np.mean(t_grad)); n_ms = float(np.mean(t_newton))
    sinks_here = hi - lo
    pairs_rank = float(n) * n / world if pair_sharded else float(sinks_here) * n
    if args.one_sided:      # forced: the one-sided sweeps run
        slots_n, slots_g, kname = SLOTS_NEWTON_1S, SLOTS_GRAD_1S, "sweep_kernel<GradientPolicy> (one-sided gradient sweep, Eq. 27)"
    else:
        slots_n, slots_g, kname = SLOTS_NEWTON, SLOTS_GRAD, "sym_kernel<SymGradient> (pair-symmetric gradient sweep, Eq. 27)"
    roof = {"bound": "alu", "kernel": kname,
            "achieved": pairs_rank * FLOPS_GRAD / (g_ms * 1e-3) / 1e12, "peak": peak_tflops,
            "unit": "TFLOP/s",
            # dram__bytes_read+write of ONE band launch (gradient band 3 of 13) from the committed
            # ncu --set full capture, profiles/sym_ncu_full_r1b.md; bands 1-3 measured 0.51 / 0.86 /
            # 1.30 GB, a whole sweep ~26 GB (the B-side partial sums) = ~20 GB/s: ALU-bound
            "traffic": None if args.one_sided else 1.3047e9,
            "traffic_scope": "one band launch of 13 per sweep (profiles/sym_ncu_full_r1b.md)",
            "peak_source": f"derived: {SM_COUNT} SMs x {FP64_LANES_PER_SM} FP64 lanes x 2 x "
                           f"{sm_max_mhz:.0f} MHz ({peak_src} sm_max_mhz); HBM peak n/a",
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

    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True,
           "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": f"Plummer sphere N={n}, equal masses, G=1, seed 2 (config 3): full "
                                  "self acc+gradient pass + kick + drift per step",
                      "l2": "flushed between timed iterations (256 MB fill)",
                      "parallelism": "1 GPU" if world == 1 else (
                          f"tile pairs of the symmetric sweeps sharded over {world} ranks, all-reduce of a "
                          "and of g" if pair_sharded else
                          f"sinks sharded over {world} ranks, all-gather of a between the sweeps")},
           "gflops": value * (FLOPS_NEWTON + FLOPS_GRAD) / 1e9,
           "flops_convention": "Newton 18 + gradient 34 = 52 flops per ordered pair (FMA=2, add/mul=1, rsqrt=1)",
           "breakdown_ms": {"newton+pack+reduce": n_ms, "gradient+pack+reduce": g_ms,
                            "kick+drift": float(np.mean(t_upd))},
           "gpu_launches": int(launches), "clocks": clocks, "roofline": roof,
           "cpu_baseline": cpu, "e2e": e2e}
    if world == 1 and not args.no_rows:
        out["other_rows"] = measure_rows(fr, frost, torch, dev, flush, hbm_peak, hhs=not args.no_hhs)
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--n", type=int, default=1 << 20)
    ap.add_argument("--impl", default="frost", choices=["frost", "reference"])
    ap.add_argument("--cpu-sinks", type=int, default=6144)
    ap.add_argument("--one-sided", action="store_true", help="force the one-sided sweeps (no pair symmetry)")
    ap.add_argument("--ref-sinks", type=int, default=1024)
    ap.add_argument("--warmup-ref", type=int, default=1)
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-rows", action="store_true", help="skip the side measurements of the O(N) rows")
    ap.add_argument("--no-hhs", action="store_true", help="skip the config-5 HHS-FSI step (about 15 s)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_frost(args)


if __name__ == "__main__":
    main()
