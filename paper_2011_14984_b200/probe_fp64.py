"""Print the FP64 issue-model table of this GPU (times frost_fp64_probe modes with CUDA events).

    python -m paper_2011_14984_b200.probe_fp64

One line per probe: issue cycles per FP64 warp instruction per SM sub-partition at the max SM clock
(2.0 = the nominal rate of a 16-lane FP64 pipe).  See DESIGN.md "FP64 issue model".
"""
import json
import os
import sys

import torch

import paper_2011_14984_b200 as frost

MODES = [
    (1, "DADD, 2 distinct register pairs", 0),
    (2, "DMUL, 2 distinct register pairs", 0),
    (6, "DFMA, 2 register pairs + immediate", 0),
    (0, "DFMA, 1 register pair + 2 loop-invariant pairs (.reuse)", 0),
    (4, "DFMA, 3 distinct register pairs", 0),
    (5, "DFMA triples sharing one operand, adjacent (.reuse) [48 of 64] + 16 DADD", 0),
    (3, "mix: DFMA(2 pairs) / DADD / DMUL", 0),
    (7, "DADD + 12 integer-ALU instr per 16 FP64 instr", 12),
    (8, "DADD + 2 MUFU.RSQ64H per 16 FP64 instr", 2),
    (9, "DADD + 4 LDS.128 per 16 FP64 instr", 4),
]


def main():
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    mhz = 1965.0
    p = os.path.join(root, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        mhz = json.load(open(p)).get("sm_max_mhz", mhz)
    fr = frost.Frost(0)
    scratch = torch.zeros(148 * 8 * 256 * 2, dtype=torch.float64, device="cuda")
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    print(f"# {torch.cuda.get_device_name(0)}, {sms} SMs, cycles at {mhz:.0f} MHz; 4 CTAs x 256 threads per SM")
    print(f"# {'probe':78s} cyc/FP64-inst  extra cyc per extra instr")
    base = None
    for mode, name, extras in MODES:
        fr.fp64_probe(mode, 2000, 4, scratch); torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(); ninst = fr.fp64_probe(mode, 40000, 4, scratch); b.record(); torch.cuda.synchronize()
        sec = a.elapsed_time(b) * 1e-3
        warp_inst_per_smsp = ninst / 32 / (sms * 4)
        cyc = sec * mhz * 1e6 / warp_inst_per_smsp
        if mode == 1:
            base = cyc
        extra = "" if not extras else f"{(cyc - base) * 16 / extras:6.2f}"
        print(f"  {name:78s} {cyc:6.3f}        {extra}")
    # dependent-chain latency: 1 CTA of 8 warps per SM (2 warps per sub-partition), one chain per thread
    for mode, name in ((10, "DFMA"), (11, "DADD")):
        fr.fp64_probe(mode, 2000, 1, scratch); torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        iters = 40000
        a.record(); fr.fp64_probe(mode, iters, 1, scratch); b.record(); torch.cuda.synchronize()
        cyc = a.elapsed_time(b) * 1e-3 * mhz * 1e6 / (iters * 64)
        print(f"  dependent {name} chain, 2 warps per sub-partition: {cyc:6.2f} cycles per instruction (latency)")
    fr.close()


if __name__ == "__main__":
    sys.exit(main())
