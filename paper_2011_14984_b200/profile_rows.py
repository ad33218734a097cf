"""Launches every kernel family of the path once or twice at a fixed size so that ncu can capture
them (profiles/*.md name the exact command):  python -m paper_2011_14984_b200.profile_rows [N]
                                               python -m paper_2011_14984_b200.profile_rows subtree 8

The O(N) kernels (gather/pack, kick, drift, partition) run on N = 2^20 particles after an L2 flush;
the time-step sweeps (plain symmetric, one-sided, pruned) on min(N, 65536) particles."""
import sys

import torch

import frost_inputs as fi
import paper_2011_14984_b200 as frost


def subtree(n):
    """The device-resident subtree kernel on a set of n/2 hard binaries (a latency-bound case)."""
    import numpy as np
    pos, vel, mass, pairs = fi.star_cluster(4096, 4, binary_fraction=0.6)
    sel = pairs[: n // 2].ravel()
    dev = torch.device("cuda", 0)
    p = torch.as_tensor(np.ascontiguousarray(pos[:, sel])).to(dev)
    v = torch.as_tensor(np.ascontiguousarray(vel[:, sel])).to(dev)
    m = torch.as_tensor(mass[sel].copy()).to(dev)
    fr = frost.Frost(0)
    for _ in range(2):
        st = fr.hhs_step(p.clone(), v.clone(), m, 2.0 ** -12)
    torch.cuda.synchronize()
    print("hierarchy entries:", sum(st["entries"]), "depth:", st["depth"])
    fr.close()


def main():
    if len(sys.argv) > 2 and sys.argv[1] == "subtree":
        return subtree(int(sys.argv[2]))
    n = int(sys.argv[1]) if len(sys.argv) > 1 else 1 << 20
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


if __name__ == "__main__":
    main()
