"""frost_acc_noalloc -- the one entry point of the library that allocates nothing -- against the
ordinary path (frost_forces with FROST_ACC through a context).

Why it exists: a frost context grows its scratch with cudaMalloc whenever a sweep needs more, and some
callers cannot live with that -- an application whose memory pool owns the whole device, a loop that
cannot take the device-wide synchronisation of a cudaFree, a program held to a memory budget fixed at
start-up.  frost_acc_noalloc keeps its scratch in a static device array inside the library instead
(6.5 MiB per GPU, n <= 16384) and the caller passes inputs and output only.

What is checked: two calls in a row give, each time, the accelerations of the existing path within the
tolerance the parity tests use for a_i (1e-12 |a_i| per component).  The second call is SMALLER than the
first and uses other particles, G and softening, so that anything the first call left behind in the
shared array -- stale records in the padding, stale partial sums of slices the second call does not
use -- would show up.  Sizes are ragged (not a multiple of the 128-sink block or the 256-record tile).
Sizes beyond the limit must be refused with a message that names it, without touching the output.

This file sorts last on purpose (pytest -x stops at the first failure; a failure here must not hide
the parity tests) and depends on no state of the other tests: the first call in a process does the
one-time address look-up itself, whether or not a context was ever created before it."""
import numpy as np
import pytest
import torch

import frost_inputs as fi

pytestmark = pytest.mark.gpu

TOL_A = 1e-12      # north_star's tolerance for a_i, per component against |a_i| (tests/test_gpu_parity.py)


def dev(a):
    return torch.as_tensor(np.ascontiguousarray(a)).cuda()


def vec_err(x, ref):
    nrm = np.linalg.norm(ref, axis=0)
    return float((np.abs(x - ref).max(axis=0) / nrm).max())


def existing_path(frost, pos, mass, G, eps2):
    fr = frost.Frost()
    try:
        fr.set_params(G=G, eps2=eps2)
        acc, _ = fr.forces(pos, mass, flags=frost.ACC)
        torch.cuda.synchronize()
        return acc.cpu().numpy()
    finally:
        fr.close()


def test_two_calls_in_a_row_match_the_existing_path():
    import paper_2011_14984_b200 as frost
    cases = [(9001, 11, 1.0, 0.0), (1237, 12, 2.5, 1e-4)]      # (n, seed, G, eps2): large, then small
    results = []
    for n, seed, G, eps2 in cases:
        p, _, m = fi.plummer(n, seed)
        pos, mass = dev(p), dev(m)
        out = torch.full_like(pos, float("nan"))                 # the caller's output buffer
        frost.acc_noalloc(pos, mass, out, G=G, eps2=eps2)        # back to back: no sync in between
        results.append((pos, mass, out, G, eps2))
    torch.cuda.synchronize()
    for pos, mass, out, G, eps2 in results:
        ref = existing_path(frost, pos, mass, G, eps2)
        got = out.cpu().numpy()
        assert np.isfinite(got).all()
        err = vec_err(got, ref)
        print(f"noalloc n={mass.numel()}: max |da|/|a| = {err:.2e}")
        assert err < TOL_A, err


def test_same_input_twice_is_bitwise_repeatable_and_respects_ld():
    import paper_2011_14984_b200 as frost
    n, ld = 3000, 3072
    p, _, m = fi.plummer(n, 13)
    pos = torch.zeros((3, ld), dtype=torch.float64, device="cuda")
    pos[:, :n] = dev(p)
    mass = dev(m)
    a1 = torch.full_like(pos, -7.0)
    a2 = torch.full_like(pos, -7.0)
    frost.acc_noalloc(pos, mass, a1)
    frost.acc_noalloc(pos, mass, a2)
    torch.cuda.synchronize()
    assert torch.equal(a1, a2)
    assert (a1[:, n:] == -7.0).all()                             # entries beyond n untouched
    ref = existing_path(frost, pos, mass, 1.0, 0.0)
    assert vec_err(a1[:, :n].cpu().numpy(), ref[:, :n]) < TOL_A


def test_sizes_beyond_the_static_scratch_are_refused():
    import paper_2011_14984_b200 as frost
    nmax = frost.noalloc_max_n()
    assert nmax == 16384
    n = nmax + 1
    pos = torch.zeros((3, n), dtype=torch.float64, device="cuda")
    mass = torch.ones(n, dtype=torch.float64, device="cuda")
    out = torch.full_like(pos, 3.0)
    with pytest.raises(frost.FrostError, match="FROST_NOALLOC_MAX_N"):
        frost.acc_noalloc(pos, mass, out)
    torch.cuda.synchronize()
    assert (out == 3.0).all()
    # the limit itself is served
    p, _, m = fi.plummer(nmax, 14)
    pos, mass = dev(p), dev(m)
    out = torch.empty_like(pos)
    frost.acc_noalloc(pos, mass, out)
    torch.cuda.synchronize()
    ref = existing_path(frost, pos, mass, 1.0, 0.0)
    assert vec_err(out.cpu().numpy(), ref) < TOL_A
