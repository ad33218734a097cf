"""ctypes marshalling for oracle/frost_oracle.c (argument passing only; no arithmetic here).

Arrays are numpy float64, C-contiguous, shape (3, ld) for vectors and (n,) for scalars; index
arrays are int32 or None (= all particles).  Functions that update state do so IN PLACE.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

ACC, GRAD, MUTUAL = 1, 2, 4
MAX_LEVELS = 64

_lib = None


class HHSStats(C.Structure):
    _fields_ = [("depth", C.c_int32), ("reserved", C.c_int32),
                ("entries", C.c_int64 * MAX_LEVELS), ("n_slow", C.c_int64 * MAX_LEVELS),
                ("n_fast", C.c_int64 * MAX_LEVELS), ("pairs_newton", C.c_int64),
                ("pairs_gradient", C.c_int64), ("pairs_timestep", C.c_int64),
                ("n_comp", C.c_int64 * MAX_LEVELS), ("n_kepler", C.c_int64)]

    def as_dict(self):
        d = self.depth
        return {"depth": d, "entries": list(self.entries[: d + 1]),
                "n_slow": list(self.n_slow[: d + 1]), "n_fast": list(self.n_fast[: d + 1]),
                "pairs_newton": self.pairs_newton, "pairs_gradient": self.pairs_gradient,
                "pairs_timestep": self.pairs_timestep, "n_comp": list(self.n_comp[: d + 1]),
                "n_kepler": self.n_kepler}


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.oracle_sym_factor.restype = C.c_double
        _lib.oracle_sym_factor.argtypes = [C.c_double]
    return _lib


def _d(a):
    assert a.dtype == np.float64 and a.flags.c_contiguous, "float64 C-contiguous array expected"
    return a.ctypes.data_as(C.c_void_p)


def _i(idx):
    if idx is None:
        return None, 0
    idx = np.ascontiguousarray(idx, dtype=np.int32)
    return idx, idx.size


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _check(rc, what):
    if rc != 0:
        raise RuntimeError(f"{what} failed with status {rc}")


def num_threads() -> int:
    return lib().oracle_num_threads()


def set_num_threads(t: int) -> None:
    lib().oracle_set_num_threads(C.c_int(t))


def sym_factor(q: float) -> float:
    return lib().oracle_sym_factor(C.c_double(q))


def forces(pos, mass, sink_idx=None, source_idx=None, G=1.0, eps2=0.0, flags=ACC | GRAD,
           acc=None, grad=None):
    """Returns (acc, grad) planes of shape (3, ld); entries outside the swept sets are untouched
    (zero if the arrays were created here)."""
    ld = pos.shape[1]
    n = mass.shape[0]
    if acc is None:
        acc = np.zeros((3, ld))
    if grad is None:
        grad = np.zeros((3, ld))
    si, ns = _i(sink_idx)
    so, nso = _i(source_idx)
    rc = lib().oracle_forces(C.c_int(n), C.c_int(ld), _d(pos), _d(mass), _ptr(si), C.c_int(ns),
                             _ptr(so), C.c_int(nso), C.c_double(G), C.c_double(eps2), _d(acc),
                             _d(grad), C.c_int(flags))
    _check(rc, "oracle_forces")
    return acc, grad


def gradient_termsum(pos, mass, acc, sink_idx=None, source_idx=None, G=1.0, eps2=0.0):
    """T_i = 2G sum_j |term_ij| of Eq. 27 for the sinks (shape (ld,), zero elsewhere): the
    magnitude sum behind the forward-error gate of the gradient parity tests."""
    ld = pos.shape[1]
    n = mass.shape[0]
    out = np.zeros(ld)
    si, ns = _i(sink_idx)
    so, nso = _i(source_idx)
    rc = lib().oracle_gradient_termsum(C.c_int(n), C.c_int(ld), _d(pos), _d(mass), _ptr(si),
                                       C.c_int(ns), _ptr(so), C.c_int(nso), C.c_double(G),
                                       C.c_double(eps2), _d(acc), _d(out))
    _check(rc, "oracle_gradient_termsum")
    return out


def timesteps(pos, vel, mass, idx=None, G=1.0, eta_ff=0.2, eta_fb=0.2, tau_pivot=1.0,
              eta_in_q=True, tau=None, bins=None):
    ld = pos.shape[1]
    n = mass.shape[0]
    if tau is None:
        tau = np.full(ld, np.inf)
    if bins is None:
        bins = np.zeros(ld, dtype=np.int32)
    ii, ni = _i(idx)
    rc = lib().oracle_timesteps(C.c_int(n), C.c_int(ld), _d(pos), _d(vel), _d(mass), _ptr(ii),
                                C.c_int(ni), C.c_double(G), C.c_double(eta_ff),
                                C.c_double(eta_fb), C.c_int(1 if eta_in_q else 0),
                                C.c_double(tau_pivot), _d(tau), _ptr(bins))
    _check(rc, "oracle_timesteps")
    return tau, bins


def timesteps_sampled(pos, vel, mass, sel, idx=None, G=1.0, eta_ff=0.2, eta_fb=0.2, tau_pivot=1.0,
                      eta_in_q=True):
    """tau and bin of the sinks in `sel` only, each against every member of the level `idx`."""
    ld = pos.shape[1]
    n = mass.shape[0]
    tau = np.full(ld, np.inf)
    bins = np.zeros(ld, dtype=np.int32)
    ii, ni = _i(idx)
    ss, nsel = _i(sel)
    rc = lib().oracle_timesteps_sampled(C.c_int(n), C.c_int(ld), _d(pos), _d(vel), _d(mass),
                                        _ptr(ii), C.c_int(ni), _ptr(ss), C.c_int(nsel),
                                        C.c_double(G), C.c_double(eta_ff), C.c_double(eta_fb),
                                        C.c_int(1 if eta_in_q else 0), C.c_double(tau_pivot),
                                        _d(tau), _ptr(bins))
    _check(rc, "oracle_timesteps_sampled")
    return tau, bins


def pair_timestep(xi, vi, mi, xj, vj, mj, G=1.0, eta_ff=0.2, eta_fb=0.2, eta_in_q=True):
    out = (C.c_double * 2)()
    arr = lambda v: (C.c_double * 3)(*[float(t) for t in v])
    lib().oracle_pair_timestep(arr(xi), arr(vi), C.c_double(mi), arr(xj), arr(vj), C.c_double(mj),
                               C.c_double(G), C.c_double(eta_ff), C.c_double(eta_fb),
                               C.c_int(1 if eta_in_q else 0), out)
    return out[0], out[1]


def kick(vel, acc, grad=None, idx=None, c=1.0, kappa=0.0):
    ld = vel.shape[1]
    ii, ni = _i(idx)
    rc = lib().oracle_kick(C.c_int(ld), C.c_int(ld), _d(vel), _d(acc), _ptr(grad), _ptr(ii),
                           C.c_int(ni), C.c_double(c), C.c_double(kappa))
    _check(rc, "oracle_kick")


def drift(pos, vel, idx=None, c=1.0):
    ld = pos.shape[1]
    ii, ni = _i(idx)
    rc = lib().oracle_drift(C.c_int(ld), C.c_int(ld), _d(pos), _d(vel), _ptr(ii), C.c_int(ni),
                            C.c_double(c))
    _check(rc, "oracle_drift")


def fsi_step(pos, vel, mass, dt, idx=None, G=1.0, eps2=0.0):
    ld = pos.shape[1]
    n = mass.shape[0]
    ii, ni = _i(idx)
    rc = lib().oracle_fsi_step(C.c_int(n), C.c_int(ld), _d(pos), _d(vel), _d(mass), _ptr(ii),
                               C.c_int(ni), C.c_double(dt), C.c_double(G), C.c_double(eps2))
    _check(rc, "oracle_fsi_step")


def hhs_step(pos, vel, mass, dt_top, G=1.0, eps2=0.0, eta_ff=0.2, eta_fb=0.2, eta_in_q=True,
             max_depth=64, frozen_level=None, split_max=0, frozen_comp=None, kepler=False):
    """One HHS-FSI step (Alg. 3).  split_max > 0: entries with at most split_max members split
    their fast set into the connected components of the fast pairs (O6s in frost_oracle.c)."""
    ld = pos.shape[1]
    n = mass.shape[0]
    st = HHSStats()
    fl, _ = _i(frozen_level)
    fc, _ = _i(frozen_comp)
    rc = lib().oracle_hhs_split_step(C.c_int(n), C.c_int(ld), _d(pos), _d(vel), _d(mass),
                                     C.c_double(dt_top), C.c_double(G), C.c_double(eps2),
                                     C.c_double(eta_ff), C.c_double(eta_fb),
                                     C.c_int(1 if eta_in_q else 0), C.c_int(max_depth), _ptr(fl),
                                     C.c_int(split_max), _ptr(fc), C.c_int(1 if kepler else 0),
                                     C.byref(st))
    _check(rc, "oracle_hhs_split_step")
    return st.as_dict()


def kepler_relative(mu, dt, r, v):
    """Relative position and velocity (length-3 arrays) advanced by dt along the Kepler flow of mu."""
    rr = np.ascontiguousarray(r, dtype=np.float64).copy()
    vv = np.ascontiguousarray(v, dtype=np.float64).copy()
    _check(lib().oracle_kepler_relative(C.c_double(mu), C.c_double(dt), _d(rr), _d(vv)), "oracle_kepler_relative")
    return rr, vv


def components(pos, vel, mass, tau_pivot, idx=None, G=1.0, eta_ff=0.2, eta_fb=0.2, eta_in_q=True):
    """Component label (smallest member index; -1 = no fast pair) of every member of the level `idx`,
    shape (ld,), entries outside the level are -2."""
    ld = pos.shape[1]
    n = mass.shape[0]
    label = np.full(ld, -2, dtype=np.int32)
    ii, ni = _i(idx)
    rc = lib().oracle_components(C.c_int(n), C.c_int(ld), _d(pos), _d(vel), _d(mass), _ptr(ii),
                                 C.c_int(ni), C.c_double(G), C.c_double(eta_ff), C.c_double(eta_fb),
                                 C.c_int(1 if eta_in_q else 0), C.c_double(tau_pivot), _ptr(label))
    _check(rc, "oracle_components")
    return label


def forces_masked(pos, mass, idx, label, G=1.0, eps2=0.0, flags=ACC | GRAD, acc=None, grad=None):
    """Eq. 42-44 on the pair set {(i, j) in idx^2 : label_i != label_j} (label indexed globally)."""
    ld = pos.shape[1]
    n = mass.shape[0]
    if acc is None:
        acc = np.zeros((3, ld))
    if grad is None:
        grad = np.zeros((3, ld))
    ii, ni = _i(idx)
    lab = np.ascontiguousarray(label, dtype=np.int32)
    rc = lib().oracle_forces_masked(C.c_int(n), C.c_int(ld), _d(pos), _d(mass), _ptr(ii), C.c_int(ni),
                                    _ptr(lab), C.c_double(G), C.c_double(eps2), _d(acc), _d(grad),
                                    C.c_int(flags))
    _check(rc, "oracle_forces_masked")
    return acc, grad


def diagnostics(pos, vel, mass, G=1.0, eps2=0.0):
    """Returns dict(T, U, E, P(3), L(3))."""
    ld = pos.shape[1]
    n = mass.shape[0]
    out = np.zeros(8)
    rc = lib().oracle_diagnostics(C.c_int(n), C.c_int(ld), _d(pos), _d(vel), _d(mass),
                                  C.c_double(G), C.c_double(eps2), _d(out))
    _check(rc, "oracle_diagnostics")
    return {"T": out[0], "U": out[1], "E": out[0] + out[1], "P": out[2:5].copy(),
            "L": out[5:8].copy()}
