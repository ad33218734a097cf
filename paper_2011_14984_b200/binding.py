"""ctypes binding with the same names as include/frost.h (argument marshalling only).

Tensors are torch CUDA tensors: vectors float64 of shape (3, ld) C-contiguous (three SoA planes),
mass/tau float64 (n,), index lists int32 (k,) or None for "all particles".
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import torch

ACC, GRAD, MUTUAL, ACCUMULATE = 1, 2, 4, 8
MAX_LEVELS = 64

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libfrost_b200.so")
_lib = None

# every symbol include/frost.h declares (tests/test_abi.py checks the header against this list)
exported_symbols = [
    "frost_create", "frost_destroy", "frost_set_params", "frost_forces", "frost_forces_host",
    "frost_timesteps", "frost_partition", "frost_kick", "frost_drift", "frost_fsi_step",
    "frost_hhs_step", "frost_gather_pack", "frost_launch_count", "frost_last_cuda_error",
    "frost_strerror", "frost_version", "frost_set_tuning", "frost_set_symmetric",
    "frost_diagnostics", "frost_set_shard", "frost_fsi_steps", "frost_set_overlap",
    "frost_set_split", "frost_forces_masked", "frost_set_pair_path",
    "frost_set_gradient_guard", "frost_set_equal_mass_path",
    "frost_set_kepler", "frost_acc_noalloc", "frost_noalloc_max_n",
]


class FrostError(RuntimeError):
    pass


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


def library_path() -> str:
    return _LIB_PATH


def load_library():
    """Load libfrost_b200.so (built in-tree by build.py).  Raises if it is missing: there is no
    fallback implementation."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise FrostError(f"{_LIB_PATH} is missing: run `python -m paper_2011_14984_b200.build` "
                         "(or __graft_entry__.build()); there is no CPU fallback")
    lib = C.CDLL(_LIB_PATH)
    vp, i32, f64 = C.c_void_p, C.c_int, C.c_double
    lib.frost_create.argtypes = [C.POINTER(vp), i32, vp]
    lib.frost_destroy.argtypes = [vp]
    lib.frost_set_params.argtypes = [vp, f64, f64, f64, f64, i32]
    lib.frost_set_tuning.argtypes = [vp, i32, i32, i32, i32]
    lib.frost_set_symmetric.argtypes = [vp, i32, i32]
    lib.frost_set_shard.argtypes = [vp, i32, i32]
    lib.frost_set_overlap.argtypes = [vp, i32]
    lib.frost_set_split.argtypes = [vp, i32]
    lib.frost_set_pair_path.argtypes = [vp, i32]
    lib.frost_set_gradient_guard.argtypes = [vp, i32]
    lib.frost_set_equal_mass_path.argtypes = [vp, i32]
    lib.frost_set_kepler.argtypes = [vp, i32]
    lib.frost_forces_masked.argtypes = [vp, i32, i32, vp, vp, vp, i32, vp, vp, vp]
    lib.frost_diagnostics.argtypes = [vp, i32, i32, vp, vp, vp, vp, vp]
    lib.frost_forces.argtypes = [vp, i32, i32, vp, vp, vp, vp, i32, vp, i32, vp, vp, i32]
    lib.frost_forces_host.argtypes = [vp, i32, i32, vp, vp, vp, i32, vp, i32, vp, vp, i32]
    lib.frost_timesteps.argtypes = [vp, i32, i32, vp, vp, vp, vp, i32, f64, vp, vp]
    lib.frost_partition.argtypes = [vp, i32, vp, vp, i32, f64, vp, vp, vp]
    lib.frost_kick.argtypes = [vp, i32, i32, vp, vp, vp, vp, i32, f64, f64]
    lib.frost_drift.argtypes = [vp, i32, i32, vp, vp, vp, i32, f64]
    lib.frost_fsi_step.argtypes = [vp, i32, i32, vp, vp, vp, vp, i32, f64]
    lib.frost_fsi_steps.argtypes = [vp, i32, i32, vp, vp, vp, vp, i32, f64, i32]
    lib.frost_hhs_step.argtypes = [vp, i32, i32, vp, vp, vp, f64, vp]
    lib.frost_gather_pack.argtypes = [vp, i32, i32, vp, vp, vp, i32, i32, vp]
    lib.frost_acc_noalloc.argtypes = [i32, vp, i32, i32, vp, vp, f64, f64, vp, C.POINTER(C.c_int)]
    lib.frost_noalloc_max_n.argtypes = []
    lib.frost_launch_count.argtypes = [vp]
    lib.frost_launch_count.restype = C.c_int64
    lib.frost_last_cuda_error.argtypes = [vp]
    lib.frost_strerror.argtypes = [i32]
    lib.frost_strerror.restype = C.c_char_p
    lib.frost_version.restype = C.c_char_p
    _lib = lib
    return lib


def _p(t: Optional[torch.Tensor]):
    return None if t is None else C.c_void_p(t.data_ptr())


def _vec(t: torch.Tensor, name: str):
    if not (t.is_cuda and t.dtype == torch.float64 and t.dim() == 2 and t.shape[0] == 3
            and t.is_contiguous()):
        raise FrostError(f"{name}: expected a contiguous CUDA float64 tensor of shape (3, ld)")
    return t


def _idx(t: Optional[torch.Tensor], name: str):
    if t is None:
        return None, 0
    if not (t.is_cuda and t.dtype == torch.int32 and t.dim() == 1 and t.is_contiguous()):
        raise FrostError(f"{name}: expected a contiguous CUDA int32 vector or None")
    if t.numel() == 0:      # an empty list is not "all particles": pass a non-NULL pointer, count 0
        return torch.zeros(1, dtype=torch.int32, device=t.device), 0
    return t, t.numel()


def noalloc_max_n() -> int:
    """Largest n frost_acc_noalloc accepts (its scratch is a fixed static device array)."""
    return int(load_library().frost_noalloc_max_n())


def acc_noalloc(pos, mass, out_acc, G=1.0, eps2=0.0, stream: Optional[torch.cuda.Stream] = None):
    """frost_acc_noalloc: Newtonian accelerations of all particles (Eq. 24) written into the
    caller's out_acc, for callers that must not allocate device memory (a pool that owns the device, a
    loop that cannot afford cudaFree's synchronisation, a fixed memory budget).  No context, no
    cudaMalloc anywhere on the path -- which is why out_acc is a required argument here: this wrapper
    creates no tensor either.  n <= noalloc_max_n(); calls that overlap on the GPU race on the library's
    one static scratch array; make the first call on a device outside stream capture (frost.h)."""
    lib = load_library()
    _vec(pos, "pos"); _vec(out_acc, "out_acc")
    if out_acc.shape != pos.shape or out_acc.device != pos.device or mass.device != pos.device:
        raise FrostError("acc_noalloc: pos, mass and out_acc must share device and plane stride")
    dev = pos.device.index
    if stream is None:
        stream = torch.cuda.current_stream(dev)
    err = C.c_int(0)
    rc = lib.frost_acc_noalloc(dev, C.c_void_p(stream.cuda_stream), mass.numel(), pos.shape[1], _p(pos),
                               _p(mass), G, eps2, _p(out_acc), C.byref(err))
    if rc != 0:
        raise FrostError(f"frost_acc_noalloc: {lib.frost_strerror(rc).decode()} "
                         f"(status {rc}, cudaError {err.value})")
    return out_acc


class Frost:
    """One context = one device + one stream + scratch (frost_create / frost_destroy)."""

    def __init__(self, device: int = 0, stream: Optional[torch.cuda.Stream] = None):
        self.lib = load_library()
        if not torch.cuda.is_available():
            raise FrostError("no CUDA device: the frost path has no CPU fallback")
        if stream is None:
            stream = torch.cuda.current_stream(device)
        self.stream = stream
        self.device = device
        h = C.c_void_p()
        self._check(self.lib.frost_create(C.byref(h), device, C.c_void_p(stream.cuda_stream)),
                    "frost_create")
        self.h = h

    def close(self):
        if getattr(self, "h", None):
            self.lib.frost_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc: int, what: str):
        if rc != 0:
            cuda = self.lib.frost_last_cuda_error(self.h) if getattr(self, "h", None) else 0
            raise FrostError(f"{what}: {self.lib.frost_strerror(rc).decode()} "
                             f"(status {rc}, cudaError {cuda})")

    # -- parameters ------------------------------------------------------------------------
    def set_params(self, G=1.0, eps2=0.0, eta_ff=0.2, eta_fb=0.2, max_depth=64):
        self._check(self.lib.frost_set_params(self.h, G, eps2, eta_ff, eta_fb, max_depth),
                    "frost_set_params")

    def set_tuning(self, sinks_per_thread=0, source_slices=0, small_set_max=-1, subtree_one_cta=0):
        self._check(self.lib.frost_set_tuning(self.h, sinks_per_thread, source_slices,
                                              small_set_max, subtree_one_cta),
                    "frost_set_tuning")

    def set_symmetric(self, mode=0, scratch_mib=0):
        """0 = auto, 1 = one-sided sweeps only, 2 = pair-symmetric sweeps whenever applicable;
        scratch_mib caps the B-side scratch (0 = default 4096 MiB)."""
        self._check(self.lib.frost_set_symmetric(self.h, mode, scratch_mib), "frost_set_symmetric")

    def set_shard(self, rank=0, world=1):
        """This context's share of the symmetric sweeps (partial sums; add them across ranks)."""
        self._check(self.lib.frost_set_shard(self.h, rank, world), "frost_set_shard")

    def set_overlap(self, on=1):
        """1 (default): fsi(S) of a host-driven hierarchy entry runs on a side stream concurrently
        with the recursion into F; 0: back to back on the context's stream (same bits)."""
        self._check(self.lib.frost_set_overlap(self.h, on), "frost_set_overlap")

    def set_split(self, split_max=0):
        """split_max > 0: hierarchy entries with at most split_max members recurse into the connected
        components of their fast pairs one by one (frost.h: frost_set_split); 0 (default): Alg. 3."""
        self._check(self.lib.frost_set_split(self.h, split_max), "frost_set_split")

    def set_kepler(self, on=0):
        """1: two-body components of a split entry follow their exact Kepler orbit over the entry's half
        step instead of being recursed into (needs set_split, eps2 = 0); 0 (default)."""
        self._check(self.lib.frost_set_kepler(self.h, on), "frost_set_kepler")

    def set_equal_mass_path(self, on=1):
        """1 (default): large pair-symmetric force sweeps take their equal-mass variant when every mass
        of the swept lists is the same (decided on the device; bitwise the same sums); 0: never."""
        self._check(self.lib.frost_set_equal_mass_path(self.h, on), "frost_set_equal_mass_path")

    def set_gradient_guard(self, on=0):
        """0 (default): large pair-symmetric gradient sweeps run unguarded with a gated guarded repair
        pass; 1: the coincident-pair guard stays in the loop (frost.h: frost_set_gradient_guard)."""
        self._check(self.lib.frost_set_gradient_guard(self.h, on), "frost_set_gradient_guard")

    def set_pair_path(self, on=1):
        """1 (default): two-body hierarchy entries of the subtree kernels run on one thread with both
        bodies in registers; 0: on the warp team (same bits)."""
        self._check(self.lib.frost_set_pair_path(self.h, on), "frost_set_pair_path")

    def launch_count(self) -> int:
        return int(self.lib.frost_launch_count(self.h))

    # -- the path --------------------------------------------------------------------------
    def forces(self, pos, mass, sink_idx=None, source_idx=None, out_acc=None, out_grad=None,
               flags=ACC | GRAD, vel=None):
        _vec(pos, "pos")
        ld, n = pos.shape[1], mass.numel()
        if out_acc is None:
            out_acc = torch.zeros_like(pos)
        if out_grad is None and (flags & GRAD):
            out_grad = torch.zeros_like(pos)
        si, ns = _idx(sink_idx, "sink_idx")
        so, nso = _idx(source_idx, "source_idx")
        self._check(self.lib.frost_forces(self.h, n, ld, _p(pos), _p(vel), _p(mass), _p(si), ns,
                                          _p(so), nso, _p(_vec(out_acc, "out_acc")),
                                          _p(out_grad), flags), "frost_forces")
        return out_acc, out_grad

    def forces_masked(self, pos, mass, label, idx=None, out_acc=None, out_grad=None, grad=True):
        """Eq. 42-44 over the pairs of the list whose labels (int32, by list position) differ."""
        _vec(pos, "pos")
        ld, n = pos.shape[1], mass.numel()
        if out_acc is None:
            out_acc = torch.zeros_like(pos)
        if out_grad is None and grad:
            out_grad = torch.zeros_like(pos)
        ii, ni = _idx(idx, "idx")
        lab, nl = _idx(label, "label")
        if nl != (ni if idx is not None else n):
            raise FrostError("label: one entry per list position expected")
        self._check(self.lib.frost_forces_masked(self.h, n, ld, _p(pos), _p(mass), _p(ii), ni, _p(lab),
                                                 _p(_vec(out_acc, "out_acc")), _p(out_grad if grad else None)),
                    "frost_forces_masked")
        return out_acc, out_grad

    def forces_host(self, pos, mass, sink_idx=None, source_idx=None, out_acc=None, out_grad=None,
                    flags=ACC | GRAD):
        """Host-buffer entry (CPU tensors, ideally pinned): copies in, sweeps, copies out."""
        ld, n = pos.shape[1], mass.numel()
        if out_acc is None:
            out_acc = torch.zeros_like(pos)
        if out_grad is None and (flags & GRAD):
            out_grad = torch.zeros_like(pos)
        ns = 0 if sink_idx is None else sink_idx.numel()
        nso = 0 if source_idx is None else source_idx.numel()
        self._check(self.lib.frost_forces_host(self.h, n, ld, _p(pos), _p(mass), _p(sink_idx), ns,
                                               _p(source_idx), nso, _p(out_acc), _p(out_grad),
                                               flags), "frost_forces_host")
        return out_acc, out_grad

    def timesteps(self, pos, vel, mass, idx=None, tau_pivot=1.0, out_tau=None, out_bin=None,
                  want_bins=True):
        _vec(pos, "pos"); _vec(vel, "vel")
        ld, n = pos.shape[1], mass.numel()
        if out_tau is None:
            out_tau = torch.full((ld,), float("inf"), dtype=torch.float64, device=pos.device)
        if out_bin is None and want_bins:
            out_bin = torch.zeros((ld,), dtype=torch.int32, device=pos.device)
        ii, ni = _idx(idx, "idx")
        self._check(self.lib.frost_timesteps(self.h, n, ld, _p(pos), _p(vel), _p(mass), _p(ii), ni,
                                             tau_pivot, _p(out_tau), _p(out_bin)), "frost_timesteps")
        return out_tau, out_bin

    def partition(self, tau, tau_pivot, idx=None):
        n = tau.numel()
        ii, ni = _idx(idx, "idx")
        k = n if ii is None else ni
        slow = torch.empty((max(k, 1),), dtype=torch.int32, device=tau.device)
        fast = torch.empty((max(k, 1),), dtype=torch.int32, device=tau.device)
        counts = (C.c_int32 * 2)()
        self._check(self.lib.frost_partition(self.h, n, _p(tau), _p(ii), ni, tau_pivot, _p(slow),
                                             _p(fast), counts), "frost_partition")
        return slow[: counts[0]], fast[: counts[1]]

    def kick(self, vel, acc, grad=None, idx=None, c=1.0, kappa=0.0):
        _vec(vel, "vel")
        ii, ni = _idx(idx, "idx")
        self._check(self.lib.frost_kick(self.h, vel.shape[1], vel.shape[1], _p(vel), _p(acc),
                                        _p(grad), _p(ii), ni, c, kappa), "frost_kick")

    def drift(self, pos, vel, idx=None, c=1.0):
        _vec(pos, "pos")
        ii, ni = _idx(idx, "idx")
        self._check(self.lib.frost_drift(self.h, pos.shape[1], pos.shape[1], _p(pos), _p(vel),
                                         _p(ii), ni, c), "frost_drift")

    def fsi_step(self, pos, vel, mass, dt, idx=None):
        _vec(pos, "pos"); _vec(vel, "vel")
        ii, ni = _idx(idx, "idx")
        self._check(self.lib.frost_fsi_step(self.h, mass.numel(), pos.shape[1], _p(pos), _p(vel),
                                            _p(mass), _p(ii), ni, dt), "frost_fsi_step")

    def fsi_steps(self, pos, vel, mass, dt, n_steps, idx=None):
        _vec(pos, "pos"); _vec(vel, "vel")
        ii, ni = _idx(idx, "idx")
        self._check(self.lib.frost_fsi_steps(self.h, mass.numel(), pos.shape[1], _p(pos), _p(vel),
                                             _p(mass), _p(ii), ni, dt, n_steps), "frost_fsi_steps")

    def hhs_step(self, pos, vel, mass, dt_top):
        _vec(pos, "pos"); _vec(vel, "vel")
        st = HHSStats()
        self._check(self.lib.frost_hhs_step(self.h, mass.numel(), pos.shape[1], _p(pos), _p(vel),
                                            _p(mass), dt_top, C.byref(st)), "frost_hhs_step")
        return st.as_dict()

    def diagnostics(self, pos, vel, mass, out_phi=None):
        """dict(T, U, E, P(3), L(3)) of all particles, computed on the device (frost_diagnostics)."""
        _vec(pos, "pos"); _vec(vel, "vel")
        out = (C.c_double * 8)()
        self._check(self.lib.frost_diagnostics(self.h, mass.numel(), pos.shape[1], _p(pos), _p(vel),
                                               _p(mass), _p(out_phi), out), "frost_diagnostics")
        o = list(out)
        return {"T": o[0], "U": o[1], "E": o[0] + o[1], "P": o[2:5], "L": o[5:8]}

    def gather_pack(self, pos, mass, idx=None, n_pad=None):
        _vec(pos, "pos")
        ii, ni = _idx(idx, "idx")
        k = mass.numel() if ii is None else ni
        if n_pad is None:
            n_pad = k
        out = torch.empty((n_pad, 4), dtype=torch.float64, device=pos.device)
        self._check(self.lib.frost_gather_pack(self.h, mass.numel(), pos.shape[1], _p(pos),
                                               _p(mass), _p(ii), ni, n_pad, _p(out)),
                    "frost_gather_pack")
        return out
