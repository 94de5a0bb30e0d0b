"""Thin Python binding of liblsm (include/lsm.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels behind the C ABI; PyTorch is used for device
memory (`torch.empty(..., device="cuda")`) and streams (`torch.cuda.current_stream()`), nothing else.
There is no CPU fallback: if liblsm.so is missing or there is no CUDA device, calls raise.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_PKG = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_PKG, "liblsm.so")

ISING, NE_HEATBATH, NE_METROPOLIS, EA, POTTS = 0, 1, 2, 3, 4
KERNEL_AUTO, KERNEL_GENERIC, KERNEL_TILED, KERNEL_RESIDENT, KERNEL_SMALL, KERNEL_SLAB, KERNEL_BULK = 0, 1, 2, 3, 4, 5, 6
OK, ERR_ARG, ERR_UNSUPPORTED, ERR_CUDA, ERR_WORKSPACE, ERR_STATE, ERR_LIMIT = 0, -1, -2, -3, -4, -5, -6
NOALLOC_MAX_SWEEPS = 4096     # LSM_NOALLOC_MAX_SWEEPS of include/lsm.h

# name -> (restype, argtypes); every symbol include/lsm.h declares
_vp, _i32, _i64, _u64, _dbl, _sz = (ctypes.c_void_p, ctypes.c_int, ctypes.c_int64, ctypes.c_uint64,
                                    ctypes.c_double, ctypes.c_size_t)
_P = ctypes.POINTER
SIGNATURES = {
    "lsm_workspace_bytes": (_i32, [_i32, _i32, _i32, _i32, _P(_sz)]),
    "lsm_create": (_i32, [_i32, _i32, _i32, _i32, _dbl, _dbl, _dbl, _u64, _vp, _sz, _vp, _P(_vp)]),
    "lsm_destroy": (_i32, [_vp]),
    "lsm_sweep": (_i32, [_vp, _i64, _vp]),
    "lsm_sweep_record": (_i32, [_vp, _i64, _vp, _vp]),
    "lsm_sweep_record_host": (_i32, [_vp, _i64, _vp, _vp, _vp]),
    "lsm_sweep_record_host_async": (_i32, [_vp, _i64, _vp, _vp, _vp]),
    "lsm_sweep_record_host_noalloc": (_i32, [_vp, _i64, _vp, _vp]),
    "lsm_stage_spins_host": (_i32, [_vp, _vp, _vp, _vp]),
    "lsm_sweep_random_tile": (_i32, [_vp, _i64, _i32, _i32, _vp, _vp]),
    "lsm_sweep_random_tile_balanced": (_i32, [_vp, _i64, _i32, _i32, _vp, _vp]),
    "lsm_batch_workspace_bytes": (_i32, [_i32, _i32, _i32, _i32, _i32, _P(_sz)]),
    "lsm_batch_create": (_i32, [_i32, _i32, _i32, _i32, _i32, _dbl, _dbl, _vp, _vp, _vp, _sz, _vp, _P(_vp)]),
    "lsm_batch_destroy": (_i32, [_vp]),
    "lsm_batch_size": (_i32, [_vp, _P(_i32)]),
    "lsm_batch_replica": (_i32, [_vp, _i32, _P(_vp)]),
    "lsm_batch_sweep": (_i32, [_vp, _i64, _vp]),
    "lsm_batch_sweep_record": (_i32, [_vp, _i64, _vp, _vp]),
    "lsm_batch_sweep_random_tile": (_i32, [_vp, _i64, _i32, _i32, _i32, _vp, _vp]),
    "lsm_batch_set_temperatures": (_i32, [_vp, _vp]),
    "lsm_batch_set_tracking": (_i32, [_vp, _i32, _vp]),
    "lsm_batch_set_cluster": (_i32, [_vp, _i32]),
    "lsm_batch_measure_int": (_i32, [_vp, _vp, _vp]),
    "lsm_batch_get_launch_count": (_i32, [_vp, _P(_u64)]),
    "lsm_measure": (_i32, [_vp, _P(_dbl), _P(_i64)]),
    "lsm_measure_int": (_i32, [_vp, _P(_i64), _P(_i64), _P(_u64)]),
    "lsm_measure_full": (_i32, [_vp, _P(_i64), _P(_i64)]),
    "lsm_persistence": (_i32, [_vp, _P(_i64), _P(_i64)]),
    "lsm_reset_reference": (_i32, [_vp, _vp]),
    "lsm_set_tracking": (_i32, [_vp, _i32, _vp]),
    "lsm_get_spins": (_i32, [_vp, _vp, _vp]),
    "lsm_get_spins_host": (_i32, [_vp, _vp, _vp, _vp]),
    "lsm_set_spins": (_i32, [_vp, _vp, _u64, _vp]),
    "lsm_set_spins_host": (_i32, [_vp, _vp, _vp, _u64, _vp]),
    "lsm_set_bonds": (_i32, [_vp, _vp, _vp]),
    "lsm_get_bonds": (_i32, [_vp, _vp, _vp]),
    "lsm_set_temperature": (_i32, [_vp, _dbl]),
    "lsm_get_thresholds": (_i32, [_vp, _P(_u64), _P(_i32)]),
    "lsm_set_kernel": (_i32, [_vp, _i32]),
    "lsm_get_kernel": (_i32, [_vp, _P(_i32)]),
    "lsm_set_temporal_depth": (_i32, [_vp, _i32]),
    "lsm_get_temporal_depth": (_i32, [_vp, _P(_i32)]),
    "lsm_get_launch_count": (_i32, [_vp, _P(_u64)]),
    "lsm_binder_u4": (_i32, [_vp, _i64, _P(_dbl)]),
    "lsm_heat_capacity": (_i32, [_vp, _i64, _i64, _dbl, _dbl, _dbl, _P(_dbl)]),
    "lsm_series_means": (_i32, [_vp, _i64, _i64, _dbl, _dbl, _P(_dbl), _P(_dbl)]),
    "lsm_phi": (_i32, [_i64, _i64, _dbl, _P(_dbl)]),
    "lsm_persistence_fraction": (_i32, [_i64, _i64, _P(_dbl)]),
    "lsm_energy": (_i32, [_i32, _dbl, _dbl, _i64, _i64, _P(_dbl)]),
    "lsm_philox_device": (_i32, [_vp, _vp, _i64, _vp]),
    "lsm_philox_throughput": (_i32, [_i32, _i32, _vp, _vp]),
    "lsm_strerror": (ctypes.c_char_p, [_i32]),
    "lsm_last_cuda_error": (ctypes.c_char_p, []),
}

_lib = None


def lib_path() -> str:
    return _LIB_PATH


def load():
    """dlopen liblsm.so and bind every declared symbol.  Raises if the library is missing:
    the product path never falls back to anything else."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise RuntimeError(
                f"{_LIB_PATH} not found: build it with `python -m paper_1209_0296_b200.build` "
                "(there is no CPU fallback)")
        L = ctypes.CDLL(_LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(L, name)
            fn.restype = res
            fn.argtypes = args
        _lib = L
    return _lib


class LsmError(RuntimeError):
    def __init__(self, code, where):
        L = load()
        msg = L.lsm_strerror(code).decode()
        if code == ERR_CUDA:
            msg += " -- " + L.lsm_last_cuda_error().decode()
        super().__init__(f"{where}: {msg} ({code})")
        self.code = code


def _check(code, where):
    if code != OK:
        raise LsmError(code, where)


def _stream_ptr(stream, device=None):
    import torch

    s = torch.cuda.current_stream(device) if stream is None else stream
    return ctypes.c_void_p(s.cuda_stream)


def _on_device(fn):
    """Run a Lattice method with the lattice's GPU current: the library launches on the calling thread's current
    device, and the default stream is that device's current stream."""
    import functools

    @functools.wraps(fn)
    def wrapped(self, *a, **kw):
        import torch

        with torch.cuda.device(self.device):
            return fn(self, *a, **kw)
    return wrapped


def workspace_bytes(dims, L, two_S=1, model=ISING) -> int:
    n = _sz()
    _check(load().lsm_workspace_bytes(dims, L, two_S, model, ctypes.byref(n)), "lsm_workspace_bytes")
    return int(n.value)


class Lattice:
    """One lattice = one lsm_t handle plus the torch-owned device workspace behind it."""

    def __init__(self, dims, L, two_S=1, model=ISING, J=1.0, h=0.0, T=1.0, seed=0, device="cuda:0", stream=None):
        import torch

        if not torch.cuda.is_available():
            raise RuntimeError("liblsm needs a CUDA device (there is no CPU fallback)")
        self._lib = load()
        self.dims, self.L, self.two_S, self.model = int(dims), int(L), int(two_S), int(model)
        self.J, self.h, self.T, self.seed = float(J), float(h), float(T), int(seed)
        self.device = torch.device(device)
        self.N = self.L ** self.dims
        nbytes = workspace_bytes(dims, L, two_S, model)
        self._h = None
        self._last_stream = None
        with torch.cuda.device(self.device):
            self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            off = (-self._ws.data_ptr()) % 256
            self._ws_ptr = self._ws.data_ptr() + off
            h_ = _vp()
            _check(self._lib.lsm_create(self.dims, self.L, self.two_S, self.model, self.J, self.h, self.T,
                                        self.seed, _vp(self._ws_ptr), nbytes, self._sp(stream),
                                        ctypes.byref(h_)), "lsm_create")
        self._h = h_
        self._scratch = None

    def _sp(self, stream):
        import torch

        self._last_stream = torch.cuda.current_stream(self.device) if stream is None else stream
        return ctypes.c_void_p(self._last_stream.cuda_stream)

    # ------------------------------------------------------------------ life cycle
    @_on_device
    def close(self):
        if getattr(self, "_h", None):
            if self._last_stream is not None:
                self._last_stream.synchronize()      # work may still be in flight on a stream other than the allocator's
            self._lib.lsm_destroy(self._h)
            self._h = None
            self._ws = None
            self._scratch = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _dev_scratch(self, nbytes):
        import torch

        if self._scratch is None or self._scratch.numel() < nbytes:
            self._scratch = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        return self._scratch

    # ------------------------------------------------------------------ sweeps
    @_on_device
    def sweep(self, n=1, stream=None):
        _check(self._lib.lsm_sweep(self._h, int(n), self._sp(stream)), "lsm_sweep")

    @_on_device
    def sweep_record(self, n, out=None, stream=None):
        """n sweeps; returns a device int64 tensor [n, 2] = (B, M) after each sweep (asynchronous)."""
        import torch

        if out is None:
            out = torch.empty((int(n), 2), dtype=torch.int64, device=self.device)
        assert out.is_cuda and out.dtype == torch.int64 and out.is_contiguous() and out.numel() >= 2 * int(n)
        _check(self._lib.lsm_sweep_record(self._h, int(n), _vp(out.data_ptr()), self._sp(stream)),
               "lsm_sweep_record")
        return out

    @_on_device
    def sweep_random_tile(self, n=1, b=32, lam=16, record=False, out=None, stream=None, balanced=False):
        """North-East model: n sweeps of the paper's corrected algorithm: random picks of `lam`
        threads in tiles of b x b spins; balanced=True: its balance-preserving variant.
        record=True returns the device [n, 2] series (0, M)."""
        import torch

        if record and out is None:
            out = torch.empty((int(n), 2), dtype=torch.int64, device=self.device)
        ptr = _vp(out.data_ptr()) if out is not None else None
        fn = self._lib.lsm_sweep_random_tile_balanced if balanced else self._lib.lsm_sweep_random_tile
        _check(fn(self._h, int(n), int(b), int(lam), ptr, self._sp(stream)),
               "lsm_sweep_random_tile_balanced" if balanced else "lsm_sweep_random_tile")
        return out

    @_on_device
    def sweep_record_host(self, n, h_obs=None, stream=None):
        """n sweeps with the (B, M) series delivered into a HOST array (pinned torch tensor or numpy)."""
        import torch

        if h_obs is None:
            h_obs = torch.empty((int(n), 2), dtype=torch.int64).pin_memory()
        ptr = h_obs.data_ptr() if hasattr(h_obs, "data_ptr") else h_obs.ctypes.data
        sc = self._dev_scratch(16 * max(int(n), 1))
        _check(self._lib.lsm_sweep_record_host(self._h, int(n), _vp(ptr), _vp(sc.data_ptr()), self._sp(stream)),
               "lsm_sweep_record_host")
        return h_obs

    @_on_device
    def sweep_record_host_async(self, n, h_obs, d_scratch, stream=None):
        """n sweeps; the (B, M) series lands in the pinned host tensor h_obs once `stream` has been synchronised."""
        _check(self._lib.lsm_sweep_record_host_async(self._h, int(n), _vp(h_obs.data_ptr()), _vp(d_scratch.data_ptr()),
                                                     self._sp(stream)), "lsm_sweep_record_host_async")
        return h_obs

    @_on_device
    def sweep_record_host_noalloc(self, n, h_obs=None, stream=None):
        """n sweeps with the (B, M) series delivered into a HOST array, for callers that cannot allocate device memory
        (a plug-in under somebody else's memory pool, a loop that cannot afford cudaMalloc's device-wide synchronisation,
        a spent memory quota): the device-side staging of the series is a fixed 64 KiB array inside liblsm.so instead of a
        tensor, so this method creates no device tensor and the library call allocates nothing.  n is limited to
        NOALLOC_MAX_SWEEPS (LsmError with code ERR_LIMIT beyond; split the run).  One array per GPU for all lattices:
        do not let two such calls overlap on one GPU.  h_obs: int64 [n, 2] numpy array or host tensor (default: a
        fresh numpy array)."""
        if h_obs is None:
            h_obs = np.empty((int(n), 2), dtype=np.int64)
        ptr = h_obs.data_ptr() if hasattr(h_obs, "data_ptr") else h_obs.ctypes.data
        _check(self._lib.lsm_sweep_record_host_noalloc(self._h, int(n), _vp(ptr), self._sp(stream)),
               "lsm_sweep_record_host_noalloc")
        return h_obs

    @_on_device
    def stage_spins_host(self, h_in, d_stage, copy_stream):
        """Upload only (pinned host tensor -> device staging tensor) on copy_stream; install with set_spins(d_stage, t)."""
        assert h_in.numel() == self.N and d_stage.numel() == self.N and d_stage.is_cuda
        _check(self._lib.lsm_stage_spins_host(self._h, _vp(h_in.data_ptr()), _vp(d_stage.data_ptr()),
                                              ctypes.c_void_p(copy_stream.cuda_stream)), "lsm_stage_spins_host")

    # ------------------------------------------------------------------ observables
    @_on_device
    def measure(self):
        E, M = _dbl(), _i64()
        _check(self._lib.lsm_measure(self._h, ctypes.byref(E), ctypes.byref(M)), "lsm_measure")
        return float(E.value), int(M.value)

    @_on_device
    def measure_int(self):
        B, M, t = _i64(), _i64(), _u64()
        _check(self._lib.lsm_measure_int(self._h, ctypes.byref(B), ctypes.byref(M), ctypes.byref(t)),
               "lsm_measure_int")
        return int(B.value), int(M.value), int(t.value)

    @_on_device
    def measure_full(self):
        B, M = _i64(), _i64()
        _check(self._lib.lsm_measure_full(self._h, ctypes.byref(B), ctypes.byref(M)), "lsm_measure_full")
        return int(B.value), int(M.value)

    @_on_device
    def persistence(self):
        a, b = _i64(), _i64()
        _check(self._lib.lsm_persistence(self._h, ctypes.byref(a), ctypes.byref(b)), "lsm_persistence")
        return int(a.value), int(b.value)

    @_on_device
    def reset_reference(self, stream=None):
        _check(self._lib.lsm_reset_reference(self._h, self._sp(stream)), "lsm_reset_reference")

    @_on_device
    def set_tracking(self, on, stream=None):
        _check(self._lib.lsm_set_tracking(self._h, 1 if on else 0, self._sp(stream)), "lsm_set_tracking")

    # ------------------------------------------------------------------ configuration I/O
    @_on_device
    def get_spins(self, out=None, stream=None):
        import torch

        if out is None:
            out = torch.empty(self.N, dtype=torch.int8, device=self.device)
        assert out.is_cuda and out.dtype == torch.int8 and out.numel() == self.N and out.is_contiguous()
        _check(self._lib.lsm_get_spins(self._h, _vp(out.data_ptr()), self._sp(stream)), "lsm_get_spins")
        return out

    @_on_device
    def get_spins_host(self, h_out=None, stream=None):
        if h_out is None:
            h_out = np.empty(self.N, dtype=np.int8)
        ptr = h_out.data_ptr() if hasattr(h_out, "data_ptr") else h_out.ctypes.data
        sc = self._dev_scratch(self.N)
        _check(self._lib.lsm_get_spins_host(self._h, _vp(ptr), _vp(sc.data_ptr()), self._sp(stream)),
               "lsm_get_spins_host")
        return h_out

    @_on_device
    def set_spins(self, d_in, sweep_counter, stream=None):
        import torch

        assert d_in.is_cuda and d_in.dtype == torch.int8 and d_in.numel() == self.N and d_in.is_contiguous()
        _check(self._lib.lsm_set_spins(self._h, _vp(d_in.data_ptr()), int(sweep_counter), self._sp(stream)),
               "lsm_set_spins")

    @_on_device
    def set_spins_host(self, h_in, sweep_counter, stream=None):
        if hasattr(h_in, "data_ptr"):
            ptr, n = h_in.data_ptr(), h_in.numel()
        else:
            h_in = np.ascontiguousarray(h_in, dtype=np.int8)
            ptr, n = h_in.ctypes.data, h_in.size
        assert n == self.N
        sc = self._dev_scratch(self.N)
        _check(self._lib.lsm_set_spins_host(self._h, _vp(ptr), _vp(sc.data_ptr()), int(sweep_counter),
                                            self._sp(stream)), "lsm_set_spins_host")

    @_on_device
    def set_bonds(self, d_tau, stream=None):
        """EA model: device int8 [dims, N], +1 / -1 per bond (site i, direction +a)."""
        import torch

        assert d_tau.is_cuda and d_tau.dtype == torch.int8 and d_tau.numel() == self.dims * self.N and d_tau.is_contiguous()
        _check(self._lib.lsm_set_bonds(self._h, _vp(d_tau.data_ptr()), self._sp(stream)), "lsm_set_bonds")

    @_on_device
    def get_bonds(self, stream=None):
        import torch

        out = torch.empty((self.dims, self.N), dtype=torch.int8, device=self.device)
        _check(self._lib.lsm_get_bonds(self._h, _vp(out.data_ptr()), self._sp(stream)), "lsm_get_bonds")
        return out

    @_on_device
    def set_temperature(self, T):
        _check(self._lib.lsm_set_temperature(self._h, float(T)), "lsm_set_temperature")
        self.T = float(T)

    @_on_device
    def thresholds(self):
        buf = (_u64 * 128)()
        n = _i32()
        _check(self._lib.lsm_get_thresholds(self._h, buf, ctypes.byref(n)), "lsm_get_thresholds")
        return [int(buf[i]) for i in range(n.value)]

    # ------------------------------------------------------------------ kernel family / counters
    @_on_device
    def set_kernel(self, family):
        _check(self._lib.lsm_set_kernel(self._h, int(family)), "lsm_set_kernel")

    @property
    @_on_device
    def kernel(self):
        k = _i32()
        _check(self._lib.lsm_get_kernel(self._h, ctypes.byref(k)), "lsm_get_kernel")
        return int(k.value)

    @_on_device
    def set_temporal_depth(self, depth):
        """Half-sweeps between two boundary exchanges of the slab family (0: default); results do not depend on it."""
        _check(self._lib.lsm_set_temporal_depth(self._h, int(depth)), "lsm_set_temporal_depth")

    @property
    @_on_device
    def temporal_depth(self):
        d = _i32()
        _check(self._lib.lsm_get_temporal_depth(self._h, ctypes.byref(d)), "lsm_get_temporal_depth")
        return int(d.value)

    @property
    @_on_device
    def launch_count(self):
        n = _u64()
        _check(self._lib.lsm_get_launch_count(self._h, ctypes.byref(n)), "lsm_get_launch_count")
        return int(n.value)


class Batch:
    """R lattices of one shape with per-replica temperature and seed, swept by one launch (lsm_batch_*).

    `replica(r)` is a Lattice view of replica r (borrowed handle) for get_spins / persistence / thresholds ..."""

    def __init__(self, dims, L, T, seeds, two_S=1, model=ISING, J=1.0, h=0.0, device="cuda:0", stream=None):
        import torch

        if not torch.cuda.is_available():
            raise RuntimeError("liblsm needs a CUDA device (there is no CPU fallback)")
        self._lib = load()
        self.T = [float(t) for t in T]
        self.seeds = [int(x) for x in seeds]
        assert len(self.T) == len(self.seeds) and len(self.T) >= 1
        self.R = len(self.T)
        self.dims, self.L, self.two_S, self.model, self.J, self.h = int(dims), int(L), int(two_S), int(model), float(J), float(h)
        self.device = torch.device(device)
        self.N = self.L ** self.dims
        n = _sz()
        _check(self._lib.lsm_batch_workspace_bytes(self.R, self.dims, self.L, self.two_S, self.model, ctypes.byref(n)),
               "lsm_batch_workspace_bytes")
        self._h = None
        self._last_stream = None
        with torch.cuda.device(self.device):
            self._ws = torch.empty(n.value + 256, dtype=torch.uint8, device=self.device)
            ptr = self._ws.data_ptr() + (-self._ws.data_ptr()) % 256
            Ta = (ctypes.c_double * self.R)(*self.T)
            Sa = (ctypes.c_uint64 * self.R)(*self.seeds)
            h_ = _vp()
            _check(self._lib.lsm_batch_create(self.R, self.dims, self.L, self.two_S, self.model, self.J, self.h, Ta, Sa,
                                              _vp(ptr), n.value, self._sp(stream), ctypes.byref(h_)), "lsm_batch_create")
        self._h = h_
        self._views = {}

    def _sp(self, stream):
        import torch

        self._last_stream = torch.cuda.current_stream(self.device) if stream is None else stream
        return ctypes.c_void_p(self._last_stream.cuda_stream)

    @_on_device
    def close(self):
        if getattr(self, "_h", None):
            if self._last_stream is not None:
                self._last_stream.synchronize()
            for v in self._views.values():
                v._h = None                      # borrowed handles die with the batch
            self._views = {}
            self._lib.lsm_batch_destroy(self._h)
            self._h = None
            self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def replica(self, r):
        """Lattice view of replica r (borrowed: closing it does nothing)."""
        if r not in self._views:
            h_ = _vp()
            _check(self._lib.lsm_batch_replica(self._h, int(r), ctypes.byref(h_)), "lsm_batch_replica")
            v = Lattice.__new__(Lattice)
            v._lib, v._h, v._ws, v._scratch, v._last_stream = self._lib, h_, None, None, None
            v.dims, v.L, v.two_S, v.model, v.J, v.h = self.dims, self.L, self.two_S, self.model, self.J, self.h
            v.T, v.seed, v.device, v.N = self.T[r], self.seeds[r], self.device, self.N
            v.close = lambda: None
            self._views[r] = v
        return self._views[r]

    @_on_device
    def sweep(self, n=1, stream=None):
        _check(self._lib.lsm_batch_sweep(self._h, int(n), self._sp(stream)), "lsm_batch_sweep")

    @_on_device
    def sweep_record(self, n, out=None, stream=None):
        """n sweeps of every replica; device int64 [R, n, 2] = (B, M) of replica r after sweep k."""
        import torch

        if out is None:
            out = torch.empty((self.R, int(n), 2), dtype=torch.int64, device=self.device)
        assert out.is_cuda and out.dtype == torch.int64 and out.is_contiguous() and out.numel() >= 2 * int(n) * self.R
        _check(self._lib.lsm_batch_sweep_record(self._h, int(n), _vp(out.data_ptr()), self._sp(stream)),
               "lsm_batch_sweep_record")
        return out

    @_on_device
    def sweep_random_tile(self, n=1, b=32, lam=16, record=False, out=None, stream=None, balanced=False):
        """North-East batches: n sweeps of the paper's corrected algorithm (balanced=True: its
        balance-preserving variant) on every replica, each launch covering the tiles of all replicas.
        record=True returns the device [R, n, 2] series (0, M)."""
        import torch

        if record and out is None:
            out = torch.empty((self.R, int(n), 2), dtype=torch.int64, device=self.device)
        ptr = _vp(out.data_ptr()) if out is not None else None
        _check(self._lib.lsm_batch_sweep_random_tile(self._h, int(n), int(b), int(lam), 1 if balanced else 0, ptr,
                                                     self._sp(stream)), "lsm_batch_sweep_random_tile")
        return out

    @_on_device
    def set_temperatures(self, T):
        T = [float(t) for t in T]
        assert len(T) == self.R
        _check(self._lib.lsm_batch_set_temperatures(self._h, (ctypes.c_double * self.R)(*T)), "lsm_batch_set_temperatures")
        self.T = T
        for r, v in self._views.items():
            v.T = T[r]

    @_on_device
    def set_tracking(self, on, stream=None):
        _check(self._lib.lsm_batch_set_tracking(self._h, 1 if on else 0, self._sp(stream)), "lsm_batch_set_tracking")

    def set_cluster(self, blocks_per_replica):
        _check(self._lib.lsm_batch_set_cluster(self._h, int(blocks_per_replica)), "lsm_batch_set_cluster")

    @_on_device
    def measure_int(self):
        """[(B, M)] of every replica's current configuration (synchronises once)."""
        Bv, Mv = (ctypes.c_int64 * self.R)(), (ctypes.c_int64 * self.R)()
        _check(self._lib.lsm_batch_measure_int(self._h, Bv, Mv), "lsm_batch_measure_int")
        return [(int(Bv[r]), int(Mv[r])) for r in range(self.R)]

    @property
    def launch_count(self):
        n = _u64()
        _check(self._lib.lsm_batch_get_launch_count(self._h, ctypes.byref(n)), "lsm_batch_get_launch_count")
        return int(n.value)


# ---------------------------------------------------------------------- derived doubles (host math in the library)
def binder_u4(obs) -> float:
    a = np.ascontiguousarray(obs, dtype=np.int64).reshape(-1, 2)
    out = _dbl()
    _check(load().lsm_binder_u4(_vp(a.ctypes.data), a.shape[0], ctypes.byref(out)), "lsm_binder_u4")
    return float(out.value)


def heat_capacity(obs, N, J, h, T) -> float:
    a = np.ascontiguousarray(obs, dtype=np.int64).reshape(-1, 2)
    out = _dbl()
    _check(load().lsm_heat_capacity(_vp(a.ctypes.data), a.shape[0], int(N), float(J), float(h), float(T),
                                    ctypes.byref(out)), "lsm_heat_capacity")
    return float(out.value)


def series_means(obs, N, J, h) -> tuple[float, float]:
    """(<E>/N, <|M|>/N) of a recorded (B, M) series."""
    a = np.ascontiguousarray(obs, dtype=np.int64).reshape(-1, 2)
    e, m = _dbl(), _dbl()
    _check(load().lsm_series_means(_vp(a.ctypes.data), a.shape[0], int(N), float(J), float(h), ctypes.byref(e),
                                   ctypes.byref(m)), "lsm_series_means")
    return float(e.value), float(m.value)


def phi(overlap, N, c) -> float:
    out = _dbl()
    _check(load().lsm_phi(int(overlap), int(N), float(c), ctypes.byref(out)), "lsm_phi")
    return float(out.value)


def persistence_fraction(never_changed, N) -> float:
    out = _dbl()
    _check(load().lsm_persistence_fraction(int(never_changed), int(N), ctypes.byref(out)), "lsm_persistence_fraction")
    return float(out.value)


def energy(model, J, h, B, M) -> float:
    out = _dbl()
    _check(load().lsm_energy(int(model), float(J), float(h), int(B), int(M), ctypes.byref(out)), "lsm_energy")
    return float(out.value)


# ---------------------------------------------------------------------- test hooks
def philox_device(ctr_key):
    """ctr_key: int array [n, 6] (c0..c3, k0, k1) -> uint32 array [n, 4] computed by the device Philox."""
    import torch

    a = torch.as_tensor(np.ascontiguousarray(ctr_key, dtype=np.uint32).view(np.int32)).cuda()
    out = torch.empty((a.shape[0], 4), dtype=torch.int32, device=a.device)
    _check(load().lsm_philox_device(_vp(a.data_ptr()), _vp(out.data_ptr()), a.shape[0], _stream_ptr(None)),
           "lsm_philox_device")
    return out.cpu().numpy().view(np.uint32)


def philox_throughput(blocks, calls, stream=None):
    """Enqueue the register-only Philox loop; returns the sink tensor (keeps it alive)."""
    import torch

    sink = torch.empty(blocks * 256, dtype=torch.int32, device="cuda")
    _check(load().lsm_philox_throughput(int(blocks), int(calls), _vp(sink.data_ptr()), _stream_ptr(stream)),
           "lsm_philox_throughput")
    return sink
