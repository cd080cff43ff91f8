"""ctypes binding of libafqmc.so (include/afqmc.h).  Argument marshalling only: every step
of the path runs in the library's CUDA kernels.  There is no CPU fallback: if the library is
missing or cannot be loaded, importing this module raises.

Arrays may be torch CUDA tensors (device pointers) or NumPy arrays / CPU tensors (host
pointers, staged inside the library call).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libafqmc.so")

EXPORTS = ["afqmc_create", "afqmc_step", "afqmc_local_energy", "afqmc_get_overlaps",
           "afqmc_get_constants", "afqmc_debug_read", "afqmc_launch_count", "afqmc_sync",
           "afqmc_last_error", "afqmc_destroy", "afqmc_measure_fp64_peak", "afqmc_set_profiling",
           "afqmc_get_stage_times", "afqmc_population_control", "afqmc_estimators", "afqmc_run_block",
           "afqmc_set_block_graph", "afqmc_shard_setup_partial", "afqmc_shard_setup_finish",
           "afqmc_shard_get_buffers", "afqmc_shard_ipc_export", "afqmc_shard_ipc_open", "afqmc_shard_ipc_close",
           "afqmc_shard_set_peers", "afqmc_shard_theta", "afqmc_shard_vhs", "afqmc_shard_propagate",
           "afqmc_shard_energy", "afqmc_shard_energy_finish", "afqmc_shard_setup_reduce", "afqmc_exchange_plan", "afqmc_exchange_plan_pin",
           "afqmc_reorthonormalise", "afqmc_qr_shifted_passes", "afqmc_comb_static",
           "afqmc_exchange_plan_unpin"]

COMB_STATIC_MAX_WALKERS = 65536      # AFQMC_COMB_STATIC_MAX_WALKERS of include/afqmc.h

STAGES = ["overlap_theta", "force_bias", "field_shift", "vhs", "one_body", "taylor", "overlap_new",
          "weight", "reortho", "e_theta", "exchange", "e_reduce", "e1_build", "pop_control", "estimators",
          "shard_exchange", "shard_reduce", "fused_step", "fused_energy"]


class AfqmcParams(C.Structure):
    _fields_ = [("struct_size", C.c_int32), ("M", C.c_int32), ("n_alpha", C.c_int32),
                ("n_beta", C.c_int32), ("n_chol", C.c_int32), ("max_walkers", C.c_int32),
                ("walker_kind", C.c_int32), ("taylor_order", C.c_int32),
                ("ortho_every", C.c_int32), ("e_shift_auto", C.c_int32),
                ("e_shift", C.c_double), ("stream", C.c_void_p), ("pack_chol", C.c_int32),
                ("group_size", C.c_int32), ("group_rank", C.c_int32), ("mixed_precision", C.c_int32),
                ("complex_chol", C.c_int32), ("kernel_path", C.c_int32), ("complex_trial", C.c_int32),
                ("tuning_flags", C.c_int32), ("xbar_bound", C.c_double), ("ehyb_bound", C.c_double)]


def _load():
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} not found: build it with `python -m paper_2406_16238_b200.build` "
                          "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp, i32, i64, dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_double
    lib.afqmc_create.argtypes = [vp, vp, vp, C.POINTER(AfqmcParams), C.POINTER(vp)]
    lib.afqmc_create.restype = i32
    lib.afqmc_step.argtypes = [vp, vp, vp, vp, dbl, i32]
    lib.afqmc_step.restype = i32
    lib.afqmc_local_energy.argtypes = [vp, vp, vp, i32]
    lib.afqmc_local_energy.restype = i32
    lib.afqmc_get_overlaps.argtypes = [vp, vp]
    lib.afqmc_get_overlaps.restype = i32
    lib.afqmc_get_constants.argtypes = [vp, vp]
    lib.afqmc_get_constants.restype = i32
    lib.afqmc_debug_read.argtypes = [vp, i32, vp]
    lib.afqmc_debug_read.restype = i64
    lib.afqmc_launch_count.argtypes = [vp]
    lib.afqmc_launch_count.restype = i64
    lib.afqmc_sync.argtypes = [vp]
    lib.afqmc_sync.restype = i32
    lib.afqmc_last_error.argtypes = [vp]
    lib.afqmc_last_error.restype = C.c_char_p
    lib.afqmc_destroy.argtypes = [vp]
    lib.afqmc_destroy.restype = None
    lib.afqmc_set_profiling.argtypes = [vp, i32]
    lib.afqmc_set_profiling.restype = i32
    lib.afqmc_get_stage_times.argtypes = [vp, vp, vp, i32]
    lib.afqmc_get_stage_times.restype = i32
    lib.afqmc_population_control.argtypes = [vp, vp, vp, vp, i32, vp]
    lib.afqmc_population_control.restype = i32
    lib.afqmc_estimators.argtypes = [vp, vp, vp, vp, i32]
    lib.afqmc_estimators.restype = i32
    lib.afqmc_run_block.argtypes = [vp, vp, vp, vp, vp, dbl, i32, i32, i32, vp, vp]
    lib.afqmc_run_block.restype = i32
    lib.afqmc_set_block_graph.argtypes = [vp, i32]
    lib.afqmc_set_block_graph.restype = i64
    u64 = C.c_uint64
    for name, args in [("afqmc_shard_setup_partial", [vp, vp]), ("afqmc_shard_setup_finish", [vp, vp]),
                       ("afqmc_shard_get_buffers", [vp, vp]), ("afqmc_shard_ipc_export", [vp, i32, vp]),
                       ("afqmc_shard_ipc_open", [vp, vp, vp]), ("afqmc_shard_ipc_close", [u64]),
                       ("afqmc_shard_set_peers", [vp, vp]), ("afqmc_shard_theta", [vp, vp, i32, i32]),
                       ("afqmc_shard_vhs", [vp, vp, dbl, i32]), ("afqmc_shard_propagate", [vp, vp, vp, dbl, i32]),
                       ("afqmc_shard_energy", [vp, i32]), ("afqmc_shard_energy_finish", [vp, vp, i32])]:
        getattr(lib, name).argtypes = args
        getattr(lib, name).restype = i32
    lib.afqmc_shard_setup_reduce.argtypes = [vp, i32, i64, vp]
    lib.afqmc_shard_setup_reduce.restype = i32
    lib.afqmc_measure_fp64_peak.argtypes = [dbl, vp]
    lib.afqmc_measure_fp64_peak.restype = i32
    lib.afqmc_reorthonormalise.argtypes = [vp, vp, vp, i32]
    lib.afqmc_reorthonormalise.restype = i32
    lib.afqmc_qr_shifted_passes.argtypes = [vp]
    lib.afqmc_qr_shifted_passes.restype = i64
    lib.afqmc_comb_static.argtypes = [vp, vp, vp, i32, vp, C.c_char_p, i32]
    lib.afqmc_comb_static.restype = i32
    lib.afqmc_exchange_plan.argtypes = [i32, i32, i32, C.c_char_p, i32]
    lib.afqmc_exchange_plan.restype = i32
    lib.afqmc_exchange_plan_pin.argtypes = [i32] * 10
    lib.afqmc_exchange_plan_pin.restype = i32
    lib.afqmc_exchange_plan_unpin.argtypes = [i32, i32, i32]
    lib.afqmc_exchange_plan_unpin.restype = i32
    return lib


lib = _load()


class AfqmcError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libafqmc error {code}: {msg}")
        self.code = code


def _ptr(a):
    """Raw address of a torch tensor or a NumPy array (must be contiguous)."""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        if not a.flags["C_CONTIGUOUS"]:
            raise ValueError("array must be C-contiguous")
        return a.ctypes.data
    if hasattr(a, "data_ptr"):
        if not a.is_contiguous():
            raise ValueError("tensor must be contiguous")
        return a.data_ptr()
    raise TypeError(f"unsupported array type {type(a)}")


def measure_fp64_peak(ms=200.0):
    """(DMMA TFLOP/s, DFMA TFLOP/s, SM MHz) from register-only issue loops."""
    out = np.zeros(3)
    rc = lib.afqmc_measure_fp64_peak(float(ms), out.ctypes.data)
    if rc != 0:
        raise AfqmcError(rc, "afqmc_measure_fp64_peak")
    return tuple(out)


def comb_static(weights, xi, map_out, nw=None, stream=None):
    """afqmc_comb_static: the population-control comb for callers that cannot allocate device memory - no handle, no
    cudaMalloc; the running sum lives in a 512 KiB array built into the library (at most COMB_STATIC_MAX_WALKERS
    walkers).  `weights` (float64, in/out), `xi` (one float64) and `map_out` (int32) are CUDA tensors on one GPU;
    `stream` is a raw cudaStream_t of that GPU (None: its default stream).  Asynchronous; calls that may overlap on
    one GPU share the array and must be ordered by the caller."""
    n = int(weights.shape[0]) if nw is None else int(nw)
    buf = C.create_string_buffer(512)
    rc = lib.afqmc_comb_static(_ptr(weights), _ptr(xi), _ptr(map_out), n, stream, buf, len(buf))
    if rc != 0:
        raise AfqmcError(rc, buf.value.decode())


def exchange_plan(ns, M, pair=False):
    """(useful fraction of the issued DMMA blocks, description) of the exchange kernel's tile plan."""
    buf = C.create_string_buffer(512)
    rc = lib.afqmc_exchange_plan(int(ns), int(M), int(bool(pair)), buf, 512)
    if rc < 0:
        raise AfqmcError(rc, "afqmc_exchange_plan")
    return rc * 1e-6, buf.value.decode()


def exchange_plan_pin(ns, M, pair, warps, mi, ni, wm, G, Wn, epi_warps=3):
    """Pin the exchange kernel's tile plan for (ns, M, pair); call before creating handles.  False if it does not fit."""
    return lib.afqmc_exchange_plan_pin(int(ns), int(M), int(bool(pair)), int(warps), int(mi), int(ni), int(wm),
                                       int(G), int(Wn), int(epi_warps)) == 0


def exchange_plan_unpin(ns=0, M=0, pair=False):
    """Forget the pinned exchange plan of (ns, M, pair); ns = 0: every pin of this process."""
    rc = lib.afqmc_exchange_plan_unpin(int(ns), int(M), 1 if pair else 0)
    if rc != 0:
        raise AfqmcError(rc, "afqmc_exchange_plan_unpin")


class AFQMC:
    """Handle wrapper with the same calls as the C ABI."""

    def __init__(self, h1, L_chol, trial, *, M, n_alpha, n_beta, n_chol, max_walkers,
                 walker_kind, taylor_order=6, ortho_every=0, e_shift=None, stream=None, pack_chol=False,
                 group_size=0, group_rank=0, mixed_precision=False, complex_chol=False, kernel_path=0,
                 complex_trial=False, xbar_bound=0.0, ehyb_bound=0.0, tuning_flags=0):
        p = AfqmcParams()
        p.struct_size = C.sizeof(AfqmcParams)
        p.M, p.n_alpha, p.n_beta, p.n_chol = M, n_alpha, n_beta, n_chol
        p.max_walkers, p.walker_kind = max_walkers, walker_kind
        p.taylor_order, p.ortho_every = taylor_order, ortho_every
        p.e_shift_auto = 1 if e_shift is None else 0
        p.e_shift = 0.0 if e_shift is None else float(e_shift)
        p.stream = stream
        p.pack_chol = 1 if pack_chol else 0
        p.group_size, p.group_rank = int(group_size), int(group_rank)
        p.mixed_precision = 1 if mixed_precision else 0
        p.complex_chol = 1 if complex_chol else 0
        p.kernel_path = int(kernel_path)
        p.complex_trial = 1 if complex_trial else 0
        p.xbar_bound, p.ehyb_bound = float(xbar_bound), float(ehyb_bound)
        p.tuning_flags = int(tuning_flags)
        # L_chol is borrowed by the library (only during create when pack_chol is set)
        self._keep = (h1, None if (pack_chol or mixed_precision or complex_chol) else L_chol, trial)
        self.M, self.n_chol, self.max_walkers = M, n_chol, max_walkers
        self.Nt = n_alpha if walker_kind == 0 else n_alpha + n_beta
        h = C.c_void_p()
        rc = lib.afqmc_create(_ptr(h1), _ptr(L_chol), _ptr(trial), C.byref(p), C.byref(h))
        if rc != 0:
            raise AfqmcError(rc, lib.afqmc_last_error(None).decode())
        self._h = h

    def _check(self, rc):
        if rc != 0:
            raise AfqmcError(rc, lib.afqmc_last_error(self._h).decode())

    def step(self, walkers, weights, aux_fields, dt, nw=None):
        nw = int(walkers.shape[0]) if nw is None else nw
        self._check(lib.afqmc_step(self._h, _ptr(walkers), _ptr(weights), _ptr(aux_fields), float(dt), nw))

    def local_energy(self, walkers, E_out, nw=None):
        nw = int(walkers.shape[0]) if nw is None else nw
        self._check(lib.afqmc_local_energy(self._h, _ptr(walkers), _ptr(E_out), nw))

    def reorthonormalise(self, walkers, detR_out=None, nw=None):
        nw = int(walkers.shape[0]) if nw is None else nw
        self._check(lib.afqmc_reorthonormalise(self._h, _ptr(walkers), _ptr(detR_out), nw))

    def qr_shifted_passes(self):
        v = int(lib.afqmc_qr_shifted_passes(self._h))
        if v < 0:
            self._check(v)
        return v

    def population_control(self, walkers, weights, xi, map_out=None, nw=None):
        """xi: array/tensor holding one double in [0, 1) (host or device)."""
        nw = int(walkers.shape[0]) if nw is None else nw
        self._check(lib.afqmc_population_control(self._h, _ptr(walkers), _ptr(weights), _ptr(xi), nw,
                                                 _ptr(map_out)))

    def estimators(self, weights, E, est_out, nw=None):
        nw = int(weights.shape[0]) if nw is None else nw
        self._check(lib.afqmc_estimators(self._h, _ptr(weights), _ptr(E), _ptr(est_out), nw))

    def run_block(self, walkers, weights, aux_fields, xi, dt, pop_every, E_out=None, est_out=None, nw=None):
        """aux_fields [n_steps][nw][n_chol]; xi [n_steps // pop_every] doubles (None if pop_every = 0)."""
        nw = int(walkers.shape[0]) if nw is None else nw
        n_steps = int(aux_fields.shape[0])
        self._check(lib.afqmc_run_block(self._h, _ptr(walkers), _ptr(weights), _ptr(aux_fields), _ptr(xi),
                                        float(dt), nw, n_steps, int(pop_every), _ptr(E_out), _ptr(est_out)))

    def set_block_graph(self, on=-1):
        """Switch CUDA-graph replay of run_block on/off (-1: query only); returns graph launches so far."""
        n = lib.afqmc_set_block_graph(self._h, int(on))
        if n < 0:
            self._check(int(n))
        return int(n)

    def get_overlaps(self, out):
        self._check(lib.afqmc_get_overlaps(self._h, _ptr(out)))

    def constants(self):
        out = np.zeros(3)
        self._check(lib.afqmc_get_constants(self._h, out.ctypes.data))
        return dict(E_const=out[0], e_shift=out[1], e_trial=out[2])

    def debug_read(self, which):
        n = lib.afqmc_debug_read(self._h, which, None)
        if n < 0:
            self._check(int(n))
        out = np.empty(int(n))
        r = lib.afqmc_debug_read(self._h, which, out.ctypes.data)
        if r < 0:
            self._check(int(r))
        return out

    # ---- distributed Hamiltonian (group_size > 1): the afqmc_shard_* phases, same names ----
    def shard_setup_partial(self):
        out = np.empty(self.M * self.M + 2)
        self._check(lib.afqmc_shard_setup_partial(self._h, out.ctypes.data))
        return out

    @staticmethod
    def shard_setup_reduce(parts):
        """Member-order sum of the partials [G][M*M + 2] (done inside the library)."""
        a = np.ascontiguousarray(parts, dtype=np.float64)
        out = np.empty(a.shape[1])
        rc = lib.afqmc_shard_setup_reduce(a.ctypes.data, a.shape[0], a.shape[1], out.ctypes.data)
        if rc != 0:
            raise AfqmcError(rc, "afqmc_shard_setup_reduce")
        return out

    def shard_ipc_open(self, handle_bytes):
        """Map a peer's exported buffer on this member's device; returns the device address."""
        out = np.zeros(1, dtype=np.uint64)
        hb = np.frombuffer(handle_bytes, dtype=np.uint8).copy()
        rc = lib.afqmc_shard_ipc_open(self._h, hb.ctypes.data, out.ctypes.data)
        if rc != 0:
            raise AfqmcError(rc, lib.afqmc_last_error(None).decode())
        return int(out[0])

    def shard_setup_finish(self, total):
        self._check(lib.afqmc_shard_setup_finish(self._h, _ptr(total)))

    def shard_get_buffers(self):
        out = np.zeros(4, dtype=np.uint64)
        self._check(lib.afqmc_shard_get_buffers(self._h, out.ctypes.data))
        return out

    def shard_ipc_export(self, which):
        buf = np.zeros(64, dtype=np.uint8)
        self._check(lib.afqmc_shard_ipc_export(self._h, int(which), buf.ctypes.data))
        return buf

    def shard_set_peers(self, addrs):
        a = np.ascontiguousarray(addrs, dtype=np.uint64)
        self._check(lib.afqmc_shard_set_peers(self._h, a.ctypes.data))

    def shard_theta(self, walkers, for_energy=False, nw=None):
        nw = int(walkers.shape[0]) if nw is None else nw
        self._check(lib.afqmc_shard_theta(self._h, _ptr(walkers), nw, 1 if for_energy else 0))

    def shard_vhs(self, aux_local, dt, nw):
        self._check(lib.afqmc_shard_vhs(self._h, _ptr(aux_local), float(dt), int(nw)))

    def shard_propagate(self, walkers, weights, dt, nw=None):
        nw = int(walkers.shape[0]) if nw is None else nw
        self._check(lib.afqmc_shard_propagate(self._h, _ptr(walkers), _ptr(weights), float(dt), nw))

    def shard_energy(self, nw):
        self._check(lib.afqmc_shard_energy(self._h, int(nw)))

    def shard_energy_finish(self, E_out, nw=None):
        nw = int(E_out.shape[0]) if nw is None else nw
        self._check(lib.afqmc_shard_energy_finish(self._h, _ptr(E_out), nw))

    def set_profiling(self, on):
        self._check(lib.afqmc_set_profiling(self._h, 1 if on else 0))

    def stage_times(self, reset=False):
        """{stage: (total ms, brackets)} since the last reset (synchronises the stream)."""
        ms = np.zeros(len(STAGES))
        n = np.zeros(len(STAGES), dtype=np.int64)
        self._check(lib.afqmc_get_stage_times(self._h, ms.ctypes.data, n.ctypes.data, 1 if reset else 0))
        return {k: (float(ms[i]), int(n[i])) for i, k in enumerate(STAGES)}

    def launch_count(self):
        return int(lib.afqmc_launch_count(self._h))

    def sync(self):
        self._check(lib.afqmc_sync(self._h))

    def close(self):
        if getattr(self, "_h", None):
            lib.afqmc_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
