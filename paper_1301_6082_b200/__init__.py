"""paper_1301_6082_b200 - thin Python binding of libpcpd.so (include/pcpd.h).

Argument marshalling only: every step of the path (RNG, masks, schedule, update
rule, density reduction) runs in the CUDA kernels of csrc/.  PyTorch is used for
device memory (its CUDA caching allocator is installed as the library's
allocator) and for the stream (torch's current stream), nothing else.  There is
no CPU fallback: if libpcpd.so is missing or no B200 is present, calls raise.

Names follow the C ABI: pcpd_create / pcpd_init / pcpd_run / pcpd_density ...
"""
from __future__ import annotations

import atexit
import ctypes as C
import os
import weakref

import numpy as np

from .shard import gather_counts, max_over_ranks, shard_words  # noqa: F401

PCPD, TCPD, QCPD, CPD = 0, 1, 2, 3
CONNECTED = 0x200    # OR into `variant`: the paper's connected multispin lattice (PCPD_VARIANT_CONNECTED)
PMASK_PAPER = 0x100  # OR into `variant`: the paper's own annihilation mask (PCPD_VARIANT_PMASK_PAPER)
# with PMASK_PAPER: decorrelation bound b of the paper's mask family (default 1/4) - PCPD_VARIANT_PMASK_BOUND_*
PMASK_BOUND_HALF, PMASK_BOUND_ONE, PMASK_BOUND_3_4 = 0x400, 0x800, 0xC00
INIT_FULL, INIT_BERNOULLI, INIT_EMPTY = 0, 1, 2
DEFAULT_TS, DEFAULT_D, DEFAULT_A = 2048, 64, 4
STATIC_SERIES_MAX_COUNTS = 524288   # PCPD_STATIC_SERIES_MAX_COUNTS of include/pcpd.h

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpcpd.so")

# every symbol include/pcpd.h declares
EXPORTS = (
    "pcpd_set_allocator", "pcpd_set_stream", "pcpd_create", "pcpd_create_ex", "pcpd_create_scan", "pcpd_init", "pcpd_run",
    "pcpd_density", "pcpd_pair_density", "pcpd_get_lattice", "pcpd_set_lattice", "pcpd_schedule_info",
    "pcpd_thresholds", "pcpd_sweep", "pcpd_set_sweep", "pcpd_synchronize", "pcpd_destroy", "pcpd_last_error",
    "pcpd_launch_count", "pcpd_microbench", "pcpd_jit_state", "pcpd_jit_message", "pcpd_jit_launch_count",
    "pcpd_jit_selftest", "pcpd_split_launch_count", "pcpd_step_from_host", "pcpd_run_series", "pcpd_delta_eff",
    "pcpd_run_series_static", "pcpd_step_from_host_columns",
)

_ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p)
_FREE_FN = C.CFUNCTYPE(None, C.c_void_p)

_lib = None
_keepalive = []
_live = weakref.WeakSet()  # open handles; closed at interpreter exit while torch's allocator is still alive


@atexit.register
def _close_all():
    for h in list(_live):
        try:
            h.close()
        except Exception:
            pass


class PcpdError(RuntimeError):
    pass


def load_library() -> C.CDLL:
    """dlopen the in-tree libpcpd.so and declare the signatures.  Fails loudly
    when the extension has not been built (python -m paper_1301_6082_b200.build)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise PcpdError(f"{LIB_PATH} is missing: run `python -m paper_1301_6082_b200.build` (no CPU fallback exists)")
    L = C.CDLL(LIB_PATH)
    u32p, u64p = C.POINTER(C.c_uint32), C.POINTER(C.c_uint64)
    L.pcpd_set_allocator.argtypes = [_ALLOC_FN, _FREE_FN]
    L.pcpd_set_allocator.restype = C.c_int
    L.pcpd_set_stream.argtypes = [C.c_void_p, C.c_void_p]
    L.pcpd_set_stream.restype = C.c_int
    L.pcpd_create.argtypes = [C.c_uint64, C.c_uint64, C.c_double, C.c_double, C.c_uint64, C.c_int]
    L.pcpd_create.restype = C.c_void_p
    L.pcpd_create_ex.argtypes = [C.c_uint64, C.c_uint64, C.c_double, C.c_double, C.c_uint64, C.c_int,
                                 C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint64]
    L.pcpd_create_ex.restype = C.c_void_p
    L.pcpd_create_scan.argtypes = [C.c_uint64, C.c_uint64, C.c_void_p, C.c_void_p, C.c_uint64, C.c_int,
                                   C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint64]
    L.pcpd_create_scan.restype = C.c_void_p
    L.pcpd_init.argtypes = [C.c_void_p, C.c_int]
    L.pcpd_init.restype = C.c_int
    L.pcpd_run.argtypes = [C.c_void_p, C.c_uint64]
    L.pcpd_run.restype = C.c_int
    L.pcpd_density.argtypes = [C.c_void_p, C.c_void_p]
    L.pcpd_density.restype = C.c_int
    L.pcpd_pair_density.argtypes = [C.c_void_p, C.c_void_p]
    L.pcpd_pair_density.restype = C.c_int
    L.pcpd_get_lattice.argtypes = [C.c_void_p, C.c_void_p]
    L.pcpd_get_lattice.restype = C.c_int
    L.pcpd_set_lattice.argtypes = [C.c_void_p, C.c_void_p]
    L.pcpd_set_lattice.restype = C.c_int
    L.pcpd_schedule_info.argtypes = [C.c_void_p, u32p, u32p, u32p, u32p]
    L.pcpd_schedule_info.restype = C.c_int
    L.pcpd_thresholds.argtypes = [C.c_void_p, u64p, u64p]
    L.pcpd_thresholds.restype = C.c_int
    L.pcpd_sweep.argtypes = [C.c_void_p]
    L.pcpd_sweep.restype = C.c_uint64
    L.pcpd_set_sweep.argtypes = [C.c_void_p, C.c_uint64]
    L.pcpd_set_sweep.restype = C.c_int
    L.pcpd_synchronize.argtypes = [C.c_void_p]
    L.pcpd_synchronize.restype = C.c_int
    L.pcpd_destroy.argtypes = [C.c_void_p]
    L.pcpd_destroy.restype = None
    L.pcpd_last_error.argtypes = []
    L.pcpd_last_error.restype = C.c_char_p
    L.pcpd_launch_count.argtypes = []
    L.pcpd_launch_count.restype = C.c_uint64
    L.pcpd_microbench.argtypes = [C.c_int, C.c_uint32, C.POINTER(C.c_double)]
    L.pcpd_microbench.restype = C.c_int
    L.pcpd_jit_state.argtypes = [C.c_void_p]
    L.pcpd_jit_state.restype = C.c_int
    L.pcpd_jit_message.argtypes = []
    L.pcpd_jit_message.restype = C.c_char_p
    L.pcpd_jit_launch_count.argtypes = []
    L.pcpd_jit_launch_count.restype = C.c_uint64
    L.pcpd_jit_selftest.argtypes = [C.c_int, C.c_uint32, C.c_uint32, u64p]
    L.pcpd_jit_selftest.restype = C.c_int
    L.pcpd_run_series.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, C.c_void_p, C.c_void_p]
    L.pcpd_run_series.restype = C.c_int
    L.pcpd_step_from_host.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, C.c_void_p]
    L.pcpd_step_from_host.restype = C.c_int
    L.pcpd_step_from_host_columns.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, C.c_void_p]
    L.pcpd_step_from_host_columns.restype = C.c_int
    L.pcpd_split_launch_count.argtypes = [C.c_void_p]
    L.pcpd_split_launch_count.restype = C.c_uint64
    L.pcpd_run_series_static.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, C.c_void_p, C.c_void_p]
    L.pcpd_run_series_static.restype = C.c_int
    L.pcpd_delta_eff.argtypes = [C.c_void_p, C.c_uint64, C.c_void_p, C.c_uint64, C.c_uint64, C.c_uint32, C.c_void_p, C.c_void_p]
    L.pcpd_delta_eff.restype = C.c_int
    _lib = L
    return L


def _install_torch_allocator(L: C.CDLL) -> None:
    """PyTorch for device memory: route the library's allocations through
    torch's CUDA caching allocator."""
    if _keepalive:
        return
    import torch

    def _alloc(nbytes, stream):
        try:
            return torch.cuda.caching_allocator_alloc(int(nbytes), stream=int(stream or 0))
        except Exception:
            return None

    def _free(ptr):
        torch.cuda.caching_allocator_delete(ptr)

    a, f = _ALLOC_FN(_alloc), _FREE_FN(_free)
    _keepalive.extend([a, f])
    L.pcpd_set_allocator(a, f)


def _err(L) -> str:
    return (L.pcpd_last_error() or b"").decode()


def _check(L, rc):
    if rc != 0:
        raise PcpdError(f"libpcpd error {rc}: {_err(L)}")


def launch_count() -> int:
    return int(load_library().pcpd_launch_count())


def jit_launch_count() -> int:
    return int(load_library().pcpd_jit_launch_count())


def jit_message() -> str:
    return (load_library().pcpd_jit_message() or b"").decode()


def jit_selftest(variant: int, T_d: int, T_p: int) -> int:
    """Compile (NVRTC, no device needed) the sweep kernel specialised on the thresholds; returns the cubin size."""
    L = load_library()
    n = C.c_uint64(0)
    _check(L, L.pcpd_jit_selftest(int(variant), int(T_d), int(T_p), C.byref(n)))
    return int(n.value)


def microbench(kind: int, iters: int = 2000) -> float:
    L = load_library()
    out = C.c_double()
    _check(L, L.pcpd_microbench(kind, iters, C.byref(out)))
    return out.value


def delta_eff(times, series, L, half_window=1):
    """pcpd_delta_eff: (rho[k], delta_eff[k]) of a density series: rho = mean count / L,
    delta_eff = -d ln rho / d ln t as a central log-log difference over +- half_window records (NaN at the ends).
    `series` is counts[len(times), n_replicas] as pcpd_run_series returns it (particle or pair counts)."""
    lib = load_library()
    t = np.ascontiguousarray(times, dtype=np.uint64)
    c = np.ascontiguousarray(series, dtype=np.uint32)
    if c.ndim != 2 or c.shape[0] != len(t):
        raise ValueError("series must be counts[len(times), n_replicas]")
    rho, dl = np.empty(len(t)), np.empty(len(t))
    _check(lib, lib.pcpd_delta_eff(t.ctypes.data, len(t), c.ctypes.data, c.shape[1], int(L), int(half_window),
                                   rho.ctypes.data, dl.ctypes.data))
    return rho, dl


class Pcpd:
    """One simulation handle (pcpd_t).  Methods mirror the C ABI one to one."""

    def __init__(self, L, n_replicas, d, p, seed, variant=PCPD, Ts=None, D=None, A=None, word_offset=0):
        import torch

        if not torch.cuda.is_available():
            raise PcpdError("no CUDA device: the PCPD path has no CPU fallback")
        lib = load_library()
        _install_torch_allocator(lib)
        self._lib = lib
        torch.cuda.current_stream()  # make sure the context exists
        if np.ndim(d) or np.ndim(p):   # per-word-column probabilities: pcpd_create_scan
            W = int(n_replicas) // 64
            dw = np.ascontiguousarray(np.broadcast_to(np.asarray(d, dtype=np.float64), (W,)))
            pw = np.ascontiguousarray(np.broadcast_to(np.asarray(p, dtype=np.float64), (W,)))
            h = lib.pcpd_create_scan(L, n_replicas, dw.ctypes.data, pw.ctypes.data, seed, variant, Ts or DEFAULT_TS,
                                     D or DEFAULT_D, A or DEFAULT_A, word_offset)
        elif Ts is None and D is None and A is None and word_offset == 0:
            h = lib.pcpd_create(L, n_replicas, d, p, seed, variant)
        else:
            h = lib.pcpd_create_ex(L, n_replicas, d, p, seed, variant, Ts or DEFAULT_TS, D or DEFAULT_D,
                                   A or DEFAULT_A, word_offset)
        if not h:
            raise PcpdError(f"pcpd_create failed: {_err(lib)}")
        self._h = h
        _live.add(self)
        self.L, self.n_replicas, self.W = int(L), int(n_replicas), int(n_replicas) // 64
        self.use_current_stream()

    # -- plumbing
    def use_current_stream(self):
        import torch

        _check(self._lib, self._lib.pcpd_set_stream(self._h, torch.cuda.current_stream().cuda_stream))

    def close(self):
        if getattr(self, "_h", None):
            self._lib.pcpd_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- the path
    def init(self, mode=INIT_FULL):
        _check(self._lib, self._lib.pcpd_init(self._h, mode))

    def run(self, n_sweeps):
        _check(self._lib, self._lib.pcpd_run(self._h, n_sweeps))

    def density(self, out=None) -> np.ndarray:
        out = np.empty(self.n_replicas, dtype=np.uint32) if out is None else out
        _check(self._lib, self._lib.pcpd_density(self._h, out.ctypes.data))
        return out

    def run_series(self, times, pairs=False):
        """Advance to each of the ascending absolute sweep indices `times` and record the per-replica counts there
        (pcpd_run_series: one read-back for the whole series).  Returns counts[len(times), n_replicas], and the pair
        counts as well if pairs is true."""
        t = np.ascontiguousarray(times, dtype=np.uint64)
        cnt = np.empty((len(t), self.n_replicas), dtype=np.uint32)
        pr = np.empty((len(t), self.n_replicas), dtype=np.uint32) if pairs else None
        _check(self._lib, self._lib.pcpd_run_series(self._h, t.ctypes.data, len(t), cnt.ctypes.data,
                                                    pr.ctypes.data if pairs else None))
        return (cnt, pr) if pairs else cnt

    def run_series_static(self, times, pairs=False):
        """pcpd_run_series_static: run_series with the device-side records in the library's fixed static buffer - no
        allocation on the device (at most STATIC_SERIES_MAX_COUNTS counts per call; one call at a time per GPU)."""
        t = np.ascontiguousarray(times, dtype=np.uint64)
        cnt = np.empty((len(t), self.n_replicas), dtype=np.uint32)
        pr = np.empty((len(t), self.n_replicas), dtype=np.uint32) if pairs else None
        _check(self._lib, self._lib.pcpd_run_series_static(self._h, t.ctypes.data, len(t), cnt.ctypes.data,
                                                           pr.ctypes.data if pairs else None))
        return (cnt, pr) if pairs else cnt

    def pair_density(self, out=None) -> np.ndarray:
        out = np.empty(self.n_replicas, dtype=np.uint32) if out is None else out
        _check(self._lib, self._lib.pcpd_pair_density(self._h, out.ctypes.data))
        return out

    def get_lattice(self, out=None) -> np.ndarray:
        out = np.empty((self.L, self.W), dtype=np.uint64) if out is None else out
        _check(self._lib, self._lib.pcpd_get_lattice(self._h, out.ctypes.data))
        return out

    def set_lattice(self, words):
        a = np.ascontiguousarray(words, dtype=np.uint64)
        if a.size != self.L * self.W:
            raise ValueError("lattice must hold L*W uint64 words in canonical order [i][w]")
        _check(self._lib, self._lib.pcpd_set_lattice(self._h, a.ctypes.data))

    def get_lattice_ptr(self, host_ptr: int):
        _check(self._lib, self._lib.pcpd_get_lattice(self._h, host_ptr))

    def set_lattice_ptr(self, host_ptr: int):
        _check(self._lib, self._lib.pcpd_set_lattice(self._h, host_ptr))

    def step_from_host_ptr(self, host_lattice_ptr: int, n_sweeps: int, host_counts_ptr: int = 0):
        """set_lattice + run(n_sweeps) + density with the upload pipelined against the sweeps (pcpd_step_from_host)."""
        _check(self._lib, self._lib.pcpd_step_from_host(self._h, host_lattice_ptr, int(n_sweeps), host_counts_ptr or None))

    def step_from_host_columns_ptr(self, host_columns_ptr: int, n_sweeps: int, host_counts_ptr: int = 0):
        """pcpd_step_from_host_columns: the same step from a column-major host lattice [w][i] (contiguous chunk copies)."""
        _check(self._lib, self._lib.pcpd_step_from_host_columns(self._h, host_columns_ptr, int(n_sweeps), host_counts_ptr or None))

    def density_ptr(self, host_ptr: int):
        _check(self._lib, self._lib.pcpd_density(self._h, host_ptr))

    def schedule_info(self) -> dict:
        v = [C.c_uint32() for _ in range(4)]
        _check(self._lib, self._lib.pcpd_schedule_info(self._h, *[C.byref(x) for x in v]))
        return dict(Ts=v[0].value, D=v[1].value, A=v[2].value, K=v[3].value)

    def thresholds(self):
        a, b = C.c_uint64(), C.c_uint64()
        _check(self._lib, self._lib.pcpd_thresholds(self._h, C.byref(a), C.byref(b)))
        return a.value, b.value

    @property
    def sweep(self) -> int:
        return int(self._lib.pcpd_sweep(self._h))

    @sweep.setter
    def sweep(self, t):
        _check(self._lib, self._lib.pcpd_set_sweep(self._h, t))

    def split_launch_count(self) -> int:
        """column_kernel launches of this handle (small / mid-size path: 1 per sweep; 0: fused kernel)."""
        return int(self._lib.pcpd_split_launch_count(self._h))

    def jit_state(self) -> int:
        """1: sweeps run the threshold-specialised kernel; 0: not tried / not applicable; -1: unavailable."""
        return int(self._lib.pcpd_jit_state(self._h))

    def synchronize(self):
        _check(self._lib, self._lib.pcpd_synchronize(self._h))
