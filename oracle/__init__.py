"""ctypes binding of the plain-C CPU oracle (oracle/pcpd_oracle.c).

TEST INFRASTRUCTURE ONLY: may be imported by tests/, __graft_entry__.smoke()
and bench.py's cpu_baseline / --impl reference legs.  The product package
(paper_1301_6082_b200) never imports this module and shares no code with it.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pcpd_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")

STREAM_MISC, STREAM_DIFF, STREAM_ANNI, STREAM_SHIFT, STREAM_INIT = 0, 1, 2, 3, 4


def build(force: bool = False) -> str:
    """gcc -O2 (as the paper's CPU code) -> oracle/liboracle.so."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(
            ["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-Wall", "-Wextra", "-o", tmp, _SRC, "-lm"]
        )
        os.replace(tmp, _LIB)
    return _LIB


_lib = None
_lib_lock = threading.Lock()   # (tests run oracle handles on many threads: build and load once)


def lib() -> C.CDLL:
    global _lib
    if _lib is not None:
        return _lib
    with _lib_lock:
        if _lib is not None:
            return _lib
        return _load()


def _load() -> C.CDLL:
    global _lib
    L = C.CDLL(build())
    u8p, u32p, u64p = C.POINTER(C.c_uint8), C.POINTER(C.c_uint32), C.POINTER(C.c_uint64)
    L.oracle_philox4x32_10.argtypes = [u32p, u32p, u32p]
    L.oracle_philox4x32_10.restype = None
    L.oracle_threshold.argtypes = [C.c_double]
    L.oracle_threshold.restype = C.c_uint64
    L.oracle_lane_uniforms.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32, C.c_int, u32p]
    L.oracle_lane_uniforms.restype = None
    L.oracle_paper_pmask.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint64, u8p]
    L.oracle_paper_pmask.restype = None
    L.oracle_paper_pmask_bound.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint64, C.c_int, u8p]
    L.oracle_paper_pmask_bound.restype = None
    L.oracle_pmask_gate_threshold.argtypes = [C.c_double, C.c_int]
    L.oracle_pmask_gate_threshold.restype = C.c_uint64
    L.oracle_bernoulli_mask.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint64, u8p]
    L.oracle_bernoulli_mask.restype = None
    L.oracle_single_attempt.argtypes = [C.c_int, C.c_uint32, u8p, C.c_uint32, C.c_int, C.c_int, C.c_int]
    L.oracle_single_attempt.restype = None
    L.oracle_create.argtypes = [C.c_uint64, C.c_double, C.c_double, C.c_uint64, C.c_int,
                                C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32, u32p]
    L.oracle_create.restype = C.c_void_p
    L.oracle_destroy.argtypes = [C.c_void_p]
    L.oracle_destroy.restype = None
    L.oracle_set_reverse_order.argtypes = [C.c_void_p, C.c_int]
    L.oracle_set_reverse_order.restype = None
    L.oracle_sweep.argtypes = [C.c_void_p]
    L.oracle_sweep.restype = C.c_uint32
    L.oracle_set_sweep.argtypes = [C.c_void_p, C.c_uint32]
    L.oracle_set_sweep.restype = None
    L.oracle_thresholds.argtypes = [C.c_void_p, u64p, u64p]
    L.oracle_thresholds.restype = None
    L.oracle_set_word_probabilities.argtypes = [C.c_void_p, C.c_uint32, C.c_double, C.c_double]
    L.oracle_set_word_probabilities.restype = C.c_int
    L.oracle_stats.argtypes = [C.c_void_p, u64p]
    L.oracle_stats.restype = None
    L.oracle_init.argtypes = [C.c_void_p, C.c_int]
    L.oracle_init.restype = C.c_int
    L.oracle_run.argtypes = [C.c_void_p, C.c_uint64]
    L.oracle_run.restype = C.c_int
    L.oracle_shifts.argtypes = [C.c_void_p, C.c_uint32, u32p, u32p]
    L.oracle_shifts.restype = None
    L.oracle_counts.argtypes = [C.c_void_p, u32p]
    L.oracle_counts.restype = None
    L.oracle_pair_counts.argtypes = [C.c_void_p, u32p]
    L.oracle_pair_counts.restype = None
    L.oracle_get_words.argtypes = [C.c_void_p, u64p]
    L.oracle_get_words.restype = None
    L.oracle_set_words.argtypes = [C.c_void_p, u64p]
    L.oracle_set_words.restype = None
    L.oracle_literal_run.argtypes = [C.c_int, C.c_uint32, C.c_uint32, C.c_double, C.c_double, C.c_uint64,
                                     u8p, C.c_uint32, u32p, u32p]
    L.oracle_literal_run.restype = C.c_int
    _lib = L
    return _lib


def _p(a: np.ndarray, ct):
    return a.ctypes.data_as(C.POINTER(ct))


def philox4x32_10(ctr, key) -> np.ndarray:
    c = np.asarray(ctr, dtype=np.uint32).copy()
    k = np.asarray(key, dtype=np.uint32).copy()
    out = np.zeros(4, dtype=np.uint32)
    lib().oracle_philox4x32_10(_p(c, C.c_uint32), _p(k, C.c_uint32), _p(out, C.c_uint32))
    return out


def threshold(q: float) -> int:
    return int(lib().oracle_threshold(float(q)))


def lane_uniforms(seed, slot, sweep, word, stream, K=32) -> np.ndarray:
    U = np.zeros(64, dtype=np.uint32)
    lib().oracle_lane_uniforms(seed, slot, sweep, word, stream, K, _p(U, C.c_uint32))
    return U


def bernoulli_mask(seed, slot, sweep, word, stream, T) -> np.ndarray:
    m = np.zeros(64, dtype=np.uint8)
    lib().oracle_bernoulli_mask(seed, slot, sweep, word, stream, T, _p(m, C.c_uint8))
    return m


def paper_pmask(seed, slot, sweep, word, T4p) -> np.ndarray:
    """The paper's partially correlated annihilation mask (oracle_paper_pmask)."""
    m = np.zeros(64, dtype=np.uint8)
    lib().oracle_paper_pmask(seed, slot, sweep, word, T4p, _p(m, C.c_uint8))
    return m


def paper_pmask_bound(seed, slot, sweep, word, Tg, code) -> np.ndarray:
    """The paper's annihilation mask family (oracle_paper_pmask_bound): code 0 b = 1/4, 1 b = 1/2, 2 b = 1, 3 b = 3/4."""
    m = np.zeros(64, dtype=np.uint8)
    lib().oracle_paper_pmask_bound(seed, slot, sweep, word, Tg, code, _p(m, C.c_uint8))
    return m


def pmask_gate_threshold(p: float, code: int) -> int:
    """floor((p / b) 2^32) of the word-wide draw for bound code `code`; 2^64 - 1 if p >= b or the code is invalid."""
    return int(lib().oracle_pmask_gate_threshold(float(p), int(code)))


PMASK_BOUNDS = {0: 0.25, 1: 0.5, 2: 1.0, 3: 0.75}   # bound code -> b
PMASK_BOUND_SHIFT = 10   # variant bits 10-11 hold the bound code (with PMASK_PAPER)
CONNECTED = 0x200    # variant flag: the paper's connected multispin lattice (64 lanes = one ring of 64 L sites)
PMASK_PAPER = 0x100  # variant flag: the paper's own annihilation mask (needs p < 1/4)


def single_attempt(variant, q, i, Dm, Pm, Fm) -> np.ndarray:
    """Returns the ring after one attempt at site i (q: sequence of 0/1)."""
    a = np.asarray(q, dtype=np.uint8).copy()
    lib().oracle_single_attempt(variant, len(a), _p(a, C.c_uint8), i, int(Dm), int(Pm), int(Fm))
    return a


class Oracle:
    """SD2(T_s, D, A) schedule run of the word columns `words` (default: all)."""

    def __init__(self, L, n_replicas, d, p, seed, variant=0, Ts=2048, D=64, A=4, words=None):
        if n_replicas % 64 or n_replicas <= 0:
            raise ValueError("n_replicas must be a positive multiple of 64")
        self.W_full = n_replicas // 64
        self.words = np.arange(self.W_full, dtype=np.uint32) if words is None else np.asarray(words, dtype=np.uint32).copy()
        self.L, self.nwords = int(L), len(self.words)
        self._h = lib().oracle_create(L, d, p, seed, variant, Ts, D, A, self.nwords, _p(self.words, C.c_uint32))
        if not self._h:
            raise ValueError("oracle_create: invalid arguments")

    def close(self):
        if self._h:
            lib().oracle_destroy(self._h)
            self._h = None

    __del__ = close

    def init(self, mode):
        if lib().oracle_init(self._h, mode) != 0:
            raise ValueError("bad init mode")

    def run(self, n):
        rc = lib().oracle_run(self._h, n)
        if rc != 0:
            raise RuntimeError(f"oracle_run failed ({rc})")

    @property
    def sweep(self):
        return lib().oracle_sweep(self._h)

    @sweep.setter
    def sweep(self, t):
        lib().oracle_set_sweep(self._h, t)

    def set_reverse_order(self, rev):
        lib().oracle_set_reverse_order(self._h, int(rev))

    def thresholds(self):
        a, b = C.c_uint64(), C.c_uint64()
        lib().oracle_thresholds(self._h, C.byref(a), C.byref(b))
        return a.value, b.value

    def set_word_probabilities(self, k, d, p):
        """Column k (index into `words`) uses (d, p) from now on (oracle_set_word_probabilities, C11)."""
        if lib().oracle_set_word_probabilities(self._h, k, float(d), float(p)) != 0:
            raise ValueError("oracle_set_word_probabilities: invalid arguments")

    def stats(self) -> dict:
        s = np.zeros(5, dtype=np.uint64)
        lib().oracle_stats(self._h, _p(s, C.c_uint64))
        k = ("attempt_words", "planes_needed_D", "planes_needed_P", "blocks_needed_D", "blocks_needed_P")
        return dict(zip(k, (int(v) for v in s)))

    def shifts(self, t, S):
        Sigma = C.c_uint32()
        sig = np.zeros(S, dtype=np.uint32)
        lib().oracle_shifts(self._h, t, C.byref(Sigma), _p(sig, C.c_uint32))
        return Sigma.value, sig

    def counts(self) -> np.ndarray:
        out = np.zeros(self.nwords * 64, dtype=np.uint32)
        lib().oracle_counts(self._h, _p(out, C.c_uint32))
        return out

    def pair_counts(self) -> np.ndarray:
        out = np.zeros(self.nwords * 64, dtype=np.uint32)
        lib().oracle_pair_counts(self._h, _p(out, C.c_uint32))
        return out

    def get_words(self) -> np.ndarray:
        out = np.zeros((self.L, self.nwords), dtype=np.uint64)
        lib().oracle_get_words(self._h, _p(out, C.c_uint64))
        return out

    def set_words(self, words):
        a = np.ascontiguousarray(words, dtype=np.uint64)
        assert a.shape == (self.L, self.nwords)
        lib().oracle_set_words(self._h, _p(a, C.c_uint64))


def literal_run(variant, L, R, d, p, seed, q0, rec_times):
    """Literal Algorithm 1. q0: uint8[R, L]; returns
    (counts uint32[n_rec, R], final q)."""
    q = np.ascontiguousarray(q0, dtype=np.uint8).copy()
    assert q.shape == (R, L)
    rt = np.asarray(rec_times, dtype=np.uint32).copy()
    out = np.zeros((len(rt), R), dtype=np.uint32)
    rc = lib().oracle_literal_run(variant, L, R, d, p, seed, _p(q, C.c_uint8), len(rt), _p(rt, C.c_uint32), _p(out, C.c_uint32))
    if rc != 0:
        raise ValueError("oracle_literal_run: invalid arguments")
    return out, q
