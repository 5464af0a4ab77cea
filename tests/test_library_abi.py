"""CPU-side checks of the boundary: libpcpd.so builds for sm_100a, loads, and
exports every symbol include/pcpd.h declares; argument errors that are detected
before any device work; host-side helpers.  No compute calls (no GPU here)."""
import ctypes as C
import os
import re

import pytest

import workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1301_6082_b200 import build, load_library

    build.build()
    return load_library()


def test_header_symbols_are_exported(lib):
    import paper_1301_6082_b200 as pk

    hdr = open(os.path.join(ROOT, "include", "pcpd.h")).read()
    declared = set(re.findall(r"\b(pcpd_[a-z_]+)\s*\(", hdr))
    declared -= {"pcpd_alloc_fn", "pcpd_free_fn"}
    assert declared == set(pk.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), name


def test_argument_errors_without_device(lib):
    # all of these are rejected before the device is touched
    bad = [
        (1024, 63, 0.5, 0.1, 1, 0),     # replicas not a multiple of 64
        (1024, 0, 0.5, 0.1, 1, 0),
        (1000, 64, 0.5, 0.1, 1, 0),     # L not a multiple of D = 64
        (1024, 64, 1.5, 0.1, 1, 0),     # d out of range
        (1024, 64, 0.5, float("nan"), 1, 0),
        (1024, 64, 0.5, 0.1, 1, 7),     # variant
        (1 << 32, 64, 0.5, 0.1, 1, 0),  # L >= 2^32
        (2048 + 64, 64, 0.5, 0.1, 1, 0),  # L % T_s != 0
    ]
    for args in bad:
        assert not lib.pcpd_create(*args)
        assert lib.pcpd_last_error()
    assert not lib.pcpd_create_ex(1024, 64, 0.5, 0.1, 1, 0, 256, 64, 5, 0)   # A does not divide D
    assert not lib.pcpd_create_ex(1024, 64, 0.5, 0.1, 1, 1, 256, 8, 4, 0)    # TCPD needs D >= 9
    assert not lib.pcpd_create_ex(1024, 64, 0.5, 0.1, 1, 0, 96, 64, 4, 0)    # D does not divide T_s
    assert lib.pcpd_run(None, 1) < 0 and lib.pcpd_init(None, 0) < 0
    assert lib.pcpd_density(None, None) < 0
    lib.pcpd_destroy(None)  # NULL-safe


@pytest.mark.parametrize("variant,Td,Tp", [(0, 0xCCCCCCCC, 0x1EB851EB), (1, 0x80000000, 0x0CCCCCCC), (2, 1, 0xFFFFFFFF),
                                           (3, 0, 0x4CCCCCCC)])
def test_run_time_specialisation_compiles_for_sm_100a(lib, variant, Td, Tp):
    """csrc/jit.cu: the device source embedded in the library compiles with NVRTC for sm_100a with the
    thresholds as template constants (needs libnvrtc, no device)."""
    n = C.c_uint64(0)
    rc = lib.pcpd_jit_selftest(variant, Td, Tp, C.byref(n))
    if rc != 0 and b"libnvrtc not found" in lib.pcpd_last_error():
        pytest.skip("libnvrtc is not installed here")
    assert rc == 0, lib.pcpd_last_error()
    assert n.value > 10_000  # a cubin, not an empty image


def test_no_cpu_fallback_without_gpu():
    import torch

    if torch.cuda.is_available():
        pytest.skip("GPU present")
    import paper_1301_6082_b200 as pk

    with pytest.raises(pk.PcpdError):
        pk.Pcpd(1024, 64, 0.5, 0.15, 1)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1301_6082_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "oracle/" not in src.replace(
                    "shares nothing with oracle/", "").replace("used by oracle/", ""), f
    osrc = open(os.path.join(ROOT, "oracle", "pcpd_oracle.c")).read()
    assert "#include \"" not in osrc  # only system headers
    assert "paper_1301_6082_b200" not in open(os.path.join(ROOT, "oracle", "__init__.py")).read().replace(
        "(paper_1301_6082_b200)", "")


def test_delta_eff_on_the_papers_scaling_form(lib):
    """pcpd_delta_eff (host-side analysis): on rho(t) = c1 t^-delta + c2 t^-2delta (eq. (2)) the
    effective exponent is -d ln rho / d ln t = delta (c1 t^-delta + 2 c2 t^-2delta) / rho; the library's central
    log-log difference must reproduce it (to the O(h^2) of the difference and the rounding of the counts), and a pure
    power law exactly.  The definition is also written out in numpy and compared element by element."""
    import numpy as np

    import paper_1301_6082_b200 as pk

    L, R = 1 << 22, 128
    times = np.array([t for t in wl.record_times(10_000) if t > 0], dtype=np.uint64)
    tt = times.astype(np.float64)
    delta, c1, c2 = 0.2, 0.9, -0.35
    rho_true = c1 * tt ** -delta + c2 * tt ** (-2 * delta)
    rng = np.random.Generator(np.random.PCG64(5))
    counts = np.round(rho_true[:, None] * L * (1 + 1e-4 * rng.standard_normal((len(tt), R)))).astype(np.uint32)
    for m in (1, 3):
        rho, de = pk.delta_eff(times, counts, L, half_window=m)
        assert np.allclose(rho, counts.astype(np.float64).mean(axis=1) / L, rtol=1e-13)
        # the definition, written out
        ref = np.full(len(tt), np.nan)
        for k in range(m, len(tt) - m):
            ref[k] = -np.log(rho[k + m] / rho[k - m]) / np.log(tt[k + m] / tt[k - m])
        assert np.array_equal(np.isnan(de), np.isnan(ref)) and np.isnan(de[:m]).all() and np.isnan(de[-m:]).all()
        assert np.allclose(de[m:-m], ref[m:-m], rtol=1e-12)
        # against the analytic derivative at the window's log-midpoint
        tm = np.sqrt(tt[2 * m:] * tt[:-2 * m])
        exact = delta * (c1 * tm ** -delta + 2 * c2 * tm ** (-2 * delta)) / (c1 * tm ** -delta + c2 * tm ** (-2 * delta))
        sel = tt[m:-m] >= 20            # (below, the record times are integers a factor 1.1 .. 2 apart: O(h^2) is not small)
        assert np.max(np.abs(de[m:-m][sel] - exact[sel])) < 2e-3
    # a pure power law gives delta at every interior point
    pure = np.round(0.7 * tt[:, None] ** -0.159 * L * np.ones((1, 4))).astype(np.uint32)
    _, de = pk.delta_eff(times, pure, L, 2)
    assert np.allclose(de[2:-2], 0.159, atol=2e-6)
    # degenerate windows: t = 0, repeated times, zero density -> NaN, not an error
    t2 = np.array([0, 1, 2, 2, 2, 4, 8], dtype=np.uint64)
    c = np.array([[9], [8], [7], [7], [7], [0], [5]], dtype=np.uint32)
    _, de = pk.delta_eff(t2, c, 16, 1)
    assert np.isnan(de[[0, 1, 3, 4, 6]]).all() and np.isfinite(de[[2, 5]]).all()
    # argument errors
    r, dl = np.empty(7), np.empty(7)
    assert lib.pcpd_delta_eff(t2.ctypes.data, 7, c.ctypes.data, 1, 16, 0, r.ctypes.data, dl.ctypes.data) < 0
    assert lib.pcpd_delta_eff(t2[::-1].copy().ctypes.data, 7, c.ctypes.data, 1, 16, 1, r.ctypes.data, dl.ctypes.data) < 0
    assert lib.pcpd_delta_eff(None, 7, c.ctypes.data, 1, 16, 1, r.ctypes.data, dl.ctypes.data) < 0


def test_record_times():
    t = wl.record_times(10_000)
    assert t[0] == 0 and t[1] == 1 and t[-1] == 10_000 and t == sorted(set(t))
    assert len(t) == 71  # the 70 distinct log-spaced integers of SURVEY.md 8(d) (10^4 among them) + t = 0
