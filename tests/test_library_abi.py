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


def test_record_times():
    t = wl.record_times(10_000)
    assert t[0] == 0 and t[1] == 1 and t[-1] == 10_000 and t == sorted(set(t))
    assert len(t) == 71  # the 70 distinct log-spaced integers of SURVEY.md 8(d) (10^4 among them) + t = 0
