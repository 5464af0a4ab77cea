"""GPU <-> oracle parity, through the C ABI (binding = argument marshalling only).

Bar: BIT-EXACT - every packed lattice word and every per-replica count equal
to the oracle's on the same seeded inputs (integer / bit work, no tolerance).
Scaled-down cases span several tiles, several word columns,
ragged shapes, the seam domain and the threshold edge cases; the BASELINE.json
configs are checked in the launch configuration bench.py times, on sampled
word columns the oracle can compute one by one (columns never interact,
oracle pin P7), per the protocol of SURVEY.md 8(d).
"""
import os
from concurrent.futures import ThreadPoolExecutor

import numpy as np
import pytest

import oracle
import workloads as wl

pytestmark = pytest.mark.gpu

NCPU = max(1, min(32, os.cpu_count() or 1))


@pytest.fixture(scope="module")
def pk():
    import paper_1301_6082_b200 as pk
    from paper_1301_6082_b200 import build

    build.build()
    return pk


def oracle_columns(cfg_kw, words, init, n_sweeps_list, words_in=None):
    """Run the oracle on word columns `words` (one thread per column; ctypes
    releases the GIL).  Returns {t: (lattice[L, len(words)], counts[len(words)*64])}."""
    def one(w):
        o = oracle.Oracle(words=[w], **cfg_kw)
        if words_in is not None:
            o.set_words(words_in[:, [w]])
        else:
            o.init(init)
        res, prev = {}, 0
        for t in n_sweeps_list:
            o.run(t - prev)
            prev = t
            res[t] = (o.get_words()[:, 0].copy(), o.counts().copy())
        return res

    with ThreadPoolExecutor(NCPU) as ex:
        cols = list(ex.map(one, words))
    out = {}
    for t in n_sweeps_list:
        out[t] = (np.stack([c[t][0] for c in cols], axis=1), np.concatenate([c[t][1] for c in cols]))
    return out


def gpu_check(pk, kw, sch, init, times, words=None, words_in=None, expect_jit=False, expect_split=None):
    W = kw["n_replicas"] // 64
    words = list(range(W)) if words is None else words
    okw = dict(kw)
    g = pk.Pcpd(kw["L"], kw["n_replicas"], kw["d"], kw["p"], kw["seed"], kw["variant"], **sch)
    info = g.schedule_info()
    ref = oracle_columns(dict(okw, Ts=info["Ts"], D=info["D"], A=info["A"]), words, init, times, words_in)
    if words_in is not None:
        g.set_lattice(words_in)
    else:
        g.init(init)
    prev = 0
    for t in times:
        g.run(t - prev)
        prev = t
        lat = g.get_lattice()
        cnt = g.density()
        rl, rc = ref[t]
        assert np.array_equal(lat[:, words], rl), f"lattice mismatch after sweep {t}"
        assert np.array_equal(cnt.reshape(W, 64)[words].ravel(), rc), f"count mismatch after sweep {t}"
        # counts agree with the lattice the GPU itself returned (all columns)
        bits = (lat[:, :, None] >> np.arange(64, dtype=np.uint64)) & np.uint64(1) if lat.size <= (1 << 18) else None
        if bits is not None:
            assert np.array_equal(bits.sum(axis=0).ravel().astype(np.uint32), cnt)
    assert g.sweep == times[-1]
    if expect_jit:  # the sweeps ran the threshold-specialised (run-time compiled) kernel, not the built-in one
        if g.jit_state() != 1 and "libnvrtc not found" in pk.jit_message():
            g.close()
            pytest.skip("libnvrtc is not installed on this box: the built-in kernel ran (and passed the checks above)")
        assert g.jit_state() == 1, pk.jit_message()
    if expect_split is not None:  # which small-problem path ran: launches per handle on the SPLIT paths
        # "column": one column_kernel per sweep; False: the fused kernel
        want = times[-1] if expect_split else 0
        assert g.split_launch_count() == want
    g.close()


def test_thresholds_and_schedule_match_oracle(pk):
    for c in wl.CONFIGS:
        g = pk.Pcpd(4096, 64, c.d, c.p, c.seed, c.variant)
        o = oracle.Oracle(4096, 64, c.d, c.p, c.seed, c.variant)
        assert g.thresholds() == o.thresholds()
        assert g.schedule_info() == dict(Ts=2048, D=64, A=4, K=32)
        g.close()


SMALL = [
    # (variant, L, R, d, p, Ts, D, A, init)            what it exercises
    (0, 1024, 64, 0.5, 0.15, 2048, 64, 4, 0),        # W=1 (Wb=1), T_s clamped to L, d = 1/2
    (0, 4096, 256, 0.1, 0.09, 2048, 64, 4, 1),       # W=4 (Wb=4), two tiles, generic d and p
    (0, 8192, 128, 0.8, 0.12, 2048, 64, 4, 0),       # W=2 (Wb=2)
    (0, 2048, 192, 0.3, 0.2, 512, 64, 8, 1),         # W=3 (Wb=1), 4 tiles, A=8
    (0, 640, 320, 0.25, 0.75, 128, 32, 2, 1),        # W=5, ragged L = 5 tiles of 128
    (0, 384, 512, 0.5, 0.15, 64, 64, 64, 0),         # degenerate schedule T_s = D = A (n=1, S=1)
    (0, 112, 64, 0.37, 0.21, 56, 7, 1, 1),           # smallest legal PCPD domain D = 7
    (1, 4096, 256, 0.5, 0.05, 2048, 64, 4, 0),       # TCPD, cfg5 shape
    (1, 1152, 128, 0.2, 0.3, 576, 9, 3, 1),          # TCPD, smallest legal domain D = 9 (n = 64: generic block kernel)
    (0, 147, 64, 0.37, 0.21, 49, 7, 1, 1),           # odd L and T_s: 64-bit tile copy path
    (1, 4096, 128, 0.5, 0.05, 1024, 32, 2, 1),       # TCPD, n = 32 lanes, A = 2 batches
    (1, 2048, 768, 0.6, 0.1, 1024, 128, 16, 1),      # TCPD, W=12, D=128
    (0, 1024, 128, 0.0, 0.3, 512, 64, 4, 1),         # d = 0 (T_d = 0)
    (0, 1024, 128, 1.0, 0.3, 512, 64, 4, 1),         # d = 1 (T_d = 2^32): only swaps
    (0, 1024, 128, 0.4, 0.0, 512, 64, 4, 1),         # p = 0: no annihilation
    (0, 1024, 128, 0.4, 1.0, 512, 64, 4, 1),         # p = 1: every reacting pair annihilates
    (0, 1024, 128, 2.0 ** -32, 1 - 2.0 ** -32, 512, 64, 4, 1),  # T = 1 and T = 2^32 - 1: all 32 planes matter
    (0x100, 4096, 256, 0.75, 0.12, 2048, 64, 4, 0),  # the paper's annihilation mask (Alg. 2 l.12-13), dyadic d
    (0x100, 2048, 192, 0.3, 0.2, 512, 64, 8, 1),     # same, generic d (lazy DIFF tail), Bernoulli start
    (0x101, 4096, 128, 0.5, 0.05, 2048, 64, 4, 0),   # same on TCPD
    (2, 4096, 128, 0.5, 0.03, 2048, 64, 4, 0),       # QCPD, 6-site footprint
    (2, 1408, 128, 0.3, 0.1, 704, 11, 1, 1),         # QCPD, smallest legal domain D = 11 (n = 64: block kernel)
    (0x102, 2048, 64, 0.25, 0.05, 1024, 32, 2, 1),   # QCPD with the paper's annihilation mask
    (3, 4096, 128, 0.5, 0.3, 2048, 64, 4, 0),        # CPD (contact process with diffusion, DP class), 3-site footprint
    (3, 640, 64, 0.2, 0.4, 320, 5, 1, 1),            # CPD, smallest legal domain D = 5 (n = 64: block kernel)
    (0x203, 2048, 64, 0.25, 0.2, 1024, 32, 2, 1),    # CPD on the connected lattice
    (0, 2048, 64, 0.3, 0.12, 2048, 64, 1, 1),        # A = 1: S = 64 sub-steps (more than one group of 32 shifts per sweep)
    (0x200, 4096, 256, 0.3, 0.12, 2048, 64, 4, 1),   # the paper's connected multispin lattice (bit rotation at the ring wrap)
    (0x200, 1024, 64, 0.5, 0.15, 2048, 64, 4, 0),    # same, single tile = whole ring (T_s clamped to L)
    (0x300, 147, 64, 0.37, 0.21, 49, 7, 1, 1),       # same + paper mask, odd L and T_s (64-bit tile copy path)
    (0x201, 1152, 128, 0.2, 0.3, 576, 9, 3, 1),      # same on TCPD through the block kernel (n = 64)
    (0x500, 4096, 256, 0.75, 0.4, 2048, 64, 4, 0),   # the paper's mask family: bound b = 1/2 (one raw word), p < 1/2
    (0x900, 2048, 192, 0.3, 0.6, 512, 64, 8, 1),     # b = 1: no decorrelation bits, fully correlated lanes
    (0xD01, 4096, 128, 0.5, 0.7, 2048, 64, 4, 0),    # b = 3/4 (two raw words ORed, gate 4p/3) on TCPD
    (0, 4096, 128, 0.5, 0.15, 2048, 256, 8, 0),      # SD2(2048, 256, 8): the schedule without measurable bias; 8 domains per tile
    (0, 8192, 64, 0.8, 0.12, 2048, 128, 4, 1),       # SD2(2048, 128, 4): 16 domains per tile, S = 32 sub-steps
]


@pytest.mark.parametrize("split", ["auto", "0"])
@pytest.mark.parametrize("case", SMALL, ids=[f"case{i}" for i in range(len(SMALL))])
def test_small_cases_bit_exact_every_sweep(pk, case, split, monkeypatch):
    """Every word and count after every sweep.  split = auto: these sizes run column_kernel (producer warps + two
    half-word update warps in one block per tile column) wherever the warp kernel applies (at most 32 domains per tile);
    split = 0: the fused warp kernel (or the generic block kernel for more than 32 domains per tile)."""
    variant, L, R, d, p, Ts, D, A, init = case
    if split != "auto":
        monkeypatch.setenv("PCPD_SPLIT", split)
    kw = dict(L=L, n_replicas=R, d=d, p=p, seed=1000 + L + R, variant=variant)
    warp = min(Ts, L) // D <= 32
    gpu_check(pk, kw, dict(Ts=Ts, D=D, A=A), init, list(range(1, 7)),
              expect_split=(False if split == "0" or not warp else "column" if split == "auto" else split))


# cases of SMALL the warp kernel runs (at most 32 domains per tile) with neither threshold equal to 2^32
JIT_CASES = [0, 1, 2, 3, 4, 5, 6, 7, 9, 10, 11, 12, 14, 16, 17, 18, 19, 20, 22, 23, 25, 26, 27, 29, 31, 32, 33, 34, 35]


@pytest.mark.parametrize("idx", JIT_CASES, ids=[f"case{i}" for i in JIT_CASES])
def test_threshold_specialised_kernel_bit_exact_every_sweep(pk, idx, monkeypatch):
    """The run-time compiled sweep kernel (T_d, T_p as template constants; csrc/jit.cu), forced on at small
    sizes with PCPD_JIT=force: same bar as the built-in kernel - every word and count after every sweep."""
    monkeypatch.setenv("PCPD_JIT", "force")
    variant, L, R, d, p, Ts, D, A, init = SMALL[idx]
    kw = dict(L=L, n_replicas=R, d=d, p=p, seed=1000 + L + R, variant=variant)
    n0 = pk.jit_launch_count()
    gpu_check(pk, kw, dict(Ts=Ts, D=D, A=A), init, list(range(1, 7)), expect_jit=True)
    assert pk.jit_launch_count() - n0 == 6


def test_specialised_and_builtin_kernels_agree_at_full_size(pk, monkeypatch):
    """cfg4 and cfg5 whole lattices: the run-time specialised kernel (default at this size) against the
    built-in generic-threshold kernel (PCPD_JIT=0)."""
    for name in ("cfg4", "cfg5"):
        c = wl.BY_NAME[name]
        res = []
        for mode in ("1", "0"):
            monkeypatch.setenv("PCPD_JIT", mode)
            g = pk.Pcpd(c.L, c.n_replicas, c.d, c.p, c.seed, c.variant)
            g.init(c.init)
            g.run(3)
            if mode == "1" and g.jit_state() != 1 and "libnvrtc not found" in pk.jit_message():
                g.close()
                pytest.skip("libnvrtc is not installed on this box")
            assert g.jit_state() == (1 if mode == "1" else 0), pk.jit_message()
            res.append((g.get_lattice(), g.density()))
            g.close()
        monkeypatch.delenv("PCPD_JIT")
        assert np.array_equal(res[0][0], res[1][0]) and np.array_equal(res[0][1], res[1][1])


def test_hand_built_lattice_and_seed_high_bits(pk):
    L, R = 2048, 256
    w0 = wl.random_lattice_words(L, R // 64, 0.3, seed=77)
    kw = dict(L=L, n_replicas=R, d=0.45, p=0.13, seed=0xDEADBEEF12345678, variant=0)
    gpu_check(pk, kw, dict(Ts=1024, D=64, A=4), None, [1, 2, 5], words_in=w0)


def test_invariants_on_gpu(pk):
    # absorbing state, d = 1 conservation, run splitting, set/get round trip, pair counts
    g = pk.Pcpd(4096, 256, 0.4, 0.2, 5, 0)
    g.init(pk.INIT_EMPTY)
    g.run(3)
    assert not g.get_lattice().any() and not g.density().any()
    g.close()
    g = pk.Pcpd(4096, 256, 1.0, 0.2, 5, 0)
    w0 = wl.random_lattice_words(4096, 4, 0.4, seed=1)
    g.set_lattice(w0)
    assert np.array_equal(g.get_lattice(), w0)
    c0 = g.density()
    g.run(4)
    assert np.array_equal(g.density(), c0) and not np.array_equal(g.get_lattice(), w0)
    g.close()
    a = pk.Pcpd(4096, 256, 0.3, 0.1, 9, 0)
    b = pk.Pcpd(4096, 256, 0.3, 0.1, 9, 0)
    a.init(1)
    b.init(1)
    a.run(7)
    b.run(3)
    b.run(4)
    assert np.array_equal(a.get_lattice(), b.get_lattice())
    lat = a.get_lattice()
    pairs = ((lat & np.roll(lat, -1, axis=0))[:, :, None] >> np.arange(64, dtype=np.uint64)) & np.uint64(1)
    assert np.array_equal(a.pair_density(), pairs.sum(axis=0).ravel().astype(np.uint32))
    o = oracle.Oracle(4096, 256, 0.3, 0.1, 9, 0)
    o.set_words(lat)
    assert np.array_equal(a.pair_density(), o.pair_counts())
    # checkpoint / resume: lattice + sweep counter is the whole state (C7)
    c = pk.Pcpd(4096, 256, 0.3, 0.1, 9, 0)
    c.set_lattice(b.get_lattice())
    c.sweep = 7
    a.run(2)
    c.run(2)
    assert np.array_equal(a.get_lattice(), c.get_lattice())
    for h in (a, b, c):
        h.close()


def test_mid_size_handle_runs_the_column_kernel(pk):
    """Up to 768 tile columns (generic thresholds; 384 with one short threshold) the default is column_kernel, with 8
    producer warps per block from 149 columns on (several blocks share an SM): sampled columns against the oracle at 256
    and 768 tile columns; above the limit the handle runs the fused kernel, run-time specialised."""
    for W, words in ((8, [0, 5, 7]), (24, [3, 23])):   # 32 tiles x W columns
        kw = dict(L=65536, n_replicas=64 * W, d=0.1, p=0.09, seed=2, variant=0)
        gpu_check(pk, kw, {}, 1, [1, 2, 3], words=words, expect_split="column")
    kw = dict(L=65536, n_replicas=64 * 32, d=0.1, p=0.09, seed=2, variant=0)       # 1024 columns
    gpu_check(pk, kw, {}, 1, [1, 2], words=[31], expect_split=False, expect_jit=True)
    kw = dict(L=65536, n_replicas=64 * 16, d=0.5, p=0.152, seed=3, variant=0)      # 512 columns, d = 1/2: above its limit of 384
    gpu_check(pk, kw, {}, 0, [1, 2], words=[0, 15], expect_split=False, expect_jit=True)
    kw = dict(L=65536, n_replicas=64 * 12, d=0.5, p=0.152, seed=3, variant=0)      # 384 columns, d = 1/2: column kernel
    gpu_check(pk, kw, {}, 0, [1, 2], words=[11], expect_split="column")


def test_counter_jumps_and_reinit_on_the_column_kernel(pk, monkeypatch):
    """Re-initialising and setting the sweep counter backwards, forwards and to the last legal sweep must give what the
    fused kernel gives for the same sequence of calls (lattice + counter is the whole state, C7)."""
    def sequence(g):
        out = []
        g.init(1); g.run(3); out.append(g.get_lattice())
        g.init(1); g.run(2); out.append(g.get_lattice())
        g.sweep = 9; g.run(1); g.run(2); out.append(g.get_lattice())
        g.sweep = 4; g.run(3); out.append(g.get_lattice())
        g.sweep = 2 ** 32 - 2; g.run(1); out.append(g.get_lattice())   # last legal sweep
        return out
    res = []
    for mode in ("1", "0"):
        monkeypatch.setenv("PCPD_SPLIT", mode)
        g = pk.Pcpd(4096, 192, 0.3, 0.12, 11, 0)
        res.append(sequence(g))
        assert (g.split_launch_count() > 0) == (mode == "1")
        g.close()
    for x, y in zip(*res):
        assert np.array_equal(x, y)


def test_pipelined_step_from_host_equals_the_plain_sequence(pk, monkeypatch):
    """pcpd_step_from_host (upload cut into column chunks, copy of chunk c+1 overlapping the sweeps of chunk c) must
    give exactly what set_lattice + run + density give: forced 4-column chunks with a ragged last chunk at a small
    size (also against the oracle), and the default 8-column chunks at cfg5's size."""
    monkeypatch.setenv("PCPD_STEP_CHUNK", "4")
    L, R = 4096, 64 * 6
    w0 = wl.random_lattice_words(L, R // 64, 0.5, seed=3)
    a = pk.Pcpd(L, R, 0.3, 0.12, 21, 0)
    b = pk.Pcpd(L, R, 0.3, 0.12, 21, 0)
    a.set_lattice(w0); a.sweep = 5; a.run(3)
    b.sweep = 5
    cnt = np.empty(R, dtype=np.uint32)
    b.step_from_host_ptr(w0.ctypes.data, 3, cnt.ctypes.data)
    assert b.sweep == 8
    assert np.array_equal(a.get_lattice(), b.get_lattice()) and np.array_equal(a.density(), cnt)
    o = oracle.Oracle(L, R, 0.3, 0.12, 21, 0)
    o.set_words(w0); o.sweep = 5; o.run(3)
    assert np.array_equal(b.get_lattice(), o.get_words()) and np.array_equal(cnt, o.counts())
    # the column-major variant (contiguous chunk copies straight into the lattice), same forced ragged chunks
    c2 = pk.Pcpd(L, R, 0.3, 0.12, 21, 0)
    c2.sweep = 5
    cols = np.ascontiguousarray(w0.T)
    cnt2 = np.empty(R, dtype=np.uint32)
    c2.step_from_host_columns_ptr(cols.ctypes.data, 3, cnt2.ctypes.data)
    assert c2.sweep == 8 and np.array_equal(c2.get_lattice(), o.get_words()) and np.array_equal(cnt2, o.counts())
    a.close(); b.close(); c2.close()
    monkeypatch.delenv("PCPD_STEP_CHUNK")
    # unchunked (small handle: the column kernel runs), per-word thresholds
    s1 = pk.Pcpd(L, R, 0.3, 0.12, 21, 0)
    s1.sweep = 5
    s1.step_from_host_columns_ptr(cols.ctypes.data, 3, cnt2.ctypes.data)
    assert np.array_equal(s1.get_lattice(), o.get_words()) and np.array_equal(cnt2, o.counts()) and s1.split_launch_count() == 3
    s1.close()
    c = wl.BY_NAME["cfg5"]
    import torch
    host = torch.empty((c.L, c.W), dtype=torch.int64).pin_memory()
    hn = host.numpy().view(np.uint64)
    hn[:] = wl.random_lattice_words(c.L, c.W, 0.6, seed=4)
    a = pk.Pcpd(c.L, c.n_replicas, c.d, c.p, c.seed, c.variant)
    b = pk.Pcpd(c.L, c.n_replicas, c.d, c.p, c.seed, c.variant)
    a.set_lattice_ptr(host.data_ptr()); a.run(2)
    cnt = np.empty(c.n_replicas, dtype=np.uint32)
    b.step_from_host_ptr(host.data_ptr(), 2, cnt.ctypes.data)
    assert np.array_equal(a.get_lattice(), b.get_lattice()) and np.array_equal(a.density(), cnt)
    hostc = torch.empty((c.W, c.L), dtype=torch.int64).pin_memory()
    hostc.numpy().view(np.uint64)[:] = hn.T
    d = pk.Pcpd(c.L, c.n_replicas, c.d, c.p, c.seed, c.variant)
    cnt3 = np.empty(c.n_replicas, dtype=np.uint32)
    d.step_from_host_columns_ptr(hostc.data_ptr(), 2, cnt3.ctypes.data)     # default chunking: 3 columns of 512 tiles each
    assert np.array_equal(a.get_lattice(), d.get_lattice()) and np.array_equal(cnt, cnt3)
    a.close(); b.close(); d.close()


def test_run_series_equals_run_and_density_in_a_loop(pk):
    """pcpd_run_series (records kept on the device, one read-back) against the oracle's counts at the same times and
    against pcpd_run + pcpd_density / pcpd_pair_density in a loop; argument errors."""
    L, R = 4096, 128
    times = [0, 1, 2, 2, 5, 9]
    a = pk.Pcpd(L, R, 0.3, 0.12, 31, 0)
    b = pk.Pcpd(L, R, 0.3, 0.12, 31, 0)
    o = oracle.Oracle(L, R, 0.3, 0.12, 31, 0)
    a.init(1); b.init(1); o.init(1)
    cnt, pr = a.run_series(times, pairs=True)
    assert a.sweep == 9
    for k, t in enumerate(times):
        b.run(t - b.sweep)
        o.run(t - o.sweep)
        assert np.array_equal(cnt[k], b.density()) and np.array_equal(pr[k], b.pair_density())
        assert np.array_equal(cnt[k], o.counts()) and np.array_equal(pr[k], o.pair_counts())
    assert np.array_equal(a.run_series([9, 12]), np.stack([b.density(), (b.run(3), b.density())[1]]))
    with pytest.raises(pk.PcpdError):
        a.run_series([11])          # behind the counter
    with pytest.raises(pk.PcpdError):
        a.run_series([13, 12])      # not ascending
    a.close(); b.close()


def test_word_offset_shards_equal_one_big_run(pk):
    kw = dict(d=0.3, p=0.12, seed=31, variant=0)
    big = pk.Pcpd(2048, 512, **kw)
    big.init(1)
    big.run(3)
    full = big.get_lattice()
    for rank in range(2):
        w0, w1 = pk.shard_words(8, 2, rank)
        s = pk.Pcpd(2048, 64 * (w1 - w0), **kw, word_offset=w0)
        s.init(1)
        s.run(3)
        assert np.array_equal(s.get_lattice(), full[:, w0:w1])
        assert np.array_equal(s.density(), big.density()[64 * w0:64 * w1])
        s.close()
    big.close()


def test_cfg1_every_sweep(pk):
    c = wl.BY_NAME["cfg1"]
    kw = dict(L=c.L, n_replicas=c.n_replicas, d=c.d, p=c.p, seed=c.seed, variant=c.variant)
    gpu_check(pk, kw, {}, c.init, list(range(1, c.sweeps + 1)))


def test_cfg2_prefix(pk):
    c = wl.BY_NAME["cfg2"]
    kw = dict(L=c.L, n_replicas=c.n_replicas, d=c.d, p=c.p, seed=c.seed, variant=c.variant)
    horizon = 32 if NCPU >= 4 else 8
    times = [t for t in wl.record_times(c.sweeps) if 0 < t <= horizon]
    gpu_check(pk, kw, {}, c.init, times)


# SURVEY.md 8(d) "Parity protocol at scale", in the suite the driver runs: configs 3, 4, 5 at their full sizes in the launch
# configuration bench.py times - ALL word columns after sweeps 1 and 2, then `deep` columns spread over [0, W) out to t = 8.
@pytest.mark.parametrize("name,deep", [("cfg3", [0, 4, 9, 13, 18, 22, 27, 31]), ("cfg5", [0, 2, 4, 6, 9, 11, 13, 15]),
                                       ("cfg4", [0, 4, 9, 13, 18, 22, 27, 31])])
def test_full_size_configs_all_columns(pk, name, deep):
    """Every word of the full-size lattice and every count after sweeps 1 and 2 (all columns; the oracle computes them
    one by one - columns never interact, pin P7), then eight columns spread over the handle out to t = 8.  The GPU
    snapshots are taken first; the oracle columns are then run on all host cores and compared as they finish, so at
    most NCPU columns of oracle state (64 L bytes each) are alive at a time."""
    c = wl.BY_NAME[name]
    all_times, deep_times = [1, 2], [1, 2, 4, 8]
    g = pk.Pcpd(c.L, c.n_replicas, c.d, c.p, c.seed, c.variant)
    info = g.schedule_info()
    g.init(c.init)
    n0 = pk.jit_launch_count()
    lat, cnt = {}, {}
    for t in deep_times:
        g.run(t - g.sweep)
        cnt[t] = g.density().reshape(c.W, 64)
        full = g.get_lattice()
        lat[t] = full if t in all_times else np.ascontiguousarray(full[:, deep])   # keep only what will be compared
        del full
    jit_state, jit_launches = g.jit_state(), pk.jit_launch_count() - n0
    g.close()

    def one(w):
        o = oracle.Oracle(c.L, c.n_replicas, c.d, c.p, c.seed, c.variant, Ts=info["Ts"], D=info["D"], A=info["A"], words=[w])
        o.init(c.init)
        bad = []
        for t in (deep_times if w in deep else all_times):
            o.run(t - o.sweep)
            col = lat[t][:, w] if t in all_times else lat[t][:, deep.index(w)]
            if not np.array_equal(o.get_words()[:, 0], col):
                bad.append(("lattice", w, t))
            if not np.array_equal(o.counts(), cnt[t][w]):
                bad.append(("counts", w, t))
        o.close()
        return bad

    order = deep + [w for w in range(c.W) if w not in deep]    # the long columns first
    with ThreadPoolExecutor(NCPU) as ex:
        bad = [b for r in ex.map(one, order) for b in r]
    assert not bad, bad[:10]
    # the sweeps ran the run-time specialised kernel (the one bench.py times at this size)
    if jit_state != 1 and "libnvrtc not found" in pk.jit_message():
        pytest.skip("libnvrtc is not installed on this box: the built-in kernel ran (and passed every check above)")
    assert jit_state == 1, pk.jit_message()
    assert jit_launches == deep_times[-1]


def test_philox_block_via_init_stream(pk):
    """The device Philox against the KAT-pinned oracle block function on the
    INIT stream (C8), 2^16 blocks with seed words in both key halves."""
    seed = 0x0123456789ABCDEF
    g = pk.Pcpd(16384, 256, 0.5, 0.1, seed, 0, word_offset=1000)
    g.init(pk.INIT_BERNOULLI)
    lat = g.get_lattice()
    o = oracle.Oracle(16384, 64 * 1004, 0.5, 0.1, seed, 0, words=[1000, 1001, 1002, 1003])
    o.init(wl.INIT_BERNOULLI)
    assert np.array_equal(lat, o.get_words())
    g.close()


def test_error_behaviour_of_the_boundary(pk):
    """include/pcpd.h: every invalid argument is refused with a message, nothing is silently clamped
    except T_s > L; the sweep counter refuses to pass 2^32 - 1."""
    bad = [
        dict(L=4096, n_replicas=100, d=0.5, p=0.1),            # n_replicas not a multiple of 64
        dict(L=4096, n_replicas=0, d=0.5, p=0.1),
        dict(L=4100, n_replicas=64, d=0.5, p=0.1),             # L not a multiple of D
        dict(L=32, n_replicas=64, d=0.5, p=0.1),               # L < D
        dict(L=4096, n_replicas=64, d=1.5, p=0.1),
        dict(L=4096, n_replicas=64, d=0.5, p=float("nan")),
        dict(L=4096, n_replicas=64, d=0.5, p=0.1, variant=7),  # unknown variant
        dict(L=4096, n_replicas=64, d=0.5, p=0.25, variant=pk.PMASK_PAPER),   # paper mask needs p < 1/4
        dict(L=4096, n_replicas=64, d=0.5, p=0.5, variant=pk.PMASK_PAPER | pk.PMASK_BOUND_HALF),   # ... p < b in general
        dict(L=4096, n_replicas=64, d=0.5, p=0.75, variant=pk.PMASK_PAPER | pk.PMASK_BOUND_3_4),
        dict(L=4096, n_replicas=64, d=0.5, p=1.0, variant=pk.PMASK_PAPER | pk.PMASK_BOUND_ONE),
        dict(L=4096, n_replicas=64, d=0.5, p=0.1, variant=pk.PMASK_BOUND_HALF),   # bound bits without the mask flag
        dict(L=5120, n_replicas=64, d=0.5, p=0.1),             # L % T_s != 0 (T_s = 2048 not clamped: L > T_s)
        dict(L=4096, n_replicas=64, d=0.5, p=0.1, Ts=2048, D=64, A=5),   # A does not divide D
        dict(L=4096, n_replicas=64, d=0.5, p=0.1, Ts=2048, D=6, A=2),    # D < 2*Rr + 3
    ]
    for kw in bad:
        kw = dict(dict(seed=1, variant=0), **kw)
        with pytest.raises(pk.PcpdError) as e:
            pk.Pcpd(**kw)
        assert len(str(e.value)) > 20, kw
    g = pk.Pcpd(1024, 64, 0.5, 0.1, 1, 0)          # T_s clamped to L
    assert g.schedule_info()["Ts"] == 1024
    g.sweep = 2 ** 32 - 2
    g.init(pk.INIT_FULL)
    assert g.sweep == 0                             # init resets the counter
    g.sweep = 2 ** 32 - 2
    g.run(1)
    with pytest.raises(pk.PcpdError):
        g.run(1)
    with pytest.raises(pk.PcpdError):
        g.sweep = 2 ** 32
    with pytest.raises(pk.PcpdError):
        g.init(9)
    g.close()


def test_two_independent_kernels_agree_at_full_size(pk, monkeypatch):
    """Beyond the oracle's horizon (SURVEY.md 8(d) 'self-consistency'): the production warp-per-tile
    kernel and the generic block-per-tile kernel (different thread mapping, barriers, tile layout,
    Philox code path and compare code) must give the identical lattice on a full-size config.
    compute-sanitizer is closed on this pool, so this doubles as the memory-safety check: an
    out-of-bounds or racing shared-memory access in either kernel would show up as a mismatch."""
    c = wl.BY_NAME["cfg3"]
    res = []
    for force in ("0", "1"):
        monkeypatch.setenv("PCPD_FORCE_BLOCK_KERNEL", force)
        g = pk.Pcpd(c.L, c.n_replicas, c.d, c.p, c.seed, c.variant)
        g.init(c.init)
        g.run(3)
        res.append((g.get_lattice(), g.density(), g.pair_density()))
        g.close()
    monkeypatch.delenv("PCPD_FORCE_BLOCK_KERNEL")
    assert np.array_equal(res[0][0], res[1][0])
    assert np.array_equal(res[0][1], res[1][1]) and np.array_equal(res[0][2], res[1][2])
    # and a generic-threshold case with lazy tails on both streams, Bernoulli start
    res = []
    for force in ("0", "1"):
        monkeypatch.setenv("PCPD_FORCE_BLOCK_KERNEL", force)
        g = pk.Pcpd(1 << 18, 512, 0.8, 0.12, 4, 0)
        g.init(pk.INIT_BERNOULLI)
        g.run(5)
        res.append(g.get_lattice())
        g.close()
    monkeypatch.delenv("PCPD_FORCE_BLOCK_KERNEL")
    assert np.array_equal(res[0], res[1])


def test_P8_phase_behaviour_smoke(pk):
    """Qualitative only (pin P8; PAPER.md:41 and Fig. 1, p_c(d = 0.75) = 0.191789(2)):
    well below p_c the density settles on a plateau (active phase), well above it decays towards the
    single absorbing state.  Not a parity test - the paper's precision needs L = 2^18 and t ~ 10^7."""
    L, R, d = 1 << 16, 256, 0.75
    rho = {}
    for p in (0.10, 0.30):
        g = pk.Pcpd(L, R, d, p, 12, pk.PCPD)
        g.init(pk.INIT_FULL)
        series = []
        for _ in range(4):
            g.run(500)
            series.append(float(g.density().mean()) / L)
        rho[p] = series
        g.close()
    active, absorbing = rho[0.10], rho[0.30]
    assert active[-1] > 0.2 and abs(active[-1] - active[-2]) < 0.02 * active[-1]      # plateau
    assert absorbing[-1] < 0.05 and absorbing[-1] < absorbing[0]                          # decay
    assert active[-1] > 5 * absorbing[-1]


LONG = os.environ.get("PCPD_LONG_PARITY") == "1"


@pytest.mark.skipif(not LONG, reason="long parity run (oracle needs ~40 min of host time): set PCPD_LONG_PARITY=1")
@pytest.mark.parametrize("name,words,times", [
    ("cfg2", None, "all"),                                  # the whole run: all 4 columns, every record time up to 10^4
    ("cfg3", [0, 16, 31], [1, 2, 4, 8, 16, 32, 64]),
    ("cfg5", [0, 8, 15], [1, 2, 4, 8, 16, 32, 64]),
    ("cfg4", [0, 31], [1, 2, 4, 8, 16, 32]),
])
def test_long_parity_protocol(pk, name, words, times):
    """SURVEY.md 8(d) parity protocol beyond the default suite's horizon: cfg2 in full (lattice and counts at every
    log-spaced record time of the 10^4 sweeps), cfg3/4/5 on sampled word columns out to t = 64 (32)."""
    c = wl.BY_NAME[name]
    kw = dict(L=c.L, n_replicas=c.n_replicas, d=c.d, p=c.p, seed=c.seed, variant=c.variant)
    if times == "all":
        times = [t for t in wl.record_times(c.sweeps) if t > 0]
    gpu_check(pk, kw, {}, c.init, times, words=words)


def test_handles_created_from_two_threads(pk):
    """include/pcpd.h: pcpd_create* are thread-safe (first-use configuration and the allocator pair are serialised) and
    distinct handles are independent: two host threads create, run and destroy handles concurrently; each result equals
    the single-threaded one.  pcpd_set_allocator is refused while handles are alive."""
    import threading

    import torch

    def work(seed, out):
        with torch.cuda.stream(torch.cuda.Stream()):
            res = []
            for rep in range(4):
                g = pk.Pcpd(4096, 128, 0.3, 0.12, seed + rep, 0)
                g.init(1)
                g.run(3)
                res.append((g.get_lattice(), g.density()))
                g.close()
            out[seed] = res

    out = {}
    th = [threading.Thread(target=work, args=(s, out)) for s in (100, 200)]
    for t in th:
        t.start()
    for t in th:
        t.join()
    for seed in (100, 200):
        assert len(out[seed]) == 4
        for rep in range(4):
            g = pk.Pcpd(4096, 128, 0.3, 0.12, seed + rep, 0)
            g.init(1)
            g.run(3)
            assert np.array_equal(g.get_lattice(), out[seed][rep][0]) and np.array_equal(g.density(), out[seed][rep][1])
            if rep == 0:
                lib = pk.load_library()
                assert lib.pcpd_set_allocator(pk._ALLOC_FN(), pk._FREE_FN()) < 0    # back to cudaMalloc: not under a live handle
                assert b"alive" in lib.pcpd_last_error()
            g.close()


def test_pair_density_on_the_connected_lattice(pk):
    """C10: on the connected multispin lattice the right neighbour of (site L-1, lane j) is (site 0, lane j+1) of the
    same word column; pcpd_pair_density and the pair series of pcpd_run_series close the ring that way (the oracle's
    pair counts are pinned to the unrolled ring on the CPU side)."""
    L, R = 2048, 192
    for variant in (pk.PCPD | pk.CONNECTED, pk.PCPD):
        g = pk.Pcpd(L, R, 0.3, 0.12, 17, variant, Ts=1024, D=64, A=4)
        o = oracle.Oracle(L, R, 0.3, 0.12, 17, variant, Ts=1024, D=64, A=4)
        w0 = wl.random_lattice_words(L, R // 64, 0.5, seed=9)
        w0[0, :] |= np.uint64(0xFFFF0000FFFF0000)
        w0[L - 1, :] |= np.uint64(0x0000FFFFFFFF0000)
        g.set_lattice(w0)
        o.set_words(w0)
        assert np.array_equal(g.pair_density(), o.pair_counts())
        cnt, pr = g.run_series([0, 1, 3], pairs=True)
        for k, t in enumerate((0, 1, 3)):
            o.run(t - o.sweep)
            assert np.array_equal(cnt[k], o.counts()) and np.array_equal(pr[k], o.pair_counts()), (variant, t)
        g.close()
    a = pk.Pcpd(L, 64, 0.3, 0.12, 17, pk.PCPD | pk.CONNECTED)
    b = pk.Pcpd(L, 64, 0.3, 0.12, 17, pk.PCPD)
    w = np.zeros((L, 1), np.uint64)
    w[L - 1, 0] = np.uint64(1) << np.uint64(63)
    w[0, 0] = np.uint64(1)
    a.set_lattice(w); b.set_lattice(w)
    pa, pb = a.pair_density(), b.pair_density()
    assert pa[63] == 1 and pa.sum() == 1 and not pb.any()
    a.close(); b.close()


def test_delta_eff_of_a_near_critical_run(pk):
    """Row f1 end to end (Figs 5-6): a pcpd_run_series of particle and pair counts near the critical
    point (d = 0.5, p = 0.152; p_c(0.5) ~ 0.1524 from the analysis paper the text cites), then delta_eff on the host.
    Smoke only: both effective exponents are positive and of the magnitude the paper plots (0.1 .. 0.35) at late times,
    and the pair density lies below the particle density."""
    L, R = 1 << 16, 512
    times = [t for t in wl.record_times(2000) if t >= 1]
    g = pk.Pcpd(L, R, 0.5, 0.152, 3, pk.PCPD)
    g.init(pk.INIT_FULL)
    cnt, pr = g.run_series(times, pairs=True)
    g.close()
    rho, de = pk.delta_eff(times, cnt, L, half_window=4)
    rho2, de2 = pk.delta_eff(times, pr, L, half_window=4)
    late = [k for k, t in enumerate(times) if 200 <= t <= 1200]
    assert np.all(rho2[1:] < rho[1:]) and np.all(np.diff(rho[1:]) < 0)
    assert 0.1 < np.nanmean(de[late]) < 0.35, np.nanmean(de[late])
    assert 0.1 < np.nanmean(de2[late]) < 0.45, np.nanmean(de2[late])


def test_per_word_probabilities_scan(pk):
    """pcpd_create_scan (contract C11, next-row f4): every word column has its own (d, p); bit-exact against the
    oracle in the same mode, and column k equals the uniform GPU run with (d_k, p_k)."""
    L, W = 4096, 6
    ds = np.array([0.8, 0.5, 0.1, 1.0, 0.0, 0.3])
    ps = np.array([0.12, 0.152, 0.09, 0.3, 0.2, 0.0])
    for variant in (pk.PCPD, pk.TCPD | pk.CONNECTED):
        g = pk.Pcpd(L, 64 * W, ds, ps, 41, variant)
        o = oracle.Oracle(L, 64 * W, 0.25, 0.25, 41, variant)
        for k in range(W):
            o.set_word_probabilities(k, ds[k], ps[k])
        g.init(pk.INIT_BERNOULLI)
        o.init(1)
        for _ in range(4):
            g.run(2)
            o.run(2)
            assert np.array_equal(g.get_lattice(), o.get_words())
            assert np.array_equal(g.density(), o.counts())
        lat = g.get_lattice()
        g.close()
        if variant == pk.PCPD:
            for k in (0, 3):
                u = pk.Pcpd(L, 64, float(ds[k]), float(ps[k]), 41, variant, word_offset=k)
                u.init(pk.INIT_BERNOULLI)
                u.run(8)
                assert np.array_equal(u.get_lattice()[:, 0], lat[:, k])
                u.close()
    with pytest.raises(pk.PcpdError):
        pk.Pcpd(L, 64 * W, ds, ps, 41, pk.PCPD | pk.PMASK_PAPER)
    with pytest.raises(pk.PcpdError):
        pk.Pcpd(L, 64 * W, ds + 0.5, ps, 41, pk.PCPD)
    # a schedule the warp-per-tile-column kernel cannot run (tile column above 200 KiB) would silently ignore the
    # per-word table in the generic block kernel: refused
    with pytest.raises(pk.PcpdError):
        pk.Pcpd(25600 * 2, 64 * 2, ds[:2], ps[:2], 41, pk.PCPD, Ts=25600, D=800, A=4)
