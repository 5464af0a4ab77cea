"""Pins P0-P4, P7, P9-P12 of the CPU oracle (SURVEY.md 8(c) "What pins the oracle").

Everything here is checked against something OTHER than the oracle itself:
published Philox vectors, exact rational arithmetic, structural invariants of
eq. (1) and the master equation built from the reaction list.
CPU only (`-m "not gpu"`).
"""
import itertools
import os
from fractions import Fraction

import numpy as np
import pytest

import oracle
import workloads as wl

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


# ------------------------------------------------------------------ P0 ----
def test_P0_philox_known_answers():
    rows = [l.split() for l in open(os.path.join(GOLDEN, "philox_kat.txt")) if l.strip() and l[0] != "#"]
    assert len(rows) == 3
    for r in rows:
        v = [int(x, 16) for x in r]
        out = oracle.philox4x32_10(v[0:4], v[4:6])
        assert [int(x) for x in out] == v[6:10]


def test_P0_thresholds_exact_rational():
    for line in open(os.path.join(GOLDEN, "thresholds.txt")):
        if not line.strip() or line[0] == "#":
            continue
        q, T = line.split()
        # exact: floor of (the IEEE double nearest q) * 2^32, in rationals
        exact = (Fraction(float(q)) * (1 << 32)).__floor__()
        assert oracle.threshold(float(q)) == exact == int(T, 16)
    for bad in (-0.1, 1.0000001, float("nan")):
        assert oracle.threshold(bad) == (1 << 64) - 1


# ------------------------------------------------------------------ P0' ---
def test_P0p_lane_uniforms_are_the_planes_transposed():
    """U_j bit (31-k) = lane j of plane k; plane k = lo/hi of block k>>1 (C3),
    rebuilt here from the KAT-pinned block function with numpy bit ops."""
    seed, slot, sweep, word = 0x1234567890ABCDEF, 77, 5, 3
    for stream in (oracle.STREAM_DIFF, oracle.STREAM_ANNI):
        U = oracle.lane_uniforms(seed, slot, sweep, word, stream, 32)
        planes = []
        for m in range(16):
            x = oracle.philox4x32_10([slot, sweep, word, (stream << 24) | m],
                                     [seed & 0xFFFFFFFF, seed >> 32])
            planes.append(int(x[0]) | (int(x[1]) << 32))
            planes.append(int(x[2]) | (int(x[3]) << 32))
        for j in range(64):
            u = 0
            for k in range(32):
                u |= ((planes[k] >> j) & 1) << (31 - k)
            assert u == int(U[j])


def test_P0p_reduced_K_exhaustive_bitsliced_forms():
    """For K = 4 every (U, T): direct compare == MSB-first (lt, und) form ==
    LSB-first eager form (C3 'Equivalent bit-sliced forms').  The lanes come
    from the oracle's reduced-K uniforms so that all 16 U values occur."""
    K = 4
    seen = set()
    for slot in range(40):
        U = oracle.lane_uniforms(9, slot, 0, 0, oracle.STREAM_DIFF, K)
        seen |= set(int(u) for u in U)
        planes = [sum((((int(U[j]) >> (K - 1 - k)) & 1) << j) for j in range(64)) for k in range(K)]
        full = (1 << 64) - 1
        for T in range(0, (1 << K) + 1):
            direct = sum((1 << j) for j in range(64) if int(U[j]) < T)
            if T == (1 << K):
                assert direct == full
                continue
            lt, und = 0, full
            for k in range(K):
                bit = (T >> (K - 1 - k)) & 1
                if bit:
                    lt |= und & ~planes[k] & full
                    und &= planes[k]
                else:
                    und &= ~planes[k] & full
            assert lt == direct
            m = 0
            for k in reversed(range(K)):
                bit = (T >> (K - 1 - k)) & 1
                m = (m | (~planes[k] & full)) if bit else (m & ~planes[k] & full)
            assert m == direct
    assert seen == set(range(16))


@pytest.mark.parametrize("q", [0.5, 0.15, 0.09, 0.8, 0.0, 1.0])
def test_P0p_mask_frequency(q):
    T = oracle.threshold(q)
    n_masks = 4000  # 256k lanes
    ones = 0
    for slot in range(n_masks):
        ones += int(oracle.bernoulli_mask(42, slot, 7, 1, oracle.STREAM_ANNI, T).sum())
    n = 64 * n_masks
    pr = T / 2.0 ** 32
    sigma = (n * pr * (1 - pr)) ** 0.5
    assert abs(ones - n * pr) <= 4 * sigma + 1e-9


def test_P0p_streams_and_words_are_distinct():
    a = oracle.lane_uniforms(1, 0, 0, 0, oracle.STREAM_DIFF)
    assert not np.array_equal(a, oracle.lane_uniforms(1, 0, 0, 0, oracle.STREAM_ANNI))
    assert not np.array_equal(a, oracle.lane_uniforms(1, 1, 0, 0, oracle.STREAM_DIFF))
    assert not np.array_equal(a, oracle.lane_uniforms(1, 0, 1, 0, oracle.STREAM_DIFF))
    assert not np.array_equal(a, oracle.lane_uniforms(1, 0, 0, 1, oracle.STREAM_DIFF))
    assert not np.array_equal(a, oracle.lane_uniforms(2, 0, 0, 0, oracle.STREAM_DIFF))
    assert not np.array_equal(a, oracle.lane_uniforms(1 << 32, 0, 0, 0, oracle.STREAM_DIFF))


# ------------------------------------------------------------------ P1-P3 -
SCHEDULES = [dict(Ts=2048, D=64, A=4), dict(Ts=64, D=64, A=64), dict(Ts=32, D=16, A=2)]


@pytest.mark.parametrize("variant", [wl.PCPD, wl.TCPD, wl.QCPD, wl.CPD])
@pytest.mark.parametrize("sch", SCHEDULES)
def test_P1_empty_lattice_is_absorbing(variant, sch):
    o = oracle.Oracle(128, 128, 0.3, 0.2, 11, variant, **sch)
    o.init(wl.INIT_EMPTY)
    o.run(5)
    assert not o.get_words().any() and not o.counts().any()


@pytest.mark.parametrize("variant", [wl.PCPD, wl.TCPD, wl.QCPD, wl.CPD])
@pytest.mark.parametrize("sch", SCHEDULES)
def test_P2_d_equals_one_conserves_particles(variant, sch):
    o = oracle.Oracle(128, 128, 1.0, 0.3, 12, variant, **sch)
    w0 = wl.random_lattice_words(128, 2, 0.4, seed=5)
    o.set_words(w0)
    c0 = o.counts()
    for _ in range(4):
        o.run(1)
        assert np.array_equal(o.counts(), c0)
    assert not np.array_equal(o.get_words(), w0)  # it did move


@pytest.mark.parametrize("variant", [wl.PCPD, wl.TCPD, wl.QCPD])
def test_P3_isolated_particles_never_react(variant):
    # one particle per replica: count stays 1 for any d, p
    L = 128
    o = oracle.Oracle(L, 64, 0.4, 0.3, 13, variant, Ts=64, D=32, A=4)
    w0 = np.zeros((L, 1), dtype=np.uint64)
    rng = np.random.default_rng(0)
    for j in range(64):
        w0[rng.integers(0, L), 0] |= np.uint64(1) << np.uint64(j)
    o.set_words(w0)
    for _ in range(6):
        o.run(1)
        assert np.all(o.counts() == 1)
    # d = 0: any state without adjacent pairs (triples) is frozen bit for bit
    o = oracle.Oracle(L, 128, 0.0, 0.3, 14, variant, Ts=64, D=32, A=4)
    w0 = wl.isolated_particles_words(L, 2, 4, seed=3)
    o.set_words(w0)
    o.run(4)
    assert np.array_equal(o.get_words(), w0)


def test_P3_tcpd_pairs_frozen_at_d0_but_pcpd_reacts():
    L = 64
    w0 = np.zeros((L, 1), dtype=np.uint64)
    full = np.uint64(0xFFFFFFFFFFFFFFFF)
    for i in range(0, L, 8):
        w0[i, 0] = full
        w0[i + 1, 0] = full  # isolated pairs, no triples
    t = oracle.Oracle(L, 64, 0.0, 0.3, 15, wl.TCPD, Ts=64, D=16, A=4)
    t.set_words(w0)
    t.run(3)
    assert np.array_equal(t.get_words(), w0)
    p = oracle.Oracle(L, 64, 0.0, 0.3, 15, wl.PCPD, Ts=64, D=16, A=4)
    p.set_words(w0)
    p.run(3)
    assert not np.array_equal(p.get_words(), w0)


# ------------------------------------------------------------------ P4 ----
def _bits(s, L):
    return [(s >> i) & 1 for i in range(L)]


def _state(bits):
    return sum(b << i for i, b in enumerate(bits))


def master_matrix(variant, L, d, p):
    """One-attempt transition matrix P[s, s'] built from eq. (1)'s REACTION
    LIST alone (TCPD: BASELINE.json config 5), exact rationals:
    every bond/site i is selected with probability 1/L; hop at rate d if exactly
    one end occupied; pair (triple) -> empty at p(1-d); creation at each EMPTY
    outer neighbour at (1-p)(1-d)/2; diagonal by normalisation."""
    n = 1 << L
    P = [[Fraction(0)] * n for _ in range(n)]
    k = 1 if variant == wl.CPD else 2 + variant  # cluster size: 2 PCPD, 3 TCPD, 4 QCPD, 1 CPD
    for s in range(n):
        b = _bits(s, L)
        for i in range(L):
            cluster = [(i + m) % L for m in range(k)]
            lo, hi = (i - 1) % L, (i + k) % L
            i1 = (i + 1) % L
            if b[i] != b[i1]:
                nb = list(b)
                nb[i], nb[i1] = b[i1], b[i]
                P[s][_state(nb)] += d / L
            if all(b[c] for c in cluster):
                nb = list(b)
                for c in cluster:
                    nb[c] = 0
                P[s][_state(nb)] += p * (1 - d) / L
                for tgt in (lo, hi):
                    if not b[tgt]:
                        nb = list(b)
                        nb[tgt] = 1
                        P[s][_state(nb)] += (1 - p) * (1 - d) / 2 / L
        P[s][s] += 1 - sum(P[s])
    return P


def oracle_matrix(variant, L, d, p):
    n = 1 << L
    P = [[Fraction(0)] * n for _ in range(n)]
    half = Fraction(1, 2)
    for s in range(n):
        b = _bits(s, L)
        for i in range(L):
            for Dm, Pm, Fm in itertools.product((0, 1), repeat=3):
                wgt = (d if Dm else 1 - d) * (p if Pm else 1 - p) * half / L
                out = oracle.single_attempt(variant, b, i, Dm, Pm, Fm)
                P[s][_state([int(x) for x in out])] += wgt
    return P


@pytest.mark.parametrize("variant,L", [(wl.PCPD, 4), (wl.PCPD, 5), (wl.PCPD, 6), (wl.TCPD, 5), (wl.TCPD, 6),
                                       (wl.QCPD, 6), (wl.QCPD, 7), (wl.CPD, 3), (wl.CPD, 4), (wl.CPD, 5)])
def test_P4_master_equation_enumeration(variant, L):
    d, p = Fraction(3, 10), Fraction(7, 40)
    assert master_matrix(variant, L, d, p) == oracle_matrix(variant, L, d, p)  # exact rationals


def test_P4_fission_side_follows_alg1():
    # G8: Fm = 1 (r3 < 1/2) -> fission LOW (q_{i-1})
    q = [0, 1, 1, 0, 0, 0]
    assert list(oracle.single_attempt(wl.PCPD, q, 1, 0, 0, 1)) == [1, 1, 1, 0, 0, 0]
    assert list(oracle.single_attempt(wl.PCPD, q, 1, 0, 0, 0)) == [0, 1, 1, 1, 0, 0]
    # G3: diffusion has priority, a pair under Dm does not react
    assert list(oracle.single_attempt(wl.PCPD, q, 1, 1, 1, 1)) == q
    assert list(oracle.single_attempt(wl.PCPD, q, 1, 0, 1, 1)) == [0, 0, 0, 0, 0, 0]
    assert list(oracle.single_attempt(wl.PCPD, q, 2, 1, 0, 0)) == [0, 1, 0, 1, 0, 0]
    # periodic wrap (G2)
    assert list(oracle.single_attempt(wl.PCPD, [1, 0, 0, 0, 0, 1], 5, 0, 0, 1)) == [1, 0, 0, 0, 1, 1]
    assert list(oracle.single_attempt(wl.PCPD, [1, 0, 0, 0, 0, 1], 5, 0, 0, 0)) == [1, 1, 0, 0, 0, 1]


@pytest.mark.parametrize("variant,L", [(wl.PCPD, 6), (wl.TCPD, 6), (wl.QCPD, 6), (wl.CPD, 5)])
def test_P4_literal_mode_mean_density_vs_master_equation(variant, L):
    """E[count] after n = 1, 2, 3 time units (n*L attempts) from P^(nL) (floats
    from the exact-rational matrix) vs the literal Alg. 1 Monte Carlo mean."""
    d, p = 0.3, 0.175
    P = np.array([[float(x) for x in row] for row in
                  master_matrix(variant, L, Fraction(3, 10), Fraction(7, 40))])
    pop = np.array([bin(s).count("1") for s in range(1 << L)], dtype=float)
    R = 200_000
    q0 = np.ones((R, L), dtype=np.uint8)
    counts, _ = oracle.literal_run(variant, L, R, d, p, 99, q0, [0, 1, 2, 3])
    v = np.zeros(1 << L)
    v[(1 << L) - 1] = 1.0
    for n in range(4):
        exact_mean = v @ pop
        exact_var = v @ pop ** 2 - exact_mean ** 2
        mc = counts[n].mean()
        assert abs(mc - exact_mean) <= 4.5 * (exact_var / R) ** 0.5 + 1e-12, (n, mc, exact_mean)
        v = v @ np.linalg.matrix_power(P, L)


# ------------------------------------------------------------------ P7 ----
@pytest.mark.parametrize("variant", [wl.PCPD, wl.TCPD, wl.QCPD, wl.CPD])
def test_P7_run_splitting_loop_order_word_subsets(variant):
    kw = dict(L=256, n_replicas=256, d=0.3, p=0.12, seed=21, variant=variant, Ts=128, D=32, A=4)
    a = oracle.Oracle(**kw)
    a.init(wl.INIT_BERNOULLI)
    a.run(5)
    b = oracle.Oracle(**kw)
    b.init(wl.INIT_BERNOULLI)
    b.run(2)
    b.run(3)
    assert np.array_equal(a.get_words(), b.get_words()) and a.sweep == b.sweep == 5
    c = oracle.Oracle(**kw)
    c.set_reverse_order(1)
    c.init(wl.INIT_BERNOULLI)
    c.run(5)
    assert np.array_equal(a.get_words(), c.get_words())
    s = oracle.Oracle(**kw, words=[3, 1])
    s.init(wl.INIT_BERNOULLI)
    s.run(5)
    assert np.array_equal(a.get_words()[:, [3, 1]], s.get_words())
    assert np.array_equal(a.counts().reshape(4, 64)[[3, 1]].ravel(), s.counts())
    # set/get round trip and counts = column popcounts
    w = a.get_words()
    bits = (w[:, :, None] >> np.arange(64, dtype=np.uint64)) & np.uint64(1)
    assert np.array_equal(bits.sum(axis=0).ravel().astype(np.uint32), a.counts())
    s2 = oracle.Oracle(**kw)
    s2.set_words(w)
    assert np.array_equal(s2.get_words(), w)


def _bits_of(words):
    return ((words[:, :, None] >> np.arange(64, dtype=np.uint64)) & np.uint64(1)).astype(np.uint32)   # [L, W, 64]


def test_P7_pair_counts_against_numpy_including_the_ring_closure():
    """oracle_pair_counts = sum_i q(i) q(i+1 mod L) per replica, against numpy on the packed words;
    states built so that a dropped or wrong ring closure (site L-1 -> site 0) changes the answer."""
    L, W = 96, 3
    o = oracle.Oracle(L, 64 * W, 0.3, 0.1, 3, wl.PCPD, Ts=96, D=32, A=4)
    for trial, w in enumerate([wl.random_lattice_words(L, W, 0.5, seed=11), wl.random_lattice_words(L, W, 0.8, seed=12)]):
        w[0, :] |= np.uint64(0x00FF00FF00FF00FF)      # plenty of (L-1, 0) pairs ...
        w[L - 1, :] |= np.uint64(0x0F0F0F0F0F0F0F0F)
        w[1, :] &= ~np.uint64(0xFFFF)                 # ... that are not mirrored by (0, 1) pairs
        o.set_words(w)
        expect = _bits_of(w & np.roll(w, -1, axis=0)).sum(axis=0).ravel()
        assert np.array_equal(o.pair_counts(), expect), trial
        no_wrap = _bits_of(w[:-1] & w[1:]).sum(axis=0).ravel()
        assert not np.array_equal(expect, no_wrap)   # the closure did matter in this state
    # only the closure pair: one particle at site L-1 and one at site 0 in lane 7
    w = np.zeros((L, W), np.uint64)
    w[0, 1] = w[L - 1, 1] = np.uint64(1 << 7)
    o.set_words(w)
    pc = o.pair_counts()
    assert pc[64 + 7] == 1 and pc.sum() == 1
    # full lattice: L pairs per replica; empty: none
    o.init(wl.INIT_FULL)
    assert np.all(o.pair_counts() == L)
    o.init(wl.INIT_EMPTY)
    assert not o.pair_counts().any()


def test_P7_pair_counts_on_the_connected_lattice_are_those_of_the_long_ring():
    """C10: a word column is ONE ring of 64 L sites (strand position lane*L + site); the successor of (site L-1,
    lane j) is (site 0, lane j+1 mod 64).  The ring is unrolled here with numpy and its adjacent pairs counted by the
    lane of their left site."""
    L, W = 64, 2
    w = wl.random_lattice_words(L, W, 0.6, seed=21)
    o = oracle.Oracle(L, 64 * W, 0.3, 0.1, 3, wl.PCPD | oracle.CONNECTED, Ts=64, D=32, A=4)
    o.set_words(w)
    bits = _bits_of(w)                                              # [L, W, 64]
    for k in range(W):
        ring = bits[:, k, :].T.reshape(-1)                          # position lane*L + site
        pairs = ring & np.roll(ring, -1)
        assert np.array_equal(o.pair_counts()[64 * k:64 * (k + 1)], pairs.reshape(64, L).sum(axis=1))
    # a lone pair across the lane seam: (site L-1, lane 63) and (site 0, lane 0) are neighbours on the ring
    w = np.zeros((L, W), np.uint64)
    w[L - 1, 0] = np.uint64(1) << np.uint64(63)
    w[0, 0] = np.uint64(1)
    o.set_words(w)
    pc = o.pair_counts()
    assert pc[63] == 1 and pc.sum() == 1
    i = oracle.Oracle(L, 64 * W, 0.3, 0.1, 3, wl.PCPD, Ts=64, D=32, A=4)   # independent lanes: not neighbours
    i.set_words(w)
    assert not i.pair_counts().any()


# ----------------------------------------------------------------- P12 ----
# The oracle's instrumentation (SURVEY.md 8(d) "lazy-needed count": planes / Philox blocks a lazy MSB-first evaluation
# needs until all 64 lanes of a mask are decided) - feeds bench.py's cpu_baseline.lazy_blocks_per_attempt_word and is
# checked against the closed form the roofline numerator uses.
def _first_deciding_plane(U, T):
    """Brute force from C3: lane j is decided at the first plane k (1-based count) where bit (31-k) of U_j differs from
    that of T; planes below T's lowest set bit never matter (a lane equal to T on all planes that matter is not < T)."""
    if T == 0 or T >= 1 << 32:
        return 0
    nq = max(k + 1 for k in range(32) if (T >> (31 - k)) & 1)
    need = 0
    for u in U:
        first = next((k + 1 for k in range(32) if ((int(u) >> (31 - k)) & 1) != ((T >> (31 - k)) & 1)), 32)
        need = max(need, min(first, nq))
    return need


@pytest.mark.parametrize("d,p", [(0.8, 0.12), (0.5, 0.152), (0.75, 2.0 ** -32), (0.0, 1.0)])
def test_P12_stats_equal_brute_force_first_differing_plane(d, p):
    L, D = 16, 16     # one tile = one domain, one word: slot g = sub-step * A + a runs over 0 .. 15
    seed, word, sweeps = 0x5EED0000BEEF, 5, 3
    o = oracle.Oracle(L, 64 * 6, d, p, seed, wl.PCPD, Ts=L, D=D, A=4, words=[word])
    o.init(wl.INIT_BERNOULLI)
    o.run(sweeps)
    Td, Tp = o.thresholds()
    exp = dict(attempt_words=0, planes_needed_D=0, planes_needed_P=0, blocks_needed_D=0, blocks_needed_P=0)
    for t in range(sweeps):
        for g in range(L):
            nd = _first_deciding_plane(oracle.lane_uniforms(seed, g, t, word, oracle.STREAM_DIFF), Td)
            npp = _first_deciding_plane(oracle.lane_uniforms(seed, g, t, word, oracle.STREAM_ANNI), Tp)
            exp["attempt_words"] += 1
            exp["planes_needed_D"] += nd
            exp["planes_needed_P"] += npp
            exp["blocks_needed_D"] += (nd + 1) // 2
            exp["blocks_needed_P"] += (npp + 1) // 2
    assert o.stats() == exp


def test_P12_hand_checked_masks():
    """Four lanes worked out by hand against T = 0b1100 << 28 (0.75): U = 0b1011... differs at plane 2, 0b1101... at
    plane 4, 0b0... at plane 1; T has two planes that matter, so the counts cap at 2."""
    T = 0xC0000000
    assert _first_deciding_plane([0xB0000000], T) == 2
    assert _first_deciding_plane([0xD0000000], T) == 2      # differs at plane 4, but planes 3.. cannot matter
    assert _first_deciding_plane([0x00000000], T) == 1
    assert _first_deciding_plane([0x00000000, 0xB0000000], T) == 2
    assert _first_deciding_plane([0x12345678], 0x12345679) == 32
    assert _first_deciding_plane([0x12345678], 0) == 0 and _first_deciding_plane([5], 1 << 32) == 0


def test_P12_stats_reproduce_the_closed_form_of_the_roofline_numerator():
    """A lane is undecided after k planes w.p. 2^-k, so a generic 64-lane mask needs sum_m [1 - (1 - 4^-m)^64] = 3.92
    blocks on average (bench.py's blocks_needed_generic): the oracle's instrumentation must agree
    within its sampling error, on cfg4's thresholds."""
    c = wl.BY_NAME["cfg4"]
    o = oracle.Oracle(2048, 64 * 4, c.d, c.p, c.seed, c.variant)
    o.init(c.init)
    o.run(2)
    st = o.stats()
    n = st["attempt_words"]
    assert n == 2 * 2048 * 4
    closed = sum(1.0 - (1.0 - 4.0 ** -m) ** 64 for m in range(16))
    assert abs(closed - 3.92) < 0.01
    # per-mask block count has a standard deviation of ~0.96
    for key in ("blocks_needed_D", "blocks_needed_P"):
        assert abs(st[key] / n - closed) < 5 * 0.96 / n ** 0.5, (key, st[key] / n, closed)
    # d = 1/2: exactly one plane, one block, per mask
    o = oracle.Oracle(2048, 64, 0.5, c.p, 1, 0)
    o.init(0)
    o.run(1)
    st = o.stats()
    assert st["planes_needed_D"] == st["blocks_needed_D"] == st["attempt_words"] == 2048


def test_init_bernoulli_is_the_init_stream():
    """C8: word(i, w) = lo of block (i, 0, w, 4<<24)."""
    o = oracle.Oracle(64, 128, 0.5, 0.1, 0xABCDEF0123, 0, Ts=64, D=16, A=4)
    o.init(wl.INIT_BERNOULLI)
    w = o.get_words()
    for i, k in [(0, 0), (5, 1), (63, 0)]:
        x = oracle.philox4x32_10([i, 0, k, 4 << 24], [0xCDEF0123, 0xAB])
        assert int(w[i, k]) == int(x[0]) | (int(x[1]) << 32)
    frac = np.unpackbits(w.view(np.uint8)).mean()
    assert abs(frac - 0.5) < 4 * 0.5 / (64 * 128) ** 0.5


def test_create_rejects_invalid():
    for kw in (dict(L=100, Ts=64, D=16, A=4), dict(L=128, Ts=64, D=24, A=4),
               dict(L=128, Ts=64, D=16, A=3), dict(L=128, Ts=6, D=6, A=2)):
        with pytest.raises(ValueError):
            oracle.Oracle(kw["L"], 64, 0.5, 0.1, 1, 0, Ts=kw["Ts"], D=kw["D"], A=kw["A"])
    with pytest.raises(ValueError):
        oracle.Oracle(128, 64, 1.5, 0.1, 1, 0)
    with pytest.raises(ValueError):
        oracle.Oracle(128, 64, 0.5, 0.1, 1, 0, Ts=8, D=8, A=2).__class__(128, 64, 0.5, 0.1, 1, 1, Ts=8, D=8, A=2)  # TCPD needs D>=9


# ------------------------------------------------------------------ P9 ----
# The paper's own annihilation mask (next-row f2; Alg. 2 lines 12-13 PAPER.md:141-142,
# section 4.3): "RNG() and RNG()" = an independent 1/4-bit per lane,
# ANDed with ONE word-wide draw that is 1 w.p. 4p.  Pinned to what the paper fixes: the
# per-lane probability is p; given the word-wide draw the lanes are independent 1/4-bits;
# two lanes are both set w.p. (1/16) 4p = p/4 (partially correlated);
# the word is empty whenever the word-wide draw fails.
def test_P9_paper_pmask_probabilities():
    p = 0.12
    T4p = oracle.threshold(4 * p)
    assert T4p == int(np.floor(4 * p * 2.0 ** 32))
    n = 40000
    masks = np.array([oracle.paper_pmask(11, s, 3, s % 7, T4p) for s in range(n)], dtype=np.float64)  # [n, 64]
    gate = masks.any(axis=1)
    # per-lane probability p: words are the independent samples (lanes of a word share the draw)
    per_word = masks.mean(axis=1)
    se = per_word.std(ddof=1) / n ** 0.5
    assert abs(per_word.mean() - p) < 4 * se, (per_word.mean(), p, se)
    # P(word-wide draw = 1) = 4p, up to the words whose 64 quarter-bits are all 0 (prob. (3/4)^64 ~ 1e-8)
    assert abs(gate.mean() - 4 * p) < 4 * (4 * p * (1 - 4 * p) / n) ** 0.5
    # given the draw, lanes are independent Bernoulli(1/4)
    g = masks[gate]
    assert abs(g.mean() - 0.25) < 4 * (0.25 * 0.75 / g.size) ** 0.5
    c = np.corrcoef(g[:, :8].T)
    assert np.all(np.abs(c - np.eye(8)) < 5 / len(g) ** 0.5)
    # two lanes both set: p/4, not p^2 (independent) and not p (fully correlated)
    both = (masks[:, 0] * masks[:, 1]).mean()
    assert abs(both - p / 4) < 4 * (p / 4 / n) ** 0.5
    # threshold edge cases: T4p = 0 never annihilates
    assert not any(oracle.paper_pmask(11, s, 3, 0, 0).any() for s in range(200))


@pytest.mark.parametrize("code", [0, 1, 2, 3])
def test_P9_paper_pmask_family_probabilities(code):
    """The family of section 4.3: per-lane independent bits that are 1 w.p. b (b = 1/4: two raw words
    ANDed; 1/2: one raw word; 1: none, "all N_r bits are set to 1 with probability p and all 0 otherwise"; 3/4: two raw
    words ORed) ANDed with ONE word-wide draw that is 1 w.p. p/b.  Pinned to what those sentences fix: lane probability p;
    gate probability p/b; given the gate the lanes are independent b-bits; two lanes are both set w.p. p b - p for
    b = 1 (fully correlated), falling to p/4 with two decorrelation bits."""
    b = oracle.PMASK_BOUNDS[code]
    p = 0.12
    Tg = oracle.pmask_gate_threshold(p, code)
    from fractions import Fraction
    q = {0: 4.0 * p, 1: 2.0 * p, 2: p, 3: 4.0 * p / 3.0}[code]           # the quotient as the paper writes it
    assert Tg == (Fraction(q) * (1 << 32)).__floor__()
    n = 40000
    masks = np.array([oracle.paper_pmask_bound(11, s, 3, s % 7, Tg, code) for s in range(n)], dtype=np.float64)   # [n, 64]
    gate = masks.any(axis=1)
    per_word = masks.mean(axis=1)                     # words are the independent samples (lanes share the draw)
    assert abs(per_word.mean() - p) < 4 * per_word.std(ddof=1) / n ** 0.5
    assert abs(gate.mean() - p / b) < 4 * (p / b * (1 - p / b) / n) ** 0.5 + 1e-7   # (+ all-zero words: (1-b)^64)
    g = masks[gate]
    if b < 1:
        assert abs(g.mean() - b) < 4 * (b * (1 - b) / g.size) ** 0.5
        c = np.corrcoef(g[:, :8].T)
        assert np.all(np.abs(c - np.eye(8)) < 5 / len(g) ** 0.5)
    else:
        assert np.all(g == 1)                         # no decorrelation: the whole word at once
    both = (masks[:, 0] * masks[:, 1]).mean()
    assert abs(both - p * b) < 4 * (p * b / n) ** 0.5
    if code == 0:                                     # Alg. 2's own form is the b = 1/4 member
        for s_ in range(50):
            assert np.array_equal(oracle.paper_pmask(11, s_, 3, 2, Tg), oracle.paper_pmask_bound(11, s_, 3, 2, Tg, 0))
    # p must lie below the bound
    assert oracle.pmask_gate_threshold(b, code) == (1 << 64) - 1
    assert oracle.pmask_gate_threshold(np.nextafter(b, 0), code) < (1 << 32)
    with pytest.raises(ValueError):
        oracle.Oracle(128, 64, 0.5, b, 1, oracle.PMASK_PAPER | (code << oracle.PMASK_BOUND_SHIFT), Ts=64, D=16, A=4)
    with pytest.raises(ValueError):
        oracle.Oracle(128, 64, 0.5, 0.1, 1, code << oracle.PMASK_BOUND_SHIFT if code else 0x1000, Ts=64, D=16, A=4)   # bound bits without the flag


def test_P9_fully_correlated_mask_empties_whole_words_in_a_run():
    """b = 1 wired into the run: with d = 0 and a full lattice an annihilation removes the pair in ALL 64 replicas of the
    word at once ("the bits are fully correlated"), so after one sweep there are sites that are empty in
    every replica (where no later fission - whose side is still drawn per lane - refilled them); with b = 1/4, 1/2 or 3/4
    the lanes annihilate independently given the gate and 64 simultaneous holes do not occur."""
    kw = dict(L=256, n_replicas=64, d=0.0, p=0.2, seed=5, Ts=64, D=16, A=16)
    empty_words = {}
    for code in range(4):
        o = oracle.Oracle(variant=oracle.PMASK_PAPER | (code << oracle.PMASK_BOUND_SHIFT), **kw)
        o.init(wl.INIT_FULL)
        o.run(1)
        empty_words[code] = int((o.get_words()[:, 0] == 0).sum())
        assert o.counts().max() < 256          # something was annihilated in every replica's ring
    assert empty_words[2] > 0 and empty_words[0] == empty_words[1] == empty_words[3] == 0, empty_words


def test_P9_paper_pmask_mode_in_run():
    """The run uses exactly that mask: a full lattice with d = 0 (no diffusion) loses particles
    only in words whose word-wide draw fired, and p >= 1/4 is rejected."""
    with pytest.raises(ValueError):
        oracle.Oracle(128, 64, 0.5, 0.25, 1, oracle.PMASK_PAPER, Ts=64, D=16, A=4)
    kw = dict(L=64, n_replicas=64, d=0.0, p=0.2, seed=5, Ts=64, D=16, A=16)
    a = oracle.Oracle(variant=oracle.PMASK_PAPER, **kw)
    b = oracle.Oracle(variant=0, **kw)
    a.init(wl.INIT_FULL)
    b.init(wl.INIT_FULL)
    a.run(1)
    b.run(1)
    # same positions and fission bits, different annihilation masks -> different states
    assert not np.array_equal(a.get_words(), b.get_words())
    assert a.counts().min() < 64  # something was annihilated at p = 0.2


# ----------------------------------------------------------------- P10 ----
# The paper's connected multispin lattice (next-row f3): the 64 bit-lanes of a
# word column are 64 consecutive segments of ONE ring of 64 L sites, joined by a bit rotation at the
# seam.  Pinned to what that sentence fixes: a particle is a random walker on the long ring (its
# strand position lane*L + site moves by small steps only, also across the seam, and it does cross);
# d = 1 conserves the particle number of the RING (the sum over the 64 lanes), not of a lane.
def test_P10_connected_lattice_single_walker_crosses_the_seam():
    L = 256
    o = oracle.Oracle(L, 64, 1.0, 0.3, 17, oracle.CONNECTED, Ts=256, D=64, A=4)
    w = np.zeros((L, 1), np.uint64)
    w[L - 1, 0] = np.uint64(1) << np.uint64(5)
    o.set_words(w)
    ring = 64 * L
    pos, lanes = 5 * L + (L - 1), {5}
    for _ in range(300):
        o.run(1)
        g = o.get_words()[:, 0]
        sites = np.nonzero(g)[0]
        assert len(sites) == 1 and bin(int(g[sites[0]])).count("1") == 1      # still exactly one particle
        lane = int(g[sites[0]]).bit_length() - 1
        new = lane * L + int(sites[0])
        step = (new - pos + ring // 2) % ring - ring // 2
        assert abs(step) < L // 4, (pos, new)      # a wrongly wired seam makes the walker jump by ~L or 2L
        pos = new
        lanes.add(lane)
    assert len(lanes) >= 2                        # it did cross the seam


def test_P10_connected_lattice_conserves_ring_not_lane():
    L = 128
    kw = dict(L=L, n_replicas=128, d=1.0, p=0.2, seed=23, Ts=128, D=32, A=4)
    w0 = wl.random_lattice_words(L, 2, 0.3, seed=5)
    a = oracle.Oracle(variant=oracle.CONNECTED, **kw)
    b = oracle.Oracle(variant=0, **kw)
    for o in (a, b):
        o.set_words(w0)
    c0 = a.counts().astype(np.int64)
    a.run(20)
    b.run(20)
    ca, cb = a.counts().astype(np.int64), b.counts().astype(np.int64)
    assert np.array_equal(cb, c0)                                   # independent lanes: each lane conserved
    assert np.array_equal(ca.reshape(2, 64).sum(axis=1), c0.reshape(2, 64).sum(axis=1))   # ring conserved
    assert not np.array_equal(ca, c0)                               # ... but particles changed lanes
    # empty lattice is absorbing in this mode too
    e = oracle.Oracle(variant=oracle.CONNECTED, **dict(kw, d=0.3))
    e.init(wl.INIT_EMPTY)
    e.run(3)
    assert not e.get_words().any()


# ----------------------------------------------------------------- P11 ----
def test_P11_per_word_probabilities_equal_uniform_runs():
    """C11 (next-row f4): with per-word-column probabilities, column k evolves exactly as in a uniform run
    with (d_k, p_k) - columns never interact and all streams are keyed by the global word index."""
    L, W = 256, 4
    ds, ps = [0.5, 0.1, 0.8, 1.0], [0.15, 0.09, 0.0, 0.3]
    sch = dict(Ts=128, D=32, A=4)
    o = oracle.Oracle(L, 64 * W, 0.25, 0.25, 77, wl.PCPD, **sch)
    for k in range(W):
        o.set_word_probabilities(k, ds[k], ps[k])
    o.init(wl.INIT_BERNOULLI)
    o.run(6)
    got = o.get_words()
    for k in range(W):
        u = oracle.Oracle(L, 64 * W, ds[k], ps[k], 77, wl.PCPD, words=[k], **sch)
        u.init(wl.INIT_BERNOULLI)
        u.run(6)
        assert np.array_equal(u.get_words()[:, 0], got[:, k]), k
    with pytest.raises(ValueError):
        o.set_word_probabilities(W, 0.5, 0.1)
    with pytest.raises(ValueError):
        o.set_word_probabilities(0, 1.5, 0.1)
