"""Pins P5 and P6 of the oracle's schedule SD2.

P6: exact operator calculation on a toy ring, written here from the text of C5
and eq. (1) with numpy (shares nothing with the oracle except the KAT-pinned
Philox block used to derive the shifts), compared with the oracle's Monte Carlo
occupation and pair probabilities, site by site.
P5: SD2 vs the literal Algorithm 1, mean density at log-spaced
times - the paper's own way of validating a modified site selection
(PAPER.md:191-197).
"""
import os

import numpy as np
import pytest

import oracle
import workloads as wl


# ------------------------------------------------------------------ P6 ----
def rule_matrix(variant, nsites, x, d, p):
    """Stochastic matrix M[s', s] of ONE attempt at domain-local pair position
    x on `nsites` sites, from eq. (1)'s reaction list."""
    k = 1 if variant == wl.CPD else 2 + variant   # cluster size: 2 PCPD, 3 TCPD, 4 QCPD, 1 CPD
    n = 1 << nsites
    M = np.zeros((n, n))
    for s in range(n):
        b = [(s >> i) & 1 for i in range(nsites)]
        stay = 1.0
        if b[x] != b[x + 1]:
            nb = list(b)
            nb[x], nb[x + 1] = b[x + 1], b[x]
            M[sum(v << i for i, v in enumerate(nb)), s] += d
            stay -= d
        if all(b[x + m] for m in range(k)):
            nb = list(b)
            for m in range(k):
                nb[x + m] = 0
            M[sum(v << i for i, v in enumerate(nb)), s] += p * (1 - d)
            stay -= p * (1 - d)
            for tgt in (x - 1, x + k):
                if not b[tgt]:
                    nb = list(b)
                    nb[tgt] = 1
                    M[sum(v << i for i, v in enumerate(nb)), s] += (1 - p) * (1 - d) / 2
                    stay -= (1 - p) * (1 - d) / 2
        M[s, s] += stay
    return M


def allowed_positions(D, Rr, c):
    """C5 step 4: x in [1, D-1-Rr] minus (seam at c) x in [c-Rr, c]."""
    xs = list(range(1, D - 1 - Rr + 1))
    if c is not None:
        xs = [x for x in xs if not (c - Rr <= x <= c)]
    return xs


def apply_on_sites(v, M, sites, L):
    t = v.reshape((2,) * L)
    # numpy axis a <-> site (L-1-a) when the state index has bit i = site i
    axes = [L - 1 - s for s in sites]
    t = np.moveaxis(t, axes[::-1], range(len(sites)))  # leading index bits: site[-1] is MSB
    shp = t.shape
    t = (M @ t.reshape(1 << len(sites), -1)).reshape(shp)
    t = np.moveaxis(t, range(len(sites)), axes[::-1])
    return np.ascontiguousarray(t).reshape(-1)


def shifts_from_contract(seed, t, S, D, Ts):
    """C5 step 1 from the KAT-pinned block function."""
    key = [seed & 0xFFFFFFFF, seed >> 32]
    sig = []
    Sigma = None
    for k in range(S):
        x = oracle.philox4x32_10([k, t, 0, 3 << 24], key)
        sig.append((int(x[0]) * D) >> 32)
        if k == 0:
            Sigma = (int(x[1]) * Ts) >> 32
    return Sigma, sig


@pytest.mark.parametrize("variant,L,Ts,D,A,sweeps", [
    (wl.PCPD, 16, 16, 8, 2, 3),
    (wl.PCPD, 16, 8, 8, 8, 3),
    (wl.PCPD, 14, 14, 7, 1, 2),
    (wl.TCPD, 18, 18, 9, 3, 3),
    (wl.QCPD, 11, 11, 11, 1, 3),     # right reach 4, smallest legal domain: the single domain always holds the seam
    (wl.QCPD, 22, 22, 11, 11, 1),    # ... and a seam-free domain beside it
    (wl.CPD, 20, 10, 5, 1, 3),       # right reach 1, smallest legal domain, two tiles of two domains
    (wl.CPD, 15, 15, 5, 5, 3),
])
def test_P6_exact_schedule_operator_on_toy_ring(variant, L, Ts, D, A, sweeps):
    d, p, seed = 0.3, 0.2, 1234
    Rr = 1 if variant == wl.CPD else 2 + variant
    n, S, ntiles = Ts // D, D // A, L // Ts
    R = 64 * 12000
    o = oracle.Oracle(L, R, d, p, seed, variant, Ts=Ts, D=D, A=A)
    o.init(wl.INIT_FULL)

    mats = {x: rule_matrix(variant, D, x, d, p) for x in range(1, D - 1 - Rr + 1)}

    def domain_op(c):
        xs = allowed_positions(D, Rr, c)
        one = sum(mats[x] for x in xs) / len(xs)
        return np.linalg.matrix_power(one, A)

    v = np.zeros(1 << L)
    v[(1 << L) - 1] = 1.0

    def marginals(v):
        """P(site i occupied) and P(sites i, i+1 mod L both occupied) for every i (state index bit i = site i,
        i.e. numpy axis L-1-i of the (2,)*L tensor)."""
        t = v.reshape((2,) * L)
        occ, pair = np.zeros(L), np.zeros(L)
        for i in range(L):
            ti = np.take(t, 1, axis=L - 1 - i)                     # axis of site j in ti: L-1-j (j > i), L-2-j (j < i)
            occ[i] = ti.sum()
            j = (i + 1) % L
            pair[i] = np.take(ti, 1, axis=(L - 1 - j) if j > i else (L - 2 - j)).sum()
        return occ, pair

    for t in range(sweeps):
        Sigma, sig = shifts_from_contract(seed, t, S, D, Ts)
        oS, osig = o.shifts(t, S)
        assert oS == Sigma and list(osig) == sig
        for k in range(S):
            for tau in range(ntiles):
                for b in range(n):
                    seam = (D - sig[k]) if (b == n - 1 and sig[k] > 0) else None
                    sites = [(Sigma + tau * Ts + (sig[k] + b * D + x) % Ts) % L for x in range(D)]
                    v = apply_on_sites(v, domain_op(seam), sites, L)
        o.run(1)
        assert abs(v.sum() - 1) < 1e-12
        words = o.get_words()  # [L, W]
        bits = ((words[:, :, None] >> np.arange(64, dtype=np.uint64)) & np.uint64(1)).astype(np.float64)
        # words (not replicas) are the independent samples (reading G12)
        occ_w = bits.mean(axis=2)                                  # [L, W]
        pair_w = (bits * np.roll(bits, -1, axis=0)).mean(axis=2)   # [L, W]
        W = occ_w.shape[1]
        occ_exact, pair_exact = marginals(v)
        for exact, samp in ((occ_exact, occ_w), (pair_exact, pair_w)):
            mean = samp.mean(axis=1)
            err = samp.std(axis=1, ddof=1) / W ** 0.5
            z = (mean - exact) / np.maximum(err, 1e-9)
            assert np.all(np.abs(z) < 4.5), (t, z)


def _translate_avg(v, L):
    """Average of a distribution over all translations of the ring (state index bit i = site i <-> axis L-1-i)."""
    t = v.reshape((2,) * L)
    acc = np.zeros_like(t)
    for s in range(L):
        acc += np.transpose(t, [(a + s) % L for a in range(L)])
    return (acc / L).reshape(-1)


def _density(v, L):
    t = v.reshape((2,) * L)
    return sum(np.take(t, 1, axis=a).sum() for a in range(L)) / L


@pytest.mark.parametrize("L,Ts,D,A", [(14, 14, 7, 1), (16, 16, 8, 2), (16, 8, 8, 2)])
def test_P5_exact_bias_of_the_schedule_on_toy_rings(L, Ts, D, A):
    """How far SD2 is from Algorithm 1, EXACTLY (no Monte Carlo): E[rho] after 1, 2, 3 sweeps from the full ring under
    (i) the literal algorithm - L attempts, each at a uniformly random site - and (ii) SD2(T_s, D, A)
    averaged over its shifts (the sub-step operator averaged over sigma; the tile shift by symmetrising over translations),
    both built from eq. (1)'s reaction list with the machinery of P6.  The schedule is an O(1/D) approximation of the
    random-sequential dynamics, not an exact re-ordering of it: at D = 7 .. 8 the expected density differs by 1 .. 3 parts
    in 10^3, of either sign depending on (T_s, D, A); DESIGN.md section 3 records the values printed here next to the
    Monte Carlo measurement at the production D = 64 (-3.5 parts in 10^4 at early times)."""
    d, p, Rr = 0.5, 0.15, 2
    n, S, ntiles = Ts // D, D // A, L // Ts
    M4 = rule_matrix(wl.PCPD, 4, 1, d, p)            # the rule on sites (i-1, i, i+1, i+2)
    mats = {x: rule_matrix(wl.PCPD, D, x, d, p) for x in range(1, D - 1 - Rr + 1)}

    def domain_op(c):
        xs = allowed_positions(D, Rr, c)
        return np.linalg.matrix_power(sum(mats[x] for x in xs) / len(xs), A)

    ops = {c: domain_op(c) for c in [None] + list(range(1, D))}

    def literal_sweep(v):
        for _ in range(L):
            v = sum(apply_on_sites(v, M4, [(i - 1 + s) % L for s in range(4)], L) for i in range(L)) / L
        return v

    def sd2_sweep(v):
        for _ in range(S):
            acc = np.zeros_like(v)
            for sigma in range(D):
                u = v
                for tau in range(ntiles):
                    for b in range(n):
                        seam = (D - sigma) if (b == n - 1 and sigma > 0) else None
                        u = apply_on_sites(u, ops[seam], [(tau * Ts + (sigma + b * D + x) % Ts) % L for x in range(D)], L)
                acc += u
            v = acc / D
        return _translate_avg(v, L)                  # the tile shift Sigma is uniform and independent from sweep to sweep

    vl = np.zeros(1 << L)
    vl[-1] = 1.0
    vs = vl.copy()
    rel = []
    for _ in range(3):
        vl, vs = literal_sweep(vl), sd2_sweep(vs)
        assert abs(vl.sum() - 1) < 1e-12 and abs(vs.sum() - 1) < 1e-12
        rel.append(_density(vs, L) / _density(vl, L) - 1)
    print(f"exact schedule bias SD2({Ts}, {D}, {A}) on L = {L}: rel =", ["%+.2e" % r for r in rel])
    assert all(1e-5 < abs(r) < 5e-3 for r in rel), rel   # present, and small: O(1/D)


def test_P6_shift_distribution_uniform():
    """sigma_k uniform on [0, D), Sigma uniform on [0, Ts) (mulhi32 of the SHIFT
    block), chi-square over many sweeps."""
    D, Ts, A = 16, 64, 4
    o = oracle.Oracle(128, 64, 0.5, 0.1, 5, 0, Ts=Ts, D=D, A=A)
    cs, cS = np.zeros(D), np.zeros(Ts)
    N = 6000
    for t in range(N):
        Sg, sg = o.shifts(t, D // A)
        cS[Sg] += 1
        for s in sg:
            cs[s] += 1
    chi_s = ((cs - cs.mean()) ** 2 / cs.mean()).sum()
    chi_S = ((cS - cS.mean()) ** 2 / cS.mean()).sum()
    assert chi_s < (D - 1) + 5 * (2 * (D - 1)) ** 0.5
    assert chi_S < (Ts - 1) + 5 * (2 * (Ts - 1)) ** 0.5


# ------------------------------------------------------------------ P5 ----
def _sd2_vs_literal(variant, L, R, d, p, times, sch, seed=7):
    W = R // 64
    o = oracle.Oracle(L, R, d, p, seed, variant, **sch)
    o.init(wl.INIT_FULL)
    sd2 = []
    prev = 0
    for t in times:
        o.run(t - prev)
        prev = t
        sd2.append(o.counts().astype(np.float64).reshape(W, 64).mean(axis=1) / L)  # per word
    sd2 = np.array(sd2)                                                       # [n_t, W]
    lit, _ = oracle.literal_run(variant & 0xff, L, R, d, p, seed + 1000, np.ones((R, L), np.uint8), times)
    lit = lit.astype(np.float64) / L                                          # [n_t, R]
    m_s, e_s = sd2.mean(axis=1), sd2.std(axis=1, ddof=1) / W ** 0.5
    m_l, e_l = lit.mean(axis=1), lit.std(axis=1, ddof=1) / R ** 0.5
    z = (m_s - m_l) / np.sqrt(e_s ** 2 + e_l ** 2)
    rel = m_s / m_l - 1
    return z, rel, m_s, m_l


@pytest.mark.slow
@pytest.mark.parametrize("d,p", [(0.5, 0.15), (0.1, 0.09)])
def test_P5_sd2_matches_literal_alg1(d, p):
    times = [1, 2, 4, 8, 16, 32, 64]
    z, rel, m_s, m_l = _sd2_vs_literal(wl.PCPD, 512, 2048, d, p, times, dict(Ts=2048, D=64, A=4))
    print("P5", d, p, "z =", np.round(z, 2), "rel =", np.round(rel, 4))
    assert np.all(np.abs(z) < 4.0), (z, rel)
    assert np.all(np.abs(rel) < 0.02), rel


@pytest.mark.slow
def test_P5_tcpd_sd2_matches_literal():
    times = [1, 2, 4, 8, 16, 32]
    z, rel, _, _ = _sd2_vs_literal(wl.TCPD, 512, 1024, 0.5, 0.05, times, dict(Ts=2048, D=64, A=4))
    print("P5 tcpd z =", np.round(z, 2), "rel =", np.round(rel, 4))
    assert np.all(np.abs(z) < 4.0), (z, rel)


@pytest.mark.slow
@pytest.mark.parametrize("code", [0, 1, 2, 3])
def test_P5_paper_pmask_sd2_matches_literal(code):
    """The paper's own experiment (rho(t) for different numbers of decorrelation bits; "adding
    decorrelation bits does not help to improve the numerical result", i.e. even the fully correlated mask showed no
    bias) repeated for every member of the mask family of section 4.3 (bounds b = 1/4, 1/2, 1 = no decorrelation, 3/4):
    rho(t) of SD2 with that mask against the literal Algorithm 1, whose draws are independent per replica.  Words are
    the independent samples (reading G12) - with b = 1 the 64 replicas of a word annihilate in unison, which makes the
    word means noisier, not biased."""
    times = [1, 2, 4, 8, 16, 32, 64]
    variant = wl.PCPD | oracle.PMASK_PAPER | (code << oracle.PMASK_BOUND_SHIFT)
    z, rel, _, _ = _sd2_vs_literal(variant, 512, 4096, 0.5, 0.15, times, dict(Ts=2048, D=64, A=4))
    print(f"P5 paper-pmask b = {oracle.PMASK_BOUNDS[code]} z =", np.round(z, 2), "rel =", np.round(rel, 4))
    assert np.all(np.abs(z) < 4.0), (z, rel)
    assert np.all(np.abs(rel) < 0.02), rel


@pytest.mark.slow
def test_P5_qcpd_sd2_matches_literal():
    times = [1, 2, 4, 8, 16, 32]
    z, rel, _, _ = _sd2_vs_literal(wl.QCPD, 512, 1024, 0.5, 0.03, times, dict(Ts=2048, D=64, A=4))
    print("P5 qcpd z =", np.round(z, 2), "rel =", np.round(rel, 4))
    assert np.all(np.abs(z) < 4.0), (z, rel)


@pytest.mark.slow
def test_P5_connected_lattice_matches_literal_on_the_long_ring():
    """Connected multispin lattice: one word column = one ring of 64 L sites.  Its
    density decay must agree with the literal Algorithm 1 run on a ring of that length (the paper:
    "we found no bias" when the sites of a register are L apart).  Words / rings are the samples."""
    L, W = 256, 32
    times = [1, 2, 4, 8, 16, 32, 64]
    o = oracle.Oracle(L, 64 * W, 0.5, 0.15, 9, wl.PCPD | oracle.CONNECTED, Ts=256, D=64, A=4)
    o.init(wl.INIT_FULL)
    sd2, prev = [], 0
    for t in times:
        o.run(t - prev)
        prev = t
        sd2.append(o.counts().astype(np.float64).reshape(W, 64).sum(axis=1) / (64 * L))
    sd2 = np.array(sd2)
    lit, _ = oracle.literal_run(wl.PCPD, 64 * L, W, 0.5, 0.15, 1009, np.ones((W, 64 * L), np.uint8), times)
    lit = lit.astype(np.float64) / (64 * L)
    m_s, e_s = sd2.mean(axis=1), sd2.std(axis=1, ddof=1) / W ** 0.5
    m_l, e_l = lit.mean(axis=1), lit.std(axis=1, ddof=1) / W ** 0.5
    z = (m_s - m_l) / np.sqrt(e_s ** 2 + e_l ** 2)
    rel = m_s / m_l - 1
    print("P5 connected z =", np.round(z, 2), "rel =", np.round(rel, 4))
    assert np.all(np.abs(z) < 4.0), (z, rel)
    assert np.all(np.abs(rel) < 0.02), rel


def high_statistics_bias(R, seed, D=64, A=4, Ts=2048, L=4096, d=0.5, p=0.15, times=(1, 2, 4, 8, 16, 32, 64, 128, 256)):
    """SD2(Ts, D, A) against the literal Algorithm 1, R replicas on each side, full start: relative
    deviation of the mean density, its standard error (words are the samples on the SD2 side, reading G12) and z, per
    record time.  One oracle thread per chunk of word columns / replicas."""
    from concurrent.futures import ThreadPoolExecutor

    W = R // 64
    times = list(times)
    nthr = max(1, min(os.cpu_count() or 1, 16))

    def sd2(words):
        o = oracle.Oracle(L, R, d, p, seed, wl.PCPD, Ts=Ts, D=D, A=A, words=list(words))
        o.init(wl.INIT_FULL)
        out, prev = [], 0
        for t in times:
            o.run(t - prev)
            prev = t
            out.append(o.counts().astype(np.float64).reshape(len(words), 64).mean(axis=1) / L)
        return np.array(out)                                   # [n_t, len(words)]

    def lit(chunk):
        r0, r1 = chunk
        c, _ = oracle.literal_run(wl.PCPD, L, r1 - r0, d, p, 1000 * seed + 7 + r0, np.ones((r1 - r0, L), np.uint8), times)
        return c.astype(np.float64) / L                        # [n_t, r1-r0]

    wchunks = np.array_split(np.arange(W), 4 * nthr)
    rchunks = [(int(a[0]) * 64, (int(a[-1]) + 1) * 64) for a in wchunks]
    with ThreadPoolExecutor(nthr) as ex:
        s = np.concatenate(list(ex.map(sd2, wchunks)), axis=1)     # [n_t, W]   words are the samples (G12)
        l = np.concatenate(list(ex.map(lit, rchunks)), axis=1)     # [n_t, R]
    m_s, e_s = s.mean(axis=1), s.std(axis=1, ddof=1) / W ** 0.5
    m_l, e_l = l.mean(axis=1), l.std(axis=1, ddof=1) / R ** 0.5
    z = (m_s - m_l) / np.sqrt(e_s ** 2 + e_l ** 2)
    rel = m_s / m_l - 1
    err = np.sqrt(e_s ** 2 + e_l ** 2) / m_l
    return times, rel, err, z


@pytest.mark.skipif(os.environ.get("PCPD_LONG_PARITY") != "1", reason="high-statistics bias run (minutes of CPU): set PCPD_LONG_PARITY=1")
def test_P5_high_statistics_bias_of_the_default_schedule():
    """The paper's own validation of a parallel schedule at higher statistics: SD2(2048, D, A)
    in its production shape against the literal Algorithm 1, t <= 256.  PCPD_P5_R replicas on each side (default
    8192), seed PCPD_P5_SEED (default 7), schedule PCPD_P5_D / PCPD_P5_A (default 64 / 4; the paper's "vary the
    work-group size" check).  Prints the relative deviation, its error and z (the numbers DESIGN.md section 3 records).
    At R = 32768 the schedule's O(1/D) bias is resolved (-3.5e-4 at t <= 4 for D = 64, z ~ -6; exact on toy rings:
    test_P5_exact_bias_of_the_schedule_on_toy_rings), so z is reported, not asserted; asserted is the documented bound
    |rel| < 1e-3 at t <= 8 and |rel| < 5e-3 everywhere."""
    R = int(os.environ.get("PCPD_P5_R", "8192"))
    seed = int(os.environ.get("PCPD_P5_SEED", "7"))
    D, A = int(os.environ.get("PCPD_P5_D", "64")), int(os.environ.get("PCPD_P5_A", "4"))
    times, rel, err, z = high_statistics_bias(R, seed, D=D, A=A)
    print(f"P5 high statistics: R = {R} per side, seed {seed}, SD2(2048, {D}, {A}); t =", times)
    print("  rel =", np.round(rel, 5))
    print("  +/- =", np.round(err, 5))
    print("  z   =", np.round(z, 2))
    early = np.array(times) <= 8
    assert np.all(np.abs(rel[early]) < 1e-3 + 4 * err[early]) and np.all(np.abs(rel) < 0.005), (z, rel)


@pytest.mark.slow
def test_P5_cpd_sd2_matches_literal():
    times = [1, 2, 4, 8, 16, 32]
    z, rel, _, _ = _sd2_vs_literal(wl.CPD, 512, 1024, 0.5, 0.3, times, dict(Ts=2048, D=64, A=4))
    print("P5 cpd z =", np.round(z, 2), "rel =", np.round(rel, 4))
    assert np.all(np.abs(z) < 4.0), (z, rel)
