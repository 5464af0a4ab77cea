"""Seeded, synthetic workload descriptions shared by the oracle tests, the GPU
parity tests and bench.py.

This module holds NONE of the method's arithmetic (no Philox, no thresholds, no
update rule, no schedule): only the parameters of BASELINE.json's five configs,
the harness-side record times (SURVEY.md §8(b) "Harness-level"), and numpy-seeded
hand-built lattices used as *inputs* to both sides.  Neither ``oracle/`` nor
``paper_1301_6082_b200/`` imports the other; both may be driven from here.

The paper runs PCPD at L = 2^18, p near p_c(d), N ~ 10^3 runs;
the configs keep that structure (power-of-two periodic rings, p near criticality
for the given d, many replicas).  No dataset stands behind them: (L, R, d, p,
init rule, seed, sweeps) determine every bit.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

PCPD = 0  # AA0/0AA->AAA, AA->00, A0<->0A   (eq. (1))
CONNECTED = 0x200    # variant flag: the paper's connected multispin lattice
PMASK_PAPER = 0x100  # variant flag: the paper's own partially correlated annihilation mask
PMASK_BOUND_HALF, PMASK_BOUND_ONE, PMASK_BOUND_3_4 = 0x400, 0x800, 0xC00   # with PMASK_PAPER: its decorrelation bound b
TCPD = 1  # AAA0/0AAA->AAAA, AAA->000, A0<->0A (BASELINE.json config 5)

QCPD = 2  # AAAA0/0AAAA->AAAAA, AAAA->0000, A0<->0A (PAPER.md:21 names it; rule by analogy with Alg. 1)
CPD = 3   # A0/0A->AA, A->0, A0<->0A: contact process with diffusion (DP class; reading of PAPER.md:15,21)

INIT_FULL = 0       # all sites occupied
INIT_BERNOULLI = 1  # i.i.d. Bernoulli(1/2) per site per replica from the handle's seed
INIT_EMPTY = 2      # absorbing state, for tests


@dataclasses.dataclass(frozen=True)
class Config:
    name: str
    variant: int
    L: int
    n_replicas: int
    d: float
    p: float
    init: int
    seed: int
    sweeps: int
    record: str  # "every" | "log20"

    @property
    def W(self) -> int:
        return self.n_replicas // 64

    @property
    def lattice_bytes(self) -> int:
        return 8 * self.L * self.W


# BASELINE.json "configs", in order.  configs[3] (index 3, "cfg4") is the one the
# metric is quoted on (L = 2^22 x 2048 replicas, 1 GiB lattice).
CONFIGS = (
    Config("cfg1", PCPD, 1024, 64, 0.5, 0.15, INIT_FULL, 1, 1000, "every"),
    Config("cfg2", PCPD, 65536, 256, 0.1, 0.09, INIT_BERNOULLI, 2, 10_000, "log20"),
    Config("cfg3", PCPD, 1 << 20, 2048, 0.5, 0.152, INIT_FULL, 3, 10_000, "log20"),
    Config("cfg4", PCPD, 1 << 22, 2048, 0.8, 0.12, INIT_FULL, 4, 2000, "log20"),
    Config("cfg5", TCPD, 1 << 20, 1024, 0.5, 0.05, INIT_FULL, 5, 10_000, "log20"),
)
# Not a BASELINE.json config: cfg4's size with the paper's own mask generation (next-row f2, DESIGN.md
# section 10): dyadic d = 3/4 (the paper's AND/OR recipe) and the partially correlated
# annihilation mask, p < 1/4.  `bench.py --config cfg4p` measures it.
EXTRA_CONFIGS = (
    Config("cfg4p", PCPD | PMASK_PAPER, 1 << 22, 2048, 0.75, 0.12, INIT_FULL, 4, 2000, "log20"),
)
BY_NAME = {c.name: c for c in CONFIGS + EXTRA_CONFIGS}


def record_times(n_sweeps: int, per_decade: int = 20) -> list[int]:
    """Log-spaced record times: the distinct integers
    floor(10^(k/per_decade) + 0.5), k = 0 .. per_decade*log10(n), plus 0 and n.
    Computed once in the harness and used for both sides, so no cross-platform
    pow() issue can creep into a parity comparison."""
    if n_sweeps <= 0:
        return [0]
    ts = {0, n_sweeps}
    k = 0
    while True:
        t = int(math.floor(10.0 ** (k / per_decade) + 0.5))
        if t > n_sweeps:
            break
        ts.add(t)
        k += 1
    return sorted(ts)


def random_lattice_words(L: int, W: int, density: float, seed: int) -> np.ndarray:
    """Hand-built input state: uint64[L, W], every bit i.i.d. Bernoulli(density)
    from numpy's PCG64 (NOT the method's generator) - an arbitrary lattice to
    feed pcpd_set_lattice / the oracle's set_words."""
    rng = np.random.Generator(np.random.PCG64(seed))
    bits = rng.random((L, W, 64)) < density
    weights = (np.uint64(1) << np.arange(64, dtype=np.uint64))
    return (bits.astype(np.uint64) * weights).sum(axis=2, dtype=np.uint64)


def isolated_particles_words(L: int, W: int, spacing: int, seed: int) -> np.ndarray:
    """uint64[L, W] with, in every replica, particles at least `spacing` sites
    apart (no adjacent pairs): per replica a random offset, then one particle
    every `spacing` sites."""
    rng = np.random.Generator(np.random.PCG64(seed))
    out = np.zeros((L, W), dtype=np.uint64)
    assert spacing >= 2 and L % spacing == 0
    for w in range(W):
        for j in range(64):
            off = int(rng.integers(0, spacing))
            out[off::spacing, w] |= np.uint64(1) << np.uint64(j)
    return out
