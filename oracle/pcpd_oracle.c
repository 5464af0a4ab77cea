/*
 * pcpd_oracle.c - plain, slow, obviously-correct CPU implementation of the
 * multispin PCPD/TCPD Monte Carlo hot path of arXiv 1301.6082 (Schram).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may build, load or call it.  It shares no code, header, table or helper with
 * paper_1301_6082_b200/csrc/ and includes nothing from it.
 *
 * Representation: ONE BYTE per site per replica, q[r*L + i] in {0,1}; ordinary
 * `if`s per replica; every Bernoulli draw is made the slow way: the lane's
 * 32-bit uniform U_j is assembled bit by bit from 32 random planes and compared
 * with `<` against the threshold.  No bit-slicing, no lazy evaluation, no
 * blocking or fusion.  Citations: PAPER.md = /root/reference/PAPER.md,
 * SURVEY.md section 8(c) items C1..C9 = the contract ("readings") restated in
 * DESIGN.md.
 *
 * Pins (tests/test_oracle_pins.py, all `-m "not gpu"`):
 *   oracle_philox4x32_10      P0  known-answer vectors (Salmon et al. SC'11)
 *   oracle_lane_uniforms/mask P0' frequency + exhaustive reduced-K compare
 *   oracle_rule_pcpd/_tcpd    P1-P4 absorbing state, d=1 conservation,
 *                                 isolated particles, master-equation enumeration
 *                                 of eq. (1) on rings L<=6
 *   oracle_literal_*          P4  exact E[rho] from the master equation
 *   oracle_paper_pmask(_bound), oracle_pmask_gate_threshold
 *                             P9  the paper's own annihilation masks (Alg. 2 l.12-13 and the
 *                                 family of section 4.3, bounds b = 1/4, 1/2, 1, 3/4): lane
 *                                 probability p, word-wide gate p/b, lanes independent b-bits
 *                                 given the gate, pair probability p b; P5 bias check vs literal
 *                                 Alg. 1 for every bound (the paper's "number of decorrelation bits")
 *   oracle_set_word_probabilities  P11 column k of a per-word run == column k of the uniform
 *                                 run with (d_k, p_k), bit for bit
 *   oracle_run (schedule SD2) P5  vs literal Alg. 1 (statistical), P6 exact toy
 *                                 operator (all four rules), P7 run splitting / loop
 *                                 order / word subsets
 *   oracle_counts / oracle_pair_counts  P7  numpy column popcounts incl. the ring closure
 *                                 (independent lanes: site L-1 -> 0; connected lattice:
 *                                 the unrolled ring of 64 L sites)
 *   planes_needed / oracle_stats  P12 brute-force "first differing plane" per lane from the
 *                                 pinned lane uniforms; closed form sum_m [1-(1-4^-m)^64]
 * Parity status: every function pinned; the *numerical values* of rho(t) at the
 * five configs are "parity unpinned by the paper" (it prints none).
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <math.h>

/* ------------------------------------------------------------------ C1 --- */
/* Philox-4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11; public algorithm).
 * multipliers M0, M1; Weyl key increments W0, W1; round:
 * (hi0,lo0) = M0*c0, (hi1,lo1) = M1*c2;
 * (c0,c1,c2,c3) <- (hi1^c1^k0, lo1, hi0^c3^k1, lo0); key bumped after each of
 * the first 9 rounds; 10 rounds. */
void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    const uint64_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
    const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = M0 * (uint64_t)c0;
        uint64_t p1 = M1 * (uint64_t)c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        if (round < 9) { k0 += W0; k1 += W1; }
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* ------------------------------------------------------------------ C2 --- */
/* Addressing: key = (seed low, seed high); counter = (slot, sweep, word,
 * stream<<24 | m).  Streams (C2): */
enum { STREAM_MISC = 0, STREAM_DIFF = 1, STREAM_ANNI = 2, STREAM_SHIFT = 3,
       STREAM_INIT = 4, STREAM_LITERAL = 5 /* oracle-only, literal Alg. 1 */ };

static void block(uint64_t seed, uint32_t slot, uint32_t sweep, uint32_t word,
                  uint32_t stream, uint32_t m, uint32_t x[4])
{
    uint32_t ctr[4] = { slot, sweep, word, (stream << 24) | m };
    uint32_t key[2] = { (uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32) };
    oracle_philox4x32_10(ctr, key, x);
}

/* mulhi32(r, n) = floor(r * n / 2^32): integer form of Alg. 1's floor(L*RNG()),
 * PAPER.md:52. */
static uint32_t mulhi32(uint32_t r, uint32_t n)
{
    return (uint32_t)(((uint64_t)r * (uint64_t)n) >> 32);
}

/* ------------------------------------------------------------------ C3 --- */
/* T = floor(q * 2^32) in double arithmetic; q = 1 -> 2^32.  Returns
 * UINT64_MAX for q outside [0,1] or NaN. */
uint64_t oracle_threshold(double q)
{
    if (!(q >= 0.0 && q <= 1.0)) return UINT64_MAX;
    return (uint64_t)floor(ldexp(q, 32));
}

/* The 64 lane uniforms of stream `stream` at (slot, sweep, word), resolution K
 * (K = 32 in the contract; smaller K only for the exhaustive pin P0').
 * Plane k (k = 0 most significant) = `lo` (k even) or `hi` (k odd) of block
 * m = k>>1, lo = x0 | x1<<32, hi = x2 | x3<<32.
 * U_j = sum_k bit_j(plane_k) * 2^(K-1-k). */
void oracle_lane_uniforms(uint64_t seed, uint32_t slot, uint32_t sweep, uint32_t word,
                          uint32_t stream, int K, uint32_t U[64])
{
    uint64_t plane[32];
    uint64_t lo = 0, hi = 0;
    for (int k = 0; k < K; ++k) {
        if ((k & 1) == 0) {                     /* a new block every 2 planes */
            uint32_t x[4];
            block(seed, slot, sweep, word, stream, (uint32_t)(k >> 1), x);
            lo = (uint64_t)x[0] | ((uint64_t)x[1] << 32);
            hi = (uint64_t)x[2] | ((uint64_t)x[3] << 32);
        }
        plane[k] = (k & 1) ? hi : lo;
    }
    for (int j = 0; j < 64; ++j) {
        uint32_t u = 0;
        for (int k = 0; k < K; ++k)
            if ((plane[k] >> j) & 1u) u += (uint32_t)1 << (K - 1 - k);
        U[j] = u;
    }
}

/* Instrumentation only (SURVEY.md 8(d) "lazy-needed count"): number of planes
 * that had to be looked at, most significant first, until every one of the 64
 * lanes is decided against the 32-bit threshold T (a lane is decided at the
 * first plane where its bit differs from T's bit; planes below T's lowest set
 * bit can never matter).  Does not influence any result. */
static int planes_needed(const uint32_t U[64], uint64_t T)
{
    if (T == 0 || T >= ((uint64_t)1 << 32)) return 0;
    uint32_t t = (uint32_t)T;
    int nq = 32 - __builtin_ctz(t);        /* planes that can matter at all */
    int need = 0;
    for (int j = 0; j < 64; ++j) {
        uint32_t diff = U[j] ^ t;
        int first = diff ? __builtin_clz(diff) + 1 : 32;  /* 1-based plane count */
        if (first > nq) first = nq;
        if (first > need) need = first;
    }
    return need;
}

/* mask lane j = [U_j < T] (strict, as Alg. 1's `r < d`). */
static void bernoulli_lanes(uint64_t seed, uint32_t slot, uint32_t sweep, uint32_t word,
                            uint32_t stream, uint64_t T, uint8_t mask[64], int *need)
{
    uint32_t U[64];
    oracle_lane_uniforms(seed, slot, sweep, word, stream, 32, U);
    for (int j = 0; j < 64; ++j) mask[j] = ((uint64_t)U[j] < T) ? 1 : 0;
    if (need) *need = planes_needed(U, T);
}

/* C4' - the paper's own annihilation masks (Alg. 2 lines 12-13; section 4.3,
 * PAPER.md:157-161), next-row f2 of SURVEY.md 8(f).  The family, in the paper's words: "all N_r bits are
 * set to 1 with probability p and all 0 otherwise ... fully correlated" (bound b = 1, no
 * decorrelation bits); then the decorrelation step: per-lane independent bits that are 1 w.p. b, ANDed
 * with ONE word-wide draw that is 1 w.p. p/b - Alg. 2's "aMask := RNG() and RNG()" gives b = 1/4
 * ("(RNG() < 4p) ? 1 : 0 ... gives either 1 or 0 equally for all N_r bits"); "in the
 * case of the bound p < 3/4, we would generate uncorrelated bits with a probability of 3/4 to be 1,
 * and use the AND operation with correlated bits that are one with probability 4p/3";
 * one raw word alone gives b = 1/2.  bound code: 0: b = 1/4 (lo AND hi), 1: b = 1/2 (lo), 2: b = 1
 * (all lanes), 3: b = 3/4 (lo OR hi), lo / hi = the two planes of ANNI block 0; the word-wide uniform
 * is x3 of the MISC block (unused by C4), compared as a 32-bit integer with Tg = floor((p/b) 2^32).
 * Lane j of the mask = dec_j and [x3 < Tg]: probability b Tg / 2^32 ~ p per lane, two lanes both set
 * w.p. b^2 Tg / 2^32 ~ p b.  Requires p < b. */
static const double PMASK_BOUND[4] = { 0.25, 0.5, 1.0, 0.75 };

/* Tg = floor((p / b) 2^32) for bound code c: the quotient p/b is formed in double the way the paper
 * writes it - 4p, 2p, p, 4p/3 - then C3's floor.  UINT64_MAX for an invalid code or p >= b. */
uint64_t oracle_pmask_gate_threshold(double p, int code)
{
    if (code < 0 || code > 3 || !(p >= 0.0 && p < PMASK_BOUND[code])) return UINT64_MAX;
    double q = code == 0 ? 4.0 * p : code == 1 ? 2.0 * p : code == 2 ? p : 4.0 * p / 3.0;
    return oracle_threshold(q);
}

void oracle_paper_pmask_bound(uint64_t seed, uint32_t slot, uint32_t sweep, uint32_t word,
                              uint64_t Tg, int code, uint8_t mask[64])
{
    uint32_t a[4], misc[4];
    block(seed, slot, sweep, word, STREAM_ANNI, 0, a);
    block(seed, slot, sweep, word, STREAM_MISC, 0, misc);
    uint64_t lo = (uint64_t)a[0] | ((uint64_t)a[1] << 32);
    uint64_t hi = (uint64_t)a[2] | ((uint64_t)a[3] << 32);
    int gate = ((uint64_t)misc[3] < Tg) ? 1 : 0;
    for (int j = 0; j < 64; ++j) {
        int l = (int)((lo >> j) & 1u), h = (int)((hi >> j) & 1u);
        int dec = code == 0 ? (l && h) : code == 1 ? l : code == 2 ? 1 : (l || h);
        mask[j] = (uint8_t)(dec && gate);
    }
}

/* Alg. 2's own form (b = 1/4), T4p = floor(4p 2^32). */
void oracle_paper_pmask(uint64_t seed, uint32_t slot, uint32_t sweep, uint32_t word,
                        uint64_t T4p, uint8_t mask[64])
{
    oracle_paper_pmask_bound(seed, slot, sweep, word, T4p, 0, mask);
}

void oracle_bernoulli_mask(uint64_t seed, uint32_t slot, uint32_t sweep, uint32_t word,
                           uint32_t stream, uint64_t T, uint8_t mask[64])
{
    bernoulli_lanes(seed, slot, sweep, word, stream, T, mask, NULL);
}

/* ------------------------------------------------------------------ C6 --- */
/* One attempted update of ONE replica at pair position x (sites given by
 * pointer so the caller does the index mapping).  Alg. 1, with
 * the readings G1 (annihilate with prob. p, ELSE fission), G3 (diffusion test
 * first, unconditional swap), G4 (fission ORs the target bit):
 *   if r1<d: swap(q_x, q_x+1)
 *   else if q_x and q_x+1: if r2<p: both := 0
 *                          else if r3<1/2: q_x-1 := 1 else q_x+2 := 1        */
void oracle_rule_pcpd(uint8_t *qm1, uint8_t *q0, uint8_t *q1, uint8_t *q2,
                      int Dm, int Pm, int Fm)
{
    if (Dm) {
        uint8_t tmp = *q0; *q0 = *q1; *q1 = tmp;          /* diffusion */
    } else if (*q0 == 1 && *q1 == 1) {
        if (Pm) { *q0 = 0; *q1 = 0; }                      /* annihilation */
        else if (Fm) { *qm1 = 1; }                         /* fission low  */
        else { *q2 = 1; }                                  /* fission high */
    }
}

/* TCPD (BASELINE.json config 5; reading G15): AAA0/0AAA -> AAAA each at rate
 * (1-p)(1-d)/2, AAA -> 000 at rate p(1-d), A0 <-> 0A at rate d; footprint
 * {x-1 .. x+3}; diffusion still swaps (x, x+1). */
void oracle_rule_tcpd(uint8_t *qm1, uint8_t *q0, uint8_t *q1, uint8_t *q2, uint8_t *q3,
                      int Dm, int Pm, int Fm)
{
    if (Dm) {
        uint8_t tmp = *q0; *q0 = *q1; *q1 = tmp;
    } else if (*q0 == 1 && *q1 == 1 && *q2 == 1) {
        if (Pm) { *q0 = 0; *q1 = 0; *q2 = 0; }
        else if (Fm) { *qm1 = 1; }
        else { *q3 = 1; }
    }
}

/* QCPD, the quadruplet contact process with diffusion the paper names as a further model the
 * algorithm extends to (next-row f4 of SURVEY.md 8(f)), by the same analogy with
 * Alg. 1 as TCPD (reading G15): AAAA0/0AAAA -> AAAAA each at rate (1-p)(1-d)/2, AAAA -> 0000 at
 * rate p(1-d), A0 <-> 0A at rate d; footprint {x-1 .. x+4}; diffusion still swaps (x, x+1). */
void oracle_rule_qcpd(uint8_t *qm1, uint8_t *q0, uint8_t *q1, uint8_t *q2, uint8_t *q3, uint8_t *q4,
                      int Dm, int Pm, int Fm)
{
    if (Dm) {
        uint8_t tmp = *q0; *q0 = *q1; *q1 = tmp;
    } else if (*q0 == 1 && *q1 == 1 && *q2 == 1 && *q3 == 1) {
        if (Pm) { *q0 = 0; *q1 = 0; *q2 = 0; *q3 = 0; }
        else if (Fm) { *qm1 = 1; }
        else { *q4 = 1; }
    }
}

/* CPD, the contact process with diffusion: the one-particle member of the family PCPD (pairs),
 * TCPD (triples), QCPD (quadruplets), which is in the directed-percolation class - this build's
 * reading of the "DP" model the paper says the algorithm extends to (it prints no
 * rule; next-row f4 of SURVEY.md 8(f)).  By the same analogy with Alg. 1: A0/0A -> AA each at rate
 * (1-p)(1-d)/2, A -> 0 at rate p(1-d), A0 <-> 0A at rate d; footprint {x-1, x, x+1}; diffusion
 * swaps (x, x+1); the fission-high target x+1 is the swap partner's site. */
void oracle_rule_cpd(uint8_t *qm1, uint8_t *q0, uint8_t *q1, int Dm, int Pm, int Fm)
{
    if (Dm) {
        uint8_t tmp = *q0; *q0 = *q1; *q1 = tmp;
    } else if (*q0 == 1) {
        if (Pm) { *q0 = 0; }
        else if (Fm) { *qm1 = 1; }
        else { *q1 = 1; }
    }
}

/* Single attempt on a periodic ring of L sites at site i (literal indexing,
 * reading G2: indices mod L).  Exposed for the master-equation pin P4. */
void oracle_single_attempt(int variant, uint32_t L, uint8_t *q, uint32_t i,
                           int Dm, int Pm, int Fm)
{
    uint32_t im1 = (i + L - 1) % L, i1 = (i + 1) % L, i2 = (i + 2) % L, i3 = (i + 3) % L, i4 = (i + 4) % L;
    if (variant == 3)      oracle_rule_cpd(&q[im1], &q[i], &q[i1], Dm, Pm, Fm);
    else if (variant == 0) oracle_rule_pcpd(&q[im1], &q[i], &q[i1], &q[i2], Dm, Pm, Fm);
    else if (variant == 1) oracle_rule_tcpd(&q[im1], &q[i], &q[i1], &q[i2], &q[i3], Dm, Pm, Fm);
    else                   oracle_rule_qcpd(&q[im1], &q[i], &q[i1], &q[i2], &q[i3], &q[i4], Dm, Pm, Fm);
}

/* --------------------------------------------------------------- handle --- */
typedef struct oracle_t {
    uint32_t L, Ts, D, A;
    int variant;               /* 0 PCPD, 1 TCPD, 2 QCPD, 3 CPD (contact process with diffusion) */
    int pmask_paper;           /* 1: the paper's own annihilation mask (C4', above) */
    int pmask_code;            /*    its bound code: 0 b = 1/4, 1 b = 1/2, 2 b = 1, 3 b = 3/4 */
    int connected;             /* 1: the paper's connected multispin lattice (C10, below) */
    uint64_t Td, Tp, T4p;
    uint64_t *Td_w, *Tp_w;     /* per simulated word column (index k): thresholds in force (C11) */
    uint64_t seed;
    uint32_t sweep;            /* C7: state = lattice + sweep counter */
    uint32_t nwords;           /* word columns simulated (subset of the full run) */
    uint32_t *words;           /* their global word indices w */
    uint8_t *q;                /* q[(k*64 + j)*L + i], k = index into words[] */
    int reverse_order;         /* P7: loop (tile, domain, word) backwards */
    /* instrumentation */
    uint64_t n_attempt_words;
    uint64_t planes_needed_D, planes_needed_P;   /* sums over attempt-words */
    uint64_t blocks_needed_D, blocks_needed_P;   /* sums of ceil(planes/2)  */
} oracle_t;

/* Ts is clamped to L when L < Ts (C5).  Returns NULL on invalid arguments:
 * D | Ts | L, A | D, D >= 2*Rr+3 (reading G18), d,p in [0,1], L < 2^32. */
oracle_t *oracle_create(uint64_t L, double d, double p, uint64_t seed, int variant,
                        uint32_t Ts, uint32_t D, uint32_t A,
                        uint32_t nwords, const uint32_t *words)
{
    /* variant = base | ORACLE_PMASK_PAPER (0x100): base 0 PCPD / 1 TCPD / 2 QCPD / 3 CPD; the flag selects the
     * paper's partially correlated annihilation mask; bits 10-11 (0x400, 0x800) give
     * its bound code (0: b = 1/4 as in Alg. 2; 1: 1/2; 2: 1; 3: 3/4), which needs p < b. */
    int pmask_paper = (variant & 0x100) ? 1 : 0;
    int pmask_code = (variant >> 10) & 3;
    /* | ORACLE_CONNECTED (0x200): the paper's connected multispin lattice, C10. */
    int connected = (variant & 0x200) ? 1 : 0;
    variant &= ~0xF00;
    if (variant < 0 || variant > 3) return NULL;
    if (!pmask_paper && pmask_code) return NULL;
    if (pmask_paper && oracle_pmask_gate_threshold(p, pmask_code) == UINT64_MAX) return NULL;
    uint32_t Rr = variant == 3 ? 1u : 2u + (uint32_t)variant;   /* right reach: 2 PCPD, 3 TCPD, 4 QCPD, 1 CPD */
    if (L == 0 || L >= ((uint64_t)1 << 32) || nwords == 0) return NULL;
    if (Ts > L) Ts = (uint32_t)L;
    if (D == 0 || A == 0 || Ts == 0) return NULL;
    if (Ts % D || L % Ts || D % A) return NULL;
    if (D < 2 * Rr + 3) return NULL;
    uint64_t Td = oracle_threshold(d), Tp = oracle_threshold(p);
    if (Td == UINT64_MAX || Tp == UINT64_MAX) return NULL;
    oracle_t *o = (oracle_t *)calloc(1, sizeof *o);
    if (!o) return NULL;
    o->L = (uint32_t)L; o->Ts = Ts; o->D = D; o->A = A; o->variant = variant;
    o->pmask_paper = pmask_paper;
    o->pmask_code = pmask_code;
    o->connected = connected;
    o->T4p = pmask_paper ? oracle_pmask_gate_threshold(p, pmask_code) : 0;   /* floor((p/b) 2^32) < 2^32 since p < b */
    o->Td = Td; o->Tp = Tp; o->seed = seed; o->sweep = 0; o->nwords = nwords;
    o->words = (uint32_t *)malloc(sizeof(uint32_t) * nwords);
    o->Td_w = (uint64_t *)malloc(sizeof(uint64_t) * nwords);
    o->Tp_w = (uint64_t *)malloc(sizeof(uint64_t) * nwords);
    if (o->Td_w && o->Tp_w)
        for (uint32_t k = 0; k < nwords; ++k) { o->Td_w[k] = Td; o->Tp_w[k] = Tp; }
    o->q = (uint8_t *)calloc((size_t)nwords * 64 * (size_t)L, 1);
    if (!o->words || !o->q || !o->Td_w || !o->Tp_w) {
        free(o->words); free(o->q); free(o->Td_w); free(o->Tp_w); free(o); return NULL;
    }
    memcpy(o->words, words, sizeof(uint32_t) * nwords);
    return o;
}

void oracle_destroy(oracle_t *o)
{
    if (!o) return;
    free(o->words); free(o->q); free(o->Td_w); free(o->Tp_w); free(o);
}

void oracle_set_reverse_order(oracle_t *o, int rev) { o->reverse_order = rev; }
uint32_t oracle_sweep(const oracle_t *o) { return o->sweep; }
void oracle_set_sweep(oracle_t *o, uint32_t t) { o->sweep = t; }
void oracle_thresholds(const oracle_t *o, uint64_t *Td, uint64_t *Tp) { *Td = o->Td; *Tp = o->Tp; }

/* C11 - per-word-column probabilities (next-row f4 of SURVEY.md 8(f): one run scans p across p_c,
 * the paper's production use is many runs per p value): simulated column k uses
 * d_k, p_k, i.e. thresholds floor(d_k 2^32), floor(p_k 2^32); everything else (schedule, streams,
 * keyed by the global word index) is unchanged, so column k evolves exactly as it would in a
 * uniform run with (d_k, p_k).  Not available with the paper's annihilation mask.  Returns -1 on
 * invalid arguments. */
int oracle_set_word_probabilities(oracle_t *o, uint32_t k, double d, double p)
{
    if (!o || k >= o->nwords || o->pmask_paper) return -1;
    uint64_t Td = oracle_threshold(d), Tp = oracle_threshold(p);
    if (Td == UINT64_MAX || Tp == UINT64_MAX) return -1;
    o->Td_w[k] = Td; o->Tp_w[k] = Tp;
    return 0;
}

void oracle_stats(const oracle_t *o, uint64_t out[5])
{
    out[0] = o->n_attempt_words;
    out[1] = o->planes_needed_D; out[2] = o->planes_needed_P;
    out[3] = o->blocks_needed_D; out[4] = o->blocks_needed_P;
}

/* ------------------------------------------------------------------ C8 --- */
/* mode 0: all ones; mode 1: word(i,w) = `lo` of block (c0=i, c1=0, c2=w,
 * c3 = INIT<<24), bit j -> replica 64w+j; mode 2: empty.  Resets sweep to 0. */
int oracle_init(oracle_t *o, int mode)
{
    if (mode < 0 || mode > 2) return -1;
    for (uint32_t k = 0; k < o->nwords; ++k) {
        uint32_t w = o->words[k];
        for (uint32_t i = 0; i < o->L; ++i) {
            uint64_t word;
            if (mode == 0) word = ~(uint64_t)0;
            else if (mode == 2) word = 0;
            else {
                uint32_t x[4];
                block(o->seed, i, 0, w, STREAM_INIT, 0, x);
                word = (uint64_t)x[0] | ((uint64_t)x[1] << 32);
            }
            for (int j = 0; j < 64; ++j)
                o->q[((size_t)k * 64 + j) * o->L + i] = (uint8_t)((word >> j) & 1u);
        }
    }
    o->sweep = 0;
    return 0;
}

/* ------------------------------------------------------------------ C5 --- */
/* One attempt of (tile tau, domain b, word index k) in sub-step ks: slot g,
 * position x from the MISC block, masks Dm/Pm/Fm per lane, rule C6 per
 * replica. */
static void attempt(oracle_t *o, uint32_t t, uint32_t Sigma, uint32_t sigma,
                    uint32_t tau, uint32_t b, uint32_t k, uint32_t g)
{
    const uint32_t L = o->L, Ts = o->Ts, D = o->D;
    const uint32_t n = Ts / D;
    const uint32_t Rr = o->variant == 3 ? 1u : 2u + (uint32_t)o->variant;
    const uint32_t w = o->words[k];

    /* C5 step 3-4: only domain n-1 with sigma > 0 wraps; seam between
     * domain-local x = c-1 and x = c, c = D - sigma. */
    int has_seam = (b == n - 1 && sigma > 0);
    int64_t c = (int64_t)D - (int64_t)sigma;
    int64_t lo = 0, hi = -1, rem = 0;
    if (has_seam) {
        lo = c - (int64_t)Rr; if (lo < 1) lo = 1;
        hi = (int64_t)D - 1 - (int64_t)Rr; if (c < hi) hi = c;
        rem = hi - lo + 1; if (rem < 0) rem = 0;
    }
    uint32_t n_allow = D - 1 - Rr - (uint32_t)rem;

    /* C4: MISC block m = 0: Fm from plane `lo`, x2 -> position, x3 unused. */
    uint32_t misc[4];
    block(o->seed, g, t, w, STREAM_MISC, 0, misc);
    uint64_t misc_lo = (uint64_t)misc[0] | ((uint64_t)misc[1] << 32);
    uint32_t u = mulhi32(misc[2], n_allow);
    int64_t x = 1 + (int64_t)u;
    if (rem > 0 && x >= lo) x += rem;

    uint8_t Dm[64], Pm[64];
    int needD = 0, needP = 0;
    bernoulli_lanes(o->seed, g, t, w, STREAM_DIFF, o->Td_w[k], Dm, &needD);
    if (o->pmask_paper) { oracle_paper_pmask_bound(o->seed, g, t, w, o->T4p, o->pmask_code, Pm); needP = 2; }
    else bernoulli_lanes(o->seed, g, t, w, STREAM_ANNI, o->Tp_w[k], Pm, &needP);
    o->n_attempt_words += 1;
    o->planes_needed_D += (uint64_t)needD; o->planes_needed_P += (uint64_t)needP;
    o->blocks_needed_D += (uint64_t)((needD + 1) / 2);
    o->blocks_needed_P += (uint64_t)((needP + 1) / 2);

    /* domain-local x' -> tile-local y = (sigma + b*D + x') mod Ts
     *                 -> global   i = (Sigma + tau*Ts + y) mod L
     * C10 - the paper's CONNECTED multispin lattice ("we connected the N_r
     * lattices of the classical approach, to form one larger lattice", sites of one register
     * the maximum distance apart; "the necessary bit-rotations to connect the
     * multi-spin lattices"; next-row f3 of SURVEY.md 8(f)): the 64 bit-lanes of a word column
     * are 64 consecutive segments of ONE ring of 64 L sites; the successor of (site L-1, lane j)
     * is (site 0, lane (j+1) mod 64).  A footprint site whose unreduced index Sigma + tau*Ts + y
     * passed L therefore belongs, for the strand that has lane j before the wrap, to lane j+1. */
    uint32_t site[6], lane_shift[6];
    for (int s = 0; s < 6; ++s) {
        uint64_t xl = (uint64_t)(x - 1 + s);                 /* x-1 .. x+4 */
        uint64_t y = ((uint64_t)sigma + (uint64_t)b * D + xl) % Ts;
        uint64_t gidx = (uint64_t)Sigma + (uint64_t)tau * Ts + y;   /* < 2L */
        site[s] = (uint32_t)(gidx % L);
        lane_shift[s] = (o->connected && gidx >= L) ? 1u : 0u;
    }

    for (int j = 0; j < 64; ++j) {
        uint8_t *qs[6];      /* the strand's six footprint sites */
        for (int s = 0; s < 6; ++s)
            qs[s] = o->q + ((size_t)k * 64 + ((uint32_t)j + lane_shift[s]) % 64) * L + site[s];
        /* mask lane j belongs to the strand that is in bit-lane j BEFORE the wrap (the word as
         * it sits in the register after the bit rotation) */
        /* Fm = mask(1/2) from plane `lo` (C4): U_j < 2^31 <=> top bit of U_j,
         * i.e. lane j of plane 0, is 0.  Fm = 1 => fission LOW (G8). */
        int Fm = ((misc_lo >> j) & 1u) == 0 ? 1 : 0;
        if (o->variant == 3)
            oracle_rule_cpd(qs[0], qs[1], qs[2], Dm[j], Pm[j], Fm);
        else if (o->variant == 0)
            oracle_rule_pcpd(qs[0], qs[1], qs[2], qs[3], Dm[j], Pm[j], Fm);
        else if (o->variant == 1)
            oracle_rule_tcpd(qs[0], qs[1], qs[2], qs[3], qs[4], Dm[j], Pm[j], Fm);
        else
            oracle_rule_qcpd(qs[0], qs[1], qs[2], qs[3], qs[4], qs[5], Dm[j], Pm[j], Fm);
    }
}

/* Schedule SD2(Ts, D, A), sweeps t0 .. t0+n-1. */
int oracle_run(oracle_t *o, uint64_t n_sweeps)
{
    const uint32_t L = o->L, Ts = o->Ts, D = o->D, A = o->A;
    const uint32_t n = Ts / D, S = D / A, ntiles = L / Ts;
    if ((uint64_t)o->sweep + n_sweeps > 0xffffffffull) return -1;
    uint32_t *sigma = (uint32_t *)malloc(sizeof(uint32_t) * S);
    if (!sigma) return -2;
    for (uint64_t it = 0; it < n_sweeps; ++it) {
        uint32_t t = o->sweep;
        /* step 1: SHIFT blocks (c0=k, c1=t, c2=0, c3=3<<24) */
        uint32_t Sigma = 0;
        for (uint32_t ks = 0; ks < S; ++ks) {
            uint32_t x[4];
            block(o->seed, ks, t, 0, STREAM_SHIFT, 0, x);
            sigma[ks] = mulhi32(x[0], D);
            if (ks == 0) Sigma = mulhi32(x[1], Ts);
        }
        /* step 3: sub-steps in order; within a sub-step all (tile, domain,
         * word) are independent (disjoint footprints), so their order is free */
        for (uint32_t ks = 0; ks < S; ++ks) {
            uint64_t nunits = (uint64_t)ntiles * n * o->nwords;
            for (uint64_t unit0 = 0; unit0 < nunits; ++unit0) {
                uint64_t unit = o->reverse_order ? nunits - 1 - unit0 : unit0;
                uint32_t k = (uint32_t)(unit % o->nwords);
                uint32_t b = (uint32_t)((unit / o->nwords) % n);
                uint32_t tau = (uint32_t)(unit / o->nwords / n);
                /* step 4: attempts a = 0..A-1 in order */
                for (uint32_t a = 0; a < A; ++a) {
                    uint32_t g = (tau * n + b) * D + ks * A + a;
                    attempt(o, t, Sigma, sigma[ks], tau, b, k, g);
                }
            }
        }
        o->sweep = t + 1;
    }
    free(sigma);
    return 0;
}

/* The shifts of sweep t, for tests (P6) and diagnostics. */
void oracle_shifts(const oracle_t *o, uint32_t t, uint32_t *Sigma, uint32_t *sigma /* [D/A] */)
{
    uint32_t S = o->D / o->A;
    for (uint32_t ks = 0; ks < S; ++ks) {
        uint32_t x[4];
        block(o->seed, ks, t, 0, STREAM_SHIFT, 0, x);
        sigma[ks] = mulhi32(x[0], o->D);
        if (ks == 0) *Sigma = mulhi32(x[1], o->Ts);
    }
}

/* ------------------------------------------------------------------ C9 --- */
/* count[64k + j] = sum_i q_j(i) for the simulated word columns. */
void oracle_counts(const oracle_t *o, uint32_t *out)
{
    for (uint32_t r = 0; r < o->nwords * 64; ++r) {
        uint32_t cnt = 0;
        const uint8_t *q = o->q + (size_t)r * o->L;
        for (uint32_t i = 0; i < o->L; ++i) cnt += q[i];
        out[r] = cnt;
    }
}

/* pair count: out[r] = sum_i q_r(i) q_next(i), the number of
 * adjacent occupied pairs whose LEFT site lies in replica lane r.  Independent replicas: the ring
 * closes inside the lane, next(L-1) = site 0 of the same lane.  Connected multispin lattice (C10,
 * PAPER.md:98-100, 118): the 64 lanes of a word column are consecutive segments of one ring of
 * 64 L sites, so the right neighbour of (site L-1, lane j) is (site 0, lane (j+1) mod 64) of the
 * same word column; the sum over a column's 64 lanes is then the pair count of that ring. */
void oracle_pair_counts(const oracle_t *o, uint32_t *out)
{
    for (uint32_t r = 0; r < o->nwords * 64; ++r) {
        uint32_t cnt = 0;
        const uint8_t *q = o->q + (size_t)r * o->L;
        for (uint32_t i = 0; i + 1 < o->L; ++i) cnt += (uint32_t)(q[i] & q[i + 1]);
        uint32_t rn = o->connected ? (r / 64) * 64 + (r % 64 + 1) % 64 : r;   /* lane holding the successor of site L-1 */
        cnt += (uint32_t)(q[o->L - 1] & o->q[(size_t)rn * o->L]);
        out[r] = cnt;
    }
}

/* Packed view in canonical order out[i*nwords + k], bit j = replica 64k+j. */
void oracle_get_words(const oracle_t *o, uint64_t *out)
{
    for (uint32_t i = 0; i < o->L; ++i)
        for (uint32_t k = 0; k < o->nwords; ++k) {
            uint64_t word = 0;
            for (int j = 0; j < 64; ++j)
                if (o->q[((size_t)k * 64 + j) * o->L + i]) word |= (uint64_t)1 << j;
            out[(size_t)i * o->nwords + k] = word;
        }
}

void oracle_set_words(oracle_t *o, const uint64_t *in)
{
    for (uint32_t i = 0; i < o->L; ++i)
        for (uint32_t k = 0; k < o->nwords; ++k) {
            uint64_t word = in[(size_t)i * o->nwords + k];
            for (int j = 0; j < 64; ++j)
                o->q[((size_t)k * 64 + j) * o->L + i] = (uint8_t)((word >> j) & 1u);
        }
}

/* ------------------------------------------------ literal Algorithm 1 ---- */
/* PAPER.md:45-70 verbatim, one replica at a time, every replica choosing its
 * own site: i = floor(L*RNG()), r1, r2, r3 -> one Philox block per attempt on
 * the oracle-only stream LITERAL, counter (attempt a, sweep t, replica r):
 * x0 -> i = mulhi32(x0, L); r1 = x1 < Td; r2 = x2 < Tp; r3 = x3 < 2^31.
 * L attempts = one time unit.  q: uint8[R][L] in/out.
 * counts_out[(rec)*R + r] = particle count of replica r after rec_times[rec]
 * sweeps (rec_times ascending, may start with 0). */
int oracle_literal_run(int variant, uint32_t L, uint32_t R, double d, double p,
                       uint64_t seed, uint8_t *q, uint32_t n_rec,
                       const uint32_t *rec_times, uint32_t *counts_out)
{
    uint64_t Td = oracle_threshold(d), Tp = oracle_threshold(p);
    if (Td == UINT64_MAX || Tp == UINT64_MAX) return -1;
    if (variant < 0 || variant > 3 || L < (variant == 3 ? 3u : 4u + (uint32_t)variant)) return -1;  /* reading G18 */
    uint32_t t = 0;
    for (uint32_t rec = 0; rec < n_rec; ++rec) {
        for (; t < rec_times[rec]; ++t)
            for (uint32_t r = 0; r < R; ++r) {
                uint8_t *qr = q + (size_t)r * L;
                for (uint32_t a = 0; a < L; ++a) {
                    uint32_t x[4];
                    block(seed, a, t, r, STREAM_LITERAL, 0, x);
                    uint32_t i = mulhi32(x[0], L);
                    int r1 = (uint64_t)x[1] < Td;
                    int r2 = (uint64_t)x[2] < Tp;
                    int r3 = x[3] < 0x80000000u;
                    oracle_single_attempt(variant, L, qr, i, r1, r2, r3);
                }
            }
        for (uint32_t r = 0; r < R; ++r) {
            uint32_t cnt = 0;
            for (uint32_t i = 0; i < L; ++i) cnt += q[(size_t)r * L + i];
            counts_out[(size_t)rec * R + r] = cnt;
        }
    }
    return 0;
}
