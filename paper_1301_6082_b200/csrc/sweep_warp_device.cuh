// sweep_warp_device.cuh - device code of sweep_warp_kernel, the production sweep kernel for sm_100a.
//
// Mapping: ONE WARP owns one (tile, word column) for a whole sweep; LANE b owns
// domain b of that tile (n = T_s / D <= 32 domains).  The column's T_s words
// live in shared memory from load to store, so the lattice crosses HBM exactly
// once in each direction per sweep (0.25 B per replica-site update), moved by
// TMA bulk copies (cp.async.bulk; one or two contiguous 16-byte-aligned runs per tile
// column, completing on the warp's own mbarrier).  Because all domains of a tile column sit
// in one warp, sub-steps need __syncwarp() only - no block barrier anywhere in
// the sweep.
//
// Per attempt a lane issues, as one basic block, 1 + NU_D + NU_P independent Philox chains
// (MISC block, the first NU_D DIFF blocks, the first NU_P ANNI blocks: none depends on the lattice
// state) written round-major so that ptxas interleaves them; the planes are compared MSB-first
// against T's bits on all 64 lanes in the signed-sum form (und chain on the ALU pipe, lt
// accumulation as IMADs on the FMA pipe); the lazy tails then run as warp-uniform loops only while
// some lane whose outcome can matter is undecided (DIFF: x or x+1 occupied; ANNI: reacting lanes).
// Philox rounds 1-3 are strength-reduced: the products that depend only on (w, t) or only on the
// slot are computed once per warp / once per attempt, leaving 16 IMAD.WIDE.U32 per block, not 20.
//
// Citations: update rule = Alg. 1 PAPER.md:45-70 in the bitwise form of Alg. 2
// PAPER.md:126-151 (typos fixed per DESIGN.md readings G5/G6); schedule SD2 and
// streams = DESIGN.md section 3 C1-C9.
// This header is compiled twice: by nvcc into libpcpd.so (generic thresholds read from the constant
// bank), and at run time by NVRTC (csrc/jit.cu) with the two thresholds T_d, T_p as template constants
// (SPEC = 1), see prefix_spec below.  It therefore includes nothing but the two project headers.
#pragma once
#include "pcpd_kernels.cuh"

// 1: the tile column of sweep_warp_kernel moves between HBM and shared memory by TMA bulk copies (cp.async.bulk);
// 0: by a coalesced 128-bit load / store loop of the warp (the round-1 form; -DPCPD_TMA_TILE=0 to compare)
#ifndef PCPD_TMA_TILE
#define PCPD_TMA_TILE 1
#endif

namespace pcpd {

namespace {

__device__ __forceinline__ uint32_t hi32(uint64_t v) { return (uint32_t)(v >> 32); }
__device__ __forceinline__ uint32_t lo32(uint64_t v) { return (uint32_t)v; }
__device__ __forceinline__ uint64_t mulw(uint32_t a, uint32_t b) { return (uint64_t)a * b; }

// Constants of one (sweep t, word w) pair: everything in rounds 1-3 that does
// not depend on the slot or on c3.
struct PhiloxWarp {
    uint32_t B;     // lo(M1 w) ^ k0[1]
    uint32_t C;     // hi(M0 c0') ^ k1[1],  c0' = hi(M1 w) ^ t ^ k0[0]
    uint32_t Dc;    // lo(M0 c0') ^ k1[2]
};

__device__ __forceinline__ PhiloxWarp philox_warp_consts(uint32_t t, uint32_t w, const RoundKeys &rk)
{
    const uint64_t p1 = mulw(PHILOX_M1, w);
    const uint32_t c0p = hi32(p1) ^ t ^ rk.k0[0];
    const uint64_t p0p = mulw(PHILOX_M0, c0p);
    PhiloxWarp pw;
    pw.B = lo32(p1) ^ rk.k0[1];
    pw.C = hi32(p0p) ^ rk.k1[1];
    pw.Dc = lo32(p0p) ^ rk.k1[2];
    return pw;
}

// Constants of one slot (attempt): 2 wide multiplies.
struct PhiloxSlot {
    uint32_t X;    // hi(M0 slot) ^ k1[0]           (c2' = X ^ c3)
    uint32_t E;    // hi(M1 c2'') ^ k0[2],  c2'' = C ^ lo(M0 slot)
    uint32_t c1;   // lo(M1 c2'')                    (c1 entering round 4)
};

__device__ __forceinline__ PhiloxSlot philox_slot_consts(uint32_t slot, const PhiloxWarp &pw, const RoundKeys &rk)
{
    const uint64_t p0 = mulw(PHILOX_M0, slot);
    const uint32_t c2pp = pw.C ^ lo32(p0);
    const uint64_t p1pp = mulw(PHILOX_M1, c2pp);
    PhiloxSlot ps;
    ps.X = hi32(p0) ^ rk.k1[0];
    ps.E = hi32(p1pp) ^ rk.k0[2];
    ps.c1 = lo32(p1pp);
    return ps;
}

// Philox-4x32-10 block of counter (slot, t, w, c3): 16 IMAD.WIDE.U32 + 18 LOP3.
__device__ __forceinline__ U4 philox_block(uint32_t c3, const PhiloxSlot &ps, const PhiloxWarp &pw,
                                           const RoundKeys &rk)
{
    // round 1 -> only c2' depends on c3; round 2: one multiply; round 3: one multiply
    const uint32_t c2p = ps.X ^ c3;
    const uint64_t p1p = mulw(PHILOX_M1, c2p);
    const uint32_t c0pp = hi32(p1p) ^ pw.B;
    const uint64_t p0pp = mulw(PHILOX_M0, c0pp);
    uint32_t c0 = ps.E ^ lo32(p1p);
    uint32_t c1 = ps.c1;
    uint32_t c2 = hi32(p0pp) ^ pw.Dc;
    uint32_t c3r = lo32(p0pp);
#pragma unroll
    for (int r = 3; r < 10; ++r) {
        const uint64_t p0 = mulw(PHILOX_M0, c0);
        const uint64_t p1 = mulw(PHILOX_M1, c2);
        const uint32_t n0 = hi32(p1) ^ c1 ^ rk.k0[r];
        const uint32_t n2 = hi32(p0) ^ c3r ^ rk.k1[r];
        c1 = lo32(p1);
        c3r = lo32(p0);
        c0 = n0;
        c2 = n2;
    }
    return U4{c0, c1, c2, c3r};
}

// N blocks of one slot at once, written round-major / chain-minor so that the N
// independent multiply chains are interleaved in the instruction stream (ptxas
// keeps source order within its window; block-after-block code leaves the FMA
// pipe waiting on one chain's latency).
template <int N>
__device__ __forceinline__ void philox_blocks(const uint32_t (&c3in)[N], const PhiloxSlot &ps, const PhiloxWarp &pw,
                                              const RoundKeys &rk, U4 *out)
{
    uint32_t c0[N], c1[N], c2[N], c3[N];
    uint64_t pa[N], pb[N];
#pragma unroll
    for (int i = 0; i < N; ++i) pa[i] = mulw(PHILOX_M1, ps.X ^ c3in[i]);
#pragma unroll
    for (int i = 0; i < N; ++i) pb[i] = mulw(PHILOX_M0, hi32(pa[i]) ^ pw.B);
#pragma unroll
    for (int i = 0; i < N; ++i) {
        c0[i] = ps.E ^ lo32(pa[i]);
        c1[i] = ps.c1;
        c2[i] = hi32(pb[i]) ^ pw.Dc;
        c3[i] = lo32(pb[i]);
    }
#pragma unroll
    for (int r = 3; r < 10; ++r) {
#pragma unroll
        for (int i = 0; i < N; ++i) {
            pa[i] = mulw(PHILOX_M0, c0[i]);
            pb[i] = mulw(PHILOX_M1, c2[i]);
        }
#pragma unroll
        for (int i = 0; i < N; ++i) {
            c0[i] = hi32(pb[i]) ^ c1[i] ^ rk.k0[r];
            c2[i] = hi32(pa[i]) ^ c3[i] ^ rk.k1[r];
            c1[i] = lo32(pb[i]);
            c3[i] = lo32(pa[i]);
        }
    }
#pragma unroll
    for (int i = 0; i < N; ++i) out[i] = U4{c0[i], c1[i], c2[i], c3[i]};
}

// Connected multispin lattice (C10): the successor of (site L-1, lane j) is
// (site 0, lane j+1), so the words of the tile sites that lie past the ring wrap are rotated right by
// one bit when the tile is loaded (bit j of the tile word = the strand that is in lane j before the
// wrap) and rotated back when it is stored.  r is 0 or 1.
__device__ __forceinline__ uint64_t rotr64(uint64_t v, uint32_t r) { return (v >> r) | (v << ((64u - r) & 63u)); }
__device__ __forceinline__ uint64_t rotl64(uint64_t v, uint32_t r) { return (v << r) | (v >> ((64u - r) & 63u)); }

// 64-lane mask state as two 32-bit halves.
struct Mask2 {
    uint32_t lo, hi;
};
__device__ __forceinline__ uint64_t m64(const Mask2 &m) { return (uint64_t)m.lo | ((uint64_t)m.hi << 32); }

// MSB-first bit-sliced compare of two planes (p0 = plane 2m, p1 = plane 2m+1; block blk = planes
// x0 | x1 << 32 and x2 | x3 << 32) against T's bits tb0, tb1 given as 32-lane masks (C3), in
// signed-sum form.  und_k (lanes still equal to T before plane k) are nested
// sets, and lt = OR_k (und_k - und_(k+1)) over the planes where T's bit is 1 = sum_k s_k * und_k with
// s_k = tb_k - tb_(k-1) in {-1, 0, +1}: the lt accumulation becomes one 32-bit IMAD per plane and half
// (FMA pipe, which has slack) and only the und chain (one LOP3 per plane and half) stays on the ALU
// pipe, the binding one.  The caller closes the sum with -tb_last * und when it stops.
__device__ __forceinline__ void cmp2h_sum(uint32_t &lt, uint32_t &und, uint32_t p0, uint32_t p1, uint32_t tb0,
                                          uint32_t tb1, int32_t s0, int32_t s1)
{
    lt += und * (uint32_t)s0;
    const uint32_t u1 = und & ~(p0 ^ tb0);
    lt += u1 * (uint32_t)s1;
    und = u1 & ~(p1 ^ tb1);
}

__device__ __forceinline__ void cmp_block_sum(Mask2 &lt, Mask2 &und, const U4 &blk, uint32_t tb0, uint32_t tb1,
                                              int32_t s0, int32_t s1)
{
    cmp2h_sum(lt.lo, und.lo, blk.x0, blk.x2, tb0, tb1, s0, s1);
    cmp2h_sum(lt.hi, und.hi, blk.x1, blk.x3, tb0, tb1, s0, s1);
}

// The paper's annihilation-mask family (section 4.3): the per-lane "decorrelation" bits of one 32-lane
// half from the two planes p0, p1 of ANNI block 0 - code 0: b = 1/4 (AND, Alg. 2 line 12), 1: 1/2 (one raw word), 2: 1
// (none: fully correlated lanes), 3: 3/4 (OR).  The word-wide gate [x3 < floor((p/b) 2^32)] is applied by the caller.
__device__ __forceinline__ uint32_t pmask_dec(uint32_t p0, uint32_t p1, uint32_t code)
{
    return code == 0u ? (p0 & p1) : code == 1u ? p0 : code == 2u ? ~0u : (p0 | p1);
}

// ---- mbarrier helpers (the producer / update-warp ring of column_kernel, column_device.cuh) ----
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
// TMA bulk copies (1-D, cp.async.bulk) of a tile column between global and shared memory: addresses and sizes are
// multiples of 16 bytes; the load completes on an mbarrier (complete_tx), the store is tracked as a bulk group.
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void bulk_s2g(void *dst, const void *src, uint32_t bytes)
{
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(smem_u32(src)), "r"(bytes) : "memory");
}

// (the suspend-time hint lets the hardware park the thread until the phase completes instead of returning at once:
// a waiting warp then takes almost no issue slots from the warps it is waiting for)
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    uint32_t done;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done)
                     : "r"(smem_u32(bar)), "r"(parity), "r"(1000000u)
                     : "memory");
    } while (!done);
}

// C5 step 3-4 for domain b in a sub-step with inner shift sigma: only domain n-1 with sigma > 0 wraps; the tile
// seam lies between domain-local c-1 and c, c = D - sigma; positions [c-Rr, c] are excluded.
struct DomainPos {
    int32_t lo, rem;
    uint32_t n_allow, dbase;  // dbase = tile-local index of domain-local 0 (before wrap)
};
__device__ __forceinline__ DomainPos domain_pos(uint32_t b, uint32_t n, uint32_t sigma, uint32_t D, uint32_t Rr)
{
    DomainPos dp;
    const bool seam = (b == n - 1) && (sigma > 0);
    const int32_t c = (int32_t)D - (int32_t)sigma;
    dp.lo = 0;
    dp.rem = 0;
    if (seam) {
        dp.lo = max(1, c - (int32_t)Rr);
        const int32_t hi = min((int32_t)D - 1 - (int32_t)Rr, c);
        dp.rem = max(0, hi - dp.lo + 1);
    }
    dp.n_allow = D - 1 - Rr - (uint32_t)dp.rem;
    dp.dbase = sigma + b * D;
    return dp;
}
// C4 / C5 step 4: position selector x2 of the MISC block -> tile-local index of footprint site x-1
__device__ __forceinline__ uint32_t footprint_start(uint32_t x2, const DomainPos &dp, uint32_t Ts)
{
    int32_t x = 1 + (int32_t)__umulhi(x2, dp.n_allow);
    if (dp.rem > 0 && x >= dp.lo) x += dp.rem;
    uint32_t y0 = dp.dbase + (uint32_t)x - 1;  // footprint x-1 .. x+Rr never straddles the seam
    if (y0 >= Ts) y0 -= Ts;
    return y0;
}

// blocks of a threshold T in [0, 2^32): ceil((32 - ctz(T)) / 2), 0 for T = 0
__host__ __device__ constexpr uint32_t nblk_of(uint32_t T)
{
    uint32_t tz = 0;
    while (tz < 32 && !((T >> tz) & 1u)) ++tz;
    return T ? (32u - tz + 1u) >> 1 : 0u;
}

// Threshold-specialised prefix compare (SPEC kernels: T is a template constant).  With T's bits known
// at compile time the planes' xor with T folds into the LOP3 truth tables, and TWO planes go through
// one LOP3 for und (the AND of the per-plane equalities) and one for lt, which runs LSB-first over the
// prefix (m_k = differs_k ? tb_k : m_(k+1), m_end = 0: an equivalent form of C3's compare): 4 LOP3 per
// block instead of 4 LOP3 + 4 IMAD.  lt is exact for the lanes decided inside the prefix and 0 for the
// lanes still equal to T, so the lazy tail starts a fresh signed sum (prev = 0).
template <uint32_t T, int NB>
__device__ __forceinline__ void prefix_spec(Mask2 &lt, Mask2 &und, const U4 *blk)
{
    uint32_t ulo = ~0u, uhi = ~0u, mlo = 0u, mhi = 0u;
#pragma unroll
    for (int k = 2 * NB - 1; k >= 0; --k) {
        const U4 &b = blk[k >> 1];
        const uint32_t plo = (k & 1) ? b.x2 : b.x0, phi = (k & 1) ? b.x3 : b.x1;
        if ((T >> (31 - k)) & 1u) {
            mlo |= ~plo; mhi |= ~phi; ulo &= plo; uhi &= phi;
        } else {
            mlo &= ~plo; mhi &= ~phi; ulo &= ~plo; uhi &= ~phi;
        }
    }
    lt = Mask2{mlo, mhi};
    und = Mask2{ulo, uhi};
}

__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}

}  // namespace

// NU_D / NU_P = number of DIFF / ANNI blocks of an attempt evaluated unconditionally (template
// parameters so that the unconditional part has no branch at all): 5 and 4 for thresholds with that
// many blocks (tuned on B200: a warp pays the maximum over its 32 lanes, so nearly every attempt
// needs that many anyway), 1 for thresholds with few planes (d = 1/2 has one), 0 for T = 0 or 2^32.
//
// SPEC = 1 (kernels compiled at run time by jit.cu): the thresholds are the template constants STD, STP
// (low 32 bits of T_d, T_p; neither threshold is 2^32) instead of P.thd / P.thp and the host tables, and
// the schedule constants T_s, D, A and the ring length L are the template constants CTS, CD, CA, CL.
template <int VARIANT, int WPB, int NU_D, int NU_P, int PMODE, int PW, int SPEC = 0, uint32_t STD = 0u, uint32_t STP = 0u,
          uint32_t CTS = 0u, uint32_t CD = 0u, uint32_t CA = 0u, uint32_t CL = 0u>
__global__ void __launch_bounds__(WPB * 32, WPB >= 7 ? 2 : 1) sweep_warp_kernel(const __grid_constant__ SweepParams P)
{
    extern __shared__ __align__(16) uint64_t smem[];  // WPB buffers of `stride` words

    constexpr uint32_t Rr = VARIANT == 3 ? 1u : 2u + VARIANT;  // right reach: 2 PCPD, 3 TCPD, 4 QCPD, 1 CPD
    // SPEC kernels also have the schedule constants and the ring length as template constants (address
    // arithmetic, seam bookkeeping and the mulhi by n_allow then work on immediates).
    const uint32_t Ts = SPEC ? CTS : P.Ts, D = SPEC ? CD : P.D, A = SPEC ? CA : P.A, L = SPEC ? CL : P.L;
    const uint32_t S = SPEC ? CD / (CA ? CA : 1u) : P.S, n = SPEC ? CTS / (CD ? CD : 1u) : P.n, t = P.t;
    // (baking the seed in as well was measured slower: 32-bit immediates in the xor chain)
    const RoundKeys &rk = P.rk;

    const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31u;
    const uint32_t ntiles = L / Ts;
    const uint32_t task = blockIdx.x * WPB + warp;
    if (task >= ntiles * P.W) return;  // warps are independent: no block-wide barrier in this kernel

    // C5 step 1: shifts from the SHIFT stream; lane j holds sigma_{k0+j} of the current group of 32 sub-steps.
    uint32_t sig_reg, Sigma;
    {
        const U4 blk = philox4x32_10(lane, t, 0u, STREAM_SHIFT, rk);
        sig_reg = __umulhi(blk.x0, D);
        Sigma = __shfl_sync(0xffffffffu, __umulhi(blk.x1, Ts), 0);
    }
    const uint32_t tau = task % ntiles, wl = task / ntiles;
    const uint32_t w = P.word_offset + wl;  // global word index (RNG key)

    // ---- C5 step 2: tile tau covers global sites (Sigma + tau*Ts + y) mod L ----
    const uint32_t start = (uint32_t)(((uint64_t)Sigma + (uint64_t)tau * Ts) % L);
    uint64_t *g = P.lat + (size_t)wl * L;             // column wl, contiguous in the site index
    const uint32_t stride = (Ts + 3u) & ~1u;          // words per warp buffer (even, >= Ts + 2)
    uint64_t *buf = smem + (size_t)warp * stride;
    const bool vec = ((L | Ts) & 1u) == 0;            // 16-byte-aligned (TMA / 128-bit) path needs even L and T_s
    const uint32_t conn = P.connected;                // 1: connected multispin lattice (C10)
    const uint32_t odd = vec ? (start & 1u) : 0u;
    uint64_t *tile = buf + odd;                       // tile[y], y in [0, Ts)
    constexpr uint32_t nud = (uint32_t)NU_D, nup = (uint32_t)NU_P;
    if (vec) {
        const uint32_t s0 = start - odd, npairs = Ts / 2 + odd;
#if PCPD_TMA_TILE
        // the warp's tile column (16-byte aligned: s0, L even) by TMA bulk copy - two pieces where it passes the ring
        // wrap - completing on the warp's own mbarrier: the copy engine moves the 16 KB, the warp issues 2 instructions
        __shared__ __align__(8) uint64_t tile_bar[WPB];
        if (lane == 0) {
            mbar_init(&tile_bar[warp], 1u);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
            const uint32_t nwords = 2u * npairs, first = min(nwords, L - s0);
            mbar_expect_tx(&tile_bar[warp], nwords * 8u);
            bulk_g2s(buf, g + s0, first * 8u, &tile_bar[warp]);
            if (first < nwords) bulk_g2s(buf + first, g, (nwords - first) * 8u, &tile_bar[warp]);
        }
        __syncwarp();
        mbar_wait(&tile_bar[warp], 0u);
#else
        const ulonglong2 *g2 = reinterpret_cast<const ulonglong2 *>(g);
        ulonglong2 *b2 = reinterpret_cast<ulonglong2 *>(buf);
#pragma unroll 8
        for (uint32_t pi = lane; pi < npairs; pi += 32) {
            uint32_t i = s0 + 2 * pi;
            if (i >= L) i -= L;
            b2[pi] = g2[i >> 1];
        }
#endif
        if (conn && s0 + 2 * npairs > L) {
            // connected lattice: rotate the words past the ring wrap in place (L and s0 are even, so
            // both words of a pair lie on the same side of the wrap)
            __syncwarp();
            for (uint32_t k2 = (L - s0) + lane; k2 < 2 * npairs; k2 += 32) buf[k2] = rotr64(buf[k2], 1u);
        }
    } else {
        for (uint32_t y = lane; y < Ts; y += 32) {
            uint32_t i = start + y;
            if (i >= L) i -= L;
            tile[y] = g[i];
        }
        if (conn && start + Ts > L) {
            __syncwarp();
            for (uint32_t y = (L - start) + lane; y < Ts; y += 32) tile[y] = rotr64(tile[y], 1u);
        }
    }
    __syncwarp();

    const PhiloxWarp pw = philox_warp_consts(t, w, rk);
    const bool act = lane < n;
    const uint32_t b = act ? lane : 0u;
    const uint32_t slot0 = (tau * n + b) * D;
    uint32_t nblkD = (P.thd.nplanes + 1u) >> 1, nblkP = (P.thp.nplanes + 1u) >> 1;
    uint32_t Td = P.thd.T32, Tp = P.thp.T32;
    bool allD = P.thd.all != 0, allP = P.thp.all != 0;
    if constexpr (SPEC) {  // thresholds are template constants
        constexpr uint32_t nbd = nblk_of(STD), nbp = nblk_of(STP);
        nblkD = nbd; nblkP = nbp; Td = STD; Tp = STP; allD = false; allP = false;
    }
    // Per-word thresholds (C11): the bit masks and signed-sum coefficients of the unconditional planes live in
    // registers for the whole task instead of the constant bank.  Planes past a word's last significant one have
    // T bit 0, which closes the signed sum at the right plane by itself.
    uint32_t tdm_r[2 * NU_D + 1], tpm_r[2 * NU_P + 1];
    int32_t sd_r[2 * NU_D + 1], sp_r[2 * NU_P + 1];
    if constexpr (PW) {
        const uint4 th = reinterpret_cast<const uint4 *>(P.thr_dev)[wl];
        Td = th.x; Tp = th.y; allD = (th.z & 1u) != 0; allP = (th.z & 2u) != 0;
        nblkD = Td ? (32u - (uint32_t)(__ffs((int)Td) - 1) + 1u) >> 1 : 0u;
        nblkP = Tp ? (32u - (uint32_t)(__ffs((int)Tp) - 1) + 1u) >> 1 : 0u;
#pragma unroll
        for (int kk = 0; kk < 2 * NU_D; ++kk) {
            const uint32_t bit = (Td >> (31 - kk)) & 1u, prev = kk ? (Td >> (32 - kk)) & 1u : 0u;
            tdm_r[kk] = 0u - bit;
            sd_r[kk] = (int32_t)bit - (int32_t)prev;
        }
#pragma unroll
        for (int kk = 0; kk < 2 * NU_P; ++kk) {
            const uint32_t bit = (Tp >> (31 - kk)) & 1u, prev = kk ? (Tp >> (32 - kk)) & 1u : 0u;
            tpm_r[kk] = 0u - bit;
            sp_r[kk] = (int32_t)bit - (int32_t)prev;
        }
    }

#pragma unroll 1
    for (uint32_t k = 0; k < S; ++k) {
        if (k != 0 && (k & 31u) == 0) sig_reg = __umulhi(philox4x32_10(k + lane, t, 0u, STREAM_SHIFT, rk).x0, D);
        const uint32_t sigma = __shfl_sync(0xffffffffu, sig_reg, k & 31u);
        const DomainPos dp = domain_pos(b, n, sigma, D, Rr);

#pragma unroll 1
        for (uint32_t a = 0; a < A; ++a) {
            // The MISC block, the first NU_D DIFF blocks and the first NU_P ANNI blocks of an attempt do not
            // depend on the lattice state (only WHICH lanes matter does): independent Philox chains, issued
            // back to back so that the FMA pipe always has several wide multiplies in flight.
            const PhiloxSlot ps = philox_slot_consts(slot0 + k * A + a, pw, rk);
            U4 blks[1 + NU_D + NU_P];
            Mask2 dlt{0u, 0u}, dund{~0u, ~0u}, plt{0u, 0u}, pund{~0u, ~0u};
            {
                uint32_t c3s[1 + NU_D + NU_P];
                c3s[0] = STREAM_MISC;
#pragma unroll
                for (int m = 0; m < NU_D; ++m) c3s[1 + m] = STREAM_DIFF | m;
#pragma unroll
                for (int m = 0; m < NU_P; ++m) c3s[1 + NU_D + m] = STREAM_ANNI | m;
                philox_blocks<1 + NU_D + NU_P>(c3s, ps, pw, rk, blks);
            }
            const U4 misc = blks[0];
            const U4 *dblk = blks + 1, *pblk = blks + 1 + NU_D;

            // C4: MISC block: Fm = ~lo (1 -> fission low, Alg. 1: r3 < 1/2), x2 -> position.
            const uint32_t y0 = footprint_start(misc.x2, dp, Ts);
            const uint64_t Fm = ~lo64(misc);
            uint64_t *q = tile + y0;
            uint64_t sa = 0, sb = 0, sc = 0, se = 0, sf = 0, sg = 0;
            if (act) {
                sa = q[0]; sb = q[1]; sc = q[2];
                if constexpr (VARIANT != 3) se = q[3];
                if constexpr (VARIANT == 1 || VARIANT == 2) sf = q[4];
                if constexpr (VARIANT == 2) sg = q[5];
            }

            // DIFF and ANNI masks (C3): the unconditional planes are compared on all 64 lanes (no
            // dependence on the state), the lazy tails only on the lanes whose outcome can matter:
            // DIFF where x or x+1 is occupied, ANNI where a pair (triple) is present and Dm = 0.
            if constexpr (SPEC) {
                prefix_spec<STD, NU_D>(dlt, dund, dblk);
                if constexpr (PMODE == 0) prefix_spec<STP, NU_P>(plt, pund, pblk);
            } else {
#pragma unroll
                for (int m = 0; m < NU_D; ++m)
                    cmp_block_sum(dlt, dund, dblk[m], PW ? tdm_r[2 * m] : P.tdm[2 * m], PW ? tdm_r[2 * m + 1] : P.tdm[2 * m + 1],
                                  PW ? sd_r[2 * m] : P.sd[2 * m], PW ? sd_r[2 * m + 1] : P.sd[2 * m + 1]);
                if constexpr (PMODE == 0) {
#pragma unroll
                    for (int m = 0; m < NU_P; ++m)
                        cmp_block_sum(plt, pund, pblk[m], PW ? tpm_r[2 * m] : P.tpm[2 * m],
                                      PW ? tpm_r[2 * m + 1] : P.tpm[2 * m + 1], PW ? sp_r[2 * m] : P.sp[2 * m],
                                      PW ? sp_r[2 * m + 1] : P.sp[2 * m + 1]);
                }
            }
            {
                const uint64_t rel = sb | sc;
                dund.lo &= (uint32_t)rel;
                dund.hi &= (uint32_t)(rel >> 32);
                uint32_t Tsh = Td << (2 * nud);  // T's bits of the next two planes on top (0 past the last plane)
                uint32_t m = nud;
                // T's bit of the last plane done (PW); SPEC: the prefix lt is exact, the tail's sum starts afresh
                int32_t prev = (NU_D > 0 && !SPEC) ? (int32_t)((Td >> (32 - 2 * NU_D)) & 1u) : 0;
                for (; m < nblkD && __any_sync(0xffffffffu, (dund.lo | dund.hi) != 0); ++m) {
                    const U4 blk = philox_block(STREAM_DIFF | m, ps, pw, rk);
                    int32_t s0, s1;
                    if constexpr (PW || SPEC) {
                        const int32_t b0 = (int32_t)(Tsh >> 31), b1 = (int32_t)((Tsh >> 30) & 1u);
                        s0 = b0 - prev; s1 = b1 - b0; prev = b1;
                    } else {
                        s0 = P.sd[2 * m]; s1 = P.sd[2 * m + 1];
                    }
                    cmp_block_sum(dlt, dund, blk, (uint32_t)((int32_t)Tsh >> 31), (uint32_t)((int32_t)(Tsh << 1) >> 31), s0, s1);
                    Tsh <<= 2;
                }
                // close the sum: lanes still equal to T after the last plane looked at are not < T
                const uint32_t cl = (PW || SPEC) ? (uint32_t)(-prev) : (uint32_t)P.cld[m];
                dlt.lo += dund.lo * cl;
                dlt.hi += dund.hi * cl;
            }
            const uint64_t Dm = allD ? ~0ull : m64(dlt);
            uint64_t react = sb & ~Dm;  // particle cluster (1, 2, 3 or 4 sites from x) present and no diffusion
            if constexpr (VARIANT != 3) react &= sc;
            if constexpr (VARIANT == 1 || VARIANT == 2) react &= se;
            if constexpr (VARIANT == 2) react &= sf;
            if constexpr (PMODE == 0) {
                pund.lo &= (uint32_t)react;
                pund.hi &= (uint32_t)(react >> 32);
                uint32_t Tsh = Tp << (2 * nup);
                uint32_t m = nup;
                int32_t prev = (NU_P > 0 && !SPEC) ? (int32_t)((Tp >> (32 - 2 * NU_P)) & 1u) : 0;
                for (; m < nblkP && __any_sync(0xffffffffu, (pund.lo | pund.hi) != 0); ++m) {
                    const U4 bk = philox_block(STREAM_ANNI | m, ps, pw, rk);
                    int32_t s0, s1;
                    if constexpr (PW || SPEC) {
                        const int32_t b0 = (int32_t)(Tsh >> 31), b1 = (int32_t)((Tsh >> 30) & 1u);
                        s0 = b0 - prev; s1 = b1 - b0; prev = b1;
                    } else {
                        s0 = P.sp[2 * m]; s1 = P.sp[2 * m + 1];
                    }
                    cmp_block_sum(plt, pund, bk, (uint32_t)((int32_t)Tsh >> 31), (uint32_t)((int32_t)(Tsh << 1) >> 31), s0, s1);
                    Tsh <<= 2;
                }
                const uint32_t cl = (PW || SPEC) ? (uint32_t)(-prev) : (uint32_t)P.clp[m];
                plt.lo += pund.lo * cl;
                plt.hi += pund.hi * cl;
            } else {
                // The paper's own annihilation mask (Alg. 2 lines 12-13):
                // an independent b-bit per lane (b = 1/4: the two planes of ANNI block 0 ANDed; pmask_dec) gated by
                // ONE word-wide draw that is 1 w.p. p/b (x3 of the MISC block against floor((p/b) * 2^32)).
                // (PMODE = 1: bound code from P.pmask_code; PMODE = 2 .. 5, the run-time specialised kernels: code PMODE - 2
                // as a compile-time constant, so that the select folds away)
                const uint32_t code = PMODE >= 2 ? (uint32_t)(PMODE - 2) : P.pmask_code;
                const uint32_t gate = misc.x3 < P.T4p ? ~0u : 0u;
                plt.lo = pmask_dec(pblk[0].x0, pblk[0].x2, code) & gate;
                plt.hi = pmask_dec(pblk[0].x1, pblk[0].x3, code) & gate;
            }
            const uint64_t Pm = (PMODE == 0 && allP) ? ~0ull : m64(plt);

            // C6 / Alg. 2, branch-free over the 64 replicas.
            uint64_t nb = (Dm & sc) | (~Dm & sb);
            uint64_t nc = (Dm & sb) | (~Dm & sc);
            const uint64_t ann = react & Pm;
            const uint64_t fis = react & ~Pm;
            nb &= ~ann;
            if constexpr (VARIANT != 3) nc &= ~ann;
            sa |= fis & Fm;
            if (act) {
                if constexpr (VARIANT == 3) {        // CPD: single particle at x; fission high -> x+1 (react lanes have Dm = 0)
                    nc |= fis & ~Fm;
                } else if constexpr (VARIANT == 0) { // PCPD: pair at x, x+1; fission high -> x+2
                    se |= fis & ~Fm;
                } else if constexpr (VARIANT == 1) { // TCPD: triple x..x+2; high -> x+3
                    se &= ~ann;
                    sf |= fis & ~Fm;
                    q[4] = sf;
                } else {                             // QCPD: quadruplet x..x+3; high -> x+4
                    se &= ~ann;
                    sf &= ~ann;
                    sg |= fis & ~Fm;
                    q[4] = sf;
                    q[5] = sg;
                }
                q[0] = sa; q[1] = nb; q[2] = nc;
                if constexpr (VARIANT != 3) q[3] = se;
            }
        }
        __syncwarp();
    }

    // ---- store the tile ----
    if (conn) {  // connected lattice: rotate the words past the ring wrap back (see the load)
        const uint32_t first = vec ? (start - odd) : start, nw = vec ? 2 * (Ts / 2 + odd) : Ts;
        uint64_t *base = vec ? buf : tile;
        if (first + nw > L) {
            for (uint32_t k2 = (L - first) + lane; k2 < nw; k2 += 32) base[k2] = rotl64(base[k2], 1u);
            __syncwarp();
        }
    }
    if (vec) {
        const uint32_t s0 = start - odd, npairs = Ts / 2 + odd;
#if PCPD_TMA_TILE
        // TMA bulk store of the 16-byte-aligned part of the buffer; an odd-aligned tile holds one foreign word at either
        // end of its buffer: those two edge pairs are left out of the bulk copy and their own words stored by hand
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // every lane: its generic-proxy writes -> async proxy
        __syncwarp();                                                   // ... all of them before lane 0 issues the copy
        if (lane == 0) {
            const uint32_t w0 = 2u * odd, w1 = 2u * npairs - 2u * odd;   // buffer words [w0, w1) go by bulk copy
            uint32_t i0 = s0 + w0;
            if (i0 >= L) i0 -= L;
            const uint32_t first = min(w1 - w0, L - i0);
            bulk_s2g(g + i0, buf + w0, first * 8u);
            if (first < w1 - w0) bulk_s2g(g, buf + w0 + first, (w1 - w0 - first) * 8u);
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
            if (odd) {
                uint32_t ia = s0 + 1u, ib = s0 + 2u * npairs - 2u;
                if (ia >= L) ia -= L;
                if (ib >= L) ib -= L;
                g[ia] = buf[1];
                g[ib] = buf[2u * npairs - 2u];
            }
            asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");   // shared memory is read before the warp exits
        }
#else
        ulonglong2 *g2 = reinterpret_cast<ulonglong2 *>(g);
        const ulonglong2 *b2 = reinterpret_cast<const ulonglong2 *>(buf);
#pragma unroll 8
        for (uint32_t pi = lane; pi < npairs; pi += 32) {
            uint32_t i = s0 + 2 * pi;
            if (i >= L) i -= L;
            if (odd && (pi == 0 || pi == npairs - 1)) {
                // edge pairs of an odd-aligned tile hold one foreign word each
                if (pi == 0) g[i + 1] = buf[1];
                else g[i] = buf[2 * pi];
            } else {
                g2[i >> 1] = b2[pi];
            }
        }
#endif
    } else {
        for (uint32_t y = lane; y < Ts; y += 32) {
            uint32_t i = start + y;
            if (i >= L) i -= L;
            g[i] = tile[y];
        }
    }
}

}  // namespace pcpd
