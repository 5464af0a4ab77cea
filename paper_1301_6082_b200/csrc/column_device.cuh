// column_device.cuh - column_kernel, the sweep kernel for small and mid-size problems.
//
// With fewer tile columns than the GPU has warp slots, one warp per tile column (sweep_warp_kernel) leaves the
// machine idle: a sweep is then the latency of ONE warp's chain of D sequential attempts per domain, each with its
// ten Philox chains.  Here ONE BLOCK owns one (tile, word column) for a sweep and splits the work by dependence:
//
//   * producer warps (all but two) compute everything of an attempt that does not depend on the lattice, which is
//     everything but the rule itself: the MISC block (fission-side mask; footprint position resolved with the
//     sub-step's inner shift and seam) and the COMPLETE masks Dm, Pm - the first NU_D DIFF and NU_P
//     ANNI blocks as interleaved Philox chains, then lazily block by block until every one of the 64 lanes of all 32
//     domains is decided (state-independent lazy evaluation: ~6.4 blocks per stream for a generic threshold) -
//     attempt j by producer j mod NPROD, into a ring of records in shared memory (one `full` mbarrier per slot);
//   * two UPDATE warps apply the attempts in order, warp h on the 32-bit half h of the 64 replica lanes (the halves
//     never interact): the tile column is kept as two planes of 32-bit words, so the update warps share no data and
//     need no synchronisation with one another between load and store.  Per attempt an update warp reads its half of
//     the record (one attempt ahead) and the 4 (5, 6, 3) footprint words and applies the bitwise rule - about 40
//     instructions, no random numbers, no vote, no branch.
//
// Lane b of an update warp owns domain b (n = T_s / D <= 32), as in sweep_warp_kernel; sub-steps synchronise with
// __syncwarp().  Same contract (C1-C9), same results bit for bit.
//
// Citations: update rule = Alg. 1 PAPER.md:45-70 in the bitwise form of Alg. 2 PAPER.md:126-151 (readings G5/G6).
#pragma once
#include "sweep_warp_device.cuh"

namespace pcpd {

namespace {

// One ring slot = the record of one attempt for the 32 domains of the tile column, split by half h:
//   rec[h][lane] = {y0, Fm.h, Dm.h, Pm.h}  (uint4)
// y0 = tile-local index of footprint site x-1; Fm = ~lo of the MISC block (1 -> fission low, Alg. 1: r3 < 1/2);
// Dm, Pm = the Bernoulli(d), Bernoulli(p) masks of C3 / C4, all lanes decided.
constexpr uint32_t COL_REC_BYTES = 2u * 32u * 16u;   // 1024
constexpr uint32_t COL_RING_PER_PRODUCER = 2u;

// Producer: the record of one attempt (Philox slot `slot_of_attempt`, C5 step 4) of domain b (C4, C5 steps 3-4, C3)
// into ring slot `slot`.
// NU_D / NU_P = DIFF / ANNI blocks evaluated unconditionally, together with the MISC block, as 1 + NU_D + NU_P
// interleaved Philox chains with compile-time plane indices (T's bit masks and signed-sum coefficients are then
// constant-bank operands, as in sweep_warp_kernel); further blocks follow lazily, one at a time, while any lane of any
// domain is still equal to T on all planes looked at.  The warp votes, so all 32 domains stop together; nothing here
// depends on the lattice.
template <int NU_D, int NU_P>
__device__ __forceinline__ void produce_column_record(const SweepParams &P, const PhiloxWarp &pw, uint32_t slot_of_attempt,
                                                      uint32_t b, uint32_t lane, uint32_t sigma, uint8_t *slot)
{
    const RoundKeys &rk = P.rk;
    const DomainPos dp = domain_pos(b, P.n, sigma, P.D, P.rr);
    const PhiloxSlot ps = philox_slot_consts(slot_of_attempt, pw, rk);
    Mask2 dlt{0u, 0u}, dund{~0u, ~0u}, plt{0u, 0u}, pund{~0u, ~0u};
    U4 blks[1 + NU_D + NU_P];
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
#pragma unroll
    for (int m = 0; m < NU_D; ++m)
        cmp_block_sum(dlt, dund, blks[1 + m], P.tdm[2 * m], P.tdm[2 * m + 1], P.sd[2 * m], P.sd[2 * m + 1]);
    const uint32_t nblkD = (P.thd.nplanes + 1u) >> 1, nblkP = (P.thp.nplanes + 1u) >> 1;
    uint32_t md = NU_D, mp = NU_P;
    for (; md < nblkD && __any_sync(0xffffffffu, (dund.lo | dund.hi) != 0u); ++md)
        cmp_block_sum(dlt, dund, philox_block(STREAM_DIFF | md, ps, pw, rk), P.tdm[2 * md], P.tdm[2 * md + 1], P.sd[2 * md],
                      P.sd[2 * md + 1]);
    {
        // close the signed sum: lanes still equal to T after the last plane looked at are not < T
        const uint32_t cl = (uint32_t)P.cld[md];
        dlt.lo += dund.lo * cl;
        dlt.hi += dund.hi * cl;
        if (P.thd.all) dlt.lo = dlt.hi = ~0u;   // T_d = 2^32: always (T_d = 0: no planes, lt stays 0)
    }
    if (!P.pmask_paper) {
#pragma unroll
        for (int m = 0; m < NU_P; ++m)
            cmp_block_sum(plt, pund, blks[1 + NU_D + m], P.tpm[2 * m], P.tpm[2 * m + 1], P.sp[2 * m], P.sp[2 * m + 1]);
        for (; mp < nblkP && __any_sync(0xffffffffu, (pund.lo | pund.hi) != 0u); ++mp)
            cmp_block_sum(plt, pund, philox_block(STREAM_ANNI | mp, ps, pw, rk), P.tpm[2 * mp], P.tpm[2 * mp + 1], P.sp[2 * mp],
                          P.sp[2 * mp + 1]);
        const uint32_t cl = (uint32_t)P.clp[mp];
        plt.lo += pund.lo * cl;
        plt.hi += pund.hi * cl;
        if (P.thp.all) plt.lo = plt.hi = ~0u;
    } else if constexpr (NU_P >= 1) {
        // the paper's own annihilation mask (Alg. 2 lines 12-13): an independent b-bit per
        // lane (b = 1/4: the two planes of ANNI block 0 ANDed; pmask_dec) gated by ONE word-wide draw that is 1 w.p. p/b
        // (x3 of the MISC block)
        const U4 &pb = blks[1 + NU_D];
        const uint32_t gate = misc.x3 < P.T4p ? ~0u : 0u;
        plt.lo = pmask_dec(pb.x0, pb.x2, P.pmask_code) & gate;
        plt.hi = pmask_dec(pb.x1, pb.x3, P.pmask_code) & gate;
    }
    const uint32_t y0 = footprint_start(misc.x2, dp, P.Ts);
    uint4 *rec = reinterpret_cast<uint4 *>(slot);
    rec[lane] = make_uint4(y0, ~misc.x0, dlt.lo, plt.lo);
    rec[32 + lane] = make_uint4(y0, ~misc.x1, dlt.hi, plt.hi);
}

__device__ __forceinline__ void named_barrier_sync(uint32_t id, uint32_t nthreads)
{
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

}  // namespace

// Block = NPROD = blockDim.x / 32 - 2 producer warps (warps 0 .. NPROD-1) + 2 update warps (the LAST two: the warp
// scheduler prefers the highest warp index among eligible warps, and the update warps' dependent chain is the
// critical path); grid = tile columns.
// Shared memory: two planes of (T_s + 2) 32-bit words | ring of COL_RING_PER_PRODUCER * NPROD records | full / empty mbarriers.
template <int VARIANT, int NU_D, int NU_P>
__global__ void __launch_bounds__(512, 1) column_kernel(const __grid_constant__ SweepParams P)
{
    extern __shared__ __align__(16) uint8_t csmem[];
    const uint32_t Ts = P.Ts, D = P.D, A = P.A, L = P.L, S = P.S, n = P.n, t = P.t;
    const RoundKeys &rk = P.rk;
    const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31u;
    const uint32_t nprod = (blockDim.x >> 5) - 2u, slots = COL_RING_PER_PRODUCER * nprod;
    const uint32_t task = blockIdx.x, ntiles = L / Ts;
    const uint32_t J = S * A;   // attempts per domain and sweep (= D)

    const uint32_t pstride = (Ts + 5u) & ~3u;   // words per plane (multiple of 4: planes stay 16-byte aligned)
    uint32_t *plane0 = reinterpret_cast<uint32_t *>(csmem);
    uint8_t *ring = csmem + (((size_t)2u * pstride * 4u + 127u) & ~(size_t)127u);
    uint64_t *fullb = reinterpret_cast<uint64_t *>(ring + (size_t)slots * COL_REC_BYTES);
    uint64_t *emptyb = fullb + slots;

    if (threadIdx.x == 0) {
        for (uint32_t c = 0; c < slots; ++c) {
            mbar_init(fullb + c, 1u);    // the producer's lane 0 arrives once its warp has written the record
            mbar_init(emptyb + c, 2u);   // lane 0 of each update warp arrives once its warp has read its half
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const uint32_t tau = task % ntiles, wl = task / ntiles;
    if (warp < nprod) {
        // ---------------------------------------------------------------- producers
        // producer `warp` takes attempts j = warp, warp + nprod, ...; all index arithmetic is kept incremental
        const uint32_t b = lane < n ? lane : 0u;
        const PhiloxWarp pw = philox_warp_consts(t, P.word_offset + wl, rk);
        const uint32_t slot0 = (tau * n + b) * D;     // C5 step 4: slot g = (tau n + b) D + k A + a = slot0 + j
        uint32_t sig = 0u, sig_group = ~0u;           // lane l holds sigma of sub-step 32 * sig_group + l (C5 step 1)
        uint32_t kk = warp / A, a = warp % A;         // sub-step and attempt within it of attempt j
        const uint32_t dk = nprod / A, da = nprod % A;
        uint32_t rslot = warp % slots, rpass = warp / slots;   // ring slot j % slots and pass j / slots (nprod <= slots)
        for (uint32_t j = warp; j < J; j += nprod) {
            if ((kk >> 5) != sig_group) {
                sig_group = kk >> 5;
                sig = __umulhi(philox4x32_10(32u * sig_group + lane, t, 0u, STREAM_SHIFT, rk).x0, D);
            }
            const uint32_t sigma = __shfl_sync(0xffffffffu, sig, kk & 31u);
            mbar_wait(emptyb + rslot, (rpass & 1u) ^ 1u);   // (a fresh barrier passes a wait on parity 1)
            produce_column_record<NU_D, NU_P>(P, pw, slot0 + j, b, lane, sigma, ring + (size_t)rslot * COL_REC_BYTES);
            __syncwarp();
            if (lane == 0) mbar_arrive(fullb + rslot);
            kk += dk; a += da;
            if (a >= A) { a -= A; ++kk; }
            rslot += nprod;
            if (rslot >= slots) { rslot -= slots; ++rpass; }
        }
        return;
    }

    // -------------------------------------------------------------------- update warps
    const uint32_t h = warp - nprod;                   // this warp's half of the 64 replica lanes
    const uint32_t utid = threadIdx.x - nprod * 32u;   // 0 .. 63 over the two update warps
    uint32_t *pl = plane0 + (size_t)h * pstride;       // pl[y], y in [0, Ts): bits 32h .. 32h+31 of tile word y
    uint32_t Sigma;
    {
        const U4 blk = philox4x32_10(0u, t, 0u, STREAM_SHIFT, rk);
        Sigma = __umulhi(blk.x1, Ts);              // C5 step 1 (tile shift); the inner shifts are the producers' business
    }
    const uint32_t start = (uint32_t)(((uint64_t)Sigma + (uint64_t)tau * Ts) % L);   // C5 step 2
    uint64_t *g = P.lat + (size_t)wl * L;
    const uint32_t conn = P.connected;
    // tile load by the 64 update threads: 64-bit words, split into the two planes
    for (uint32_t y = utid; y < Ts; y += 64u) {
        uint32_t i = start + y, rot = 0u;
        if (i >= L) { i -= L; rot = conn; }        // connected multispin lattice (C10): bit rotation past the ring wrap
        const uint64_t v = rotr64(g[i], rot);
        plane0[y] = (uint32_t)v;
        plane0[pstride + y] = (uint32_t)(v >> 32);
    }
    named_barrier_sync(1u, 64u);

    const bool act = lane < n;
    const uint4 *rec = reinterpret_cast<const uint4 *>(ring) + h * 32u + lane;   // this lane's record in slot 0

    // One attempt (C6 / Alg. 2, branch-free over the 32 replicas of this half) with record r = {y0, Fm, Dm, Pm}.
    auto attempt = [&](const uint4 &r) {
        uint32_t *q = pl + r.x;
        const uint32_t Fm = r.y, Dm = r.z, Pm = r.w;
        if (act) {
            uint32_t sa = q[0], sb = q[1], sc = q[2], se = 0u, sf = 0u, sg = 0u;
            if constexpr (VARIANT != 3) se = q[3];
            if constexpr (VARIANT == 1 || VARIANT == 2) sf = q[4];
            if constexpr (VARIANT == 2) sg = q[5];
            uint32_t react = sb & ~Dm;   // particle cluster (1, 2, 3 or 4 sites from x) present and no diffusion
            if constexpr (VARIANT != 3) react &= sc;
            if constexpr (VARIANT == 1 || VARIANT == 2) react &= se;
            if constexpr (VARIANT == 2) react &= sf;
            uint32_t nb = (Dm & sc) | (~Dm & sb);
            uint32_t nc = (Dm & sb) | (~Dm & sc);
            const uint32_t ann = react & Pm, fis = react & ~Pm;
            nb &= ~ann;
            if constexpr (VARIANT != 3) nc &= ~ann;
            sa |= fis & Fm;
            if constexpr (VARIANT == 3) {          // CPD: fission high -> x+1
                nc |= fis & ~Fm;
            } else if constexpr (VARIANT == 0) {   // PCPD: high -> x+2
                se |= fis & ~Fm;
            } else if constexpr (VARIANT == 1) {   // TCPD: high -> x+3
                se &= ~ann;
                sf |= fis & ~Fm;
                q[4] = sf;
            } else {                               // QCPD: high -> x+4
                se &= ~ann;
                sf &= ~ann;
                sg |= fis & ~Fm;
                q[4] = sf;
                q[5] = sg;
            }
            q[0] = sa; q[1] = nb; q[2] = nc;
            if constexpr (VARIANT != 3) q[3] = se;
        }
    };
    // take the record of the next attempt out of the ring (it is read one attempt ahead of its use)
    uint32_t rslot = 0u, rphase = 0u;
    auto take = [&]() -> uint4 {
        mbar_wait(fullb + rslot, rphase);
        const uint4 r = rec[(size_t)rslot * (COL_REC_BYTES / 16u)];
        __syncwarp();
        if (lane == 0) mbar_arrive(emptyb + rslot);
        if (++rslot == slots) { rslot = 0u; rphase ^= 1u; }
        return r;
    };
    uint4 r0 = take(), r1;
    uint32_t a_in_substep = 0u;
    auto end_of_attempt = [&]() {
        if (++a_in_substep == A) {                 // end of a sub-step: the domains move (C5 step 3)
            a_in_substep = 0u;
            __syncwarp();
        }
    };
    // two attempts per iteration, so that the one-ahead record alternates between two register sets
#pragma unroll 1
    for (uint32_t j = 0; j + 1u < J; j += 2u) {
        r1 = take();
        attempt(r0);
        end_of_attempt();
        if (j + 2u < J) r0 = take();
        attempt(r1);
        end_of_attempt();
    }
    if (J & 1u) attempt(r0);   // (odd D)

    // ---- store the tile: both planes back into 64-bit words ----
    named_barrier_sync(1u, 64u);
    for (uint32_t y = utid; y < Ts; y += 64u) {
        uint32_t i = start + y, rot = 0u;
        if (i >= L) { i -= L; rot = conn; }
        const uint64_t v = (uint64_t)plane0[y] | ((uint64_t)plane0[pstride + y] << 32);
        g[i] = rotl64(v, rot);
    }
}

}  // namespace pcpd
