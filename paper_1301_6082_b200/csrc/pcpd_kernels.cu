// Hand-written sm_100a kernels of the PCPD/TCPD multispin hot path
// (DESIGN.md sections 4-5): sweep (RNG + masks + schedule + bitwise rule), init,
// density (positional popcount), layout transpose.
//
// Citations: update rule = Alg. 1 PAPER.md:45-70 in the bitwise form of Alg. 2
// PAPER.md:126-151 (typos fixed per DESIGN.md readings G5/G6); schedule SD2 and
// streams = DESIGN.md section 3 C1-C9.
#include "pcpd_kernels.cuh"

namespace pcpd {

__device__ __forceinline__ uint32_t mulhi32(uint32_t r, uint32_t n) { return __umulhi(r, n); }

// ---------------------------------------------------------------------------
// Bernoulli(T / 2^32) mask by MSB-first bit-sliced comparison of the 32 random
// planes with the bits of T (C3), evaluated LAZILY: only lanes in `rel` (the
// lanes on which the outcome can matter) are resolved, and the loop stops as
// soon as every such lane is decided.  A lane is decided at the first plane
// where its bit differs from T's bit; counter-based RNG makes the skipped
// blocks free.  Returns lanes (within rel) with U < T.
// Plane k (k even) = lo64, (k odd) = hi64 of block m = k >> 1 of `stream`.
template <uint32_t STREAM>
__device__ __forceinline__ uint64_t lazy_mask(uint64_t rel, const Threshold th, uint32_t slot, uint32_t t,
                                              uint32_t w, const RoundKeys &rk)
{
    if (th.all) return rel;
    uint64_t lt = 0, und = rel;
    for (uint32_t k = 0; k < th.nplanes && und != 0; k += 2) {
        const U4 blk = philox4x32_10(slot, t, w, STREAM | (k >> 1), rk);
        // T's bit for plane k is bit (31 - k); thread-uniform.
        const uint64_t tb0 = ((th.T32 >> (31 - k)) & 1u) ? ~0ull : 0ull;
        const uint64_t tb1 = ((th.T32 >> (30 - k)) & 1u) ? ~0ull : 0ull;  // k <= 30
        uint64_t pl = lo64(blk);
        lt |= und & ~pl & tb0;   // T bit 1, lane bit 0 -> U < T
        und &= ~(pl ^ tb0);      // stays undecided only where lane bit == T bit
        pl = hi64(blk);
        lt |= und & ~pl & tb1;
        und &= ~(pl ^ tb1);
    }
    return lt;
}

// ---------------------------------------------------------------------------
// GENERIC FALLBACK (schedules with more than 32 domains per tile).  One sweep of schedule
// SD2(Ts, D, A) (C5).  Grid (L/Ts tiles, W word columns); block = n threads, thread b owns
// domain b of the block's tile column for the whole sweep; the tile column lives in shared
// memory from load to store, so the lattice crosses HBM exactly once in each direction per sweep.
template <int VARIANT>
__global__ void sweep_kernel(const __grid_constant__ SweepParams P)
{
    extern __shared__ __align__(16) uint64_t tile[];  // [Ts]
    __shared__ uint32_t s_sigma[MAX_SUBSTEPS];
    __shared__ uint32_t s_Sigma;

    constexpr uint32_t Rr = VARIANT == 3 ? 1u : 2u + VARIANT;  // right reach: 2 PCPD, 3 TCPD, 4 QCPD, 1 CPD
    const uint32_t tid = threadIdx.x, nthr = blockDim.x;
    const uint32_t tau = blockIdx.x, wg = blockIdx.y;
    const uint32_t Ts = P.Ts, D = P.D, A = P.A, S = P.S, n = P.n, L = P.L, t = P.t;

    // C5 step 1: shifts from the SHIFT stream.
    for (uint32_t k = tid; k < S; k += nthr) {
        const U4 blk = philox4x32_10(k, t, 0u, STREAM_SHIFT, P.rk);
        s_sigma[k] = mulhi32(blk.x0, D);
        if (k == 0) s_Sigma = mulhi32(blk.x1, Ts);
    }
    __syncthreads();

    // C5 step 2: tile tau covers global sites (Sigma + tau*Ts + y) mod L.
    const uint32_t start = (uint32_t)(((uint64_t)s_Sigma + (uint64_t)tau * Ts) % L);
    uint64_t *g = P.lat + (size_t)wg * L;
    for (uint32_t y = tid; y < Ts; y += nthr) {
        uint32_t i = start + y, rot = 0;
        if (i >= L) { i -= L; rot = P.connected; }  // connected multispin lattice (C10): bit rotation past the wrap
        const uint64_t v = g[i];
        tile[y] = (v >> rot) | (v << ((64u - rot) & 63u));
    }
    __syncthreads();

    const uint32_t b = tid;
    const uint32_t w = P.word_offset + wg;  // global word index (RNG key)
    const uint32_t slot0 = (tau * n + b) * D;

    for (uint32_t k = 0; k < S; ++k) {
        const uint32_t sigma = s_sigma[k];
        // C5 step 3-4: only domain n-1 with sigma > 0 wraps; seam between
        // domain-local c-1 and c, c = D - sigma; positions [c-Rr, c] are excluded.
        const bool seam = (b == n - 1) && (sigma > 0);
        const int32_t c = (int32_t)D - (int32_t)sigma;
        int32_t lo = 0, rem = 0;
        if (seam) {
            lo = max(1, c - (int32_t)Rr);
            const int32_t hi = min((int32_t)D - 1 - (int32_t)Rr, c);
            rem = max(0, hi - lo + 1);
        }
        const uint32_t n_allow = D - 1 - Rr - (uint32_t)rem;
        const uint32_t dbase = sigma + b * D;  // tile-local index of domain-local 0 (before wrap)

        for (uint32_t a = 0; a < A; ++a) {
            const uint32_t slot = slot0 + k * A + a;
            // C4: MISC block: Fm = ~lo, x2 -> position.
            const U4 misc = philox4x32_10(slot, t, w, STREAM_MISC, P.rk);
            int32_t x = 1 + (int32_t)mulhi32(misc.x2, n_allow);
            if (rem > 0 && x >= lo) x += rem;
            uint32_t y0 = dbase + (uint32_t)x - 1;  // footprint x-1 .. x+Rr never straddles the seam
            if (y0 >= Ts) y0 -= Ts;
            uint64_t *q = tile + y0;

            uint64_t sa = q[0], sb = q[1], sc = q[2];
            uint64_t se = 0, sf = 0, sg = 0;
            if constexpr (VARIANT != 3) se = q[3];
            if constexpr (VARIANT == 1 || VARIANT == 2) sf = q[4];
            if constexpr (VARIANT == 2) sg = q[5];

            // C6 / Alg. 2, branch-free over the 64 replicas.
            const uint64_t Dm = lazy_mask<STREAM_DIFF>(sb | sc, P.thd, slot, t, w, P.rk);
            uint64_t react = sb & ~Dm;  // particle cluster present and no diffusion
            if constexpr (VARIANT != 3) react &= sc;
            if constexpr (VARIANT == 1 || VARIANT == 2) react &= se;
            if constexpr (VARIANT == 2) react &= sf;
            const uint64_t Pm = lazy_mask<STREAM_ANNI>(react, P.thp, slot, t, w, P.rk);
            const uint64_t Fm = ~lo64(misc);  // 1 -> fission low (Alg. 1: r3 < 1/2)
            uint64_t nb = (Dm & sc) | (~Dm & sb);
            uint64_t nc = (Dm & sb) | (~Dm & sc);
            const uint64_t ann = react & Pm;
            const uint64_t fis = react & ~Pm;
            nb &= ~ann;
            if constexpr (VARIANT != 3) nc &= ~ann;
            sa |= fis & Fm;
            if constexpr (VARIANT == 3) {
                nc |= fis & ~Fm;
            } else if constexpr (VARIANT == 0) {
                se |= fis & ~Fm;
            } else if constexpr (VARIANT == 1) {
                se &= ~ann;
                sf |= fis & ~Fm;
                q[4] = sf;
            } else {
                se &= ~ann;
                sf &= ~ann;
                sg |= fis & ~Fm;
                q[4] = sf;
                q[5] = sg;
            }
            q[0] = sa;
            q[1] = nb;
            q[2] = nc;
            if constexpr (VARIANT != 3) q[3] = se;
        }
        __syncthreads();
    }

    // store the tile
    for (uint32_t y = tid; y < Ts; y += nthr) {
        uint32_t i = start + y, rot = 0;
        if (i >= L) { i -= L; rot = P.connected; }
        const uint64_t v = tile[y];
        g[i] = (v << rot) | (v >> ((64u - rot) & 63u));
    }
}

size_t sweep_smem_bytes(uint32_t Ts) { return (size_t)Ts * 8; }

template <int VARIANT>
static int launch_sweep_t(const SweepParams &P, cudaStream_t stream)
{
    dim3 grid(P.L / P.Ts, P.W);
    dim3 block(P.n);
    sweep_kernel<VARIANT><<<grid, block, sweep_smem_bytes(P.Ts), stream>>>(P);
    return 1;
}

// The production path is the warp-per-(tile, column) kernel of sweep_warp.cu; the block kernel
// above only serves schedules with more than 32 domains per tile.
int launch_sweep(const SweepParams &P, int variant, bool force_block_kernel, cudaStream_t stream, JitSlot *jit,
                 SplitSlot *split)
{
    if (sweep_warp_supported(P.Ts, P.D) && !force_block_kernel)
        return launch_sweep_warp(P, variant, sweep_warp_wpb(P.Ts, (uint64_t)(P.L / P.Ts) * P.W), stream, jit, split);
    return variant == 0 ? launch_sweep_t<0>(P, stream) : variant == 1 ? launch_sweep_t<1>(P, stream)
           : variant == 2 ? launch_sweep_t<2>(P, stream) : launch_sweep_t<3>(P, stream);
}

int configure_kernels()
{
    cudaError_t e;
    if ((e = cudaFuncSetAttribute(sweep_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024)) != cudaSuccess)
        return (int)e;
    if ((e = cudaFuncSetAttribute(sweep_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024)) != cudaSuccess)
        return (int)e;
    if ((e = cudaFuncSetAttribute(sweep_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024)) != cudaSuccess)
        return (int)e;
    if ((e = cudaFuncSetAttribute(sweep_kernel<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024)) != cudaSuccess)
        return (int)e;
    return configure_warp_kernels();
}

}  // namespace pcpd
