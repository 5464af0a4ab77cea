// sweep_warp.cu - host side of the two sweep kernels: sweep_warp_kernel (sweep_warp_device.cuh; large problems) and
// column_kernel (column_device.cuh; small and mid-size problems): instantiations for the generic-threshold
// kernels built into libpcpd.so, launch configuration, and the dispatch to the threshold-specialised kernels
// compiled at run time (jit.cu).
#include <cstdlib>

#include "sweep_warp_device.cuh"
#include "column_device.cuh"

namespace pcpd {

// ---------------------------------------------------------------------------
static size_t warp_smem_bytes(uint32_t Ts, int wpb) { return (size_t)wpb * ((Ts + 3u) & ~1u) * 8; }

bool sweep_warp_supported(uint32_t Ts, uint32_t D)
{
    return Ts / D <= 32 && warp_smem_bytes(Ts, 1) <= 200 * 1024;
}

// warps per block: as many as fit 227 KB / SM in at most a few blocks
int sweep_warp_wpb(uint32_t Ts, uint64_t ntasks)
{
    if (ntasks < 148ull * 14) return 1;    // small problem: one warp per block so that the warps spread over all SMs
    const size_t per = warp_smem_bytes(Ts, 1);
    if (7 * per <= 113 * 1024) return 7;   // 2 blocks x 7 warps per SM at T_s = 2048 (2 x (114800 + 1024) B)
    return 1;
}

// prefix lengths for a threshold with nblk blocks (tuned on B200 at cfg4)
#ifndef PCPD_NUD_BIG
#define PCPD_NUD_BIG 5
#endif
#ifndef PCPD_NUP_BIG
#define PCPD_NUP_BIG 4
#endif
static int nu_d_of(uint32_t nblk) { return nblk == 0 ? 0 : nblk < PCPD_NUD_BIG ? 1 : PCPD_NUD_BIG; }
static int nu_p_of(uint32_t nblk) { return nblk == 0 ? 0 : nblk < PCPD_NUP_BIG ? 1 : PCPD_NUP_BIG; }

template <int VARIANT, int WPB, int NU_D, int NU_P, int PMODE, int PW = 0>
static int warp_op(const SweepParams *P, cudaStream_t stream)
{
    if (!P)  // configure
        return (int)cudaFuncSetAttribute(sweep_warp_kernel<VARIANT, WPB, NU_D, NU_P, PMODE, PW>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         WPB >= 4 ? 116 * 1024 : 226 * 1024);
    const uint32_t ntasks = (P->L / P->Ts) * P->W;
    sweep_warp_kernel<VARIANT, WPB, NU_D, NU_P, PMODE, PW>
        <<<(ntasks + WPB - 1) / WPB, WPB * 32, warp_smem_bytes(P->Ts, WPB), stream>>>(*P);
    return 1;
}

template <int VARIANT, int WPB, int NU_D>
static int warp_op_p(int nup, const SweepParams *P, cudaStream_t stream)
{
    if (nup == -2) return warp_op<VARIANT, WPB, PCPD_NUD_BIG, PCPD_NUP_BIG, 0, 1>(P, stream);  // per-word thresholds
    if (nup == -1) return warp_op<VARIANT, WPB, NU_D, 1, 1>(P, stream);  // paper annihilation mask: ANNI block 0 only
    if (nup == 0) return warp_op<VARIANT, WPB, NU_D, 0, 0>(P, stream);
    if (nup == 1) return warp_op<VARIANT, WPB, NU_D, 1, 0>(P, stream);
    return warp_op<VARIANT, WPB, NU_D, PCPD_NUP_BIG, 0>(P, stream);
}

template <int VARIANT, int WPB>
static int warp_op_d(int nud, int nup, const SweepParams *P, cudaStream_t stream)
{
    if (nud == 0) return warp_op_p<VARIANT, WPB, 0>(nup, P, stream);
    if (nud == 1) return warp_op_p<VARIANT, WPB, 1>(nup, P, stream);
    return warp_op_p<VARIANT, WPB, PCPD_NUD_BIG>(nup, P, stream);
}

static int warp_op_any(int variant, int wpb, int nud, int nup, const SweepParams *P, cudaStream_t stream)
{
    if (variant == 3)
        return wpb == 7 ? warp_op_d<3, 7>(nud, nup, P, stream) : warp_op_d<3, 1>(nud, nup, P, stream);
    if (variant == 2)
        return wpb == 7 ? warp_op_d<2, 7>(nud, nup, P, stream) : warp_op_d<2, 1>(nud, nup, P, stream);
    if (variant == 0)
        return wpb == 7 ? warp_op_d<0, 7>(nud, nup, P, stream) : warp_op_d<0, 1>(nud, nup, P, stream);
    return wpb == 7 ? warp_op_d<1, 7>(nud, nup, P, stream) : warp_op_d<1, 1>(nud, nup, P, stream);
}

// ---- column_kernel: one block per tile column, producer warps + two update warps (column_device.cuh) ----
static size_t column_smem_bytes(uint32_t Ts, uint32_t nprod)
{
    const size_t pstride = (Ts + 5u) & ~3u, slots = (size_t)COL_RING_PER_PRODUCER * nprod;
    return ((2 * pstride * 4 + 127) & ~(size_t)127) + slots * COL_REC_BYTES + 2 * slots * 8;
}

bool column_supported(uint32_t Ts, uint32_t D) { return Ts / D <= 32 && column_smem_bytes(Ts, 2) <= 226 * 1024; }

// Up to how many tile columns column_kernel beats the fused warp kernel (run-time specialised) - measured on B200 at
// L = 65536: its time grows with the blocks per SM, the fused kernel's only with the waves of 592
// warps, and the fewer Philox blocks the thresholds need, the earlier the fused kernel wins: both thresholds long
// (generic d and p) 768 columns (82 vs 91 us); one long (d = 1/2, generic p; also TCPD) 384 (35 vs 37 us; 512: 42 vs 37);
// none (dyadic d with the paper's annihilation mask) 296 = two blocks per SM (16 vs 21 us; 384: 31 vs 21).
uint64_t column_task_limit(const SweepParams &P)
{
    const bool long_d = ((P.thd.nplanes + 1u) >> 1) >= (uint32_t)5;
    const bool long_p = !P.pmask_paper && ((P.thp.nplanes + 1u) >> 1) >= (uint32_t)5;
    return long_d && long_p ? 768u : (long_d || long_p) ? 384u : 296u;
}

// producer warps per block (measured on B200 at L = 65536, generic thresholds): 14 (a 16-warp
// block) while every tile column has an SM of its own - cfg2: 18.6 us per sweep with 14, 20.5 with 8, 26.6 with 4 -
// and 8 (a 10-warp block, six of which share an SM) beyond: 256 columns 30.8 us (4: 33.2, 14: 34.9), 512 columns
// 57.4 us (4: 63.2, 14: 67.3).
static uint32_t column_nprod(uint32_t Ts, uint64_t ntasks)
{
    if (const char *e = getenv("PCPD_COL_NPROD")) {   // tuning hook
        const int v = atoi(e);
        if (v >= 1 && v <= 14) return (uint32_t)v;
    }
    uint32_t np = ntasks <= 148 ? 14u : 8u;
    while (np > 1 && column_smem_bytes(Ts, np) > 226 * 1024) --np;
    return np;
}

// prefix lengths of the producers (5 + 5 interleaved chains beside the MISC block for thresholds with that many blocks:
// all 64 lanes of 32 domains need 6.4 blocks per stream on average; 1 for short thresholds, 0 for T = 0 or 2^32)
constexpr int COL_NU_BIG = 5;
static int col_nu_of(uint32_t nblk) { return nblk == 0 ? 0 : nblk < (uint32_t)COL_NU_BIG ? 1 : COL_NU_BIG; }

template <int VARIANT, int NU_D, int NU_P>
static int column_op(const SweepParams *P, uint32_t nprod, cudaStream_t stream)
{
    if (!P)
        return (int)cudaFuncSetAttribute(column_kernel<VARIANT, NU_D, NU_P>, cudaFuncAttributeMaxDynamicSharedMemorySize, 226 * 1024);
    column_kernel<VARIANT, NU_D, NU_P><<<(P->L / P->Ts) * P->W, (2 + nprod) * 32, column_smem_bytes(P->Ts, nprod), stream>>>(*P);
    return 1;
}

template <int VARIANT, int NU_D>
static int column_op_p(int nup, const SweepParams *P, uint32_t nprod, cudaStream_t stream)
{
    if (nup == 0) return column_op<VARIANT, NU_D, 0>(P, nprod, stream);
    if (nup == 1) return column_op<VARIANT, NU_D, 1>(P, nprod, stream);
    return column_op<VARIANT, NU_D, COL_NU_BIG>(P, nprod, stream);
}

template <int VARIANT>
static int column_op_d(int nud, int nup, const SweepParams *P, uint32_t nprod, cudaStream_t stream)
{
    if (nud == 0) return column_op_p<VARIANT, 0>(nup, P, nprod, stream);
    if (nud == 1) return column_op_p<VARIANT, 1>(nup, P, nprod, stream);
    return column_op_p<VARIANT, COL_NU_BIG>(nup, P, nprod, stream);
}

static int column_any(int variant, int nud, int nup, const SweepParams *P, uint32_t nprod, cudaStream_t stream)
{
    switch (variant) {
    case 0: return column_op_d<0>(nud, nup, P, nprod, stream);
    case 1: return column_op_d<1>(nud, nup, P, nprod, stream);
    case 2: return column_op_d<2>(nud, nup, P, nprod, stream);
    default: return column_op_d<3>(nud, nup, P, nprod, stream);
    }
}

static int launch_sweep_column(const SweepParams &P0, int variant, cudaStream_t stream, SplitSlot *split)
{
    SweepParams P = P0;
    P.rr = variant == 3 ? 1u : 2u + (uint32_t)variant;
    const int nud = col_nu_of((P.thd.nplanes + 1u) >> 1);
    const int nup = P.pmask_paper ? 1 : col_nu_of((P.thp.nplanes + 1u) >> 1);   // (paper mask: ANNI block 0 only)
    column_any(variant, nud, nup, &P, column_nprod(P.Ts, (uint64_t)(P.L / P.Ts) * P.W), stream);
    split->launches += 1;
    return 1;
}

int launch_sweep_warp(const SweepParams &P, int variant, int wpb, cudaStream_t stream, JitSlot *jit, SplitSlot *split)
{
    if (P.thr_dev) return warp_op_any(variant, wpb, PCPD_NUD_BIG, -2, &P, stream);
    if (split && split->column_mode && !(jit && jit->mode == 2)) return launch_sweep_column(P, variant, stream, split);
    const int nup = P.pmask_paper ? -1 : nu_p_of((P.thp.nplanes + 1) >> 1);
    const int nud = nu_d_of((P.thd.nplanes + 1) >> 1);
    // Threshold-specialised kernel (jit.cu): every handle the fused kernel serves by default (more tile columns than
    // column_task_limit; measured 9-10 % faster than the built-in kernel at 1024 and 2048 columns too), or every size with
    // PCPD_JIT=force.  Not
    // for T = 2^32 (d = 1 or p = 1; the template constants hold 32 bits).  If it cannot be had, the built-in
    // kernel below computes the same thing.
    const uint64_t ntasks_all = (uint64_t)(P.L / P.Ts) * P.W;
    if (jit && jit->mode && jit->state >= 0 && (jit->mode == 2 || ntasks_all > column_task_limit(P)) && !P.thd.all && !P.thp.all) {
        if (jit->state == 0) {
            // prefix lengths of the specialised kernel: all of a short threshold's blocks, else 6 DIFF / 4 ANNI (5 for
            // TCPD and QCPD) (tuned on B200 at cfg3-5: its prefix compare is cheaper than the built-in kernel's)
            JitSpec js;
            js.variant = variant; js.wpb = wpb; js.pmode = P.pmask_paper ? 2 + (int)P.pmask_code : 0;   // (bound code baked in)
            js.nud = (int)min((P.thd.nplanes + 1) >> 1, 6u);
            js.nup = P.pmask_paper ? 1 : (int)min((P.thp.nplanes + 1) >> 1, variant == 1 || variant == 2 ? 5u : 4u);
            if (const char *e = getenv("PCPD_JIT_NUD")) js.nud = atoi(e);   // tuning hooks
            if (const char *e = getenv("PCPD_JIT_NUP")) js.nup = atoi(e);
            js.Td = P.thd.T32; js.Tp = P.thp.T32; js.Ts = P.Ts; js.D = P.D; js.A = P.A; js.L = P.L;
            jit->kernel = jit_sweep_kernel(js, wpb >= 4 ? 116 * 1024 : 226 * 1024);
            jit->state = jit->kernel ? 1 : -1;
            jit->wpb = wpb;
        }
        if (jit->state == 1 && jit->wpb == wpb) {
            const uint32_t ntasks = (P.L / P.Ts) * P.W;
            if (jit_launch(jit->kernel, P, (ntasks + wpb - 1) / wpb, wpb * 32, warp_smem_bytes(P.Ts, wpb), stream) == 0)
                return 1;
            jit->state = -1;
        }
    }
    return warp_op_any(variant, wpb, nud, nup, &P, stream);
}

int configure_warp_kernels()
{
    const int nuds[3] = {0, 1, PCPD_NUD_BIG}, nups[4] = {-1, 0, 1, PCPD_NUP_BIG}, wpbs[2] = {7, 1};
    for (int variant = 0; variant < 4; ++variant)
        for (int wpb : wpbs) {
            for (int nud : nuds)
                for (int nup : nups) {
                    const int e = warp_op_any(variant, wpb, nud, nup, nullptr, nullptr);
                    if (e != 0) return e;
                }
            const int e = warp_op_any(variant, wpb, PCPD_NUD_BIG, -2, nullptr, nullptr);
            if (e != 0) return e;
        }
    for (int variant = 0; variant < 4; ++variant)
        for (int nud : {0, 1, COL_NU_BIG})
            for (int nup : {0, 1, COL_NU_BIG}) {
                const int e = column_any(variant, nud, nup, nullptr, 0, nullptr);
                if (e != 0) return e;
            }
    return 0;
}

}  // namespace pcpd
