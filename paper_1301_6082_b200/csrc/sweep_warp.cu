// sweep_warp.cu - host side of the production sweep kernel (device code: sweep_warp_device.cuh):
// instantiations for the generic-threshold kernels built into libpcpd.so, launch configuration,
// and the dispatch to the threshold-specialised kernels compiled at run time (jit.cu).
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

// ---- SPLIT path for small problems: mask_kernel (all attempts of the sweep in parallel) + consumer kernel ----
// consumer's shared memory: tile buffer, the task's J mask records (TMA bulk copies), one mbarrier per chunk
static size_t split_smem_bytes(uint32_t Ts, uint32_t J)
{
    return ((warp_smem_bytes(Ts, 1) + 127) & ~(size_t)127) + (size_t)J * MASK_REC_BYTES + MASK_MAX_CHUNKS * 8;
}

bool split_supported(uint32_t Ts, uint32_t D)   // J = S * A = D attempts per domain and sweep
{
    return sweep_warp_supported(Ts, D) && split_smem_bytes(Ts, D) <= 226 * 1024;
}

template <int VARIANT, int PMODE>
static int split_consumer_op(const SweepParams *P, cudaStream_t stream)
{
    auto kern = sweep_warp_kernel<VARIANT, 1, 0, 0, PMODE, 0, 0, 0u, 0u, 0u, 0u, 0u, 0u, 2>;
    if (!P) return (int)cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 226 * 1024);
    kern<<<(P->L / P->Ts) * P->W, 32, split_smem_bytes(P->Ts, P->S * P->A), stream>>>(*P);
    return 1;
}

static int split_consumer_any(int variant, int pmode, const SweepParams *P, cudaStream_t stream)
{
    switch (variant * 2 + pmode) {
    case 0: return split_consumer_op<0, 0>(P, stream);
    case 1: return split_consumer_op<0, 1>(P, stream);
    case 2: return split_consumer_op<1, 0>(P, stream);
    case 3: return split_consumer_op<1, 1>(P, stream);
    case 4: return split_consumer_op<2, 0>(P, stream);
    case 5: return split_consumer_op<2, 1>(P, stream);
    case 6: return split_consumer_op<3, 0>(P, stream);
    default: return split_consumer_op<3, 1>(P, stream);
    }
}

// ---- SPLIT = 3: producer warps and the update warp in ONE block per tile column (records through a shared-memory ring)
static size_t block4_smem_bytes(uint32_t Ts, int wpb)
{
    const size_t slots = (size_t)RING_PER_PRODUCER * (wpb - 1);
    return ((warp_smem_bytes(Ts, 1) + 127) & ~(size_t)127) + slots * MASK_REC_BYTES + 2 * slots * 8;
}

bool split_block_supported(uint32_t Ts, uint32_t D) { return sweep_warp_supported(Ts, D) && block4_smem_bytes(Ts, 4) <= 226 * 1024; }

template <int VARIANT, int PMODE, int WPB>
static int block4_op(const SweepParams *P, cudaStream_t stream)
{
    auto kern = sweep_warp_kernel<VARIANT, WPB, 0, 0, PMODE, 0, 0, 0u, 0u, 0u, 0u, 0u, 0u, 3>;
    if (!P) return (int)cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 226 * 1024);
    kern<<<(P->L / P->Ts) * P->W, WPB * 32, block4_smem_bytes(P->Ts, WPB), stream>>>(*P);
    return 1;
}

template <int WPB>
static int block4_any_w(int variant, int pmode, const SweepParams *P, cudaStream_t stream)
{
    switch (variant * 2 + pmode) {
    case 0: return block4_op<0, 0, WPB>(P, stream);
    case 1: return block4_op<0, 1, WPB>(P, stream);
    case 2: return block4_op<1, 0, WPB>(P, stream);
    case 3: return block4_op<1, 1, WPB>(P, stream);
    case 4: return block4_op<2, 0, WPB>(P, stream);
    case 5: return block4_op<2, 1, WPB>(P, stream);
    case 6: return block4_op<3, 0, WPB>(P, stream);
    default: return block4_op<3, 1, WPB>(P, stream);
    }
}

// (The kernel takes any number of producer warps; 8-warp blocks were measured on B200 at L = 65536 with an 8 + 8 block
// prefix: 128 columns 33 us, 256 columns 45 us, 512 columns 84 us per sweep against 41 / 47 / 69 us for 4 warps.)
static int block4_any(int variant, int pmode, const SweepParams *P, cudaStream_t stream)
{
    return block4_any_w<4>(variant, pmode, P, stream);
}

static int launch_sweep_block4(const SweepParams &P0, int variant, cudaStream_t stream, SplitSlot *split)
{
    SweepParams P = P0;
    uint32_t cap_d = 7u, cap_p = 5u;   // tuned on B200 (L = 65536, 256 .. 512 tile columns); the producers are issue-bound
    if (const char *e = getenv("PCPD_SPLIT_NUD")) cap_d = (uint32_t)atoi(e);   // tuning hooks
    if (const char *e = getenv("PCPD_SPLIT_NUP")) cap_p = (uint32_t)atoi(e);
    P.split_nud = min((P.thd.nplanes + 1u) >> 1, cap_d);
    P.split_nup = P.pmask_paper ? 1u : min((P.thp.nplanes + 1u) >> 1, cap_p);
    P.rr = variant == 3 ? 1u : 2u + (uint32_t)variant;
    block4_any(variant, P.pmask_paper ? 1 : 0, &P, stream);
    split->launches += 1;
    return 1;
}

// ---- column_kernel: one block per tile column, producer warps + two update warps (column_device.cuh) ----
static size_t column_smem_bytes(uint32_t Ts, uint32_t nprod)
{
    const size_t pstride = (Ts + 5u) & ~3u, slots = (size_t)COL_RING_PER_PRODUCER * nprod;
    return ((2 * pstride * 4 + 127) & ~(size_t)127) + slots * COL_REC_BYTES + 2 * slots * 8;
}

bool column_supported(uint32_t Ts, uint32_t D) { return Ts / D <= 32 && column_smem_bytes(Ts, 2) <= 226 * 1024; }

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

size_t split_mask_bytes(const SweepParams &P) { return (size_t)(P.L / P.Ts) * P.W * P.S * P.A * 96u * sizeof(uint4); }

// Small problems (SplitSlot::buf allocated by the API layer when the handle qualifies): two launches per sweep.
int split_setup(SplitSlot *s)
{
    // lowest priority: mask_kernel's many blocks must not delay the update kernel's, which are the critical path
    int prio_lo = 0, prio_hi = 0;
    cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi);
    if (cudaStreamCreateWithPriority(&s->aux, cudaStreamNonBlocking, prio_lo) != cudaSuccess) return -1;
    for (int i = 0; i < 2; ++i) {
        if (cudaEventCreateWithFlags(&s->ready[i], cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&s->freed[i], cudaEventDisableTiming) != cudaSuccess)
            return -1;
        s->held[i] = -1;
        s->freed_valid[i] = false;
    }
    return 0;
}

void split_teardown(SplitSlot *s)
{
    if (!s->aux) return;
    cudaStreamSynchronize(s->aux);
    for (int i = 0; i < 2; ++i) {
        if (s->ready[i]) cudaEventDestroy(s->ready[i]);
        if (s->freed[i]) cudaEventDestroy(s->freed[i]);
    }
    cudaStreamDestroy(s->aux);
    s->aux = nullptr;
}

// masks of sweep t into buf[t & 1], on the auxiliary stream, once the last reader of that buffer has finished;
// false if a stream / event operation or the launch failed (the CUDA error stays pending for the caller)
static bool split_produce(const SweepParams &P, uint32_t t, SplitSlot *split)
{
    const int i = (int)(t & 1u);
    SweepParams Q = P;
    Q.t = t;
    Q.mask_dev = split->buf[i];
    split->held[i] = -1;
    if (split->freed_valid[i] && cudaStreamWaitEvent(split->aux, split->freed[i], 0) != cudaSuccess) return false;
    const uint32_t nwarps = (Q.L / Q.Ts) * Q.W * Q.S * Q.A;
    mask_kernel<<<(nwarps + 3) / 4, 128, 0, split->aux>>>(Q);
    if (cudaPeekAtLastError() != cudaSuccess) return false;
    if (cudaEventRecord(split->ready[i], split->aux) != cudaSuccess) return false;
    split->held[i] = (int64_t)t;
    return true;
}

// Small problems: two launches per sweep; the masks of sweep t + 1 are produced while sweep t is applied.  Returns the
// number of kernels launched, or -1 if a stream / event operation failed (nothing more is launched then).
static int launch_sweep_split(const SweepParams &P0, int variant, cudaStream_t stream, SplitSlot *split)
{
    SweepParams P = P0;
    // prefix lengths: up to 8 blocks per stream - the producer is parallel over all attempts of the sweep, and every
    // tail iteration it saves the consumer is ~150 cycles on the sequential chain
    P.split_nud = min((P.thd.nplanes + 1u) >> 1, 8u);
    P.split_nup = P.pmask_paper ? 1u : min((P.thp.nplanes + 1u) >> 1, 8u);
    P.rr = variant == 3 ? 1u : 2u + (uint32_t)variant;
    const uint32_t t = P.t;
    const int i = (int)(t & 1u);
    int launched = 1;
    if (split->held[i] != (int64_t)t) {   // not prefetched (first sweep of the handle, or the counter was set)
        if (!split_produce(P, t, split)) return -1;
        ++launched;
    }
    if (t != 0xffffffffu && split->held[i ^ 1] != (int64_t)t + 1) {
        if (!split_produce(P, t + 1u, split)) return -1;
        ++launched;
    }
    if (cudaStreamWaitEvent(stream, split->ready[i], 0) != cudaSuccess) return -1;
    P.mask_dev = split->buf[i];
    split_consumer_any(variant, P.pmask_paper ? 1 : 0, &P, stream);
    if (cudaEventRecord(split->freed[i], stream) != cudaSuccess) {
        split->freed_valid[i] = false;
        split->held[i] = -1;   // the buffer's reader cannot be tracked: do not reuse its contents
        return -1;
    }
    split->freed_valid[i] = true;
    split->launches += (uint64_t)launched;
    return launched;
}

int launch_sweep_warp(const SweepParams &P, int variant, int wpb, cudaStream_t stream, JitSlot *jit, SplitSlot *split)
{
    if (P.thr_dev) return warp_op_any(variant, wpb, PCPD_NUD_BIG, -2, &P, stream);
    if (split && split->block_mode == 2 && !(jit && jit->mode == 2)) return launch_sweep_column(P, variant, stream, split);
    if (split && split->block_mode && !(jit && jit->mode == 2)) return launch_sweep_block4(P, variant, stream, split);
    if (split && split->buf[0] && !(jit && jit->mode == 2)) return launch_sweep_split(P, variant, stream, split);
    const int nup = P.pmask_paper ? -1 : nu_p_of((P.thp.nplanes + 1) >> 1);
    const int nud = nu_d_of((P.thd.nplanes + 1) >> 1);
    // Threshold-specialised kernel (jit.cu): large problems (wpb == 7), or every size with PCPD_JIT=force.  Not
    // for T = 2^32 (d = 1 or p = 1; the template constants hold 32 bits).  If it cannot be had, the built-in
    // kernel below computes the same thing.
    if (jit && jit->mode && jit->state >= 0 && (jit->mode == 2 || wpb == 7) && !P.thd.all && !P.thp.all) {
        if (jit->state == 0) {
            // prefix lengths of the specialised kernel: all of a short threshold's blocks, else 6 DIFF / 4 ANNI (5 for
            // TCPD and QCPD) (tuned on B200 at cfg3-5: its prefix compare is cheaper than the built-in kernel's)
            JitSpec js;
            js.variant = variant; js.wpb = wpb; js.pmode = P.pmask_paper ? 1 : 0;
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
        for (int pmode = 0; pmode < 2; ++pmode) {
            int e = split_consumer_any(variant, pmode, nullptr, nullptr);
            if (e == 0) e = block4_any(variant, pmode, nullptr, nullptr);
            if (e == 0 && pmode == 0)
                for (int nud : {0, 1, COL_NU_BIG})
                    for (int nup : {0, 1, COL_NU_BIG})
                        if (e == 0) e = column_any(variant, nud, nup, nullptr, 0, nullptr);
            if (e != 0) return e;
        }
    return 0;
}

}  // namespace pcpd
