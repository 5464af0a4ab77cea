// Kernel-side declarations shared by pcpd_kernels.cu (device code) and
// pcpd_api.cu (host C ABI).  Product path only; nothing here is used by oracle/.
#pragma once
#ifndef __CUDACC_RTC__
#include <cstdint>
#include <cuda_runtime.h>
#endif

#include "philox.cuh"

namespace pcpd {

constexpr uint32_t MAX_SUBSTEPS = 256;  // S = D / A

// One Bernoulli threshold (C3): T = floor(q * 2^32) in [0, 2^32].
struct Threshold {
    uint32_t T32;      // low 32 bits of T (0 when T == 2^32)
    uint32_t nplanes;  // 32 - ctz(T): planes that can matter; 0 if T == 0 or T == 2^32
    uint32_t all;      // 1 if T == 2^32 (mask = all ones)
    uint32_t pad;
};

struct SweepParams {
    uint64_t *lat;  // device, column-major [W][L]
    uint32_t L, W;  // W = local word columns of this handle
    uint32_t Ts, D, A, S, n;  // n = Ts / D domains per tile, S = D / A sub-steps
    uint32_t word_offset;     // global index of local column 0
    uint32_t t;               // sweep index
    uint32_t T4p;             // paper annihilation mask: gate threshold floor((p/b) * 2^32) (pmask_paper != 0), else 0
    Threshold thd, thp;
    RoundKeys rk;
    // T's bit for plane k (bit 31-k) as an all-ones / all-zeros 32-lane mask, precomputed on the
    // host so that the kernels read them as constant-bank operands (C3)
    uint32_t tdm[32], tpm[32];
    // Signed-sum form of the compare: with und_k the lanes still equal to T
    // before plane k (nested sets), lt = sum_k s_k * und_k with s_k = tb_k - tb_(k-1) in {-1,0,+1}
    // (tb_(-1) = tb_32 = 0); stopping after M blocks closes the sum with cl[M] = -tb_(2M-1).
    int32_t sd[34], sp[34];
    int32_t cld[18], clp[18];
    // Per-word-column thresholds (C11, pcpd_create_scan): device array [W][4] = {T_d low 32 bits, T_p low 32 bits,
    // flags (bit 0: T_d = 2^32, bit 1: T_p = 2^32), 0}; NULL in the uniform mode.
    const uint32_t *thr_dev;
    uint32_t connected;       // 1: connected multispin lattice: words of tile sites past the ring wrap are bit-rotated (C10)
    uint32_t pmask_paper;     // 1: Pm = lo & hi of ANNI block 0 & [MISC x3 < T4p]  (Alg. 2 lines 12-13)
    uint32_t rr;              // right reach of the variant's footprint: 2 PCPD, 3 TCPD, 4 QCPD, 1 CPD
    uint32_t pmask_code;      // paper annihilation mask: decorrelation bound b - 0: 1/4 (lo & hi), 1: 1/2 (lo), 2: 1 (all
                              // lanes), 3: 3/4 (lo | hi), lo / hi = the planes of ANNI block 0
};

#ifndef __CUDACC_RTC__
// Threshold-specialised sweep kernel of one handle, compiled at run time (jit.cu).
struct JitSlot {
    int mode;      // 0 off, 1 auto (large problems only), 2 always (test hook)
    int state;     // 0 not tried yet, 1 kernel ready, -1 unavailable (the built-in kernel is used)
    void *kernel;  // CUfunction
    int wpb;       // warps per block the kernel was compiled for (launches with another shape use the built-in kernel)
};

// Small / mid-size path of one handle (column_kernel, column_device.cuh).
struct SplitSlot {
    uint64_t launches;     // column_kernel launches of this handle
    int column_mode;       // 1: the handle's sweeps run column_kernel (one block per tile column)
};
bool column_supported(uint32_t Ts, uint32_t D);
uint64_t column_task_limit(const SweepParams &P);   // up to this many tile columns column_kernel is the default

// Launchers (all asynchronous on `stream`); return the number of kernels launched (launch errors surface in the
// caller's cudaGetLastError).
int launch_sweep(const SweepParams &P, int variant, bool force_block_kernel, cudaStream_t stream, JitSlot *jit,
                 SplitSlot *split);
// warp-per-(tile, column) production kernel (sweep_warp.cu)
bool sweep_warp_supported(uint32_t Ts, uint32_t D);
int sweep_warp_wpb(uint32_t Ts, uint64_t ntasks);
int launch_sweep_warp(const SweepParams &P, int variant, int wpb, cudaStream_t stream, JitSlot *jit, SplitSlot *split);
// jit.cu: compile (once per process, device and parameter set)
// sweep_warp_kernel<variant, wpb, nud, nup, pmode, 0, 1, Td, Tp, Ts, D, A, L> with NVRTC and load it; NULL if NVRTC or the driver entry points are unavailable or the compilation fails
// (message in jit_message()).  jit_launch returns a cudaError_t-like code (0 = launched).
struct JitSpec {
    int variant, wpb, nud, nup, pmode;
    uint32_t Td, Tp, Ts, D, A, L;
};
void *jit_sweep_kernel(const JitSpec &js, size_t max_smem);
int jit_launch(void *kernel, const SweepParams &P, unsigned grid, unsigned block, size_t smem, cudaStream_t stream);
const char *jit_message();
uint64_t jit_launch_count();
// compile only (no device needed): returns 0 and the cubin size; used by the CPU-side build check
int jit_compile_only(const JitSpec &js, size_t *cubin_bytes);
int configure_warp_kernels();
int launch_init(uint64_t *lat, uint32_t L, uint32_t W, uint32_t word_offset, int mode, const RoundKeys &rk,
                cudaStream_t stream);
// counts[64*w + j] (device, uint32[64*W]) must be zero on entry; pairs != 0 counts q(i) & q(next(i)), with the ring
// closure of the connected multispin lattice (C10) when connected != 0.
int launch_density(const uint64_t *lat, uint32_t L, uint32_t W, int pairs, int connected, uint32_t *counts_dev,
                   cudaStream_t stream);
// canonical [L][W] <-> device column-major [W][L]
int launch_transpose(const uint64_t *src, uint64_t *dst, uint32_t L, uint32_t W, int to_physical, cudaStream_t stream);
// Opt-in shared memory size etc.; returns cudaError_t as int.
int configure_kernels();
size_t sweep_smem_bytes(uint32_t Ts);

// microbenchmarks (microbench.cu)
int run_microbench(int kind, uint32_t iters, double *out_rate, cudaStream_t stream);
int microbench_kinds();   // kinds 0 .. microbench_kinds() - 1 exist
#endif  // !__CUDACC_RTC__

}  // namespace pcpd
