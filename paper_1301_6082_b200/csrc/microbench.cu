// Pipe-peak microbenchmarks for the INT roofline of the sweep kernel
// (SURVEY.md 8(d)): LOP3-only (ALU pipe), IMAD.WIDE.U32-only
// (FMA pipe) paired 1:1 with LOP3 as in a Philox round, plain 32-bit IMAD, and back-to-back Philox-4x32-10 blocks.  Eight
// independent chains per thread, every SM filled with 2048 threads.
#include "pcpd_kernels.cuh"

namespace pcpd {

constexpr int MB_CHAINS = 8;
constexpr int MB_THREADS = 256;
constexpr int MB_BLOCKS_PER_SM = 8;
constexpr int MB_UNROLL = 16;  // instructions per chain per loop iteration

__device__ __forceinline__ uint32_t lop3_e8(uint32_t a, uint32_t b, uint32_t c)
{
    uint32_t d;
    asm volatile("lop3.b32 %0, %1, %2, %3, 0xE8;" : "=r"(d) : "r"(a), "r"(b), "r"(c));  // majority
    return d;
}

__device__ __forceinline__ uint64_t mul_wide(uint32_t a, uint32_t b)
{
    uint64_t d;
    asm volatile("mul.wide.u32 %0, %1, %2;" : "=l"(d) : "r"(a), "r"(b));
    return d;
}

__device__ __forceinline__ uint32_t mad_lo(uint32_t a, uint32_t b, uint32_t c)
{
    uint32_t d;
    asm volatile("mad.lo.u32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
    return d;
}

__global__ void __launch_bounds__(MB_THREADS) mb_lop3(uint32_t iters, uint32_t seed, uint32_t *out)
{
    uint32_t x[MB_CHAINS];
#pragma unroll
    for (int c = 0; c < MB_CHAINS; ++c) x[c] = seed * (threadIdx.x + 1u) + 0x9E3779B9u * c;
    for (uint32_t it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < MB_UNROLL; ++u)
#pragma unroll
            for (int c = 0; c < MB_CHAINS; ++c)
                x[c] = lop3_e8(x[c], x[(c + 1) % MB_CHAINS], x[(c + 3) % MB_CHAINS]);
    }
    uint32_t r = 0;
#pragma unroll
    for (int c = 0; c < MB_CHAINS; ++c) r ^= x[c];
    if (r == 0x12345u) out[0] = r;
}

// Philox's own mix: one IMAD.WIDE.U32 (both halves live) + one 3-input xor LOP3 per step.
__global__ void __launch_bounds__(MB_THREADS) mb_wide_xor(uint32_t iters, uint32_t seed, uint32_t *out)
{
    uint32_t x[MB_CHAINS];
#pragma unroll
    for (int c = 0; c < MB_CHAINS; ++c) x[c] = seed * (threadIdx.x + 1u) + 0x9E3779B9u * c;
    for (uint32_t it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < MB_UNROLL / 2; ++u)
#pragma unroll
            for (int c = 0; c < MB_CHAINS; ++c) {
                const uint64_t p = mul_wide(x[c], PHILOX_M0);
                x[c] = (uint32_t)p ^ (uint32_t)(p >> 32) ^ seed;
            }
    }
    uint32_t r = 0;
#pragma unroll
    for (int c = 0; c < MB_CHAINS; ++c) r ^= x[c];
    if (r == 0x12345u) out[0] = r;
}

// plain 32-bit IMAD chain (FMA pipe, full rate expected)
__global__ void __launch_bounds__(MB_THREADS) mb_imad_lo(uint32_t iters, uint32_t seed, uint32_t *out)
{
    uint32_t x[MB_CHAINS];
#pragma unroll
    for (int c = 0; c < MB_CHAINS; ++c) x[c] = seed * (threadIdx.x + 1u) + 0x9E3779B9u * c;
    for (uint32_t it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < MB_UNROLL; ++u)
#pragma unroll
            for (int c = 0; c < MB_CHAINS; ++c) x[c] = mad_lo(x[c], PHILOX_M0, x[(c + 1) % MB_CHAINS]);
    }
    uint32_t r = 0;
#pragma unroll
    for (int c = 0; c < MB_CHAINS; ++c) r ^= x[c];
    if (r == 0x12345u) out[0] = r;
}

// 4 independent Philox chains per thread; each iteration feeds a block's output
// back into its counter so nothing can be hoisted.
__global__ void __launch_bounds__(MB_THREADS) mb_philox(uint32_t iters, const __grid_constant__ RoundKeys rk,
                                                       uint32_t *out)
{
    U4 s[4];
#pragma unroll
    for (int c = 0; c < 4; ++c) s[c] = U4{threadIdx.x, blockIdx.x, (uint32_t)c, 0u};
    for (uint32_t it = 0; it < iters; ++it) {
#pragma unroll
        for (int c = 0; c < 4; ++c) s[c] = philox4x32_10(s[c].x0, s[c].x1, s[c].x2, s[c].x3, rk);
    }
    uint32_t r = 0;
#pragma unroll
    for (int c = 0; c < 4; ++c) r ^= s[c].x0 ^ s[c].x1 ^ s[c].x2 ^ s[c].x3;
    if (r == 0x12345u) out[0] = r;
}

// kind 4: LOP3 and 32-bit IMAD 1:1 on independent chains (do the ALU and FMA pipes issue concurrently?)
__global__ void __launch_bounds__(MB_THREADS) mb_lop3_imad(uint32_t iters, uint32_t seed, uint32_t *out)
{
    uint32_t x[MB_CHAINS], y[MB_CHAINS];
#pragma unroll
    for (int c = 0; c < MB_CHAINS; ++c) {
        x[c] = seed * (threadIdx.x + 1u) + 0x9E3779B9u * c;
        y[c] = x[c] ^ 0x55555555u;
    }
    for (uint32_t it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < MB_UNROLL / 2; ++u)
#pragma unroll
            for (int c = 0; c < MB_CHAINS; ++c) {
                x[c] = lop3_e8(x[c], x[(c + 1) % MB_CHAINS], x[(c + 3) % MB_CHAINS]);
                y[c] = mad_lo(y[c], PHILOX_M0, y[(c + 1) % MB_CHAINS]);
            }
    }
    uint32_t r = 0;
#pragma unroll
    for (int c = 0; c < MB_CHAINS; ++c) r ^= x[c] ^ y[c];
    if (r == 0x12345u) out[0] = r;
}

// kind 5: one IMAD.WIDE.U32 + three LOP3 per step (wide multiply chain plus independent logic chains):
// the sweep kernel's mix (16 wide : 28 + overhead logic per Philox block)
__global__ void __launch_bounds__(MB_THREADS) mb_wide_3lop(uint32_t iters, uint32_t seed, uint32_t *out)
{
    uint32_t x[MB_CHAINS], y[MB_CHAINS], z[MB_CHAINS];
#pragma unroll
    for (int c = 0; c < MB_CHAINS; ++c) {
        x[c] = seed * (threadIdx.x + 1u) + 0x9E3779B9u * c;
        y[c] = x[c] ^ 0x55555555u;
        z[c] = x[c] + 77u;
    }
    for (uint32_t it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < MB_UNROLL / 4; ++u)
#pragma unroll
            for (int c = 0; c < MB_CHAINS; ++c) {
                const uint64_t p = mul_wide(x[c], PHILOX_M0);
                x[c] = lop3_e8((uint32_t)p, (uint32_t)(p >> 32), seed);
                y[c] = lop3_e8(y[c], y[(c + 1) % MB_CHAINS], z[c]);
                z[c] = lop3_e8(z[c], z[(c + 3) % MB_CHAINS], y[c]);
            }
    }
    uint32_t r = 0;
#pragma unroll
    for (int c = 0; c < MB_CHAINS; ++c) r ^= x[c] ^ y[c] ^ z[c];
    if (r == 0x12345u) out[0] = r;
}

__device__ __forceinline__ uint32_t mul_hi(uint32_t a, uint32_t b)
{
    uint32_t d;
    asm volatile("mul.hi.u32 %0, %1, %2;" : "=r"(d) : "r"(a), "r"(b));
    return d;
}
__device__ __forceinline__ uint32_t mul_lo(uint32_t a, uint32_t b)
{
    uint32_t d;
    asm volatile("mul.lo.u32 %0, %1, %2;" : "=r"(d) : "r"(a), "r"(b));
    return d;
}

// kind 6: IMAD.HI.U32 only
__global__ void __launch_bounds__(MB_THREADS) mb_imad_hi(uint32_t iters, uint32_t seed, uint32_t *out)
{
    uint32_t x[MB_CHAINS];
#pragma unroll
    for (int c = 0; c < MB_CHAINS; ++c) x[c] = seed * (threadIdx.x + 1u) + 0x9E3779B9u * c;
    for (uint32_t it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < MB_UNROLL; ++u)
#pragma unroll
            for (int c = 0; c < MB_CHAINS; ++c) x[c] = mul_hi(x[c] | 0x80000000u, PHILOX_M0);
    }
    uint32_t r = 0;
#pragma unroll
    for (int c = 0; c < MB_CHAINS; ++c) r ^= x[c];
    if (r == 0x12345u) out[0] = r;
}

// kind 7: Philox-4x32-10 with each 32x32->64 product as separate mul.hi + mul.lo
__global__ void __launch_bounds__(MB_THREADS) mb_philox_hilo(uint32_t iters, const __grid_constant__ RoundKeys rk,
                                                            uint32_t *out)
{
    U4 s[4];
    uint32_t z;  // opaque zero: keeps ptxas from fusing mul.hi + mad.lo back into IMAD.WIDE
    asm volatile("mov.b32 %0, 0;" : "=r"(z));
#pragma unroll
    for (int c = 0; c < 4; ++c) s[c] = U4{threadIdx.x, blockIdx.x, (uint32_t)c, 0u};
    for (uint32_t it = 0; it < iters; ++it) {
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            uint32_t c0 = s[c].x0, c1 = s[c].x1, c2 = s[c].x2, c3 = s[c].x3;
#pragma unroll
            for (int r = 0; r < 10; ++r) {
                const uint32_t h0 = mul_hi(c0, PHILOX_M0), l0 = mad_lo(c0, PHILOX_M0, z);
                const uint32_t h1 = mul_hi(c2, PHILOX_M1), l1 = mad_lo(c2, PHILOX_M1, z);
                c0 = h1 ^ c1 ^ rk.k0[r];
                c2 = h0 ^ c3 ^ rk.k1[r];
                c1 = l1;
                c3 = l0;
            }
            s[c] = U4{c0, c1, c2, c3};
        }
    }
    uint32_t r = 0;
#pragma unroll
    for (int c = 0; c < 4; ++c) r ^= s[c].x0 ^ s[c].x1 ^ s[c].x2 ^ s[c].x3;
    if (r == 0x12345u) out[0] = r;
}

int run_microbench(int kind, uint32_t iters, double *out_rate, cudaStream_t stream)
{
    int dev = 0, nsm = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    const int blocks = nsm * MB_BLOCKS_PER_SM;
    uint32_t *out = nullptr;
    if (cudaMalloc(&out, 4) != cudaSuccess) return -3;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const RoundKeys rk = make_round_keys(0x1234567ull);
    float best_ms = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {  // rep 0 is the warm-up
        cudaEventRecord(e0, stream);
        if (kind == 0) mb_lop3<<<blocks, MB_THREADS, 0, stream>>>(iters, 12345u + rep, out);
        else if (kind == 1) mb_wide_xor<<<blocks, MB_THREADS, 0, stream>>>(iters, 12345u + rep, out);
        else if (kind == 2) mb_imad_lo<<<blocks, MB_THREADS, 0, stream>>>(iters, 12345u + rep, out);
        else if (kind == 4) mb_lop3_imad<<<blocks, MB_THREADS, 0, stream>>>(iters, 12345u + rep, out);
        else if (kind == 5) mb_wide_3lop<<<blocks, MB_THREADS, 0, stream>>>(iters, 12345u + rep, out);
        else if (kind == 6) mb_imad_hi<<<blocks, MB_THREADS, 0, stream>>>(iters, 12345u + rep, out);
        else if (kind == 7) mb_philox_hilo<<<blocks, MB_THREADS, 0, stream>>>(iters, rk, out);
        else mb_philox<<<blocks, MB_THREADS, 0, stream>>>(iters, rk, out);
        cudaEventRecord(e1, stream);
        if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(out); return -2; }
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best_ms) best_ms = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(out);
    const double threads = (double)blocks * MB_THREADS;
    double per_thread;
    if (kind == 3 || kind == 7) per_thread = 4.0 * iters;                          // Philox blocks
    else per_thread = (double)MB_CHAINS * MB_UNROLL * iters;           // instructions
    *out_rate = threads * per_thread / (best_ms * 1e-3);
    return 0;
}

}  // namespace pcpd
