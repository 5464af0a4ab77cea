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

// ---- kinds 8 .. 15: the curve behind the INT roofline peak ----------------------------------
// One template for all mixes: per step and chain NW wide multiplies, NL three-register LOP3, NX LOP3 with ONE register
// operand (the other two are uniform: register-read pressure goes down, the ALU op stays), NI 32-bit IMAD, NA IADD3.
// With NL > 0 every wide multiply is the Philox form (immediate multiplier, addend RZ, both halves consumed by one
// LOP3 - these count among the NL); with NL = 0 a wide multiply feeds the next through both of its halves
// (IMAD.WIDE.U32 R, R.lo, R.hi, RZ), so that nothing but wide multiplies is issued.
__device__ __forceinline__ uint32_t add3(uint32_t a, uint32_t b, uint32_t c)
{
    uint32_t d;
    asm volatile("{\n\t.reg .u32 t;\n\tadd.u32 t, %1, %2;\n\tadd.u32 %0, t, %3;\n\t}" : "=r"(d) : "r"(a), "r"(b), "r"(c));
    return d;
}

template <int NW, int NL, int NX, int NI, int NA>
__global__ void __launch_bounds__(MB_THREADS) mb_mix(uint32_t iters, uint32_t seed, uint32_t *out)
{
    static_assert(NL == 0 || NL >= NW, "every Philox-form wide multiply is consumed by one of the NL LOP3");
    constexpr int STEPS = 4;   // steps per loop iteration
    uint32_t x[MB_CHAINS], y[MB_CHAINS], z[MB_CHAINS], v[MB_CHAINS], a[MB_CHAINS];
    uint64_t q[MB_CHAINS];
#pragma unroll
    for (int c = 0; c < MB_CHAINS; ++c) {
        x[c] = seed * (threadIdx.x + 1u) + 0x9E3779B9u * c;
        y[c] = x[c] ^ 0x55555555u;
        z[c] = x[c] + 77u;
        v[c] = x[c] * 3u + 1u;
        a[c] = x[c] + 0x1234567u;
        q[c] = ((uint64_t)x[c] << 32) | y[c];
    }
    for (uint32_t it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < STEPS; ++u) {
            const uint32_t ua = seed * (2u * u + 3u), ub = it + 17u * u;   // warp-uniform operands of the NX LOP3
#pragma unroll
            for (int c = 0; c < MB_CHAINS; ++c) {
                if (NL > 0) {
#pragma unroll
                    for (int w = 0; w < NW; ++w) {
                        const uint64_t p = mul_wide(x[c], (w & 1) ? PHILOX_M1 : PHILOX_M0);
                        x[c] = lop3_e8((uint32_t)p, (uint32_t)(p >> 32), seed);
                    }
#pragma unroll
                    for (int l = NW; l < NL; ++l) {
                        if (l & 1) y[c] = lop3_e8(y[c], y[(c + 1) % MB_CHAINS], z[c]);
                        else z[c] = lop3_e8(z[c], z[(c + 3) % MB_CHAINS], y[c]);
                    }
                } else {
#pragma unroll
                    for (int w = 0; w < NW; ++w) q[c] = mul_wide((uint32_t)q[c], (uint32_t)(q[c] >> 32));
                }
#pragma unroll
                for (int l = 0; l < NX; ++l) {
                    if (l & 1) y[c] = lop3_e8(y[c], ua, ub);
                    else z[c] = lop3_e8(z[c], ub, ua);
                }
#pragma unroll
                for (int l = 0; l < NI; ++l) v[c] = mad_lo(v[c], PHILOX_M0, v[(c + 1) % MB_CHAINS]);
#pragma unroll
                for (int l = 0; l < NA; ++l) a[c] = add3(a[c], a[(c + 1) % MB_CHAINS], a[(c + 5) % MB_CHAINS]);
            }
        }
    }
    uint32_t r = 0;
#pragma unroll
    for (int c = 0; c < MB_CHAINS; ++c) r ^= x[c] ^ y[c] ^ z[c] ^ v[c] ^ a[c] ^ (uint32_t)q[c] ^ (uint32_t)(q[c] >> 32);
    if (r == 0x12345u) out[0] = r;
}

struct MixKind {
    int nw, nl, nx, ni, na;
    void (*kern)(uint32_t, uint32_t, uint32_t *);
};
#define MIX(NW, NL, NX, NI, NA) MixKind{NW, NL, NX, NI, NA, mb_mix<NW, NL, NX, NI, NA>}
static const MixKind g_mix[] = {
    MIX(1, 0, 0, 0, 0),   //  8: IMAD.WIDE.U32 only (each product's two halves are the next one's operands)
    MIX(1, 2, 0, 0, 0),   //  9: wide : LOP3 = 1 : 2
    MIX(1, 4, 0, 0, 0),   // 10: 1 : 4
    MIX(1, 0, 0, 1, 0),   // 11: wide + 32-bit IMAD 1 : 1 (same pipe?)
    MIX(0, 0, 0, 0, 1),   // 12: IADD3 only
    MIX(1, 1, 2, 0, 0),   // 13: wide : LOP3 = 1 : 3 with two of the three LOP3 reading ONE register (+ two uniform operands)
    MIX(1, 1, 0, 0, 2),   // 14: wide + LOP3 + 2 IADD3
    MIX(2, 5, 0, 1, 0),   // 15: the sweep kernel's mix: 2 wide : 5 LOP3 : 1 IMAD
};
#undef MIX
constexpr int MB_MIX_FIRST = 8, MB_MIX_COUNT = (int)(sizeof(g_mix) / sizeof(g_mix[0]));

int microbench_kinds() { return MB_MIX_FIRST + MB_MIX_COUNT; }

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
        if (kind >= MB_MIX_FIRST) g_mix[kind - MB_MIX_FIRST].kern<<<blocks, MB_THREADS, 0, stream>>>(iters, 12345u + rep, out);
        else if (kind == 0) mb_lop3<<<blocks, MB_THREADS, 0, stream>>>(iters, 12345u + rep, out);
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
    if (kind >= MB_MIX_FIRST) {
        const MixKind &m = g_mix[kind - MB_MIX_FIRST];
        per_thread = (double)MB_CHAINS * 4.0 * (m.nw + m.nl + m.nx + m.ni + m.na) * iters;   // instructions as written
    } else if (kind == 3 || kind == 7) per_thread = 4.0 * iters;                          // Philox blocks
    else per_thread = (double)MB_CHAINS * MB_UNROLL * iters;           // instructions
    *out_rate = threads * per_thread / (best_ms * 1e-3);
    return 0;
}

}  // namespace pcpd
