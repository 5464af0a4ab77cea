// Init (C8), per-replica particle / pair counts (C9; positional popcount) and
// canonical <-> device layout transpose.  The device layout is column-major [W][L].  sm_100a, HBM-bound streaming
// kernels.  See DESIGN.md section 5.
#include "pcpd_kernels.cuh"

namespace pcpd {

// ------------------------------------------------------------------ init ---
// mode 0: all ones; 1: word(i, w) = lo64 of block (i, 0, w_global, INIT); 2: zeros.
__global__ void init_kernel(uint64_t *lat, uint32_t L, uint32_t W, uint32_t word_offset, int mode,
                            const __grid_constant__ RoundKeys rk)
{
    const size_t total = (size_t)L * W;
    for (size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x; p < total; p += (size_t)gridDim.x * blockDim.x) {
        // p is the physical index w * L + i
        const uint32_t i = (uint32_t)(p % L);
        const uint32_t w = (uint32_t)(p / L);
        uint64_t v;
        if (mode == 0) v = ~0ull;
        else if (mode == 2) v = 0ull;
        else v = lo64(philox4x32_10(i, 0u, word_offset + w, STREAM_INIT, rk));
        lat[p] = v;
    }
}

int launch_init(uint64_t *lat, uint32_t L, uint32_t W, uint32_t word_offset, int mode, const RoundKeys &rk,
                cudaStream_t stream)
{
    const size_t total = (size_t)L * W;
    int blocks = (int)((total + 255) / 256);
    if (blocks > 148 * 16) blocks = 148 * 16;
    init_kernel<<<blocks, 256, 0, stream>>>(lat, L, W, word_offset, mode, rk);
    return 1;
}

// ------------------------------------------------------------- transpose ---
// canonical [L][W] <-> physical column-major [W][L]: a tiled transpose through shared memory
// (32 x 32 words, padded), both sides coalesced.  Only get/set_lattice and the chunk upload of
// pcpd_step_from_host use it, never pcpd_run.
__global__ void __launch_bounds__(256) transpose_kernel(const uint64_t *__restrict__ src, uint64_t *__restrict__ dst,
                                                        uint32_t rows, uint32_t cols)
{
    // src is rows x cols row-major, dst is cols x rows row-major; blockIdx.x runs over the tiles of the longer
    // dimension (the site index: up to 2^26 tiles), blockIdx.y over those of the other (word columns)
    __shared__ uint64_t t[32][33];
    const bool rows_long = rows >= cols;
    const uint32_t c0 = (rows_long ? blockIdx.y : blockIdx.x) * 32, r0 = (rows_long ? blockIdx.x : blockIdx.y) * 32;
    const uint32_t tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    for (uint32_t j = ty; j < 32; j += 8) {
        const uint32_t r = r0 + j, c = c0 + tx;
        if (r < rows && c < cols) t[j][tx] = src[(size_t)r * cols + c];
    }
    __syncthreads();
    for (uint32_t j = ty; j < 32; j += 8) {
        const uint32_t c = c0 + j, r = r0 + tx;
        if (r < rows && c < cols) dst[(size_t)c * rows + r] = t[tx][j];
    }
}

// to_physical: src = canonical L x W, dst = physical W x L; else the other way round
int launch_transpose(const uint64_t *src, uint64_t *dst, uint32_t L, uint32_t W, int to_physical, cudaStream_t stream)
{
    const uint32_t rows = to_physical ? L : W, cols = to_physical ? W : L;
    const uint32_t tr = (rows + 31) / 32, tc = (cols + 31) / 32;
    const dim3 grid(rows >= cols ? tr : tc, rows >= cols ? tc : tr);   // grid.y <= 2048 (W <= 65535)
    transpose_kernel<<<grid, 256, 0, stream>>>(src, dst, rows, cols);
    return 1;
}

// --------------------------------------------------------------- density ---
// count[64 w + j] = sum_i bit_j(word(i, w))  (C9) - a positional popcount.
// Per thread: a carry-save adder tree turns 8 words into ones/twos/fours/eights
// bit-planes (vertical counters, 64 lanes at once), `eights` ripples into five
// higher planes; 128 words per thread -> 8 planes.  Per warp: lanes of the same
// word column add their bit-sliced counters with __shfl_xor_sync full adders.
// Then each lane expands a share of the 64 lanes' counters to integers and the
// block reduces through shared-memory atomics, one global atomic per (w, j).
constexpr int DEN_THREADS = 256;
constexpr int DEN_NPT = 128;     // words per thread (multiple of 8)
constexpr int DEN_PLANES = 13;   // 8 + up to 5 shuffle levels

__device__ __forceinline__ void csa(uint64_t &h, uint64_t &l, uint64_t a, uint64_t b, uint64_t c)
{
    const uint64_t u = a ^ b;
    h = (a & b) | (u & c);
    l = u ^ c;
}

// PAIRS = 1: pair counts, word(i) & word(next(i)); CONN = 1 (connected multispin lattice, C10): the successor of
// (site L-1, lane j) is (site 0, lane j+1), i.e. the site-0 word rotated right by one bit.
template <int PAIRS, int CONN>
__global__ void __launch_bounds__(DEN_THREADS) density_kernel(const uint64_t *__restrict__ lat, uint32_t L,
                                                              uint32_t *__restrict__ counts)
{
    __shared__ uint32_t s_cnt[64];
    const uint32_t tid = threadIdx.x;
    const uint32_t wg = blockIdx.y;
    const uint64_t *g = lat + (size_t)wg * L;
    const uint32_t s0 = blockIdx.x * (DEN_THREADS * DEN_NPT);

    if (tid < 64) s_cnt[tid] = 0;

    auto load = [&](uint32_t it) -> uint64_t {
        const uint32_t i = s0 + it * DEN_THREADS + tid;
        if (i >= L) return 0ull;
        uint64_t v = g[i];
        if (PAIRS) {
            if (i + 1 == L) {
                const uint64_t n = g[0];
                v &= CONN ? ((n >> 1) | (n << 63)) : n;
            } else {
                v &= g[i + 1];
            }
        }
        return v;
    };

    uint64_t pl[DEN_PLANES];
#pragma unroll
    for (int p = 0; p < DEN_PLANES; ++p) pl[p] = 0;
    // pl[0] ones, pl[1] twos, pl[2] fours, pl[3..7] = 8s .. 128s
#pragma unroll 1
    for (uint32_t grp = 0; grp < DEN_NPT / 8; ++grp) {
        uint64_t x[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) x[u] = load(grp * 8 + u);
        uint64_t twosA, twosB, foursA, foursB, eights;
        csa(twosA, pl[0], pl[0], x[0], x[1]);
        csa(twosB, pl[0], pl[0], x[2], x[3]);
        csa(foursA, pl[1], pl[1], twosA, twosB);
        csa(twosA, pl[0], pl[0], x[4], x[5]);
        csa(twosB, pl[0], pl[0], x[6], x[7]);
        csa(foursB, pl[1], pl[1], twosA, twosB);
        csa(eights, pl[2], pl[2], foursA, foursB);
        uint64_t carry = eights;
#pragma unroll
        for (int p = 3; p < 8; ++p) {
            const uint64_t tc = pl[p] & carry;
            pl[p] ^= carry;
            carry = tc;
        }
    }

    // warp: add the 32 lanes' counters bit-sliced
#pragma unroll
    for (int off = 16; off >= 1; off >>= 1) {
        uint64_t carry = 0;
#pragma unroll
        for (int p = 0; p < DEN_PLANES; ++p) {
            const uint64_t o = __shfl_xor_sync(0xffffffffu, pl[p], off);
            uint64_t h, l;
            csa(h, l, pl[p], o, carry);
            pl[p] = l;
            carry = h;
        }
    }
    __syncthreads();  // s_cnt zeroed

    // every lane now holds the warp total; lane q expands replica lanes j = q and q + 32
    const uint32_t q = tid % 32;
#pragma unroll
    for (uint32_t m = 0; m < 2; ++m) {
        const uint32_t j = q + m * 32;
        uint32_t cnt = 0;
#pragma unroll
        for (int p = 0; p < DEN_PLANES; ++p) cnt += (uint32_t)((pl[p] >> j) & 1ull) << p;
        if (cnt) atomicAdd(&s_cnt[j], cnt);
    }
    __syncthreads();
    if (tid < 64) {
        const uint32_t cnt = s_cnt[tid];
        if (cnt) atomicAdd(&counts[(size_t)wg * 64 + tid], cnt);
    }
}

int launch_density(const uint64_t *lat, uint32_t L, uint32_t W, int pairs, int connected, uint32_t *counts_dev,
                   cudaStream_t stream)
{
    const uint32_t sites_per_block = DEN_THREADS * DEN_NPT;
    dim3 grid((L + sites_per_block - 1) / sites_per_block, W);
    if (!pairs) density_kernel<0, 0><<<grid, DEN_THREADS, 0, stream>>>(lat, L, counts_dev);
    else if (!connected) density_kernel<1, 0><<<grid, DEN_THREADS, 0, stream>>>(lat, L, counts_dev);
    else density_kernel<1, 1><<<grid, DEN_THREADS, 0, stream>>>(lat, L, counts_dev);
    return 1;
}

}  // namespace pcpd
