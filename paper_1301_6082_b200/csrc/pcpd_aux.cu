// Init (C8), per-replica particle / pair counts (C9; positional popcount) and
// canonical <-> device layout permutation.  The device layout is column-major [W][L] (Wb = 1; the
// Wb parameter of these kernels is the general word-blocked form [W/Wb][L][Wb]).  sm_100a, HBM-bound streaming
// kernels.  See DESIGN.md section 5.
#include "pcpd_kernels.cuh"

namespace pcpd {

// physical index of (site i, local column w) in the word-blocked layout [W/Wb][L][Wb]
__device__ __forceinline__ size_t phys_index(uint32_t i, uint32_t w, uint32_t L, uint32_t Wb)
{
    return ((size_t)(w / Wb) * L + i) * Wb + (w % Wb);
}

// ------------------------------------------------------------------ init ---
// mode 0: all ones; 1: word(i, w) = lo64 of block (i, 0, w_global, INIT); 2: zeros.
__global__ void init_kernel(uint64_t *lat, uint32_t L, uint32_t W, uint32_t Wb, uint32_t word_offset, int mode,
                            const __grid_constant__ RoundKeys rk)
{
    const size_t total = (size_t)L * W;
    for (size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x; p < total; p += (size_t)gridDim.x * blockDim.x) {
        // p is the PHYSICAL index; recover (i, w)
        const uint32_t wl = (uint32_t)(p % Wb);
        const size_t r = p / Wb;
        const uint32_t i = (uint32_t)(r % L);
        const uint32_t w = (uint32_t)(r / L) * Wb + wl;
        uint64_t v;
        if (mode == 0) v = ~0ull;
        else if (mode == 2) v = 0ull;
        else v = lo64(philox4x32_10(i, 0u, word_offset + w, STREAM_INIT, rk));
        lat[p] = v;
    }
}

int launch_init(uint64_t *lat, uint32_t L, uint32_t W, int Wb, uint32_t word_offset, int mode, const RoundKeys &rk,
                cudaStream_t stream)
{
    const size_t total = (size_t)L * W;
    int blocks = (int)((total + 255) / 256);
    if (blocks > 148 * 16) blocks = 148 * 16;
    init_kernel<<<blocks, 256, 0, stream>>>(lat, L, W, (uint32_t)Wb, word_offset, mode, rk);
    return 1;
}

// --------------------------------------------------------------- permute ---
// canonical [L][W] <-> physical column-major [W][L]: a tiled transpose through shared memory
// (32 x 32 words, padded), both sides coalesced.  General word-blocked layouts (Wb > 1) take the
// simple gather below; only get/set_lattice use either, never pcpd_run.
__global__ void __launch_bounds__(256) transpose_kernel(const uint64_t *__restrict__ src, uint64_t *__restrict__ dst,
                                                        uint32_t rows, uint32_t cols)
{
    // src is rows x cols row-major, dst is cols x rows row-major
    __shared__ uint64_t t[32][33];
    const uint32_t tiles_c = (cols + 31) / 32;
    const uint32_t c0 = (blockIdx.x % tiles_c) * 32, r0 = (blockIdx.x / tiles_c) * 32;
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

__global__ void permute_kernel(const uint64_t *__restrict__ src, uint64_t *__restrict__ dst, uint32_t L, uint32_t W,
                               uint32_t Wb, int to_physical)
{
    const size_t total = (size_t)L * W;
    for (size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x; c < total; c += (size_t)gridDim.x * blockDim.x) {
        const uint32_t i = (uint32_t)(c / W), w = (uint32_t)(c % W);  // canonical index c = i*W + w
        const size_t p = phys_index(i, w, L, Wb);
        if (to_physical) dst[p] = src[c];
        else dst[c] = src[p];
    }
}

int launch_permute(const uint64_t *src, uint64_t *dst, uint32_t L, uint32_t W, int Wb, int to_physical,
                   cudaStream_t stream)
{
    if (Wb == 1) {
        // to_physical: src = canonical L x W; else src = physical W x L
        const uint32_t rows = to_physical ? L : W, cols = to_physical ? W : L;
        const uint64_t tiles = (uint64_t)((cols + 31) / 32) * ((rows + 31) / 32);
        if (tiles < (1ull << 31)) {
            transpose_kernel<<<(uint32_t)tiles, 256, 0, stream>>>(src, dst, rows, cols);
            return 1;
        }
    }
    const size_t total = (size_t)L * W;
    int blocks = (int)((total + 255) / 256);
    if (blocks > 148 * 16) blocks = 148 * 16;
    permute_kernel<<<blocks, 256, 0, stream>>>(src, dst, L, W, (uint32_t)Wb, to_physical);
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

template <int WB, int PAIRS>
__global__ void __launch_bounds__(DEN_THREADS) density_kernel(const uint64_t *__restrict__ lat, uint32_t L,
                                                              uint32_t *__restrict__ counts)
{
    __shared__ uint32_t s_cnt[64 * WB];
    constexpr uint32_t SPB = DEN_THREADS / WB;  // sites per block per iteration
    const uint32_t tid = threadIdx.x, wl = tid % WB, srow = tid / WB;
    const uint32_t wg = blockIdx.y;
    const uint64_t *g = lat + (size_t)wg * L * WB;
    const uint32_t s0 = blockIdx.x * (SPB * DEN_NPT);

    for (uint32_t k = tid; k < 64 * WB; k += DEN_THREADS) s_cnt[k] = 0;

    auto load = [&](uint32_t it) -> uint64_t {
        const uint32_t i = s0 + it * SPB + srow;
        if (i >= L) return 0ull;
        uint64_t v = g[(size_t)i * WB + wl];
        if (PAIRS) {
            const uint32_t i1 = (i + 1 == L) ? 0u : i + 1;
            v &= g[(size_t)i1 * WB + wl];
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

    // warp: add the counters of lanes with the same column (lane % WB) bit-sliced
#pragma unroll
    for (int off = 16; off >= WB; off >>= 1) {
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

    // every lane of a column group now holds that column's warp total; lane
    // q = lane / WB of the group expands lanes j = q, q + 32/WB, ...
    constexpr uint32_t GROUP = 32 / WB;
    const uint32_t q = (tid % 32) / WB;
#pragma unroll
    for (uint32_t m = 0; m < 64 / GROUP; ++m) {
        const uint32_t j = q + m * GROUP;
        uint32_t cnt = 0;
#pragma unroll
        for (int p = 0; p < DEN_PLANES; ++p) cnt += (uint32_t)((pl[p] >> j) & 1ull) << p;
        if (cnt) atomicAdd(&s_cnt[wl * 64 + j], cnt);
    }
    __syncthreads();
    for (uint32_t k = tid; k < 64 * WB; k += DEN_THREADS) {
        const uint32_t cnt = s_cnt[k];
        if (cnt) atomicAdd(&counts[(size_t)wg * WB * 64 + k], cnt);
    }
}

template <int WB>
static void launch_density_t(const uint64_t *lat, uint32_t L, uint32_t W, int pairs, uint32_t *counts,
                             cudaStream_t stream)
{
    const uint32_t sites_per_block = (DEN_THREADS / WB) * DEN_NPT;
    dim3 grid((L + sites_per_block - 1) / sites_per_block, W / WB);
    if (pairs) density_kernel<WB, 1><<<grid, DEN_THREADS, 0, stream>>>(lat, L, counts);
    else density_kernel<WB, 0><<<grid, DEN_THREADS, 0, stream>>>(lat, L, counts);
}

int launch_density(const uint64_t *lat, uint32_t L, uint32_t W, int Wb, int pairs, uint32_t *counts_dev,
                   cudaStream_t stream)
{
    if (Wb == 4) launch_density_t<4>(lat, L, W, pairs, counts_dev, stream);
    else if (Wb == 2) launch_density_t<2>(lat, L, W, pairs, counts_dev, stream);
    else launch_density_t<1>(lat, L, W, pairs, counts_dev, stream);
    return 1;
}

}  // namespace pcpd
