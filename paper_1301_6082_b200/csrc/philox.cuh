// Philox-4x32-10 counter-based generator (Salmon et al., SC'11) for sm_100a and
// the addressing of DESIGN.md section 3, C1-C2.  Device code of the product path;
// shares nothing with oracle/.
#pragma once
#ifdef __CUDACC_RTC__
// run-time compilation (jit.cu): no standard headers; NVRTC's own fixed-width built-in types
typedef unsigned char uint8_t;
typedef unsigned int uint32_t;
typedef int int32_t;
typedef unsigned long long uint64_t;
#else
#include <cstdint>
#endif

namespace pcpd {

constexpr uint32_t PHILOX_M0 = 0xD2511F53u;
constexpr uint32_t PHILOX_M1 = 0xCD9E8D57u;
constexpr uint32_t PHILOX_W0 = 0x9E3779B9u;
constexpr uint32_t PHILOX_W1 = 0xBB67AE85u;

// Streams (C2): c3 = stream << 24 | block index m.
constexpr uint32_t STREAM_MISC = 0u << 24;
constexpr uint32_t STREAM_DIFF = 1u << 24;
constexpr uint32_t STREAM_ANNI = 2u << 24;
constexpr uint32_t STREAM_SHIFT = 3u << 24;
constexpr uint32_t STREAM_INIT = 4u << 24;

// The ten round keys are thread-uniform: k_r = key + r * W.  Kept in the
// kernel-parameter constant bank so that the xor takes them as c[][] operands.
struct RoundKeys {
    uint32_t k0[10];
    uint32_t k1[10];
};

#ifndef __CUDACC_RTC__
inline RoundKeys make_round_keys(uint64_t seed)
{
    RoundKeys rk;
    uint32_t a = (uint32_t)(seed & 0xffffffffu), b = (uint32_t)(seed >> 32);
    for (int r = 0; r < 10; ++r) {
        rk.k0[r] = a;
        rk.k1[r] = b;
        a += PHILOX_W0;
        b += PHILOX_W1;
    }
    return rk;
}
#endif

struct U4 {
    uint32_t x0, x1, x2, x3;
};

// One block: 10 rounds of
//   (hi0,lo0) = M0*c0, (hi1,lo1) = M1*c2; (c0,c1,c2,c3) <- (hi1^c1^k0, lo1, hi0^c3^k1, lo0)
// 20 IMAD.WIDE.U32 + 20 LOP3 on sm_100a.
__device__ __forceinline__ U4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                            const RoundKeys &rk)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)PHILOX_M0 * c0;
        const uint64_t p1 = (uint64_t)PHILOX_M1 * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ rk.k0[r];
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ rk.k1[r];
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
        c0 = n0;
        c2 = n2;
    }
    return U4{c0, c1, c2, c3};
}

__device__ __forceinline__ uint64_t lo64(const U4 &b) { return (uint64_t)b.x0 | ((uint64_t)b.x1 << 32); }
__device__ __forceinline__ uint64_t hi64(const U4 &b) { return (uint64_t)b.x2 | ((uint64_t)b.x3 << 32); }

}  // namespace pcpd
