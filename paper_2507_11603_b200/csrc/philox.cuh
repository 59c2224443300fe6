// a1 RNG — Philox4x32-10 keyed on (seed, photon id, draw index); BASELINE.json north_star, reading A16.
// (The paper uses xoshiro128++ per work-item; the north star replaces it by a counter-based RNG.)
//   key     = (seed lo, seed hi)
//   counter = (block lo, block hi, id lo, id hi),  block = draw >> 2,  word = draw & 3
// which is cuRAND's curand_init(seed, subsequence = id, offset = 0) + curand4() layout.
#pragma once
#include <cstdint>

namespace thor {

struct U4 { uint32_t x, y, z, w; };

__device__ __forceinline__ U4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0,
                                            uint32_t k1) {
    constexpr uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(M0, c0), lo0 = M0 * c0;
        const uint32_t hi1 = __umulhi(M1, c2), lo1 = M1 * c2;
        const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += W0; k1 += W1;                       // bumped after the round == before every round but the first
    }
    return U4{c0, c1, c2, c3};
}

// u32 -> uniform in the open interval (0,1): ((r >> 9) + 0.5) 2^-23 (reading A8).  23 bits: k + 1/2 with k < 2^23 is
// exact in fp32 (24 bits would round k + 1/2 to even for k >= 2^23 and could return exactly 0.5 or 1.0).  Formed
// without an int->float conversion: the bits 0x3F800000 | k are the float 1 + k 2^-23, and subtracting 1 - 2^-24
// (representable) leaves (k + 1/2) 2^-23 exactly.
__device__ __forceinline__ float u01(uint32_t r) { return __uint_as_float((r >> 9) | 0x3F800000u) - 0.99999994039535522f; }

// One packet's draw stream.  Four cached words + the draw index; draw d is word d & 3 of block d >> 2.
struct Stream {
    uint32_t k0, k1, id_lo, id_hi;
    uint32_t w0, w1, w2, w3;
    uint64_t d;

    __device__ __forceinline__ void init(uint64_t seed, uint64_t id) {
        k0 = (uint32_t)seed; k1 = (uint32_t)(seed >> 32); id_lo = (uint32_t)id; id_hi = (uint32_t)(id >> 32);
        d = 0;
    }
    __device__ __forceinline__ uint32_t next_u32() {
        const uint32_t lane = (uint32_t)d & 3u;
        if (lane == 0u) {
            const uint64_t blk = d >> 2;
            const U4 r = philox4x32_10((uint32_t)blk, (uint32_t)(blk >> 32), id_lo, id_hi, k0, k1);
            w0 = r.x; w1 = r.y; w2 = r.z; w3 = r.w;
        }
        ++d;
        return lane == 0u ? w0 : lane == 1u ? w1 : lane == 2u ? w2 : w3;
    }
    __device__ __forceinline__ float uniform() { return u01(next_u32()); }
};

// The walk kernel's view of the same stream: whole counter blocks.  next4() returns draws 4b..4b+3 of the packet as
// uniforms and advances b, so every lane of a warp runs the ten rounds at the same program point (the per-draw
// Stream above regenerates its block on a different call in every lane: 4 of 32 lanes active, 40 % of all issued
// instructions in the round-1 profile).  Draws a step does not need are skipped, never reused.
struct BlockRng {
    uint32_t id_lo, id_hi, b_lo, b_hi;

    __device__ __forceinline__ void init(uint64_t id) {
        id_lo = (uint32_t)id; id_hi = (uint32_t)(id >> 32); b_lo = 0u; b_hi = 0u;
    }
    __device__ __forceinline__ unsigned long long id() const { return ((unsigned long long)id_hi << 32) | id_lo; }
    __device__ __forceinline__ float4 next4(uint32_t k0, uint32_t k1) {
        const U4 r = philox4x32_10(b_lo, b_hi, id_lo, id_hi, k0, k1);
        b_lo += 1u;
        b_hi += (b_lo == 0u);
        return make_float4(u01(r.x), u01(r.y), u01(r.z), u01(r.w));
    }
};

}  // namespace thor
