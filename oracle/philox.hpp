// ORACLE — TEST INFRASTRUCTURE ONLY (see constants.hpp).
//
// Philox4x32-10 counter-based generator (Salmon et al. 2011, "Parallel random numbers: as easy as 1, 2, 3").
// The paper uses xoshiro128++ per work-item (§3.4.3); BASELINE.json's north_star replaces it by
// "a counter-based Philox RNG keyed on (seed, photon id, draw index)" — DESIGN.md reading A16:
//   key     = (seed_lo, seed_hi)
//   counter = (block_lo, block_hi, id_lo, id_hi),  block = draw_index >> 2,  word = draw_index & 3.
// This is the layout of cuRAND's curand_init(seed, subsequence = photon id, offset = 0) + curand4().
#pragma once
#include <cstdint>
#include <cmath>

namespace orc {

struct Philox4 { uint32_t v[4]; };

inline Philox4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1) {
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;   // round multipliers
    const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;   // key increments (Weyl sequence)
    for (int round = 0; round < 10; ++round) {
        if (round > 0) { k0 += W0; k1 += W1; }           // key bumped before every round but the first
        const uint64_t p0 = (uint64_t)M0 * c0;
        const uint64_t p1 = (uint64_t)M1 * c2;
        const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        const uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        const uint32_t n0 = hi1 ^ c1 ^ k0;
        const uint32_t n1 = lo1;
        const uint32_t n2 = hi0 ^ c3 ^ k1;
        const uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    }
    return Philox4{{c0, c1, c2, c3}};
}

// u32 -> uniform in the OPEN interval (0,1): ((r >> 9) + 0.5) * 2^-23 (reading A8).  23 bits, not 24: k + 1/2 with
// k < 2^23 fits a 24-bit significand, so the same value is exact in fp32 and in fp64.
// The paper offers R in [0,1) and 1-R in (0,1]; the open interval keeps -ln(u) finite both ways.
inline double u32_to_uniform(uint32_t r) { return ((double)(r >> 9) + 0.5) * (1.0 / 8388608.0); }

// One packet's stream: draw d of photon `id` under `seed`.
class DrawStream {
public:
    DrawStream(uint64_t seed, uint64_t photon_id) : seed_(seed), id_(photon_id), d_(0), have_block_(~0ull) {}
    uint32_t next_u32() {
        const uint64_t block = d_ >> 2;
        if (block != have_block_) {
            cur_ = philox4x32_10((uint32_t)block, (uint32_t)(block >> 32), (uint32_t)id_, (uint32_t)(id_ >> 32),
                                 (uint32_t)seed_, (uint32_t)(seed_ >> 32));
            have_block_ = block;
        }
        const uint32_t r = cur_.v[d_ & 3];
        ++d_;
        return r;
    }
    double uniform() { return u32_to_uniform(next_u32()); }
    uint64_t draws() const { return d_; }
private:
    uint64_t seed_, id_, d_, have_block_;
    Philox4 cur_;
};

}  // namespace orc
