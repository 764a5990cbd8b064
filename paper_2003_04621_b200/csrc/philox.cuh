// Philox4x32-10 for the device path (paper ref. [70]; counter convention DESIGN.md 2.1).
// Written for this library; shares nothing with oracle/ref_ptglass.c.
#pragma once
#include <stdint.h>

namespace ptg {

constexpr uint32_t PH_M0 = 0xD2511F53u;
constexpr uint32_t PH_M1 = 0xCD9E8D57u;
constexpr uint32_t PH_W0 = 0x9E3779B9u;
constexpr uint32_t PH_W1 = 0xBB67AE85u;

// The key is the run-wide seed, so the ten round keys key + r*W are constants of the run: computed once on the
// host and passed to every kernel by value (they live in the constant bank and feed LOP3 directly).
struct RoundKeys {
    uint32_t k0[10];
    uint32_t k1[10];
};

inline RoundKeys make_round_keys(uint32_t key0, uint32_t key1)
{
    RoundKeys rk;
    for (int r = 0; r < 10; ++r) {
        rk.k0[r] = key0 + (uint32_t)r * PH_W0;
        rk.k1[r] = key1 + (uint32_t)r * PH_W1;
    }
    return rk;
}

// Counter tags: ctr = (index, step, global sample, TAG)
enum : uint32_t { DOM_J = 1, DOM_SPIN = 2, DOM_METRO = 3, DOM_SWAP = 4, DOM_HOUD = 5 };
__host__ __device__ __forceinline__ uint32_t make_tag(uint32_t domain, uint32_t aux, uint32_t chain, uint32_t idx16)
{
    return (domain << 28) | (aux << 24) | (chain << 16) | idx16;
}

// One block: 10 rounds of 2 wide multiplies (IMAD.WIDE.U32) + 2 three-input XORs (LOP3).
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              const RoundKeys &rk, uint32_t &o0, uint32_t &o1, uint32_t &o2,
                                              uint32_t &o3)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const unsigned long long p0 = (unsigned long long)PH_M0 * c0;
        const unsigned long long p1 = (unsigned long long)PH_M1 * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ rk.k0[r];
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ rk.k1[r];
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
        c0 = n0;
        c2 = n2;
    }
    o0 = c0; o1 = c1; o2 = c2; o3 = c3;
}

// The Metropolis stream (domain 3) varies only c0 between the 8 blocks of a work item: c1 = sweep number,
// c2 = global sample and c3 = tag are shared.  Round 0 therefore splits into a part that is constant per item
// (Round0Shared: one multiply for many blocks) and one multiply + XOR per block; rounds 1..9 are unchanged.
struct Round0Shared {
    uint32_t n0;      // hi(M1*c2) ^ c1 ^ k0[0]
    uint32_t n1;      // lo(M1*c2)
    uint32_t x;       // c3 ^ k1[0]
};

__device__ __forceinline__ Round0Shared philox_round0_shared(uint32_t c1, uint32_t c2, uint32_t c3, const RoundKeys &rk)
{
    const unsigned long long p1 = (unsigned long long)PH_M1 * c2;
    Round0Shared r;
    r.n0 = (uint32_t)(p1 >> 32) ^ c1 ^ rk.k0[0];
    r.n1 = (uint32_t)p1;
    r.x = c3 ^ rk.k1[0];
    return r;
}

__device__ __forceinline__ void philox4x32_10_shared(uint32_t c0, const Round0Shared &s, const RoundKeys &rk,
                                                     uint32_t &o0, uint32_t &o1, uint32_t &o2, uint32_t &o3)
{
    const unsigned long long q0 = (unsigned long long)PH_M0 * c0;
    uint32_t a0 = s.n0, a1 = s.n1, a2 = (uint32_t)(q0 >> 32) ^ s.x, a3 = (uint32_t)q0;
#pragma unroll
    for (int r = 1; r < 10; ++r) {
        const unsigned long long p0 = (unsigned long long)PH_M0 * a0;
        const unsigned long long p1 = (unsigned long long)PH_M1 * a2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ a1 ^ rk.k0[r];
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ a3 ^ rk.k1[r];
        a1 = (uint32_t)p1;
        a3 = (uint32_t)p0;
        a0 = n0;
        a2 = n2;
    }
    o0 = a0; o1 = a1; o2 = a2; o3 = a3;
}

}  // namespace ptg
