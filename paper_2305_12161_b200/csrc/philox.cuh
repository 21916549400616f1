// Philox4x32-10 for the CUDA path (D5 in DESIGN.md; Salmon et al., SC'11).
// Counter (c0,c1,c2,c3), key (k0,k1).  One round:
//   p0 = M0*c0, p1 = M1*c2 (32x32 -> 64 bit);
//   (c0,c1,c2,c3) <- (hi(p1)^c1^k0, lo(p1), hi(p0)^c3^k1, lo(p0)),
// ten rounds, the key bumped by (W0,W1) between rounds.
// Written for the SM: each round is two IMAD.WIDE.U32 (FMA pipe) and two 3-input
// LOP3 (ALU pipe); the ten round keys are computed once per launch on the host and
// read from the constant bank (struct PhiloxKeys passed by value), so the key
// schedule costs no instruction.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace ising {

constexpr uint32_t kPhiloxM0 = 0xD2511F53u;
constexpr uint32_t kPhiloxM1 = 0xCD9E8D57u;
constexpr uint32_t kPhiloxW0 = 0x9E3779B9u;
constexpr uint32_t kPhiloxW1 = 0xBB67AE85u;

struct PhiloxKeys {            // round keys k0 + r*W0, k1 + r*W1, r = 0..9
    uint32_t k0[10];
    uint32_t k1[10];
};

inline PhiloxKeys make_philox_keys(uint64_t seed)
{
    PhiloxKeys k;
    uint32_t a = (uint32_t)(seed & 0xFFFFFFFFull), b = (uint32_t)(seed >> 32);
    for (int r = 0; r < 10; ++r) {
        k.k0[r] = a;
        k.k1[r] = b;
        a += kPhiloxW0;
        b += kPhiloxW1;
    }
    return k;
}

// round keys from the constant bank (single lattice)
__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                               const PhiloxKeys &k)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)kPhiloxM0 * c0;
        const uint64_t p1 = (uint64_t)kPhiloxM1 * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k.k0[r];
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k.k1[r];
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
        c0 = n0;
        c2 = n2;
    }
    return make_uint4(c0, c1, c2, c3);
}

// key schedule in registers (batched replicas: the seed is per block); also callable on the
// host, where the launch layer draws the per-sweep colour order of the mixed cycle (D10)
__host__ __device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2,
                                                        uint32_t c3, uint32_t k0, uint32_t k1)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)kPhiloxM0 * c0;
        const uint64_t p1 = (uint64_t)kPhiloxM1 * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
        c0 = n0;
        c2 = n2;
        k0 += kPhiloxW0;
        k1 += kPhiloxW1;
    }
    return make_uint4(c0, c1, c2, c3);
}

// Counter tags (domain separation, D5/D10/D11)
constexpr uint32_t kTagTie = 0u;       // tie bits of sweep t:          counter (q, t, colour, 0)
constexpr uint32_t kTagInit = 1u;      // T = infinity start:           counter (q, 0, colour, 1)
constexpr uint32_t kTagOrder = 2u;     // mixed cycle, first colour:    counter (0, t, 0, 2), word 0 bit 0
constexpr uint32_t kTagMenger = 3u;    // Menger start, tile sign bits: counter (T >> 7, k, 0, 3)
constexpr uint32_t kTagBlock = 36u;    // mixed double checkerboard, per-block fine order: (Bi >> 7, t, 0, 36)
                                       // (tags 4..35: bit planes of the finite-T uniforms, D13)

// Mixed cycle (Supp. I.B PAPER.md:258, D10): the colour updated first in sweep t.
__host__ __device__ __forceinline__ int first_colour(uint64_t seed, uint32_t t)
{
    return (int)(philox4x32_10(0u, t, 0u, kTagOrder, (uint32_t)seed, (uint32_t)(seed >> 32)).x & 1u);
}

// Double checkerboard (Supp. I.A PAPER.md:223-240, D14): cubic blocks of edge kDcbBlock form a
// coarse checkerboard; a phase updates the sites of one coarse colour only.  For the word
// (y, z) of either fine colour, bit j is site k = 32 wi + j, x = 2k + o, so x / 8 = 8 wi + j / 4:
// the sites of coarse colour `coarse` are the bits with ((j >> 2) + (y >> 3) + (z >> 3)) & 1 ==
// coarse.  coarse < 0: no mask (plain checkerboard).
constexpr int kDcbBlock = 8;
__device__ __forceinline__ uint32_t dcb_mask(int y, int z, int coarse)
{
    if (coarse < 0) return 0xFFFFFFFFu;
    return (((y >> 3) + (z >> 3) + coarse) & 1) ? 0xF0F0F0F0u : 0x0F0F0F0Fu;
}

// Mixed-cycle double checkerboard (D15): `ffbyte` holds the first-fine-colour bits of the 8
// blocks a packed word spans (bit b = block bx = 8 wi + b).  In pass `pass` of coarse colour
// `coarse`, the colour-c sites of the word that are updated are those of the blocks with
// parity == coarse and (bit ^ pass) == c.
__device__ __forceinline__ uint32_t dcb_mixed_mask(int y, int z, int coarse, int pass, int c, uint32_t ffbyte)
{
    const uint32_t want = (c ^ pass) ? ffbyte : ~ffbyte;                       // bit == c ^ pass
    const uint32_t par = (((y >> 3) + (z >> 3) + coarse) & 1) ? 0xAAu : 0x55u;   // block parity == coarse
    uint32_t x = want & par & 0xFFu;                                           // bit b -> nibble b
    x = (x | (x << 12)) & 0x000F000Fu;
    x = (x | (x << 6)) & 0x03030303u;
    x = (x | (x << 3)) & 0x11111111u;
    return x * 0xFu;
}

// ---------------------------------------------------------------------------
// The site rule on 32 sites at once (eq. (6), D2).
// n1..n6: the six neighbour words (bit = 1 <=> spin up), s: own word, rho: tie bits.
// With U = number of up neighbours the rule is  new = [U + (s ^ rho) >= 4]:
//   U >= 4 -> up, U <= 2 -> down (Delta E < 0 flips, > 0 keeps), U = 3 (Delta E = 0)
//   -> s ^ rho, i.e. flip iff the random bit is 1.
// Seven one-bit inputs, threshold 4: two 3:2 compressors, then two majorities.
// 7 LOP3 per word.
// ---------------------------------------------------------------------------
__device__ __forceinline__ uint32_t maj3(uint32_t a, uint32_t b, uint32_t c)
{
    return (a & b) | (c & (a | b));
}

__device__ __forceinline__ uint32_t rule_word(uint32_t s, uint32_t rho, uint32_t n1, uint32_t n2,
                                              uint32_t n3, uint32_t n4, uint32_t n5, uint32_t n6)
{
    const uint32_t sa = n1 ^ n2 ^ n3, ca = maj3(n1, n2, n3);
    const uint32_t sb = n4 ^ n5 ^ n6, cb = maj3(n4, n5, n6);
    const uint32_t m = maj3(sa, sb, s ^ rho);
    return maj3(ca, cb, m);
}

}  // namespace ising
