// Generic kernels: any L % 64 == 0, any number of replicas (blockIdx.y = replica).
//  - init_spins_kernel        a1: T = infinity start from Philox(tag = 1)          (D6)
//  - halfsweep_generic_kernel a2/a3: one colour, in place, one thread per 128-spin group
//                              (eq. (6); sweep order PAPER.md:116)
// Layout D3: state[rep][colour][z][y][wi], wi = 0..L/64-1 32-bit words per row, bit j of
// word wi = site k = 32 wi + j, x = 2k + ((y+z+colour)&1).
// Neighbour geometry D4: a colour-c site (k,y,z) has its six neighbours in colour 1-c at
// (k,y+-1,z), (k,y,z+-1), (k,y,z) and (k-1,y,z) if o = (y+z+c)&1 is 0, else (k+1,y,z).
#pragma once
#include "philox.cuh"

namespace ising {

__global__ void __launch_bounds__(256)
init_spins_kernel(uint32_t *__restrict__ state, const uint64_t *__restrict__ seeds, int L)
{
    const size_t groups_per_colour = (size_t)L * L * (L >> 6) / 4;
    const size_t g = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= 2 * groups_per_colour) return;
    const int rep = blockIdx.y;
    const uint32_t c = g >= groups_per_colour ? 1u : 0u;
    const uint32_t q = (uint32_t)(g - c * groups_per_colour);
    const uint64_t seed = seeds[rep];
    const uint4 v = philox4x32_10(q, 0u, c, 1u, (uint32_t)seed, (uint32_t)(seed >> 32));
    reinterpret_cast<uint4 *>(state)[(size_t)rep * 2 * groups_per_colour + g] = v;
}

// Mixed-cycle double checkerboard (D15): bit Bi of ff[rep] = the fine colour block Bi updates
// first in sweep t = bit (Bi & 127) of Philox(counter (Bi >> 7, t, 0, 36)): word wq of the bit
// array is output word wq & 3 of the call for group wq >> 2.
__global__ void __launch_bounds__(256)
block_order_kernel(uint32_t *__restrict__ ff, size_t ff_stride, const uint64_t *__restrict__ seeds,
                   int n_words, uint32_t t)
{
    const int wq = blockIdx.x * blockDim.x + threadIdx.x;
    if (wq >= n_words) return;
    const int rep = blockIdx.y;
    const uint64_t seed = seeds[rep];
    const uint4 r = philox4x32_10((uint32_t)(wq >> 2), t, 0u, kTagBlock, (uint32_t)seed, (uint32_t)(seed >> 32));
    const int k = wq & 3;
    ff[(size_t)rep * ff_stride + wq] = k == 0 ? r.x : k == 1 ? r.y : k == 2 ? r.z : r.w;
}

// `coarse` >= 0: only the sites of that coarse colour are updated (double checkerboard, D14).
// `phase` = 0 / 1: first / second half-sweep of sweep t.  01 cycle (mixed = 0): colour = phase.
// Mixed cycle (mixed = 1, D10): colour = phase ^ first_colour(seed of the replica, t).
// Menger-sponge start (D11): the lattice is tiled from the origin by sponges of
// iteration k and edge size = 3^k (the last tile in each direction is cut at L); a site belongs
// to the sponge iff at no ternary digit position two or more of its local coordinates have the
// digit 1; tile T = (Z*nT + Y)*nT + X draws its sign from Philox(counter (T >> 7, k, 0, 3)) bit
// T & 127; sponge sites take that sign, holes the opposite.  One thread per packed word.
__global__ void __launch_bounds__(256)
init_menger_kernel(uint32_t *__restrict__ state, const uint64_t *__restrict__ seeds, int L, int k,
                   int size)
{
    const int WPR = L >> 6;
    const size_t WPC = (size_t)L * L * WPR;
    const size_t w = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (w >= 2 * WPC) return;
    const int rep = blockIdx.y;
    const uint64_t seed = seeds[rep];
    const int c = w >= WPC ? 1 : 0;
    const size_t wc = w - (size_t)c * WPC;
    const int wi = (int)(wc % WPR);
    const size_t row = wc / WPR;
    const int y = (int)(row % L), z = (int)(row / L);
    const int o = (y + z + c) & 1;
    const int nT = (L + size - 1) / size;
    const int Y = y / size, Z = z / size, v = y - Y * size, ww = z - Z * size;
    uint32_t out = 0, cached_group = 0xFFFFFFFFu;
    uint4 rnd = make_uint4(0, 0, 0, 0);
    for (int j = 0; j < 32; ++j) {
        const int x = 2 * (32 * wi + j) + o;
        const int X = x / size;
        int a = x - X * size, b = v, d = ww;
        bool solid = true;
        for (int level = 0; level < k; ++level) {
            const int ones = (a % 3 == 1) + (b % 3 == 1) + (d % 3 == 1);
            if (ones >= 2) solid = false;
            a /= 3; b /= 3; d /= 3;
        }
        // 64-bit tile index: nT^3 passes 2^32 from L = 1664 at k = 0 (the counter word is T >> 7)
        const uint64_t T = ((uint64_t)Z * (uint64_t)nT + (uint64_t)Y) * (uint64_t)nT + (uint64_t)X;
        if ((uint32_t)(T >> 7) != cached_group) {
            cached_group = (uint32_t)(T >> 7);
            rnd = philox4x32_10(cached_group, (uint32_t)k, 0u, kTagMenger, (uint32_t)seed,
                                (uint32_t)(seed >> 32));
        }
        const uint32_t word = ((T >> 5) & 3) == 0 ? rnd.x : ((T >> 5) & 3) == 1 ? rnd.y
                            : ((T >> 5) & 3) == 2 ? rnd.z : rnd.w;
        const uint32_t bit = (word >> (T & 31)) & 1u;
        out |= (solid ? bit : bit ^ 1u) << j;
    }
    state[(size_t)rep * 2 * WPC + w] = out;
}

__global__ void __launch_bounds__(256)
halfsweep_generic_kernel(uint32_t *__restrict__ state, const uint64_t *__restrict__ seeds,
                         int L, uint32_t t, int phase, int mixed, int coarse,
                         const uint32_t *__restrict__ ff = nullptr, size_t ff_stride = 0, int pass = 0)
{
    const int WPR = L >> 6;                                   // words per row
    const size_t WPC = (size_t)L * L * WPR;                   // words per colour
    const size_t g = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= WPC / 4) return;
    const int rep = blockIdx.y;
    const uint64_t seed = seeds[rep];
    const int c = mixed ? phase ^ first_colour(seed, t) : phase;
    uint32_t *own = state + (size_t)rep * 2 * WPC + (size_t)c * WPC;
    const uint32_t *oth = state + (size_t)rep * 2 * WPC + (size_t)(1 - c) * WPC;
    const uint4 rnd = philox4x32_10((uint32_t)g, t, (uint32_t)c, 0u, (uint32_t)seed,
                                    (uint32_t)(seed >> 32));
    const uint32_t rho[4] = {rnd.x, rnd.y, rnd.z, rnd.w};
    const uint4 sv = reinterpret_cast<const uint4 *>(own)[g];
    const uint32_t s[4] = {sv.x, sv.y, sv.z, sv.w};
    const int coarse_mixed = ff ? coarse ^ first_colour(seed, t) : 0;   // D15: k-th coarse colour of the drawn order
    uint32_t out[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const size_t w = 4 * g + i;
        const int wi = (int)(w % WPR);
        const size_t row = w / WPR;
        const int y = (int)(row % L);
        const int z = (int)(row / L);
        const int yp = (y + 1 == L) ? 0 : y + 1, ym = (y == 0) ? L - 1 : y - 1;
        const int zp = (z + 1 == L) ? 0 : z + 1, zm = (z == 0) ? L - 1 : z - 1;
        const uint32_t n_same = oth[w];
        const uint32_t n_yp = oth[((size_t)z * L + yp) * WPR + wi];
        const uint32_t n_ym = oth[((size_t)z * L + ym) * WPR + wi];
        const uint32_t n_zp = oth[((size_t)zp * L + y) * WPR + wi];
        const uint32_t n_zm = oth[((size_t)zm * L + y) * WPR + wi];
        uint32_t n_x;
        if (((y + z + c) & 1) == 0) {       // neighbour at k-1: bit j <- bit j-1
            const uint32_t prev = oth[row * WPR + (wi == 0 ? WPR - 1 : wi - 1)];
            n_x = (n_same << 1) | (prev >> 31);
        } else {                            // neighbour at k+1: bit j <- bit j+1
            const uint32_t next = oth[row * WPR + (wi == WPR - 1 ? 0 : wi + 1)];
            n_x = (n_same >> 1) | (next << 31);
        }
        const uint32_t upd = rule_word(s[i], rho[i], n_same, n_x, n_yp, n_ym, n_zp, n_zm);
        uint32_t m;
        if (ff) {
            // mixed-cycle double checkerboard (D15): `coarse` = 0 / 1 is the first / second coarse
            // colour of the sweep's drawn order; the block bits come from block_order_kernel
            const int nB = L >> 3;
            const size_t Bi0 = ((size_t)(z >> 3) * nB + (y >> 3)) * nB + 8 * (size_t)wi;
            const uint32_t ffbyte = (ff[(size_t)rep * ff_stride + (Bi0 >> 5)] >> (Bi0 & 31)) & 0xFFu;
            m = dcb_mixed_mask(y, z, coarse_mixed, pass, c, ffbyte);
        } else {
            m = dcb_mask(y, z, coarse);                         // double checkerboard: one coarse colour
        }
        out[i] = (upd & m) | (s[i] & ~m);
    }
    reinterpret_cast<uint4 *>(own)[g] = make_uint4(out[0], out[1], out[2], out[3]);
}

// ---------------------------------------------------------------------------------------------
// Finite-temperature Glauber half-sweep (eq. (5); reading D13).
// A site with n antiparallel neighbours flips iff u < thr[n], u its 32-bit uniform of the sweep,
// thr[n] = floor(2^32 / (1 + exp((12 - 4n)/T))) in [0, 2^32].  Bit-sliced: n is counted with two
// 3:2 compressors (c2 c1 c0), the seven class masks are one LOP3 each, and u < thr[n] is decided
// MSB first over bit planes: plane j of u for the 128 spins of a group is one Philox call
// (counter (q, t, colour, 4 + j)), the threshold's bit of that plane is a 7-entry truth table over
// n (GlauberTables, built on the host).  The loop stops as soon as no site of the warp is still
// undecided (about 13 of 32 planes on average), which is exact: later planes cannot change lt.
// ---------------------------------------------------------------------------------------------
struct GlauberTables {
    uint32_t sel[33][7];     // sel[B][n] = all ones iff bit B (32 = the 2^32 bit, .. 0) of thr[n] is set
};

__global__ void __launch_bounds__(256)
halfsweep_glauber_kernel(uint32_t *__restrict__ state, const uint64_t *__restrict__ seeds, int L,
                         uint32_t t, int phase, int mixed, const __grid_constant__ GlauberTables tb)
{
    const int WPR = L >> 6;
    const size_t WPC = (size_t)L * L * WPR;
    const size_t g = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const bool active = g < WPC / 4;
    const size_t gg = active ? g : 0;                           // idle lanes follow along (warp votes)
    const int rep = blockIdx.y;
    const uint64_t seed = seeds[rep];
    const int c = mixed ? phase ^ first_colour(seed, t) : phase;
    uint32_t *own = state + (size_t)rep * 2 * WPC + (size_t)c * WPC;
    const uint32_t *oth = state + (size_t)rep * 2 * WPC + (size_t)(1 - c) * WPC;
    const uint4 sv = reinterpret_cast<const uint4 *>(own)[gg];
    const uint32_t s[4] = {sv.x, sv.y, sv.z, sv.w};
    uint32_t cls[4][7];                                         // class masks: n == 0..6
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const size_t w = 4 * gg + i;
        const int wi = (int)(w % WPR);
        const size_t row = w / WPR;
        const int y = (int)(row % L), z = (int)(row / L);
        const int yp = (y + 1 == L) ? 0 : y + 1, ym = (y == 0) ? L - 1 : y - 1;
        const int zp = (z + 1 == L) ? 0 : z + 1, zm = (z == 0) ? L - 1 : z - 1;
        const uint32_t n_same = oth[w];
        uint32_t n_x;
        if (((y + z + c) & 1) == 0) {
            const uint32_t prev = oth[row * WPR + (wi == 0 ? WPR - 1 : wi - 1)];
            n_x = (n_same << 1) | (prev >> 31);
        } else {
            const uint32_t next = oth[row * WPR + (wi == WPR - 1 ? 0 : wi + 1)];
            n_x = (n_same >> 1) | (next << 31);
        }
        // antiparallel indicators of the six neighbours
        const uint32_t d1 = s[i] ^ n_same, d2 = s[i] ^ n_x;
        const uint32_t d3 = s[i] ^ oth[((size_t)z * L + yp) * WPR + wi];
        const uint32_t d4 = s[i] ^ oth[((size_t)z * L + ym) * WPR + wi];
        const uint32_t d5 = s[i] ^ oth[((size_t)zp * L + y) * WPR + wi];
        const uint32_t d6 = s[i] ^ oth[((size_t)zm * L + y) * WPR + wi];
        const uint32_t sa = d1 ^ d2 ^ d3, ca = maj3(d1, d2, d3);
        const uint32_t sb = d4 ^ d5 ^ d6, cb = maj3(d4, d5, d6);
        const uint32_t c0 = sa ^ sb, k1 = sa & sb;
        const uint32_t c1 = ca ^ cb ^ k1, c2 = maj3(ca, cb, k1);
#pragma unroll
        for (int n = 0; n < 7; ++n)
            cls[i][n] = ((n & 1) ? c0 : ~c0) & ((n & 2) ? c1 : ~c1) & ((n & 4) ? c2 : ~c2);
    }
    uint32_t lt[4], eq[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {                               // the 2^32 bit: u has none
        uint32_t T = 0;
#pragma unroll
        for (int n = 0; n < 7; ++n) T |= cls[i][n] & tb.sel[32][n];
        lt[i] = T;
        eq[i] = ~T;
    }
    for (int j = 0; j < 32; ++j) {
        const uint32_t alive = active ? (eq[0] | eq[1] | eq[2] | eq[3]) : 0u;
        if (!__any_sync(0xffffffffu, alive != 0u)) break;
        const uint4 rnd = philox4x32_10((uint32_t)gg, t, (uint32_t)c, 4u + (uint32_t)j, (uint32_t)seed,
                                        (uint32_t)(seed >> 32));
        const uint32_t r[4] = {rnd.x, rnd.y, rnd.z, rnd.w};
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            uint32_t T = 0;
#pragma unroll
            for (int n = 0; n < 7; ++n) T |= cls[i][n] & tb.sel[31 - j][n];
            lt[i] |= eq[i] & ~r[i] & T;
            eq[i] &= ~(r[i] ^ T);
        }
    }
    if (active)
        reinterpret_cast<uint4 *>(own)[g] = make_uint4(s[0] ^ lt[0], s[1] ^ lt[1], s[2] ^ lt[2], s[3] ^ lt[3]);
}

}  // namespace ising
