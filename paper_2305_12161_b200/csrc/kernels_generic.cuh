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
// 3:2 compressors into three bit planes (c2 c1 c0), and u < thr[n] is decided MSB first over bit
// planes: plane j of u for the 128 spins of a group is one Philox call (counter (q, t, colour,
// 4 + j)); the threshold's bit of that plane is a 7-entry truth table over n, i.e. a three-input
// boolean function of (c2, c1, c0): ONE LOP3 whose immediate is chosen by a warp-uniform switch on
// the table (GlauberTables::lut, built on the host).  The loop stops as soon as no site of the warp
// is still undecided (13-14 of 32 planes on average: each plane halves the undecided sites of the
// warp's 4096), which is exact: later planes cannot change a decided site.
// Philox: everything that does not depend on the plane is hoisted out of the loop (round 0 has one
// product, M0*q; in round 1 the product M0*c0 and in round 2 the product M1*c2 do not depend on the
// tag): 16 IMAD.WIDE + 18 LOP3 per plane; the round keys are computed once per thread.
// ---------------------------------------------------------------------------------------------
struct GlauberTables {
    uint32_t lut[33];        // bit n of lut[B] = bit B (32 = the 2^32 bit, .. 0) of thr[n], n = 0..6
};

// T = f(c2, c1, c0) word by word with the truth table `lut` (bit n = value for n = 4 c2 + 2 c1 + c0):
// one LOP3 per word whose immediate is the table, reached through a 128-entry jump table (brx.idx;
// the C++ switch is lowered to a seven-level compare tree instead, 14 instructions per dispatch).
// The 128 cases differ only in the immediate, so the preprocessor writes them: case 0xHL has the label
// GLHL and the immediate 0xHL (H = 0..7, L = 0..f).
#define ISING_GL_LBL(h, l) "GL" #h #l
#define ISING_GL_TGT(h, l) ISING_GL_LBL(h, l) ", "
#define ISING_GL_CASE(h, l)                                                                                    \
    ISING_GL_LBL(h, l) ": lop3.b32 %0, %4, %8, %13, 0x" #h #l "; lop3.b32 %1, %5, %9, %14, 0x" #h #l             \
                       "; lop3.b32 %2, %6, %10, %15, 0x" #h #l "; lop3.b32 %3, %7, %11, %16, 0x" #h #l "; bra.uni GLE;\n"
#define ISING_GL_ROW(M, h)                                                                                     \
    M(h, 0) M(h, 1) M(h, 2) M(h, 3) M(h, 4) M(h, 5) M(h, 6) M(h, 7) M(h, 8) M(h, 9) M(h, a) M(h, b) M(h, c) M(h, d) M(h, e) M(h, f)
#define ISING_GL_ALL(M)                                                                                        \
    ISING_GL_ROW(M, 0) ISING_GL_ROW(M, 1) ISING_GL_ROW(M, 2) ISING_GL_ROW(M, 3) ISING_GL_ROW(M, 4) ISING_GL_ROW(M, 5)  \
    ISING_GL_ROW(M, 6) ISING_GL_ROW(M, 7)
__device__ __forceinline__ uint4 class_select(const uint32_t lut, const uint4 c2, const uint4 c1, const uint4 c0)
{
    uint4 T;
    const uint32_t idx = lut & 127u;
    asm volatile(
        "{\n"
        // targets 0..127 in index order; GLE closes the list and is never indexed (idx < 128)
        "GLT: .branchtargets " ISING_GL_ALL(ISING_GL_TGT) "GLE;\n"
        "brx.idx %12, GLT;\n"
        ISING_GL_ALL(ISING_GL_CASE)
        "GLE:\n"
        "}\n"
        : "=r"(T.x), "=r"(T.y), "=r"(T.z), "=r"(T.w)
        : "r"(c2.x), "r"(c2.y), "r"(c2.z), "r"(c2.w), "r"(c1.x), "r"(c1.y), "r"(c1.z), "r"(c1.w), "r"(idx),
          "r"(c0.x), "r"(c0.y), "r"(c0.z), "r"(c0.w));
    return T;
}
#undef ISING_GL_ALL
#undef ISING_GL_ROW
#undef ISING_GL_CASE
#undef ISING_GL_TGT
#undef ISING_GL_LBL

// 32 x 32 -> 64 bit product as ONE IMAD.WIDE.U32 (written in PTX: inside the plane loop the C++
// form picked up a dead add per product)
__device__ __forceinline__ uint64_t mul_wide(uint32_t a, uint32_t b)
{
    uint64_t p;
    asm("mul.wide.u32 %0, %1, %2;" : "=l"(p) : "r"(a), "r"(b));
    return p;
}

__global__ void __launch_bounds__(256)
halfsweep_glauber_kernel(uint32_t *__restrict__ state, const uint64_t *__restrict__ seeds, int L,
                         uint32_t t, int phase, int mixed, const __grid_constant__ GlauberTables tb)
{
    // all indices fit 32 bits: a colour has L^3/64 <= 2^30 words
    const uint32_t WPR = (uint32_t)L >> 6, uL = (uint32_t)L;
    const uint32_t WPCu = uL * uL * WPR;
    const size_t WPC = WPCu;
    const uint32_t g = blockIdx.x * blockDim.x + threadIdx.x;
    const bool active = g < WPCu / 4;
    const uint32_t gg = active ? g : 0;                         // idle lanes follow along (warp votes)
    const int rep = blockIdx.y;
    const uint64_t seed = seeds[rep];
    const int c = mixed ? phase ^ first_colour(seed, t) : phase;
    uint32_t *own = state + (size_t)rep * 2 * WPC + (size_t)c * WPC;
    const uint32_t *oth = state + (size_t)rep * 2 * WPC + (size_t)(1 - c) * WPC;
    const uint4 sv = reinterpret_cast<const uint4 *>(own)[gg];
    const uint32_t s[4] = {sv.x, sv.y, sv.z, sv.w};
    uint32_t c0[4], c1[4], c2[4];                               // bit planes of n = antiparallel neighbours
    // n = antiparallel neighbours of the 32 sites of word i, as three bit planes (two 3:2 compressors)
    auto count = [&](int i, uint32_t n_same, uint32_t n_x, uint32_t n_yp, uint32_t n_ym, uint32_t n_zp, uint32_t n_zm) {
        const uint32_t d1 = s[i] ^ n_same, d2 = s[i] ^ n_x, d3 = s[i] ^ n_yp;
        const uint32_t d4 = s[i] ^ n_ym, d5 = s[i] ^ n_zp, d6 = s[i] ^ n_zm;
        const uint32_t sa = d1 ^ d2 ^ d3, ca = maj3(d1, d2, d3);
        const uint32_t sb = d4 ^ d5 ^ d6, cb = maj3(d4, d5, d6);
        const uint32_t k1 = sa & sb;
        c0[i] = sa ^ sb;
        c1[i] = ca ^ cb ^ k1;
        c2[i] = maj3(ca, cb, k1);
    };
    if ((WPR & 3u) == 0u) {
        // rows of a multiple of four words (L % 256 == 0): the group lies in one row, so the six
        // neighbour words of all four words come as five 128-bit loads and one edge word (D4)
        const uint32_t R4 = WPR >> 2, row = gg / R4, x4 = gg - row * R4;
        const uint32_t z = row / uL, y = row - z * uL;
        const uint32_t yp = (y + 1 == uL) ? 0 : y + 1, ym = (y == 0) ? uL - 1 : y - 1;
        const uint32_t zp = (z + 1 == uL) ? 0 : z + 1, zm = (z == 0) ? uL - 1 : z - 1;
        const uint4 *oth4 = reinterpret_cast<const uint4 *>(oth);
        const uint4 a = oth4[gg];
        const uint4 vyp = oth4[(z * uL + yp) * R4 + x4], vym = oth4[(z * uL + ym) * R4 + x4];
        const uint4 vzp = oth4[(zp * uL + y) * R4 + x4], vzm = oth4[(zm * uL + y) * R4 + x4];
        uint4 x;
        if (((y + z + (uint32_t)c) & 1u) == 0u) {           // neighbour k-1: bit j <- bit j-1
            const uint32_t edge = oth[4u * (row * R4 + (x4 == 0 ? R4 - 1 : x4 - 1)) + 3u];
            x = make_uint4((a.x << 1) | (edge >> 31), (a.y << 1) | (a.x >> 31), (a.z << 1) | (a.y >> 31),
                           (a.w << 1) | (a.z >> 31));
        } else {                                            // neighbour k+1: bit j <- bit j+1
            const uint32_t edge = oth[4u * (row * R4 + (x4 == R4 - 1 ? 0 : x4 + 1))];
            x = make_uint4((a.x >> 1) | (a.y << 31), (a.y >> 1) | (a.z << 31), (a.z >> 1) | (a.w << 31),
                           (a.w >> 1) | (edge << 31));
        }
        count(0, a.x, x.x, vyp.x, vym.x, vzp.x, vzm.x);
        count(1, a.y, x.y, vyp.y, vym.y, vzp.y, vzm.y);
        count(2, a.z, x.z, vyp.z, vym.z, vzp.z, vzm.z);
        count(3, a.w, x.w, vyp.w, vym.w, vzp.w, vzm.w);
    } else {
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const uint32_t w = 4u * gg + (uint32_t)i;
            const uint32_t row = w / WPR, wi = w - row * WPR;
            const uint32_t z = row / uL, y = row - z * uL;
            const uint32_t yp = (y + 1 == uL) ? 0 : y + 1, ym = (y == 0) ? uL - 1 : y - 1;
            const uint32_t zp = (z + 1 == uL) ? 0 : z + 1, zm = (z == 0) ? uL - 1 : z - 1;
            const uint32_t n_same = oth[w];
            uint32_t n_x;
            if (((y + z + (uint32_t)c) & 1u) == 0u) {
                const uint32_t prev = oth[row * WPR + (wi == 0 ? WPR - 1 : wi - 1)];
                n_x = (n_same << 1) | (prev >> 31);
            } else {
                const uint32_t next = oth[row * WPR + (wi == WPR - 1 ? 0 : wi + 1)];
                n_x = (n_same >> 1) | (next << 31);
            }
            count(i, n_same, n_x, oth[(z * uL + yp) * WPR + wi], oth[(z * uL + ym) * WPR + wi],
                  oth[(zp * uL + y) * WPR + wi], oth[(zm * uL + y) * WPR + wi]);
        }
    }
    // Philox4x32-10 of counter (q, t, c, 4 + j), key = seed: the plane-independent parts
    uint32_t k0r[10], k1r[10];
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        k0r[r] = (uint32_t)seed + (uint32_t)r * kPhiloxW0;
        k1r[r] = (uint32_t)(seed >> 32) + (uint32_t)r * kPhiloxW1;
    }
    const uint32_t q = gg;
    const uint64_t q0 = mul_wide(kPhiloxM0, q);                            // round 0, p0
    const uint32_t a0 = t ^ k0r[0];                                          // round-0 c0 (hi(M1*c) = 0)
    const uint32_t b0 = c ? kPhiloxM1 : 0u;                                  // round-0 c1 = lo(M1*c)
    const uint32_t x0 = (uint32_t)(q0 >> 32) ^ k1r[0];                       // round-0 c2 = x0 ^ tag
    const uint64_t pa = mul_wide(kPhiloxM0, a0);                            // round 1, p0
    const uint32_t r1c2 = (uint32_t)(pa >> 32) ^ (uint32_t)q0 ^ k1r[1];      // round-1 c2
    const uint32_t r1c3 = (uint32_t)pa;                                      // round-1 c3
    const uint64_t pb = mul_wide(kPhiloxM1, r1c2);                          // round 2, p1
    const uint4 C0 = make_uint4(c0[0], c0[1], c0[2], c0[3]), C1 = make_uint4(c1[0], c1[1], c1[2], c1[3]);
    const uint4 C2 = make_uint4(c2[0], c2[1], c2[2], c2[3]);
    uint4 lt = class_select(tb.lut[32], C2, C1, C0);            // the 2^32 bit: u has none
    uint4 eq = make_uint4(~lt.x, ~lt.y, ~lt.z, ~lt.w);
    for (int j = 0; j < 32; ++j) {
        const uint32_t alive = active ? (eq.x | eq.y | eq.z | eq.w) : 0u;
        if (!__any_sync(0xffffffffu, alive != 0u)) break;
        uint4 r;
        {
            const uint32_t tag = 4u + (uint32_t)j;
            const uint64_t p1 = mul_wide(kPhiloxM1, x0 ^ tag);            // round 1
            uint32_t v0 = (uint32_t)(p1 >> 32) ^ b0 ^ k0r[1], v1 = (uint32_t)p1;
            uint64_t p0 = mul_wide(kPhiloxM0, v0);                           // round 2 (p1 = pb)
            v0 = (uint32_t)(pb >> 32) ^ v1 ^ k0r[2];
            uint32_t v2 = (uint32_t)(p0 >> 32) ^ r1c3 ^ k1r[2];
            v1 = (uint32_t)pb;
            uint32_t v3 = (uint32_t)p0;
#pragma unroll
            for (int rr = 3; rr < 10; ++rr) {
                p0 = mul_wide(kPhiloxM0, v0);
                const uint64_t p1r = mul_wide(kPhiloxM1, v2);
                v0 = (uint32_t)(p1r >> 32) ^ v1 ^ k0r[rr];
                v2 = (uint32_t)(p0 >> 32) ^ v3 ^ k1r[rr];
                v1 = (uint32_t)p1r;
                v3 = (uint32_t)p0;
            }
            r = make_uint4(v0, v1, v2, v3);
        }
        const uint4 T = class_select(tb.lut[31 - j], C2, C1, C0);
        lt.x |= eq.x & ~r.x & T.x;  eq.x &= ~(r.x ^ T.x);
        lt.y |= eq.y & ~r.y & T.y;  eq.y &= ~(r.y ^ T.y);
        lt.z |= eq.z & ~r.z & T.z;  eq.z &= ~(r.z ^ T.z);
        lt.w |= eq.w & ~r.w & T.w;  eq.w &= ~(r.w ^ T.w);
    }
    if (active)
        reinterpret_cast<uint4 *>(own)[g] = make_uint4(s[0] ^ lt.x, s[1] ^ lt.y, s[2] ^ lt.z, s[3] ^ lt.w);
}

}  // namespace ising
