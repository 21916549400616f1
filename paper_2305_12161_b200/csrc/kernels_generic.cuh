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
__device__ __forceinline__ uint4 class_select(const uint32_t lut, const uint4 c2, const uint4 c1, const uint4 c0)
{
    uint4 T;
    const uint32_t idx = lut & 127u;
    asm volatile(
        "{\n"
        "GLT: .branchtargets GL0, GL1, GL2, GL3, GL4, GL5, GL6, GL7, GL8, GL9, GL10, GL11, GL12, GL13, GL14, GL15, GL16, GL17, GL18, GL19, GL20, GL21, GL22, GL23, GL24, GL25, GL26, GL27, GL28, GL29, GL30, GL31, GL32, GL33, GL34, GL35, GL36, GL37, GL38, GL39, GL40, GL41, GL42, GL43, GL44, GL45, GL46, GL47, GL48, GL49, GL50, GL51, GL52, GL53, GL54, GL55, GL56, GL57, GL58, GL59, GL60, GL61, GL62, GL63, GL64, GL65, GL66, GL67, GL68, GL69, GL70, GL71, GL72, GL73, GL74, GL75, GL76, GL77, GL78, GL79, GL80, GL81, GL82, GL83, GL84, GL85, GL86, GL87, GL88, GL89, GL90, GL91, GL92, GL93, GL94, GL95, GL96, GL97, GL98, GL99, GL100, GL101, GL102, GL103, GL104, GL105, GL106, GL107, GL108, GL109, GL110, GL111, GL112, GL113, GL114, GL115, GL116, GL117, GL118, GL119, GL120, GL121, GL122, GL123, GL124, GL125, GL126, GL127;\n"
        "brx.idx %12, GLT;\n"
        "GL0: lop3.b32 %0, %4, %8, %13, 0; lop3.b32 %1, %5, %9, %14, 0; lop3.b32 %2, %6, %10, %15, 0; lop3.b32 %3, %7, %11, %16, 0; bra.uni GLE;\n"
        "GL1: lop3.b32 %0, %4, %8, %13, 1; lop3.b32 %1, %5, %9, %14, 1; lop3.b32 %2, %6, %10, %15, 1; lop3.b32 %3, %7, %11, %16, 1; bra.uni GLE;\n"
        "GL2: lop3.b32 %0, %4, %8, %13, 2; lop3.b32 %1, %5, %9, %14, 2; lop3.b32 %2, %6, %10, %15, 2; lop3.b32 %3, %7, %11, %16, 2; bra.uni GLE;\n"
        "GL3: lop3.b32 %0, %4, %8, %13, 3; lop3.b32 %1, %5, %9, %14, 3; lop3.b32 %2, %6, %10, %15, 3; lop3.b32 %3, %7, %11, %16, 3; bra.uni GLE;\n"
        "GL4: lop3.b32 %0, %4, %8, %13, 4; lop3.b32 %1, %5, %9, %14, 4; lop3.b32 %2, %6, %10, %15, 4; lop3.b32 %3, %7, %11, %16, 4; bra.uni GLE;\n"
        "GL5: lop3.b32 %0, %4, %8, %13, 5; lop3.b32 %1, %5, %9, %14, 5; lop3.b32 %2, %6, %10, %15, 5; lop3.b32 %3, %7, %11, %16, 5; bra.uni GLE;\n"
        "GL6: lop3.b32 %0, %4, %8, %13, 6; lop3.b32 %1, %5, %9, %14, 6; lop3.b32 %2, %6, %10, %15, 6; lop3.b32 %3, %7, %11, %16, 6; bra.uni GLE;\n"
        "GL7: lop3.b32 %0, %4, %8, %13, 7; lop3.b32 %1, %5, %9, %14, 7; lop3.b32 %2, %6, %10, %15, 7; lop3.b32 %3, %7, %11, %16, 7; bra.uni GLE;\n"
        "GL8: lop3.b32 %0, %4, %8, %13, 8; lop3.b32 %1, %5, %9, %14, 8; lop3.b32 %2, %6, %10, %15, 8; lop3.b32 %3, %7, %11, %16, 8; bra.uni GLE;\n"
        "GL9: lop3.b32 %0, %4, %8, %13, 9; lop3.b32 %1, %5, %9, %14, 9; lop3.b32 %2, %6, %10, %15, 9; lop3.b32 %3, %7, %11, %16, 9; bra.uni GLE;\n"
        "GL10: lop3.b32 %0, %4, %8, %13, 10; lop3.b32 %1, %5, %9, %14, 10; lop3.b32 %2, %6, %10, %15, 10; lop3.b32 %3, %7, %11, %16, 10; bra.uni GLE;\n"
        "GL11: lop3.b32 %0, %4, %8, %13, 11; lop3.b32 %1, %5, %9, %14, 11; lop3.b32 %2, %6, %10, %15, 11; lop3.b32 %3, %7, %11, %16, 11; bra.uni GLE;\n"
        "GL12: lop3.b32 %0, %4, %8, %13, 12; lop3.b32 %1, %5, %9, %14, 12; lop3.b32 %2, %6, %10, %15, 12; lop3.b32 %3, %7, %11, %16, 12; bra.uni GLE;\n"
        "GL13: lop3.b32 %0, %4, %8, %13, 13; lop3.b32 %1, %5, %9, %14, 13; lop3.b32 %2, %6, %10, %15, 13; lop3.b32 %3, %7, %11, %16, 13; bra.uni GLE;\n"
        "GL14: lop3.b32 %0, %4, %8, %13, 14; lop3.b32 %1, %5, %9, %14, 14; lop3.b32 %2, %6, %10, %15, 14; lop3.b32 %3, %7, %11, %16, 14; bra.uni GLE;\n"
        "GL15: lop3.b32 %0, %4, %8, %13, 15; lop3.b32 %1, %5, %9, %14, 15; lop3.b32 %2, %6, %10, %15, 15; lop3.b32 %3, %7, %11, %16, 15; bra.uni GLE;\n"
        "GL16: lop3.b32 %0, %4, %8, %13, 16; lop3.b32 %1, %5, %9, %14, 16; lop3.b32 %2, %6, %10, %15, 16; lop3.b32 %3, %7, %11, %16, 16; bra.uni GLE;\n"
        "GL17: lop3.b32 %0, %4, %8, %13, 17; lop3.b32 %1, %5, %9, %14, 17; lop3.b32 %2, %6, %10, %15, 17; lop3.b32 %3, %7, %11, %16, 17; bra.uni GLE;\n"
        "GL18: lop3.b32 %0, %4, %8, %13, 18; lop3.b32 %1, %5, %9, %14, 18; lop3.b32 %2, %6, %10, %15, 18; lop3.b32 %3, %7, %11, %16, 18; bra.uni GLE;\n"
        "GL19: lop3.b32 %0, %4, %8, %13, 19; lop3.b32 %1, %5, %9, %14, 19; lop3.b32 %2, %6, %10, %15, 19; lop3.b32 %3, %7, %11, %16, 19; bra.uni GLE;\n"
        "GL20: lop3.b32 %0, %4, %8, %13, 20; lop3.b32 %1, %5, %9, %14, 20; lop3.b32 %2, %6, %10, %15, 20; lop3.b32 %3, %7, %11, %16, 20; bra.uni GLE;\n"
        "GL21: lop3.b32 %0, %4, %8, %13, 21; lop3.b32 %1, %5, %9, %14, 21; lop3.b32 %2, %6, %10, %15, 21; lop3.b32 %3, %7, %11, %16, 21; bra.uni GLE;\n"
        "GL22: lop3.b32 %0, %4, %8, %13, 22; lop3.b32 %1, %5, %9, %14, 22; lop3.b32 %2, %6, %10, %15, 22; lop3.b32 %3, %7, %11, %16, 22; bra.uni GLE;\n"
        "GL23: lop3.b32 %0, %4, %8, %13, 23; lop3.b32 %1, %5, %9, %14, 23; lop3.b32 %2, %6, %10, %15, 23; lop3.b32 %3, %7, %11, %16, 23; bra.uni GLE;\n"
        "GL24: lop3.b32 %0, %4, %8, %13, 24; lop3.b32 %1, %5, %9, %14, 24; lop3.b32 %2, %6, %10, %15, 24; lop3.b32 %3, %7, %11, %16, 24; bra.uni GLE;\n"
        "GL25: lop3.b32 %0, %4, %8, %13, 25; lop3.b32 %1, %5, %9, %14, 25; lop3.b32 %2, %6, %10, %15, 25; lop3.b32 %3, %7, %11, %16, 25; bra.uni GLE;\n"
        "GL26: lop3.b32 %0, %4, %8, %13, 26; lop3.b32 %1, %5, %9, %14, 26; lop3.b32 %2, %6, %10, %15, 26; lop3.b32 %3, %7, %11, %16, 26; bra.uni GLE;\n"
        "GL27: lop3.b32 %0, %4, %8, %13, 27; lop3.b32 %1, %5, %9, %14, 27; lop3.b32 %2, %6, %10, %15, 27; lop3.b32 %3, %7, %11, %16, 27; bra.uni GLE;\n"
        "GL28: lop3.b32 %0, %4, %8, %13, 28; lop3.b32 %1, %5, %9, %14, 28; lop3.b32 %2, %6, %10, %15, 28; lop3.b32 %3, %7, %11, %16, 28; bra.uni GLE;\n"
        "GL29: lop3.b32 %0, %4, %8, %13, 29; lop3.b32 %1, %5, %9, %14, 29; lop3.b32 %2, %6, %10, %15, 29; lop3.b32 %3, %7, %11, %16, 29; bra.uni GLE;\n"
        "GL30: lop3.b32 %0, %4, %8, %13, 30; lop3.b32 %1, %5, %9, %14, 30; lop3.b32 %2, %6, %10, %15, 30; lop3.b32 %3, %7, %11, %16, 30; bra.uni GLE;\n"
        "GL31: lop3.b32 %0, %4, %8, %13, 31; lop3.b32 %1, %5, %9, %14, 31; lop3.b32 %2, %6, %10, %15, 31; lop3.b32 %3, %7, %11, %16, 31; bra.uni GLE;\n"
        "GL32: lop3.b32 %0, %4, %8, %13, 32; lop3.b32 %1, %5, %9, %14, 32; lop3.b32 %2, %6, %10, %15, 32; lop3.b32 %3, %7, %11, %16, 32; bra.uni GLE;\n"
        "GL33: lop3.b32 %0, %4, %8, %13, 33; lop3.b32 %1, %5, %9, %14, 33; lop3.b32 %2, %6, %10, %15, 33; lop3.b32 %3, %7, %11, %16, 33; bra.uni GLE;\n"
        "GL34: lop3.b32 %0, %4, %8, %13, 34; lop3.b32 %1, %5, %9, %14, 34; lop3.b32 %2, %6, %10, %15, 34; lop3.b32 %3, %7, %11, %16, 34; bra.uni GLE;\n"
        "GL35: lop3.b32 %0, %4, %8, %13, 35; lop3.b32 %1, %5, %9, %14, 35; lop3.b32 %2, %6, %10, %15, 35; lop3.b32 %3, %7, %11, %16, 35; bra.uni GLE;\n"
        "GL36: lop3.b32 %0, %4, %8, %13, 36; lop3.b32 %1, %5, %9, %14, 36; lop3.b32 %2, %6, %10, %15, 36; lop3.b32 %3, %7, %11, %16, 36; bra.uni GLE;\n"
        "GL37: lop3.b32 %0, %4, %8, %13, 37; lop3.b32 %1, %5, %9, %14, 37; lop3.b32 %2, %6, %10, %15, 37; lop3.b32 %3, %7, %11, %16, 37; bra.uni GLE;\n"
        "GL38: lop3.b32 %0, %4, %8, %13, 38; lop3.b32 %1, %5, %9, %14, 38; lop3.b32 %2, %6, %10, %15, 38; lop3.b32 %3, %7, %11, %16, 38; bra.uni GLE;\n"
        "GL39: lop3.b32 %0, %4, %8, %13, 39; lop3.b32 %1, %5, %9, %14, 39; lop3.b32 %2, %6, %10, %15, 39; lop3.b32 %3, %7, %11, %16, 39; bra.uni GLE;\n"
        "GL40: lop3.b32 %0, %4, %8, %13, 40; lop3.b32 %1, %5, %9, %14, 40; lop3.b32 %2, %6, %10, %15, 40; lop3.b32 %3, %7, %11, %16, 40; bra.uni GLE;\n"
        "GL41: lop3.b32 %0, %4, %8, %13, 41; lop3.b32 %1, %5, %9, %14, 41; lop3.b32 %2, %6, %10, %15, 41; lop3.b32 %3, %7, %11, %16, 41; bra.uni GLE;\n"
        "GL42: lop3.b32 %0, %4, %8, %13, 42; lop3.b32 %1, %5, %9, %14, 42; lop3.b32 %2, %6, %10, %15, 42; lop3.b32 %3, %7, %11, %16, 42; bra.uni GLE;\n"
        "GL43: lop3.b32 %0, %4, %8, %13, 43; lop3.b32 %1, %5, %9, %14, 43; lop3.b32 %2, %6, %10, %15, 43; lop3.b32 %3, %7, %11, %16, 43; bra.uni GLE;\n"
        "GL44: lop3.b32 %0, %4, %8, %13, 44; lop3.b32 %1, %5, %9, %14, 44; lop3.b32 %2, %6, %10, %15, 44; lop3.b32 %3, %7, %11, %16, 44; bra.uni GLE;\n"
        "GL45: lop3.b32 %0, %4, %8, %13, 45; lop3.b32 %1, %5, %9, %14, 45; lop3.b32 %2, %6, %10, %15, 45; lop3.b32 %3, %7, %11, %16, 45; bra.uni GLE;\n"
        "GL46: lop3.b32 %0, %4, %8, %13, 46; lop3.b32 %1, %5, %9, %14, 46; lop3.b32 %2, %6, %10, %15, 46; lop3.b32 %3, %7, %11, %16, 46; bra.uni GLE;\n"
        "GL47: lop3.b32 %0, %4, %8, %13, 47; lop3.b32 %1, %5, %9, %14, 47; lop3.b32 %2, %6, %10, %15, 47; lop3.b32 %3, %7, %11, %16, 47; bra.uni GLE;\n"
        "GL48: lop3.b32 %0, %4, %8, %13, 48; lop3.b32 %1, %5, %9, %14, 48; lop3.b32 %2, %6, %10, %15, 48; lop3.b32 %3, %7, %11, %16, 48; bra.uni GLE;\n"
        "GL49: lop3.b32 %0, %4, %8, %13, 49; lop3.b32 %1, %5, %9, %14, 49; lop3.b32 %2, %6, %10, %15, 49; lop3.b32 %3, %7, %11, %16, 49; bra.uni GLE;\n"
        "GL50: lop3.b32 %0, %4, %8, %13, 50; lop3.b32 %1, %5, %9, %14, 50; lop3.b32 %2, %6, %10, %15, 50; lop3.b32 %3, %7, %11, %16, 50; bra.uni GLE;\n"
        "GL51: lop3.b32 %0, %4, %8, %13, 51; lop3.b32 %1, %5, %9, %14, 51; lop3.b32 %2, %6, %10, %15, 51; lop3.b32 %3, %7, %11, %16, 51; bra.uni GLE;\n"
        "GL52: lop3.b32 %0, %4, %8, %13, 52; lop3.b32 %1, %5, %9, %14, 52; lop3.b32 %2, %6, %10, %15, 52; lop3.b32 %3, %7, %11, %16, 52; bra.uni GLE;\n"
        "GL53: lop3.b32 %0, %4, %8, %13, 53; lop3.b32 %1, %5, %9, %14, 53; lop3.b32 %2, %6, %10, %15, 53; lop3.b32 %3, %7, %11, %16, 53; bra.uni GLE;\n"
        "GL54: lop3.b32 %0, %4, %8, %13, 54; lop3.b32 %1, %5, %9, %14, 54; lop3.b32 %2, %6, %10, %15, 54; lop3.b32 %3, %7, %11, %16, 54; bra.uni GLE;\n"
        "GL55: lop3.b32 %0, %4, %8, %13, 55; lop3.b32 %1, %5, %9, %14, 55; lop3.b32 %2, %6, %10, %15, 55; lop3.b32 %3, %7, %11, %16, 55; bra.uni GLE;\n"
        "GL56: lop3.b32 %0, %4, %8, %13, 56; lop3.b32 %1, %5, %9, %14, 56; lop3.b32 %2, %6, %10, %15, 56; lop3.b32 %3, %7, %11, %16, 56; bra.uni GLE;\n"
        "GL57: lop3.b32 %0, %4, %8, %13, 57; lop3.b32 %1, %5, %9, %14, 57; lop3.b32 %2, %6, %10, %15, 57; lop3.b32 %3, %7, %11, %16, 57; bra.uni GLE;\n"
        "GL58: lop3.b32 %0, %4, %8, %13, 58; lop3.b32 %1, %5, %9, %14, 58; lop3.b32 %2, %6, %10, %15, 58; lop3.b32 %3, %7, %11, %16, 58; bra.uni GLE;\n"
        "GL59: lop3.b32 %0, %4, %8, %13, 59; lop3.b32 %1, %5, %9, %14, 59; lop3.b32 %2, %6, %10, %15, 59; lop3.b32 %3, %7, %11, %16, 59; bra.uni GLE;\n"
        "GL60: lop3.b32 %0, %4, %8, %13, 60; lop3.b32 %1, %5, %9, %14, 60; lop3.b32 %2, %6, %10, %15, 60; lop3.b32 %3, %7, %11, %16, 60; bra.uni GLE;\n"
        "GL61: lop3.b32 %0, %4, %8, %13, 61; lop3.b32 %1, %5, %9, %14, 61; lop3.b32 %2, %6, %10, %15, 61; lop3.b32 %3, %7, %11, %16, 61; bra.uni GLE;\n"
        "GL62: lop3.b32 %0, %4, %8, %13, 62; lop3.b32 %1, %5, %9, %14, 62; lop3.b32 %2, %6, %10, %15, 62; lop3.b32 %3, %7, %11, %16, 62; bra.uni GLE;\n"
        "GL63: lop3.b32 %0, %4, %8, %13, 63; lop3.b32 %1, %5, %9, %14, 63; lop3.b32 %2, %6, %10, %15, 63; lop3.b32 %3, %7, %11, %16, 63; bra.uni GLE;\n"
        "GL64: lop3.b32 %0, %4, %8, %13, 64; lop3.b32 %1, %5, %9, %14, 64; lop3.b32 %2, %6, %10, %15, 64; lop3.b32 %3, %7, %11, %16, 64; bra.uni GLE;\n"
        "GL65: lop3.b32 %0, %4, %8, %13, 65; lop3.b32 %1, %5, %9, %14, 65; lop3.b32 %2, %6, %10, %15, 65; lop3.b32 %3, %7, %11, %16, 65; bra.uni GLE;\n"
        "GL66: lop3.b32 %0, %4, %8, %13, 66; lop3.b32 %1, %5, %9, %14, 66; lop3.b32 %2, %6, %10, %15, 66; lop3.b32 %3, %7, %11, %16, 66; bra.uni GLE;\n"
        "GL67: lop3.b32 %0, %4, %8, %13, 67; lop3.b32 %1, %5, %9, %14, 67; lop3.b32 %2, %6, %10, %15, 67; lop3.b32 %3, %7, %11, %16, 67; bra.uni GLE;\n"
        "GL68: lop3.b32 %0, %4, %8, %13, 68; lop3.b32 %1, %5, %9, %14, 68; lop3.b32 %2, %6, %10, %15, 68; lop3.b32 %3, %7, %11, %16, 68; bra.uni GLE;\n"
        "GL69: lop3.b32 %0, %4, %8, %13, 69; lop3.b32 %1, %5, %9, %14, 69; lop3.b32 %2, %6, %10, %15, 69; lop3.b32 %3, %7, %11, %16, 69; bra.uni GLE;\n"
        "GL70: lop3.b32 %0, %4, %8, %13, 70; lop3.b32 %1, %5, %9, %14, 70; lop3.b32 %2, %6, %10, %15, 70; lop3.b32 %3, %7, %11, %16, 70; bra.uni GLE;\n"
        "GL71: lop3.b32 %0, %4, %8, %13, 71; lop3.b32 %1, %5, %9, %14, 71; lop3.b32 %2, %6, %10, %15, 71; lop3.b32 %3, %7, %11, %16, 71; bra.uni GLE;\n"
        "GL72: lop3.b32 %0, %4, %8, %13, 72; lop3.b32 %1, %5, %9, %14, 72; lop3.b32 %2, %6, %10, %15, 72; lop3.b32 %3, %7, %11, %16, 72; bra.uni GLE;\n"
        "GL73: lop3.b32 %0, %4, %8, %13, 73; lop3.b32 %1, %5, %9, %14, 73; lop3.b32 %2, %6, %10, %15, 73; lop3.b32 %3, %7, %11, %16, 73; bra.uni GLE;\n"
        "GL74: lop3.b32 %0, %4, %8, %13, 74; lop3.b32 %1, %5, %9, %14, 74; lop3.b32 %2, %6, %10, %15, 74; lop3.b32 %3, %7, %11, %16, 74; bra.uni GLE;\n"
        "GL75: lop3.b32 %0, %4, %8, %13, 75; lop3.b32 %1, %5, %9, %14, 75; lop3.b32 %2, %6, %10, %15, 75; lop3.b32 %3, %7, %11, %16, 75; bra.uni GLE;\n"
        "GL76: lop3.b32 %0, %4, %8, %13, 76; lop3.b32 %1, %5, %9, %14, 76; lop3.b32 %2, %6, %10, %15, 76; lop3.b32 %3, %7, %11, %16, 76; bra.uni GLE;\n"
        "GL77: lop3.b32 %0, %4, %8, %13, 77; lop3.b32 %1, %5, %9, %14, 77; lop3.b32 %2, %6, %10, %15, 77; lop3.b32 %3, %7, %11, %16, 77; bra.uni GLE;\n"
        "GL78: lop3.b32 %0, %4, %8, %13, 78; lop3.b32 %1, %5, %9, %14, 78; lop3.b32 %2, %6, %10, %15, 78; lop3.b32 %3, %7, %11, %16, 78; bra.uni GLE;\n"
        "GL79: lop3.b32 %0, %4, %8, %13, 79; lop3.b32 %1, %5, %9, %14, 79; lop3.b32 %2, %6, %10, %15, 79; lop3.b32 %3, %7, %11, %16, 79; bra.uni GLE;\n"
        "GL80: lop3.b32 %0, %4, %8, %13, 80; lop3.b32 %1, %5, %9, %14, 80; lop3.b32 %2, %6, %10, %15, 80; lop3.b32 %3, %7, %11, %16, 80; bra.uni GLE;\n"
        "GL81: lop3.b32 %0, %4, %8, %13, 81; lop3.b32 %1, %5, %9, %14, 81; lop3.b32 %2, %6, %10, %15, 81; lop3.b32 %3, %7, %11, %16, 81; bra.uni GLE;\n"
        "GL82: lop3.b32 %0, %4, %8, %13, 82; lop3.b32 %1, %5, %9, %14, 82; lop3.b32 %2, %6, %10, %15, 82; lop3.b32 %3, %7, %11, %16, 82; bra.uni GLE;\n"
        "GL83: lop3.b32 %0, %4, %8, %13, 83; lop3.b32 %1, %5, %9, %14, 83; lop3.b32 %2, %6, %10, %15, 83; lop3.b32 %3, %7, %11, %16, 83; bra.uni GLE;\n"
        "GL84: lop3.b32 %0, %4, %8, %13, 84; lop3.b32 %1, %5, %9, %14, 84; lop3.b32 %2, %6, %10, %15, 84; lop3.b32 %3, %7, %11, %16, 84; bra.uni GLE;\n"
        "GL85: lop3.b32 %0, %4, %8, %13, 85; lop3.b32 %1, %5, %9, %14, 85; lop3.b32 %2, %6, %10, %15, 85; lop3.b32 %3, %7, %11, %16, 85; bra.uni GLE;\n"
        "GL86: lop3.b32 %0, %4, %8, %13, 86; lop3.b32 %1, %5, %9, %14, 86; lop3.b32 %2, %6, %10, %15, 86; lop3.b32 %3, %7, %11, %16, 86; bra.uni GLE;\n"
        "GL87: lop3.b32 %0, %4, %8, %13, 87; lop3.b32 %1, %5, %9, %14, 87; lop3.b32 %2, %6, %10, %15, 87; lop3.b32 %3, %7, %11, %16, 87; bra.uni GLE;\n"
        "GL88: lop3.b32 %0, %4, %8, %13, 88; lop3.b32 %1, %5, %9, %14, 88; lop3.b32 %2, %6, %10, %15, 88; lop3.b32 %3, %7, %11, %16, 88; bra.uni GLE;\n"
        "GL89: lop3.b32 %0, %4, %8, %13, 89; lop3.b32 %1, %5, %9, %14, 89; lop3.b32 %2, %6, %10, %15, 89; lop3.b32 %3, %7, %11, %16, 89; bra.uni GLE;\n"
        "GL90: lop3.b32 %0, %4, %8, %13, 90; lop3.b32 %1, %5, %9, %14, 90; lop3.b32 %2, %6, %10, %15, 90; lop3.b32 %3, %7, %11, %16, 90; bra.uni GLE;\n"
        "GL91: lop3.b32 %0, %4, %8, %13, 91; lop3.b32 %1, %5, %9, %14, 91; lop3.b32 %2, %6, %10, %15, 91; lop3.b32 %3, %7, %11, %16, 91; bra.uni GLE;\n"
        "GL92: lop3.b32 %0, %4, %8, %13, 92; lop3.b32 %1, %5, %9, %14, 92; lop3.b32 %2, %6, %10, %15, 92; lop3.b32 %3, %7, %11, %16, 92; bra.uni GLE;\n"
        "GL93: lop3.b32 %0, %4, %8, %13, 93; lop3.b32 %1, %5, %9, %14, 93; lop3.b32 %2, %6, %10, %15, 93; lop3.b32 %3, %7, %11, %16, 93; bra.uni GLE;\n"
        "GL94: lop3.b32 %0, %4, %8, %13, 94; lop3.b32 %1, %5, %9, %14, 94; lop3.b32 %2, %6, %10, %15, 94; lop3.b32 %3, %7, %11, %16, 94; bra.uni GLE;\n"
        "GL95: lop3.b32 %0, %4, %8, %13, 95; lop3.b32 %1, %5, %9, %14, 95; lop3.b32 %2, %6, %10, %15, 95; lop3.b32 %3, %7, %11, %16, 95; bra.uni GLE;\n"
        "GL96: lop3.b32 %0, %4, %8, %13, 96; lop3.b32 %1, %5, %9, %14, 96; lop3.b32 %2, %6, %10, %15, 96; lop3.b32 %3, %7, %11, %16, 96; bra.uni GLE;\n"
        "GL97: lop3.b32 %0, %4, %8, %13, 97; lop3.b32 %1, %5, %9, %14, 97; lop3.b32 %2, %6, %10, %15, 97; lop3.b32 %3, %7, %11, %16, 97; bra.uni GLE;\n"
        "GL98: lop3.b32 %0, %4, %8, %13, 98; lop3.b32 %1, %5, %9, %14, 98; lop3.b32 %2, %6, %10, %15, 98; lop3.b32 %3, %7, %11, %16, 98; bra.uni GLE;\n"
        "GL99: lop3.b32 %0, %4, %8, %13, 99; lop3.b32 %1, %5, %9, %14, 99; lop3.b32 %2, %6, %10, %15, 99; lop3.b32 %3, %7, %11, %16, 99; bra.uni GLE;\n"
        "GL100: lop3.b32 %0, %4, %8, %13, 100; lop3.b32 %1, %5, %9, %14, 100; lop3.b32 %2, %6, %10, %15, 100; lop3.b32 %3, %7, %11, %16, 100; bra.uni GLE;\n"
        "GL101: lop3.b32 %0, %4, %8, %13, 101; lop3.b32 %1, %5, %9, %14, 101; lop3.b32 %2, %6, %10, %15, 101; lop3.b32 %3, %7, %11, %16, 101; bra.uni GLE;\n"
        "GL102: lop3.b32 %0, %4, %8, %13, 102; lop3.b32 %1, %5, %9, %14, 102; lop3.b32 %2, %6, %10, %15, 102; lop3.b32 %3, %7, %11, %16, 102; bra.uni GLE;\n"
        "GL103: lop3.b32 %0, %4, %8, %13, 103; lop3.b32 %1, %5, %9, %14, 103; lop3.b32 %2, %6, %10, %15, 103; lop3.b32 %3, %7, %11, %16, 103; bra.uni GLE;\n"
        "GL104: lop3.b32 %0, %4, %8, %13, 104; lop3.b32 %1, %5, %9, %14, 104; lop3.b32 %2, %6, %10, %15, 104; lop3.b32 %3, %7, %11, %16, 104; bra.uni GLE;\n"
        "GL105: lop3.b32 %0, %4, %8, %13, 105; lop3.b32 %1, %5, %9, %14, 105; lop3.b32 %2, %6, %10, %15, 105; lop3.b32 %3, %7, %11, %16, 105; bra.uni GLE;\n"
        "GL106: lop3.b32 %0, %4, %8, %13, 106; lop3.b32 %1, %5, %9, %14, 106; lop3.b32 %2, %6, %10, %15, 106; lop3.b32 %3, %7, %11, %16, 106; bra.uni GLE;\n"
        "GL107: lop3.b32 %0, %4, %8, %13, 107; lop3.b32 %1, %5, %9, %14, 107; lop3.b32 %2, %6, %10, %15, 107; lop3.b32 %3, %7, %11, %16, 107; bra.uni GLE;\n"
        "GL108: lop3.b32 %0, %4, %8, %13, 108; lop3.b32 %1, %5, %9, %14, 108; lop3.b32 %2, %6, %10, %15, 108; lop3.b32 %3, %7, %11, %16, 108; bra.uni GLE;\n"
        "GL109: lop3.b32 %0, %4, %8, %13, 109; lop3.b32 %1, %5, %9, %14, 109; lop3.b32 %2, %6, %10, %15, 109; lop3.b32 %3, %7, %11, %16, 109; bra.uni GLE;\n"
        "GL110: lop3.b32 %0, %4, %8, %13, 110; lop3.b32 %1, %5, %9, %14, 110; lop3.b32 %2, %6, %10, %15, 110; lop3.b32 %3, %7, %11, %16, 110; bra.uni GLE;\n"
        "GL111: lop3.b32 %0, %4, %8, %13, 111; lop3.b32 %1, %5, %9, %14, 111; lop3.b32 %2, %6, %10, %15, 111; lop3.b32 %3, %7, %11, %16, 111; bra.uni GLE;\n"
        "GL112: lop3.b32 %0, %4, %8, %13, 112; lop3.b32 %1, %5, %9, %14, 112; lop3.b32 %2, %6, %10, %15, 112; lop3.b32 %3, %7, %11, %16, 112; bra.uni GLE;\n"
        "GL113: lop3.b32 %0, %4, %8, %13, 113; lop3.b32 %1, %5, %9, %14, 113; lop3.b32 %2, %6, %10, %15, 113; lop3.b32 %3, %7, %11, %16, 113; bra.uni GLE;\n"
        "GL114: lop3.b32 %0, %4, %8, %13, 114; lop3.b32 %1, %5, %9, %14, 114; lop3.b32 %2, %6, %10, %15, 114; lop3.b32 %3, %7, %11, %16, 114; bra.uni GLE;\n"
        "GL115: lop3.b32 %0, %4, %8, %13, 115; lop3.b32 %1, %5, %9, %14, 115; lop3.b32 %2, %6, %10, %15, 115; lop3.b32 %3, %7, %11, %16, 115; bra.uni GLE;\n"
        "GL116: lop3.b32 %0, %4, %8, %13, 116; lop3.b32 %1, %5, %9, %14, 116; lop3.b32 %2, %6, %10, %15, 116; lop3.b32 %3, %7, %11, %16, 116; bra.uni GLE;\n"
        "GL117: lop3.b32 %0, %4, %8, %13, 117; lop3.b32 %1, %5, %9, %14, 117; lop3.b32 %2, %6, %10, %15, 117; lop3.b32 %3, %7, %11, %16, 117; bra.uni GLE;\n"
        "GL118: lop3.b32 %0, %4, %8, %13, 118; lop3.b32 %1, %5, %9, %14, 118; lop3.b32 %2, %6, %10, %15, 118; lop3.b32 %3, %7, %11, %16, 118; bra.uni GLE;\n"
        "GL119: lop3.b32 %0, %4, %8, %13, 119; lop3.b32 %1, %5, %9, %14, 119; lop3.b32 %2, %6, %10, %15, 119; lop3.b32 %3, %7, %11, %16, 119; bra.uni GLE;\n"
        "GL120: lop3.b32 %0, %4, %8, %13, 120; lop3.b32 %1, %5, %9, %14, 120; lop3.b32 %2, %6, %10, %15, 120; lop3.b32 %3, %7, %11, %16, 120; bra.uni GLE;\n"
        "GL121: lop3.b32 %0, %4, %8, %13, 121; lop3.b32 %1, %5, %9, %14, 121; lop3.b32 %2, %6, %10, %15, 121; lop3.b32 %3, %7, %11, %16, 121; bra.uni GLE;\n"
        "GL122: lop3.b32 %0, %4, %8, %13, 122; lop3.b32 %1, %5, %9, %14, 122; lop3.b32 %2, %6, %10, %15, 122; lop3.b32 %3, %7, %11, %16, 122; bra.uni GLE;\n"
        "GL123: lop3.b32 %0, %4, %8, %13, 123; lop3.b32 %1, %5, %9, %14, 123; lop3.b32 %2, %6, %10, %15, 123; lop3.b32 %3, %7, %11, %16, 123; bra.uni GLE;\n"
        "GL124: lop3.b32 %0, %4, %8, %13, 124; lop3.b32 %1, %5, %9, %14, 124; lop3.b32 %2, %6, %10, %15, 124; lop3.b32 %3, %7, %11, %16, 124; bra.uni GLE;\n"
        "GL125: lop3.b32 %0, %4, %8, %13, 125; lop3.b32 %1, %5, %9, %14, 125; lop3.b32 %2, %6, %10, %15, 125; lop3.b32 %3, %7, %11, %16, 125; bra.uni GLE;\n"
        "GL126: lop3.b32 %0, %4, %8, %13, 126; lop3.b32 %1, %5, %9, %14, 126; lop3.b32 %2, %6, %10, %15, 126; lop3.b32 %3, %7, %11, %16, 126; bra.uni GLE;\n"
        "GL127: lop3.b32 %0, %4, %8, %13, 127; lop3.b32 %1, %5, %9, %14, 127; lop3.b32 %2, %6, %10, %15, 127; lop3.b32 %3, %7, %11, %16, 127; bra.uni GLE;\n"
        "GLE:\n"
        "}\n"
        : "=r"(T.x), "=r"(T.y), "=r"(T.z), "=r"(T.w)
        : "r"(c2.x), "r"(c2.y), "r"(c2.z), "r"(c2.w), "r"(c1.x), "r"(c1.y), "r"(c1.z), "r"(c1.w), "r"(idx),
          "r"(c0.x), "r"(c0.y), "r"(c0.z), "r"(c0.w));
    return T;
}

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
