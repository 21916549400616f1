// Fused full-sweep kernel, second generation (a2+a3+a4 in one launch), L in {512..4096}.
//
// Same data flow as kernels_fused.cuh (z-march, bulk-async plane tiles in a shared-memory
// ring, black at plane z then white at plane z-1 on the updated black spins, ping-pong
// src -> dst), re-organised around what the first ncu capture showed (instruction-bound:
// ALU pipe 54 %, issue 58 %, 310 warp instructions per group pair against ~185 needed):
//
//  * every thread owns TWO adjacent rows (even tile row 2p and odd row 2p+1) of one 128-spin
//    group column.  The in-row neighbour direction o = (y+z+c)&1 (D4) is then the same for
//    all threads of the CTA at a given step (even row: o = z&1, odd row: the opposite), so
//    the one-bit funnel shifts are compile-time left/right, and one of the two y-neighbours
//    of each row is already in the thread's registers (half the shared-memory reads).
//  * the march is unrolled 6 planes deep (lcm of the 3-slot register windows and the
//    2-periodic shift direction): the windows W_old[z-1..z+1], B_new[z-2..z] rotate by
//    renaming, not by moves.
//  * tiles are 2*NT/R4 rows tall (64 rows at L = 2048) with the same 2+2 halo rows, so the
//    recomputed fraction halves.
//  * Philox4x32-10: everything that depends only on (t, colour, key) is folded on the host
//    per launch (round 0 has one variable product, round 1 one), the rest reads its round
//    keys from the constant bank: 18 IMAD.WIDE + 19 LOP3 per 128 sites.
//
// Site rule: eq. (6) PAPER.md:105-108 (D2); sweep order PAPER.md:116 (D7); random bits D5.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "kernels_fused.cuh"   // mbarrier / bulk-copy helpers, rule_group
#include "philox.cuh"

namespace ising {

// Shared-memory ring depth S; prefetch distance S-1.  The depth itself does not matter (4, 5, 6 time the
// same); 6 = the unroll depth of the march makes the stage of every step a compile-time constant.
constexpr int kF2Stages = 6;

// Per-launch Philox constants (host-folded, D5): counter (q, t, colour, 0), key (k0, k1).
struct SweepConsts {
    uint32_t a0;        // round-0 output c0 = t ^ k0[0]           (hi(M1*colour) = 0)
    uint32_t r0k1;      // k1[0]:        round-0 c2 = hi(M0*q) ^ k1[0]
    uint32_t c1[2];     // (M1*colour) ^ k0[1]: round-1 c0 = hi(M1*c2) ^ c1[colour]
    uint32_t d1;        // hi(M0*a0) ^ k1[1]:   round-1 c2 = lo(M0*q) ^ d1
    uint32_t e2;        // lo(M0*a0) ^ k1[2]:   round-2 c2 = hi(M0*c0) ^ e2
    uint32_t k0[10];    // round keys
    uint32_t k1[10];
};

// `first` = colour updated first in this sweep (0 for the 01 cycle; drawn per sweep in the mixed
// cycle, D10).  The kernel's "black" role is colour `first`, its "white" role colour 1-first;
// c1[role] carries the role's colour into the Philox counter.
inline SweepConsts make_sweep_consts(uint64_t seed, uint32_t t, int first = 0)
{
    SweepConsts s;
    const PhiloxKeys k = make_philox_keys(seed);
    for (int r = 0; r < 10; ++r) {
        s.k0[r] = k.k0[r];
        s.k1[r] = k.k1[r];
    }
    s.a0 = t ^ k.k0[0];
    s.r0k1 = k.k1[0];
    s.c1[0] = (first ? kPhiloxM1 : 0u) ^ k.k0[1];
    s.c1[1] = (first ? 0u : kPhiloxM1) ^ k.k0[1];
    const uint64_t p0 = (uint64_t)kPhiloxM0 * s.a0;
    s.d1 = (uint32_t)(p0 >> 32) ^ k.k1[1];
    s.e2 = (uint32_t)p0 ^ k.k1[2];
    return s;
}

// Philox4x32-10 of counter (q, t, COL, 0) with the constants above; bit-identical to
// philox4x32_10(q, t, COL, 0, keys) (checked against the oracle by the parity tests).
template <int COL>
__device__ __forceinline__ uint4 philox_folded(const uint32_t q, const SweepConsts &k)
{
    // round 0: p0 = M0*q, p1 = M1*COL (constant, hi = 0)
    const uint64_t q0 = (uint64_t)kPhiloxM0 * q;
    uint32_t c2 = (uint32_t)(q0 >> 32) ^ k.r0k1;
    // round 1: p0 = M0*a0 (constant), p1 = M1*c2
    const uint64_t p1a = (uint64_t)kPhiloxM1 * c2;
    uint32_t c0 = (uint32_t)(p1a >> 32) ^ k.c1[COL];
    uint32_t c1 = (uint32_t)p1a;
    c2 = (uint32_t)q0 ^ k.d1;
    // round 2: c3 = lo(M0*a0) folded into e2
    uint32_t c3;
    {
        const uint64_t p0 = (uint64_t)kPhiloxM0 * c0;
        const uint64_t p1 = (uint64_t)kPhiloxM1 * c2;
        c0 = (uint32_t)(p1 >> 32) ^ c1 ^ k.k0[2];
        c2 = (uint32_t)(p0 >> 32) ^ k.e2;
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
    }
#pragma unroll
    for (int r = 3; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)kPhiloxM0 * c0;
        const uint64_t p1 = (uint64_t)kPhiloxM1 * c2;
        c0 = (uint32_t)(p1 >> 32) ^ c1 ^ k.k0[r];
        c2 = (uint32_t)(p0 >> 32) ^ c3 ^ k.k1[r];
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
    }
    return make_uint4(c0, c1, c2, c3);
}

// x-neighbour word with a compile-time direction (D4): O = 0 -> neighbour k-1, edge = word 3
// of the previous group of the row; O = 1 -> neighbour k+1, edge = word 0 of the next group.
template <int O>
__device__ __forceinline__ uint4 xshift_t(const uint4 w, const uint32_t edge)
{
    uint4 r;
    if (O == 0) {
        r.x = __funnelshift_l(edge, w.x, 1);
        r.y = __funnelshift_l(w.x, w.y, 1);
        r.z = __funnelshift_l(w.y, w.z, 1);
        r.w = __funnelshift_l(w.z, w.w, 1);
    } else {
        r.x = __funnelshift_r(w.x, w.y, 1);
        r.y = __funnelshift_r(w.y, w.z, 1);
        r.z = __funnelshift_r(w.z, w.w, 1);
        r.w = __funnelshift_r(w.w, edge, 1);
    }
    return r;
}

template <int O>
__device__ __forceinline__ uint4 xneigh(const uint4 w, const int lane_prev, const int lane_next)
{
    const uint32_t edge = __shfl_sync(0xffffffffu, O ? w.x : w.w, O ? lane_next : lane_prev);
    return xshift_t<O>(w, edge);
}

// Register windows of one thread: [slot][row]; the slot <-> plane assignment rotates with the
// step phase PH = k mod 3 (W: slot PH = z-1, PH+1 = z, PH+2 = z+1; B_new: PH = z-2, PH+1 = z-1,
// PH+2 = z), all indices compile-time after unrolling.
__device__ __forceinline__ bool elect_one()
{
    uint32_t p;
    asm volatile("{\n.reg .pred e;\nelect.sync _|e, 0xffffffff;\nselp.u32 %0, 1, 0, e;\n}\n" : "=r"(p));
    return p != 0;
}

struct F2Win {
    uint4 W[3][2];
    uint4 B[3][2];
};

struct F2Ctx {
    const uint4 *Wst, *Bst;     // shared-memory ring [S][PLANE]
    uint4 *nb;                  // [2][PLANE] B_new planes for the y+-1 exchange
    uint64_t *bars;
    uint4 *dstB, *dstW;         // colour bases of the destination state
    int si0, si_ym, si_yp;      // own position (row 2p) / row 2p-1 / row 2p+2 in a plane tile
    int lane_prev, lane_next;
    uint32_t qrow, qplane;      // Philox group index of (row 2p, x4) inside a plane; groups/plane
    bool ok0, ok1;              // rows whose results this CTA stores
    int nz;
};

// U = position of the step in the 6-step unrolled march (k = 6 lap + U).  With a ring of 3 or 6 stages
// the stage of the step, and with it every shared-memory address, is base + immediate; the mbarrier
// parity is U/3 (S = 3) or the parity of the lap (S = 6).  The exchange plane index is U & 1.
// DCB (double checkerboard, Supp. I.A PAPER.md:223-240): only some blocks are updated in this launch;
// mB / mW are the bit masks of their sites in the four words of this thread's group column (its two
// rows lie in the same block row) at the black plane z and at the white plane z-1; the other sites
// keep their old value (they are the frozen halo of the blocks being updated).
//   DCB = 1 (01 cycle, D14): the blocks of one coarse colour.
//   DCB = 2 (mixed cycle, D15): the blocks of one coarse colour whose drawn first fine colour is the
//           launch's `first` (bit array ff from block_order_kernel); the launch's role order (black
//           role = colour `first`) is then each of these blocks' own order.
__device__ __forceinline__ uint4 keep_unmasked(const uint4 upd, const uint4 old, const uint4 m)
{
    return make_uint4((upd.x & m.x) | (old.x & ~m.x), (upd.y & m.y) | (old.y & ~m.y),
                      (upd.z & m.z) | (old.z & ~m.z), (upd.w & m.w) | (old.w & ~m.w));
}

// bit n of the byte -> nibble n of the word (a block of edge 8 spans four bits of a packed word)
__device__ __forceinline__ uint32_t byte_to_nibbles(uint32_t x)
{
    x = (x | (x << 12)) & 0x000F000Fu;
    x = (x | (x << 6)) & 0x03030303u;
    x = (x | (x << 3)) & 0x11111111u;
    return x * 0xFu;
}

template <int R4, int PLANE, int U, int DCB>
__device__ __forceinline__ void f2_step(F2Win &w, const F2Ctx &c, const int k, const uint32_t qb,
                                        const uint32_t qw, const uint32_t lap_parity,
                                        const SweepConsts &keys, const uint4 mB, const uint4 mW)
{
    constexpr int S = kF2Stages;
    constexpr int PH = U % 3, O = U & 1;
    constexpr int M = PH % 3, Z = (PH + 1) % 3, P = (PH + 2) % 3;
    constexpr bool kStatic = (S == 3 || S == 6);
    const int s = kStatic ? U % S : k % S;
    const uint32_t par = S == 3 ? (uint32_t)(U / 3) : S == 6 ? lap_parity : (uint32_t)((k / S) & 1);
    mbar_wait(smem_u32(&c.bars[s]), par);
    const uint4 *Wnew = c.Wst + s * PLANE;
    const uint4 *Bold = c.Bst + s * PLANE;
    const uint4 *Wz = c.Wst + (kStatic ? (U + S - 1) % S : (k + S - 1) % S) * PLANE;   // plane z of W_old
    w.W[P][0] = Wnew[c.si0];
    w.W[P][1] = Wnew[c.si0 + R4];
    const uint4 Bo0 = Bold[c.si0], Bo1 = Bold[c.si0 + R4];
    // ---- black update at plane z (colour 0); even row: o = O, odd row: o = 1-O ----
    {
        const uint4 Wym = Wz[c.si_ym], Wyp = Wz[c.si_yp];
        const uint32_t q = qb;                                    // group of (row 2p, x4) in plane z
        const uint4 rho0 = philox_folded<0>(q, keys);
        const uint4 rho1 = philox_folded<0>(q + R4, keys);
        const uint4 Wx0 = xneigh<O>(w.W[Z][0], c.lane_prev, c.lane_next);
        const uint4 Wx1 = xneigh<1 - O>(w.W[Z][1], c.lane_prev, c.lane_next);
        w.B[P][0] = rule_group(Bo0, rho0, w.W[Z][0], Wx0, Wym, w.W[Z][1], w.W[M][0], w.W[P][0]);
        w.B[P][1] = rule_group(Bo1, rho1, w.W[Z][1], Wx1, w.W[Z][0], Wyp, w.W[M][1], w.W[P][1]);
        if (DCB) {
            w.B[P][0] = keep_unmasked(w.B[P][0], Bo0, mB);
            w.B[P][1] = keep_unmasked(w.B[P][1], Bo1, mB);
        }
        uint4 *nbw = c.nb + O * PLANE + c.si0;
        nbw[0] = w.B[P][0];
        nbw[R4] = w.B[P][1];
        if (k >= 3 && k < 3 + c.nz) {
            uint4 *d = c.dstB + (size_t)q;
            if (c.ok0) d[0] = w.B[P][0];
            if (c.ok1) d[R4] = w.B[P][1];
        }
    }
    // ---- white update at plane z-1 (colour 1) on the updated black spins ----
    {
        const uint4 *Bz = c.nb + (1 - O) * PLANE;                // B_new[z-1], written last step
        const uint4 Bym = Bz[c.si_ym], Byp = Bz[c.si_yp];
        const uint32_t q = qw;                                    // the same group in plane z-1
        const uint4 rho0 = philox_folded<1>(q, keys);
        const uint4 rho1 = philox_folded<1>(q + R4, keys);
        const uint4 Bx0 = xneigh<O>(w.B[Z][0], c.lane_prev, c.lane_next);
        const uint4 Bx1 = xneigh<1 - O>(w.B[Z][1], c.lane_prev, c.lane_next);
        uint4 nW0 = rule_group(w.W[M][0], rho0, w.B[Z][0], Bx0, Bym, w.B[Z][1], w.B[M][0], w.B[P][0]);
        uint4 nW1 = rule_group(w.W[M][1], rho1, w.B[Z][1], Bx1, w.B[Z][0], Byp, w.B[M][1], w.B[P][1]);
        if (DCB) {
            nW0 = keep_unmasked(nW0, w.W[M][0], mW);
            nW1 = keep_unmasked(nW1, w.W[M][1], mW);
        }
        if (k >= 4) {
            uint4 *d = c.dstW + (size_t)q;
            if (c.ok0) d[0] = nW0;
            if (c.ok1) d[R4] = nW1;
        }
    }
}

__host__ __device__ constexpr int f2_row_lanes(int r4) { return r4 <= 1 ? 1 : r4 <= 2 ? 2 : r4 <= 4 ? 4 : r4 <= 8 ? 8 : r4 <= 16 ? 16 : 32; }

// Grid: blockIdx.x = y tile (RPT stored rows each, RPT even), blockIdx.y = z chunk.
// Chunk boundaries are odd planes, so the first marched plane z0 = zs-3 is even and the
// in-row direction of the even tile row at step k is k & 1.
// DCB: `coarse` = the coarse colour updated by this launch.  01 cycle (DCB = 1, D14): a sweep is the
// launch for coarse 0 followed by the one for coarse 1, each dark sites then light sites.  Mixed
// cycle (DCB = 2, D15): for each coarse colour in the drawn order, one launch with first = 0 and one
// with first = 1, each masked to the blocks that drew that fine order (ff: bit Bi of the block-order
// array of this sweep, word (bz nB + by) R4 + x4 for the 32 blocks a group column spans).
template <int R4, int NT, int DCB>
__global__ void __launch_bounds__(NT, 2)
fused2_sweep_kernel(const uint4 *__restrict__ src, uint4 *__restrict__ dst, const int L,
                    const int RPT, const int nzc, const int first, const int coarse,
                    const uint32_t *__restrict__ ff, const __grid_constant__ SweepConsts keys)
{
    // R4 = groups per row (L / 256); a row takes RL = the next power of two lanes of a warp (L = 1536:
    // 6 groups on 8 lanes; the two spare lanes of a row repeat its last group and store nothing)
    constexpr int RL = f2_row_lanes(R4);
    constexpr int TY = 2 * NT / RL;    // rows in the tile (incl. 2+2 halo rows)
    constexpr int PLANE = TY * R4;     // uint4 per plane tile
    constexpr int S = kF2Stages, D = S - 1;
    static_assert(RL <= 32, "a row must fit a warp");

    extern __shared__ __align__(128) uint4 smem[];
    uint4 *Wst = smem;                     // [S][PLANE]  W_old planes
    uint4 *Bst = smem + S * PLANE;         // [S][PLANE]  B_old planes
    uint4 *nb = smem + 2 * S * PLANE;      // [2][PLANE]  B_new planes (y+-1 exchange)
    uint64_t *bars = reinterpret_cast<uint64_t *>(nb + 2 * PLANE);

    const int tid = threadIdx.x, lane = tid & 31;
    const int x4l = tid & (RL - 1), p = tid / RL;    // lane inside the row, row pair
    const int x4 = (R4 != RL && x4l >= R4) ? R4 - 1 : x4l;   // group column
    const bool spare = R4 != RL && x4l >= R4;
    const int ry = 2 * p;                            // even tile row of this thread
    const int jt = blockIdx.x, zc = blockIdx.y;
    // chunk borders have the parity of 1-first, so that (z0 + first) is even for z0 = zs-3 and
    // the in-row direction o = (y + z + colour) & 1 of the even tile row at step k is k & 1
    const int b0 = (int)((long long)L * zc / nzc), b1 = zc + 1 == nzc ? L : (int)((long long)L * (zc + 1) / nzc);
    const int zs = first ? (b0 & ~1) : (b0 | 1);
    const int ze = first ? (b1 & ~1) : (b1 | 1);
    const int nz = ze - zs;
    const int K = nz + 4;                  // steps: 2 window fills, nz+1 black, nz white
    int ybase = jt * RPT - 2;
    if (ybase < 0) ybase += L;
    int y = ybase + ry;
    if (y >= L) y -= L;
    const size_t G = (size_t)L * L * R4;   // groups per colour

    F2Ctx c;
    c.Wst = Wst;
    c.Bst = Bst;
    c.nb = nb;
    c.bars = bars;
    const uint4 *srcB = src + (first ? G : 0), *srcW = src + (first ? 0 : G);
    c.dstB = dst + (first ? G : 0);
    c.dstW = dst + (first ? 0 : G);
    // keep the two store bases as plain 64-bit values (address = base + 16 q: one LEA pair per store)
    asm volatile("" : "+l"(c.dstB), "+l"(c.dstW));
    c.si0 = ry * R4 + x4;
    c.si_ym = ry > 0 ? c.si0 - R4 : c.si0;
    c.si_yp = ry + 2 < TY ? c.si0 + 2 * R4 : c.si0;
    c.lane_prev = (lane & ~(RL - 1)) | (x4 == 0 ? R4 - 1 : x4 - 1);
    c.lane_next = (lane & ~(RL - 1)) | (x4 == R4 - 1 ? 0 : x4 + 1);
    c.qrow = (uint32_t)(y * R4 + x4);
    c.qplane = (uint32_t)(L * R4);
    c.ok0 = !spare && (ry >= 2) && (ry - 2 < RPT) && (jt * RPT + ry - 2 < L);
    c.ok1 = !spare && (ry + 1 - 2 < RPT) && (ry + 1 < TY - 2) && (jt * RPT + ry + 1 - 2 < L) && (ry >= 2);
    c.nz = nz;

    if (tid == 0) {
        for (int s = 0; s < S; ++s) mbar_init(smem_u32(&bars[s]), 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // producer (thread 0): stage k holds W_old[z0+1+k] and B_old[z0+k], z0 = zs-3 (periodic).
    // Stages are issued in order, so the plane indices and pointers advance incrementally
    // (no division in the loop).  No proxy fence is needed before re-filling a stage: its last
    // generic-proxy accesses were loads that completed before the __syncthreads.
    const int n1 = min(TY, L - ybase);     // rows before the periodic wrap in y
    const uint32_t bytes1 = (uint32_t)n1 * R4 * 16u, bytes2 = (uint32_t)(TY - n1) * R4 * 16u;
    const size_t plane_u4 = (size_t)L * R4;
    int pzw = ((zs - 2) % L + L) % L, pzb = ((zs - 3) % L + L) % L, pk = 0;
    const uint4 *pgw = srcW + (size_t)pzw * plane_u4;
    const uint4 *pgb = srcB + (size_t)pzb * plane_u4;
    // The whole of warp 0 runs the producer: its state is then warp-uniform (uniform registers and
    // datapath, no per-thread copies of the pointers), and one elected lane issues the copies.
    const bool prod_warp = __shfl_sync(0xffffffffu, tid >> 5, 0) == 0;
    auto issue_next = [&]() {
        const int s = pk % S;
        const uint32_t bar = smem_u32(&bars[s]);
        if (elect_one()) {
            mbar_expect_tx(bar, 2u * (uint32_t)PLANE * 16u);
            bulk_g2s(smem_u32(Wst + s * PLANE), pgw + (size_t)ybase * R4, bytes1, bar);
            bulk_g2s(smem_u32(Bst + s * PLANE), pgb + (size_t)ybase * R4, bytes1, bar);
            if (bytes2) {
                bulk_g2s(smem_u32(Wst + s * PLANE + n1 * R4), pgw, bytes2, bar);
                bulk_g2s(smem_u32(Bst + s * PLANE + n1 * R4), pgb, bytes2, bar);
            }
        }
        ++pk;
        pgw += plane_u4;
        pgb += plane_u4;
        if (++pzw == L) { pzw = 0; pgw = srcW; }
        if (++pzb == L) { pzb = 0; pgb = srcB; }
    };
    if (prod_warp)
        for (int k = 0; k < D && k < K; ++k) issue_next();

    F2Win w;
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int r = 0; r < 2; ++r) {
            w.W[i][r] = make_uint4(0, 0, 0, 0);
            w.B[i][r] = make_uint4(0, 0, 0, 0);
        }
    int z = zs - 3;                        // plane of the black update (even)
    if (z < 0) z += L;
    int k = 0;
    // Philox / store group index of this thread's even row in the black plane z (qb) and in the white
    // plane z-1 (qw = the previous step's qb), kept incrementally
    uint32_t qb = (uint32_t)z * c.qplane + c.qrow;
    uint32_t qw = (uint32_t)(z == 0 ? L - 1 : z - 1) * c.qplane + c.qrow;
    // double checkerboard: bits j of a word with ((j >> 2) + (y >> 3) + (z >> 3)) & 1 == coarse (philox.cuh)
    const uint32_t ycoarse = DCB ? (uint32_t)((y >> 3) + coarse) : 0u;
    const uint32_t ffrow = DCB == 2 ? (uint32_t)(y >> 3) * (uint32_t)R4 + (uint32_t)x4 : 0u;
    const uint32_t ffplane = (uint32_t)(L >> 3) * (uint32_t)R4;          // ff words per block plane
    uint4 mB = make_uint4(0xFFFFFFFFu, 0xFFFFFFFFu, 0xFFFFFFFFu, 0xFFFFFFFFu), mW = mB;

#define F2_STEP(U)                                                            \
    {                                                                         \
        if (k >= K) break;                                                    \
        if (DCB) {                                                            \
            mW = mB;                  /* the white plane z-1 was the previous step's black plane */ \
            const uint32_t odd = (ycoarse + (uint32_t)(z >> 3)) & 1u;         \
            if (DCB == 1) {                                                   \
                const uint32_t m = odd ? 0xF0F0F0F0u : 0x0F0F0F0Fu;           \
                mB = make_uint4(m, m, m, m);                                  \
            } else {                                                          \
                uint32_t fw = __ldg(ff + (uint32_t)(z >> 3) * ffplane + ffrow);  \
                fw = (first ? fw : ~fw) & (odd ? 0xAAAAAAAAu : 0x55555555u);  \
                mB = make_uint4(byte_to_nibbles(fw & 0xFFu), byte_to_nibbles((fw >> 8) & 0xFFu),  \
                                byte_to_nibbles((fw >> 16) & 0xFFu), byte_to_nibbles(fw >> 24));   \
            }                                                                 \
        }                                                                     \
        f2_step<R4, PLANE, U, DCB>(w, c, k, qb, qw, lap_parity, keys, mB, mW); \
        __syncthreads();                                                      \
        if (prod_warp && pk < K) issue_next();                                \
        ++k;                                                                  \
        z = (z + 1 == L) ? 0 : z + 1;                                         \
        qw = qb;                                                              \
        qb = z == 0 ? c.qrow : qb + c.qplane;                                 \
    }
    for (uint32_t lap_parity = 0;; lap_parity ^= 1u) {
        F2_STEP(0)
        F2_STEP(1)
        F2_STEP(2)
        F2_STEP(3)
        F2_STEP(4)
        F2_STEP(5)
    }
#undef F2_STEP
}

// ---------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------
inline bool fused2_supported(int L) { return L == 512 || L == 1024 || L == 1536 || L == 2048 || L == 4096; }

template <int R4, int NT>
inline cudaError_t plan_fused2_t(FusedPlan &plan, int L, int sm_count)
{
    constexpr int TY = 2 * NT / f2_row_lanes(R4);
    constexpr int PLANE = TY * R4;
    constexpr size_t smem = (size_t)PLANE * 16 * (2 * kF2Stages + 2) + kF2Stages * 8;
    cudaError_t e = cudaFuncSetAttribute(fused2_sweep_kernel<R4, NT, 0>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(fused2_sweep_kernel<R4, NT, 1>,
                                 cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(fused2_sweep_kernel<R4, NT, 2>,
                                 cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int occ = 0, occ1 = 0, occ2 = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fused2_sweep_kernel<R4, NT, 0>, NT, smem);
    if (e == cudaSuccess)
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ1, fused2_sweep_kernel<R4, NT, 1>, NT, smem);
    if (e == cudaSuccess)
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ2, fused2_sweep_kernel<R4, NT, 2>, NT, smem);
    if (occ1 < occ) occ = occ1;                // one launch shape for all three
    if (occ2 < occ) occ = occ2;
    if (e != cudaSuccess) return e;
    if (occ < 1) occ = 1;
    const int tyo = TY - 4;                        // stored rows per tile (even)
    int nty = (L + tyo - 1) / tyo;
    int RPT = (L + nty - 1) / nty;
    RPT += RPT & 1;                                // even, so that ybase is even
    nty = (L + RPT - 1) / RPT;
    int nzc = (sm_count * occ) / nty;
    if (nzc < 1) nzc = 1;
    if (nzc > L / 8) nzc = L / 8;
    plan.nty = nty;
    plan.RPT = RPT;
    plan.nzc = nzc;
    plan.ready = true;
    return cudaSuccess;
}

template <int R4, int NT>
inline cudaError_t launch_fused2_t(const uint32_t *src, uint32_t *dst, int L, int first, int coarse,
                                   const uint32_t *ff, const SweepConsts &keys, const FusedPlan &plan,
                                   cudaStream_t stream)
{
    constexpr int TY = 2 * NT / f2_row_lanes(R4);
    constexpr int PLANE = TY * R4;
    constexpr size_t smem = (size_t)PLANE * 16 * (2 * kF2Stages + 2) + kF2Stages * 8;
    dim3 grid((unsigned)plan.nty, (unsigned)plan.nzc);
    if (coarse < 0)
        fused2_sweep_kernel<R4, NT, 0><<<grid, NT, smem, stream>>>(
            reinterpret_cast<const uint4 *>(src), reinterpret_cast<uint4 *>(dst), L, plan.RPT, plan.nzc,
            first, 0, nullptr, keys);
    else if (!ff)
        fused2_sweep_kernel<R4, NT, 1><<<grid, NT, smem, stream>>>(
            reinterpret_cast<const uint4 *>(src), reinterpret_cast<uint4 *>(dst), L, plan.RPT, plan.nzc,
            first, coarse, nullptr, keys);
    else
        fused2_sweep_kernel<R4, NT, 2><<<grid, NT, smem, stream>>>(
            reinterpret_cast<const uint4 *>(src), reinterpret_cast<uint4 *>(dst), L, plan.RPT, plan.nzc,
            first, coarse, ff, keys);
    return cudaGetLastError();
}

inline cudaError_t plan_fused2(FusedPlan &plan, int L, int sm_count)
{
    switch (L) {
        case 512:  return plan_fused2_t<2, 128>(plan, L, sm_count);
        case 1024: return plan_fused2_t<4, 256>(plan, L, sm_count);
        case 1536: return plan_fused2_t<6, 256>(plan, L, sm_count);
        case 2048: return plan_fused2_t<8, 256>(plan, L, sm_count);
        case 4096: return plan_fused2_t<16, 256>(plan, L, sm_count);
        default:   return cudaErrorInvalidValue;
    }
}

// coarse < 0: the plain checkerboard sweep; coarse = 0 / 1: the double-checkerboard launch that
// updates that coarse colour only (D14), or with ff (the sweep's block-order bits, D15) only its
// blocks whose first fine colour is `first`.
inline cudaError_t launch_fused2_sweep(const uint32_t *src, uint32_t *dst, int L, uint32_t t,
                                       uint64_t seed, int first, const FusedPlan &plan,
                                       cudaStream_t stream, int coarse = -1, const uint32_t *ff = nullptr)
{
    const SweepConsts keys = make_sweep_consts(seed, t, first);
    switch (L) {
        case 512:  return launch_fused2_t<2, 128>(src, dst, L, first, coarse, ff, keys, plan, stream);
        case 1024: return launch_fused2_t<4, 256>(src, dst, L, first, coarse, ff, keys, plan, stream);
        case 1536: return launch_fused2_t<6, 256>(src, dst, L, first, coarse, ff, keys, plan, stream);
        case 2048: return launch_fused2_t<8, 256>(src, dst, L, first, coarse, ff, keys, plan, stream);
        case 4096: return launch_fused2_t<16, 256>(src, dst, L, first, coarse, ff, keys, plan, stream);
        default:   return cudaErrorInvalidValue;
    }
}

}  // namespace ising
