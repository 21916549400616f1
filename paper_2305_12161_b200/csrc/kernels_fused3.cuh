// EXPERIMENT, FROZEN.  Kept as the evidence that the sweep is bound by the SM, not by HBM (half the DRAM
// traffic per sweep, no gain in time: profiles/r1g_fused3_full.md).  Opt-in only
// (ISING3D_VARIANT_FUSED3), oracle-tested as it stands, but not developed further: later work on fused2
// (instruction trims, double checkerboard, L = 1536, activity hand-over) was not brought over, and
// bench.py no longer offers it.
//
// Two sweeps per launch (temporal blocking of a2+a3+a4), L in {1024, 2048}, cycle 01.
//
// kernels_fused2.cuh moves N/4 bytes per sweep and sits between its memory time and its compute
// time.  Here one CTA carries TWO levels of the same z-march:
//   level 1 (threads 0..NT-1)    sweep t   : planes of the source state from the bulk-async ring,
//                                            results B1[z], W1[z-1] into a shared-memory ring;
//   level 2 (threads NT..2NT-1)  sweep t+1 : reads B1 / W1 from that ring exactly as level 1 reads
//                                            the source planes, stores the result to the destination.
// The state after sweep t never goes to HBM: N/4 bytes per TWO sweeps.  Each level is the
// fused2 step (two rows per thread, 6-step unroll, host-folded Philox constants); the levels
// run warp-specialised and decoupled by the ring, each with its own named barrier for the
// y+-1 exchange.
//
// Geometry.  Tile = TY rows; level 1 loses 2+2 rows to the y halo (as in fused2), level 2 two
// more on each side: TY-8 rows stored.  Level 2 marches z0' = z0 + DZ (DZ = 2, same parity, so
// the compile-time in-row directions agree) and consumes, at its step k', W1 of relative plane
// k'+DZ+1 and B1, W1 of relative plane k'+DZ; level 1 produces B1[k] and W1[k-1] at step k.
//   level 2 step k' needs level 1 steps <= k'+DZ+2 done        (l1_done >= k'+DZ+3)
//   level 1 step k  needs level 2 steps <= k-SM-DZ   done      (l2_done >= k-SM-DZ+1)
// with SM the ring depth in planes.  Thread 0 of each level checks the other level's step
// counter before its level's barrier; the barrier publishes the observation to its level.
//
// Site rule: eq. (6) PAPER.md:105-108 (D2); sweep order PAPER.md:116 (D7); random bits D5.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "kernels_fused2.cuh"

namespace ising {

constexpr int kF3Mid = 8;                   // SM: planes of B1 / W1 kept in shared memory
constexpr int kF3Stages = 3;                // S: bulk-copy ring depth of level 1
constexpr int kF3Dz = 2;                    // DZ

__device__ __forceinline__ void named_bar_sync(const int id, const int count)
{
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(count) : "memory");
}
__device__ __forceinline__ void step_publish(int *p, const int v)
{
    asm volatile("st.release.cta.shared.s32 [%0], %1;" ::"r"(smem_u32(p)), "r"(v) : "memory");
}
__device__ __forceinline__ void step_wait(int *p, const int v)
{
    int cur;
    do {
        asm volatile("ld.acquire.cta.shared.s32 %0, [%1];" : "=r"(cur) : "r"(smem_u32(p)) : "memory");
    } while (cur < v);
}

struct F3Ctx {
    uint4 *inW, *inB;           // [S][PLANE]   source planes (bulk ring), level 1
    uint4 *midW, *midB;         // [SM][PLANE]  W1 / B1 planes
    uint4 *nb;                  // [2][PLANE]   B2 planes for the y+-1 exchange of level 2
    uint64_t *bars;
    uint4 *dstB, *dstW;
    int si0, si_ym, si_yp;
    int lane_prev, lane_next;
    uint32_t qrow, qplane;
    bool ok0, ok1;
    int nz;
};

// Level 1, step k (black at plane z, white at z-1): B1[z] -> midB[mk], W1[z-1] -> midW[mkm1]
// (mk = k mod SM, mkm1 = (k-1) mod SM).  midB doubles as the y+-1 exchange buffer of level 1.
template <int R4, int PLANE, int PH, int O>
__device__ __forceinline__ void f3_level1(F2Win &w, const F3Ctx &c, const int k, const int z,
                                          const int mk, const int mkm1, const SweepConsts &keys)
{
    constexpr int S = kF3Stages;
    constexpr int M = PH % 3, Z = (PH + 1) % 3, P = (PH + 2) % 3;
    const int s = k % S;
    mbar_wait(smem_u32(&c.bars[s]), (uint32_t)((k / S) & 1));
    const uint4 *Wnew = c.inW + s * PLANE;
    const uint4 *Bold = c.inB + s * PLANE;
    const uint4 *Wz = c.inW + ((k + S - 1) % S) * PLANE;
    w.W[P][0] = Wnew[c.si0];
    w.W[P][1] = Wnew[c.si0 + R4];
    const uint4 Bo0 = Bold[c.si0], Bo1 = Bold[c.si0 + R4];
    {
        const uint4 Wym = Wz[c.si_ym], Wyp = Wz[c.si_yp];
        const uint32_t q = (uint32_t)z * c.qplane + c.qrow;
        const uint4 rho0 = philox_folded<0>(q, keys);
        const uint4 rho1 = philox_folded<0>(q + R4, keys);
        const uint4 Wx0 = xneigh<O>(w.W[Z][0], c.lane_prev, c.lane_next);
        const uint4 Wx1 = xneigh<1 - O>(w.W[Z][1], c.lane_prev, c.lane_next);
        w.B[P][0] = rule_group(Bo0, rho0, w.W[Z][0], Wx0, Wym, w.W[Z][1], w.W[M][0], w.W[P][0]);
        w.B[P][1] = rule_group(Bo1, rho1, w.W[Z][1], Wx1, w.W[Z][0], Wyp, w.W[M][1], w.W[P][1]);
        uint4 *mb = c.midB + mk * PLANE + c.si0;
        mb[0] = w.B[P][0];
        mb[R4] = w.B[P][1];
    }
    {
        const uint4 *Bz = c.midB + mkm1 * PLANE;                 // B1[z-1], written last step
        const uint4 Bym = Bz[c.si_ym], Byp = Bz[c.si_yp];
        const int zw = z == 0 ? (int)(c.qplane / R4) - 1 : z - 1;
        const uint32_t q = (uint32_t)zw * c.qplane + c.qrow;
        const uint4 rho0 = philox_folded<1>(q, keys);
        const uint4 rho1 = philox_folded<1>(q + R4, keys);
        const uint4 Bx0 = xneigh<O>(w.B[Z][0], c.lane_prev, c.lane_next);
        const uint4 Bx1 = xneigh<1 - O>(w.B[Z][1], c.lane_prev, c.lane_next);
        uint4 *mw = c.midW + mkm1 * PLANE + c.si0;
        mw[0] = rule_group(w.W[M][0], rho0, w.B[Z][0], Bx0, Bym, w.B[Z][1], w.B[M][0], w.B[P][0]);
        mw[R4] = rule_group(w.W[M][1], rho1, w.B[Z][1], Bx1, w.B[Z][0], Byp, w.B[M][1], w.B[P][1]);
    }
}

// Level 2, step k (black at plane z, white at z-1) on the planes of level 1:
// W1[z+1] = midW[mn], B1[z] = midB[mz], W1[z] (y neighbours) = midW[mz].
template <int R4, int PLANE, int PH, int O>
__device__ __forceinline__ void f3_level2(F2Win &w, const F3Ctx &c, const int k, const int z,
                                          const int mz, const int mn, const SweepConsts &keys)
{
    constexpr int M = PH % 3, Z = (PH + 1) % 3, P = (PH + 2) % 3;
    const uint4 *Wnew = c.midW + mn * PLANE;
    const uint4 *Bold = c.midB + mz * PLANE;
    const uint4 *Wz = c.midW + mz * PLANE;
    w.W[P][0] = Wnew[c.si0];
    w.W[P][1] = Wnew[c.si0 + R4];
    const uint4 Bo0 = Bold[c.si0], Bo1 = Bold[c.si0 + R4];
    {
        const uint4 Wym = Wz[c.si_ym], Wyp = Wz[c.si_yp];
        const uint32_t q = (uint32_t)z * c.qplane + c.qrow;
        const uint4 rho0 = philox_folded<0>(q, keys);
        const uint4 rho1 = philox_folded<0>(q + R4, keys);
        const uint4 Wx0 = xneigh<O>(w.W[Z][0], c.lane_prev, c.lane_next);
        const uint4 Wx1 = xneigh<1 - O>(w.W[Z][1], c.lane_prev, c.lane_next);
        w.B[P][0] = rule_group(Bo0, rho0, w.W[Z][0], Wx0, Wym, w.W[Z][1], w.W[M][0], w.W[P][0]);
        w.B[P][1] = rule_group(Bo1, rho1, w.W[Z][1], Wx1, w.W[Z][0], Wyp, w.W[M][1], w.W[P][1]);
        uint4 *nbw = c.nb + (k & 1) * PLANE + c.si0;
        nbw[0] = w.B[P][0];
        nbw[R4] = w.B[P][1];
        if (k >= 3 && k < 3 + c.nz) {
            uint4 *d = c.dstB + (size_t)q;
            if (c.ok0) d[0] = w.B[P][0];
            if (c.ok1) d[R4] = w.B[P][1];
        }
    }
    {
        const uint4 *Bz = c.nb + ((k - 1) & 1) * PLANE;
        const uint4 Bym = Bz[c.si_ym], Byp = Bz[c.si_yp];
        const int zw = z == 0 ? (int)(c.qplane / R4) - 1 : z - 1;
        const uint32_t q = (uint32_t)zw * c.qplane + c.qrow;
        const uint4 rho0 = philox_folded<1>(q, keys);
        const uint4 rho1 = philox_folded<1>(q + R4, keys);
        const uint4 Bx0 = xneigh<O>(w.B[Z][0], c.lane_prev, c.lane_next);
        const uint4 Bx1 = xneigh<1 - O>(w.B[Z][1], c.lane_prev, c.lane_next);
        const uint4 nW0 =
            rule_group(w.W[M][0], rho0, w.B[Z][0], Bx0, Bym, w.B[Z][1], w.B[M][0], w.B[P][0]);
        const uint4 nW1 =
            rule_group(w.W[M][1], rho1, w.B[Z][1], Bx1, w.B[Z][0], Byp, w.B[M][1], w.B[P][1]);
        if (k >= 4) {
            uint4 *d = c.dstW + (size_t)q;
            if (c.ok0) d[0] = nW0;
            if (c.ok1) d[R4] = nW1;
        }
    }
}

// Grid: blockIdx.x = y tile (RPT = TY-8 stored rows, even), blockIdx.y = z chunk [zs, ze) with
// odd borders (cycle 01: colour 0 first in both sweeps).  Level 1 covers [zs-2, ze+2).
template <int R4, int NT>
__global__ void __launch_bounds__(2 * NT, 1)
fused3_sweep2_kernel(const uint4 *__restrict__ src, uint4 *__restrict__ dst, const int L,
                     const int RPT, const int nzc, const __grid_constant__ SweepConsts keys1,
                     const __grid_constant__ SweepConsts keys2)
{
    constexpr int TY = 2 * NT / R4;
    constexpr int PLANE = TY * R4;
    constexpr int S = kF3Stages, D = S - 1, SM = kF3Mid, DZ = kF3Dz;
    static_assert(R4 <= 32 && (32 % R4) == 0, "a row must fit a warp");
    static_assert(SM >= 5, "the two levels need slack");

    extern __shared__ __align__(128) uint4 smem[];
    F3Ctx c;
    c.inW = smem;
    c.inB = c.inW + S * PLANE;
    c.midW = c.inB + S * PLANE;
    c.midB = c.midW + SM * PLANE;
    c.nb = c.midB + SM * PLANE;
    c.bars = reinterpret_cast<uint64_t *>(c.nb + 2 * PLANE);
    int *l1_done = reinterpret_cast<int *>(c.bars + S);
    int *l2_done = l1_done + 1;

    const int level = threadIdx.x >= NT ? 1 : 0;
    const int tid = threadIdx.x - level * NT, lane = tid & 31;
    const int x4 = tid & (R4 - 1), p = tid / R4;
    const int ry = 2 * p;
    const int jt = blockIdx.x, zc = blockIdx.y;
    const int b0 = (int)((long long)L * zc / nzc), b1 = zc + 1 == nzc ? L : (int)((long long)L * (zc + 1) / nzc);
    const int zs = b0 | 1, ze = b1 | 1;
    const int nz = ze - zs;
    const int K2 = nz + 4;                 // level 2 steps (as fused2)
    const int K1 = K2 + DZ + 2;            // level 1 runs DZ + 2 steps ahead at least
    int ybase = jt * RPT - 4;
    if (ybase < 0) ybase += L;
    int y = ybase + ry;
    if (y >= L) y -= L;
    const size_t G = (size_t)L * L * R4;

    c.dstB = dst;
    c.dstW = dst + G;
    c.si0 = ry * R4 + x4;
    c.si_ym = ry > 0 ? c.si0 - R4 : c.si0;
    c.si_yp = ry + 2 < TY ? c.si0 + 2 * R4 : c.si0;
    c.lane_prev = (lane & ~(R4 - 1)) | ((lane - 1) & (R4 - 1));
    c.lane_next = (lane & ~(R4 - 1)) | ((lane + 1) & (R4 - 1));
    c.qrow = (uint32_t)(y * R4 + x4);
    c.qplane = (uint32_t)(L * R4);
    c.ok0 = (ry >= 4) && (ry - 4 < RPT) && (ry < TY - 4) && (jt * RPT + ry - 4 < L);
    c.ok1 = (ry >= 4) && (ry + 1 - 4 < RPT) && (ry + 1 < TY - 4) && (jt * RPT + ry + 1 - 4 < L);
    c.nz = nz;

    if (threadIdx.x == 0) {
        for (int s = 0; s < S; ++s) mbar_init(smem_u32(&c.bars[s]), 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        *l1_done = 0;
        *l2_done = 0;
    }
    __syncthreads();

    F2Win w;
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int r = 0; r < 2; ++r) {
            w.W[i][r] = make_uint4(0, 0, 0, 0);
            w.B[i][r] = make_uint4(0, 0, 0, 0);
        }

    if (level == 0) {
        // ---------------- level 1: sweep t, source planes -> midB / midW ----------------
        const int n1 = min(TY, L - ybase);
        const uint32_t bytes1 = (uint32_t)n1 * R4 * 16u, bytes2 = (uint32_t)(TY - n1) * R4 * 16u;
        const size_t plane_u4 = (size_t)L * R4;
        const int z0 = ((zs - DZ - 3) % L + L) % L;            // even
        int pzw = (z0 + 1) % L, pzb = z0, pk = 0;
        const uint4 *srcB = src, *srcW = src + G;
        const uint4 *pgw = srcW + (size_t)pzw * plane_u4;
        const uint4 *pgb = srcB + (size_t)pzb * plane_u4;
        auto issue_next = [&]() {
            const int s = pk % S;
            const uint32_t bar = smem_u32(&c.bars[s]);
            mbar_expect_tx(bar, 2u * (uint32_t)PLANE * 16u);
            bulk_g2s(smem_u32(c.inW + s * PLANE), pgw + (size_t)ybase * R4, bytes1, bar);
            bulk_g2s(smem_u32(c.inB + s * PLANE), pgb + (size_t)ybase * R4, bytes1, bar);
            if (bytes2) {
                bulk_g2s(smem_u32(c.inW + s * PLANE + n1 * R4), pgw, bytes2, bar);
                bulk_g2s(smem_u32(c.inB + s * PLANE + n1 * R4), pgb, bytes2, bar);
            }
            ++pk;
            pgw += plane_u4;
            pgb += plane_u4;
            if (++pzw == L) { pzw = 0; pgw = srcW; }
            if (++pzb == L) { pzb = 0; pgb = srcB; }
        };
        if (tid == 0)
            for (int k = 0; k < D && k < K1; ++k) issue_next();

        int z = z0, k = 0, mk = 0, mkm1 = SM - 1;
#define F3_STEP1(PH, O)                                                               \
    {                                                                                 \
        if (k >= K1) break;                                                           \
        f3_level1<R4, PLANE, PH, O>(w, c, k, z, mk, mkm1, keys1);                     \
        /* step k+1 overwrites B1[k+1-SM], W1[k-SM]: level 2 is past them */          \
        if (tid == 0 && k + 1 < K1) step_wait(l2_done, k + 1 - SM - DZ + 1);          \
        named_bar_sync(1, NT);                                                        \
        if (tid == 0) {                                                               \
            step_publish(l1_done, k + 1);                                             \
            if (pk < K1) issue_next();                                                \
        }                                                                             \
        ++k;                                                                          \
        z = (z + 1 == L) ? 0 : z + 1;                                                 \
        mkm1 = mk;                                                                    \
        mk = (mk + 1 == SM) ? 0 : mk + 1;                                             \
    }
        for (;;) {
            F3_STEP1(0, 0)
            F3_STEP1(1, 1)
            F3_STEP1(2, 0)
            F3_STEP1(0, 1)
            F3_STEP1(1, 0)
            F3_STEP1(2, 1)
        }
#undef F3_STEP1
    } else {
        // ---------------- level 2: sweep t+1, midB / midW -> destination ----------------
        int z = ((zs - 3) % L + L) % L;                        // z0 + DZ, even
        int k = 0, mz = DZ % SM, mn = (DZ + 1) % SM;
        if (tid == 0) step_wait(l1_done, DZ + 3);
        named_bar_sync(2, NT);
#define F3_STEP2(PH, O)                                                               \
    {                                                                                 \
        if (k >= K2) break;                                                           \
        f3_level2<R4, PLANE, PH, O>(w, c, k, z, mz, mn, keys2);                       \
        if (tid == 0 && k + 1 < K2) step_wait(l1_done, k + 1 + DZ + 3);               \
        named_bar_sync(2, NT);                                                        \
        if (tid == 0) step_publish(l2_done, k + 1);                                   \
        ++k;                                                                          \
        z = (z + 1 == L) ? 0 : z + 1;                                                 \
        mz = mn;                                                                      \
        mn = (mn + 1 == SM) ? 0 : mn + 1;                                             \
    }
        for (;;) {
            F3_STEP2(0, 0)
            F3_STEP2(1, 1)
            F3_STEP2(2, 0)
            F3_STEP2(0, 1)
            F3_STEP2(1, 0)
            F3_STEP2(2, 1)
        }
#undef F3_STEP2
    }
}

// ---------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------
inline bool fused3_supported(int L) { return L == 1024 || L == 2048; }

template <int R4, int NT>
inline cudaError_t plan_fused3_t(FusedPlan &plan, int L, int sm_count)
{
    constexpr int TY = 2 * NT / R4;
    constexpr int PLANE = TY * R4;
    constexpr size_t smem =
        (size_t)PLANE * 16 * (2 * kF3Stages + 2 * kF3Mid + 2) + kF3Stages * 8 + 16;
    cudaError_t e = cudaFuncSetAttribute(fused3_sweep2_kernel<R4, NT>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const int tyo = TY - 8;                        // stored rows per tile (even)
    int nty = (L + tyo - 1) / tyo;
    int RPT = (L + nty - 1) / nty;
    RPT += RPT & 1;
    nty = (L + RPT - 1) / RPT;
    int nzc = sm_count / nty;                      // one CTA per SM
    if (nzc < 1) nzc = 1;
    if (nzc > L / 16) nzc = L / 16;
    plan.nty = nty;
    plan.RPT = RPT;
    plan.nzc = nzc;
    plan.ready = true;
    return cudaSuccess;
}

template <int R4, int NT>
inline cudaError_t launch_fused3_t(const uint32_t *src, uint32_t *dst, int L, const SweepConsts &k1,
                                   const SweepConsts &k2, const FusedPlan &plan, cudaStream_t stream)
{
    constexpr int TY = 2 * NT / R4;
    constexpr int PLANE = TY * R4;
    constexpr size_t smem =
        (size_t)PLANE * 16 * (2 * kF3Stages + 2 * kF3Mid + 2) + kF3Stages * 8 + 16;
    dim3 grid((unsigned)plan.nty, (unsigned)plan.nzc);
    fused3_sweep2_kernel<R4, NT><<<grid, 2 * NT, smem, stream>>>(
        reinterpret_cast<const uint4 *>(src), reinterpret_cast<uint4 *>(dst), L, plan.RPT, plan.nzc,
        k1, k2);
    return cudaGetLastError();
}

inline cudaError_t plan_fused3(FusedPlan &plan, int L, int sm_count)
{
    switch (L) {
        case 1024: return plan_fused3_t<4, 256>(plan, L, sm_count);
        case 2048: return plan_fused3_t<8, 256>(plan, L, sm_count);
        default:   return cudaErrorInvalidValue;
    }
}

// sweeps t and t+1 (cycle 01) of the state `src` into `dst`
inline cudaError_t launch_fused3_sweep2(const uint32_t *src, uint32_t *dst, int L, uint32_t t,
                                        uint64_t seed, const FusedPlan &plan, cudaStream_t stream)
{
    const SweepConsts k1 = make_sweep_consts(seed, t, 0), k2 = make_sweep_consts(seed, t + 1, 0);
    switch (L) {
        case 1024: return launch_fused3_t<4, 256>(src, dst, L, k1, k2, plan, stream);
        case 2048: return launch_fused3_t<8, 256>(src, dst, L, k1, k2, plan, stream);
        default:   return cudaErrorInvalidValue;
    }
}

}  // namespace ising
