// Fused full-sweep kernel (a2+a3+a4 in one launch): black half-sweep, then white half-sweep
// on the updated black spins, marching along z with a register window, for one lattice
// with L in {256, 512, 1024, 2048, 4096} (row = R4 = L/256 128-bit groups, a power of two).
//
// Why fused: the two half-sweeps of one sweep read and write each colour
// once (3 N/8 bytes per sweep if done separately); doing white at plane z-1 right after
// black at plane z is available on chip moves N/4 bytes per sweep instead (+ halo).
//
// Data flow per CTA (tile = TY consecutive rows y, all x, a chunk [zs,ze) of planes):
//   - src/dst are ping-pong copies of the packed state (D3), so no CTA ever reads a word
//     another CTA writes in the same launch.
//   - One elected thread streams plane tiles {W_old[z+1], B_old[z]} (each one contiguous
//     TY*R4*16 bytes in HBM) into a ring of shared-memory stages with 1-D bulk async
//     copies (cp.async.bulk, complete_tx on an mbarrier) D stages ahead of the consumers.
//   - Every thread owns one 128-spin group position (row ry, group x4) and keeps
//     W_old[z-1..z+1] and B_new[z-2..z] of that position in registers; the y+-1 neighbours
//     come from the shared-memory planes, the x+-1 neighbour bit across groups from a warp
//     shuffle (rows are assigned to warps by parity so the shift direction is warp-uniform).
//   - step z: B_new[z] = rule(B_old[z]; W_old at (z-1, z+1, y-1, y+1, same, x-shift)),
//             W_new[z-1] = rule(W_old[z-1]; B_new at (z-2, z, y-1, y+1, same, x-shift)).
//   - Halo: rows 0,1 and TY-2,TY-1 of the tile and 2 planes before / 1 after the chunk are
//     recomputed by the neighbouring CTAs (B_new there is needed as input for W_new).
// Random bits: Philox4x32-10(key = seed, counter = (group, t, colour, 0)) (D5), one call
// per 128 sites per colour, round keys in the constant bank.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "philox.cuh"

namespace ising {

constexpr int kFusedStages = 4;   // shared-memory ring depth S; prefetch distance D = S-1

__device__ __forceinline__ uint32_t smem_u32(const void *p)
{
    return (uint32_t)__cvta_generic_to_shared(p);
}

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}

__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes)
                 : "memory");
}

__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    uint32_t done;
    do {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n"
            : "=r"(done)
            : "r"(bar), "r"(parity)
            : "memory");
    } while (!done);
}

// 1-D bulk async copy global -> shared (SASS: UBLKCP), bytes % 16 == 0, 16-byte aligned.
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
        ::"r"(dst), "l"(src), "r"(bytes), "r"(bar)
        : "memory");
}

// x-neighbour word of a 128-bit group (D4): o = 0 -> neighbour k-1 (bit j <- bit j-1),
// o = 1 -> neighbour k+1.  `edge` is word 3 of the previous group (o = 0) or word 0 of the
// next group (o = 1) of the same row, periodic.
__device__ __forceinline__ uint4 xshift(const uint4 w, const int o, const uint32_t edge)
{
    uint4 r;
    if (o == 0) {
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

__device__ __forceinline__ uint4 rule_group(const uint4 s, const uint4 rho, const uint4 a,
                                            const uint4 b, const uint4 c, const uint4 d,
                                            const uint4 e, const uint4 f)
{
    uint4 r;
    r.x = rule_word(s.x, rho.x, a.x, b.x, c.x, d.x, e.x, f.x);
    r.y = rule_word(s.y, rho.y, a.y, b.y, c.y, d.y, e.y, f.y);
    r.z = rule_word(s.z, rho.z, a.z, b.z, c.z, d.z, e.z, f.z);
    r.w = rule_word(s.w, rho.w, a.w, b.w, c.w, d.w, e.w, f.w);
    return r;
}

template <int NT>
struct FusedOcc {
    static constexpr int value = NT <= 256 ? 3 : (NT <= 512 ? 2 : 1);
};

template <int R4, int NT>
__global__ void __launch_bounds__(NT, FusedOcc<NT>::value)
fused_sweep_kernel(const uint4 *__restrict__ src, uint4 *__restrict__ dst, const int L,
                   const uint32_t t, const int RPT, const int nzc,
                   const __grid_constant__ PhiloxKeys keys)
{
    constexpr int TY = NT / R4;        // rows in the tile (incl. 2+2 halo rows)
    constexpr int RW = 32 / R4;        // rows per warp
    constexpr int PLANE = TY * R4;     // uint4 per plane tile
    constexpr int S = kFusedStages, D = S - 1;
    static_assert((NT / 32) % 2 == 0, "need an even number of warps (row parity split)");

    extern __shared__ __align__(128) uint4 smem[];
    uint4 *Wst = smem;                     // [S][PLANE]  W_old planes
    uint4 *Bst = smem + S * PLANE;         // [S][PLANE]  B_old planes
    uint4 *nb = smem + 2 * S * PLANE;      // [2][PLANE]  B_new planes (y+-1 exchange)
    uint64_t *bars = reinterpret_cast<uint64_t *>(nb + 2 * PLANE);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int x4 = lane & (R4 - 1), rl = lane / R4;
    const int ry = 2 * ((warp >> 1) * RW + rl) + (warp & 1);   // tile row, parity = warp & 1
    const int jt = blockIdx.x, zc = blockIdx.y;
    const int zs = (int)((long long)L * zc / nzc);
    const int ze = (int)((long long)L * (zc + 1) / nzc);
    const int nz = ze - zs;
    const int K = nz + 4;                  // steps: 2 warm-up loads, nz+1 black, nz white
    int ybase = jt * RPT - 2;
    if (ybase < 0) ybase += L;
    int y = ybase + ry;
    if (y >= L) y -= L;
    const bool store_row = (ry >= 2) && (ry - 2 < RPT) && (jt * RPT + ry - 2 < L);
    const size_t G = (size_t)L * L * R4;   // groups per colour
    const int si = ry * R4 + x4;           // position inside a plane tile
    const int si_ym = ry > 0 ? si - R4 : si;
    const int si_yp = ry < TY - 1 ? si + R4 : si;
    const int lane_prev = (lane & ~(R4 - 1)) | ((lane - 1) & (R4 - 1));
    const int lane_next = (lane & ~(R4 - 1)) | ((lane + 1) & (R4 - 1));
    const uint32_t qrow = (uint32_t)(y * R4 + x4);   // group index of (y, x4) inside a plane
    const uint32_t qplane = (uint32_t)(L * R4);      // groups per plane

    if (tid == 0) {
        for (int s = 0; s < S; ++s) mbar_init(smem_u32(&bars[s]), 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // producer: stage k holds W_old[zs-2+k] and (k >= 2) B_old[zs-3+k]
    const int n1 = min(TY, L - ybase);     // rows before the periodic wrap in y
    auto issue = [&](int k) {
        const int s = k % S;
        int zw = zs - 2 + k;
        zw = (zw % L + L) % L;
        int zb = zs - 3 + k;
        zb = (zb % L + L) % L;
        const uint32_t bar = smem_u32(&bars[s]);
        const uint32_t bytes = (uint32_t)PLANE * 16u;
        mbar_expect_tx(bar, k >= 2 ? 2 * bytes : bytes);
        const uint4 *gw = src + G + ((size_t)zw * L) * R4;
        bulk_g2s(smem_u32(Wst + s * PLANE), gw + (size_t)ybase * R4, (uint32_t)n1 * R4 * 16u, bar);
        if (n1 < TY)
            bulk_g2s(smem_u32(Wst + s * PLANE + n1 * R4), gw, (uint32_t)(TY - n1) * R4 * 16u, bar);
        if (k >= 2) {
            const uint4 *gb = src + ((size_t)zb * L) * R4;
            bulk_g2s(smem_u32(Bst + s * PLANE), gb + (size_t)ybase * R4, (uint32_t)n1 * R4 * 16u, bar);
            if (n1 < TY)
                bulk_g2s(smem_u32(Bst + s * PLANE + n1 * R4), gb, (uint32_t)(TY - n1) * R4 * 16u, bar);
        }
    };
    if (tid == 0)
        for (int k = 0; k < D && k < K; ++k) issue(k);

    uint4 Wm = make_uint4(0, 0, 0, 0), W0 = Wm, Wp = Wm;       // W_old[z-1], [z], [z+1]
    uint4 nBm2 = Wm, nBm1 = Wm, nB0 = Wm;                      // B_new[z-2], [z-1], [z]
    int z = zs - 3;                                            // plane of the black update
    if (z < 0) z += L;
    // o = (y + z) & 1 for black at plane z and for white at plane z-1 (D4); warp-uniform
    int o = (y + z) & 1;

    for (int k = 0; k < K; ++k) {
        const int s = k % S;
        mbar_wait(smem_u32(&bars[s]), (uint32_t)((k / S) & 1));
        Wm = W0;
        W0 = Wp;
        Wp = Wst[s * PLANE + si];
        if (k >= 2) {
            // ---- black update at plane z (colour 0) ----
            const uint4 Bo = Bst[s * PLANE + si];
            const uint4 *Wz = Wst + ((k - 1) % S) * PLANE;     // plane z of W_old
            const uint4 Wym = Wz[si_ym], Wyp = Wz[si_yp];
            const uint32_t edge_w =
                __shfl_sync(0xffffffffu, o ? W0.x : W0.w, o ? lane_next : lane_prev);
            const uint4 Wx = xshift(W0, o, edge_w);
            const uint4 rho_b =
                philox4x32_10((uint32_t)z * qplane + qrow, t, 0u, 0u, keys);
            nBm2 = nBm1;
            nBm1 = nB0;
            nB0 = rule_group(Bo, rho_b, W0, Wx, Wym, Wyp, Wm, Wp);
            nb[(k & 1) * PLANE + si] = nB0;
            if (store_row && k >= 3 && k < 3 + nz) dst[((size_t)z * L + y) * R4 + x4] = nB0;
        }
        if (k >= 4) {
            // ---- white update at plane z-1 (colour 1) on the updated black spins ----
            const int zw1 = z == 0 ? L - 1 : z - 1;
            const uint4 *Bz = nb + ((k - 1) & 1) * PLANE;      // B_new[z-1], written last step
            const uint4 Bym = Bz[si_ym], Byp = Bz[si_yp];
            const uint32_t edge_b =
                __shfl_sync(0xffffffffu, o ? nBm1.x : nBm1.w, o ? lane_next : lane_prev);
            const uint4 Bx = xshift(nBm1, o, edge_b);
            const uint4 rho_w =
                philox4x32_10((uint32_t)zw1 * qplane + qrow, t, 1u, 0u, keys);
            const uint4 nW = rule_group(Wm, rho_w, nBm1, Bx, Bym, Byp, nBm2, nB0);
            if (store_row) dst[G + ((size_t)zw1 * L + y) * R4 + x4] = nW;
        }
        __syncthreads();
        if (tid == 0 && k + D < K) {
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            issue(k + D);
        }
        z = (z + 1 == L) ? 0 : z + 1;
        o ^= 1;
    }
}

// ---------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------
inline bool fused_supported(int L)
{
    return L == 256 || L == 512 || L == 1024 || L == 2048 || L == 4096;
}

// Launch shape of a fused sweep kernel for one (L, device): computed once per handle at its first
// sweep and kept in the handle (no process-wide state: distinct handles are independent).
struct FusedPlan {
    int nty = 0, RPT = 0, nzc = 0;
    bool ready = false;
};

template <int R4, int NT>
inline cudaError_t plan_fused_t(FusedPlan &plan, int L, int sm_count)
{
    constexpr int TY = NT / R4;
    constexpr int PLANE = TY * R4;
    constexpr size_t smem = (size_t)PLANE * 16 * (2 * kFusedStages + 2) + kFusedStages * 8;
    // per device and idempotent; the CUDA runtime serialises concurrent callers
    cudaError_t e = cudaFuncSetAttribute(fused_sweep_kernel<R4, NT>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int occ = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fused_sweep_kernel<R4, NT>, NT, smem);
    if (e != cudaSuccess) return e;
    if (occ < 1) occ = 1;
    const int tyo = TY - 4;
    plan.nty = (L + tyo - 1) / tyo;
    plan.RPT = (L + plan.nty - 1) / plan.nty;
    int nzc = (sm_count * occ) / plan.nty;
    if (nzc < 1) nzc = 1;
    if (nzc > L / 8) nzc = L / 8;
    plan.nzc = nzc;
    plan.ready = true;
    return cudaSuccess;
}

template <int R4, int NT>
inline cudaError_t launch_fused_t(const uint32_t *src, uint32_t *dst, int L, uint32_t t,
                                  const PhiloxKeys &keys, const FusedPlan &plan, cudaStream_t stream)
{
    constexpr int TY = NT / R4;
    constexpr int PLANE = TY * R4;
    constexpr size_t smem = (size_t)PLANE * 16 * (2 * kFusedStages + 2) + kFusedStages * 8;
    dim3 grid((unsigned)plan.nty, (unsigned)plan.nzc);
    fused_sweep_kernel<R4, NT><<<grid, NT, smem, stream>>>(
        reinterpret_cast<const uint4 *>(src), reinterpret_cast<uint4 *>(dst), L, t, plan.RPT,
        plan.nzc, keys);
    return cudaGetLastError();
}

inline cudaError_t plan_fused(FusedPlan &plan, int L, int sm_count)
{
    switch (L) {
        case 256:  return plan_fused_t<1, 256>(plan, L, sm_count);
        case 512:  return plan_fused_t<2, 256>(plan, L, sm_count);
        case 1024: return plan_fused_t<4, 256>(plan, L, sm_count);
        case 2048: return plan_fused_t<8, 256>(plan, L, sm_count);
        case 4096: return plan_fused_t<16, 512>(plan, L, sm_count);
        default:   return cudaErrorInvalidValue;
    }
}

inline cudaError_t launch_fused_sweep(const uint32_t *src, uint32_t *dst, int L, uint32_t t,
                                      const PhiloxKeys &keys, const FusedPlan &plan, cudaStream_t stream)
{
    switch (L) {
        case 256:  return launch_fused_t<1, 256>(src, dst, L, t, keys, plan, stream);
        case 512:  return launch_fused_t<2, 256>(src, dst, L, t, keys, plan, stream);
        case 1024: return launch_fused_t<4, 256>(src, dst, L, t, keys, plan, stream);
        case 2048: return launch_fused_t<8, 256>(src, dst, L, t, keys, plan, stream);
        case 4096: return launch_fused_t<16, 512>(src, dst, L, t, keys, plan, stream);
        default:   return cudaErrorInvalidValue;
    }
}

}  // namespace ising
