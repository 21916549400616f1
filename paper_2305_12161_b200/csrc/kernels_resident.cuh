// Shared-memory-resident multi-sweep kernel for small lattices (L = 64, 128, 256): a5 for the
// workloads whose lattice fits on chip (config 1: L = 64, 32 KiB; config 3: 64 x L = 128,
// 256 KiB each; BASELINE.json).
//
// One thread-block CLUSTER per replica.  The CS CTAs of a cluster split the lattice into z slabs
// of PZ = L/CS planes; a CTA keeps both colours of its slab in shared memory for the whole
// launch, plus one halo plane below and above per colour.  A launch runs n_sweeps sweeps:
//     for t:  for colour c in (0, 1):                       (D7)
//         update the own planes of colour c in place (reads colour 1-c only, so no hazard; D2),
//         the first / last own plane is also stored into the halo slot of the CTA below / above
//         through distributed shared memory (st to the mapped address of the peer CTA),
//         cluster barrier (release/acquire): the peers' halo stores are visible.
// The state is read from HBM once and written back once per launch; between sweeps nothing
// leaves the SMs.  Launch overhead (2 launches per sweep in the generic path) disappears.
//
// Thread work: one 128-spin group (D5) of the colour being updated = 4 consecutive words of a
// plane.  WPR = L/64 words per row: a group is 4 rows (WPR = 1), 2 rows (2) or 1 row (4).
// Neighbour words (D4): the same group position in the other colour at planes z-1, z, z+1
// (3 LDS.128) and the previous / next group of plane z (2 LDS.128) give y-1 / y+1 and, inside
// the row, the word that supplies the edge bit of the one-bit x shift.
// Random bits: Philox4x32-10, counter (q, t, c, 0), key = the replica's seed (D5); the ten round
// keys live in registers.
#pragma once
#include <cstdint>
#include <type_traits>
#include <cooperative_groups.h>
#include <cuda_runtime.h>

#include "philox.cuh"

namespace ising {

namespace cg = cooperative_groups;

constexpr int kResThreads = 512;

template <int WPR>
__device__ __forceinline__ uint4 res_update_group(const uint4 own, const uint4 prv, const uint4 sam,
                                                  const uint4 nxt, const uint4 zm, const uint4 zp,
                                                  const uint4 rho, const int par, const int y0,
                                                  const int z, const int coarse)
{
    // cmb[4 + i] = word i of the same group position, other colour, plane z; cmb[0..3] the
    // previous group of the plane, cmb[8..11] the next one (periodic in y)
    const uint32_t cmb[12] = {prv.x, prv.y, prv.z, prv.w, sam.x, sam.y, sam.z, sam.w,
                              nxt.x, nxt.y, nxt.z, nxt.w};
    const uint32_t s[4] = {own.x, own.y, own.z, own.w};
    const uint32_t r4[4] = {rho.x, rho.y, rho.z, rho.w};
    const uint32_t m[4] = {zm.x, zm.y, zm.z, zm.w};
    const uint32_t p[4] = {zp.x, zp.y, zp.z, zp.w};
    uint32_t out[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const uint32_t n_same = cmb[4 + i];
        const uint32_t n_yp = cmb[4 + i + WPR], n_ym = cmb[4 + i - WPR];
        // row-local word index and the words before / after it in the (periodic) row
        const int wi = i % WPR, row0 = 4 + i - wi;
        const uint32_t w_prev = cmb[row0 + (wi + WPR - 1) % WPR];
        const uint32_t w_next = cmb[row0 + (wi + 1) % WPR];
        // o = (y + z + c) & 1 (D4): par = (y0 + z + c) & 1 for the group's first row y0
        const int o = (par + i / WPR) & 1;
        const uint32_t n_x = o ? __funnelshift_r(n_same, w_next, 1)     // neighbour k+1
                               : __funnelshift_l(w_prev, n_same, 1);    // neighbour k-1
        const uint32_t upd = rule_word(s[i], r4[i], n_same, n_x, n_yp, n_ym, p[i], m[i]);
        const uint32_t msk = dcb_mask(y0 + i / WPR, z, coarse);   // double checkerboard phases (D14)
        out[i] = (upd & msk) | (s[i] & ~msk);
    }
    return make_uint4(out[0], out[1], out[2], out[3]);
}

// Grid: (CS, n_rep), cluster (CS, 1, 1).  Dynamic shared memory: 2 * (PZ + 2) planes.
template <int WPR>
__global__ void __launch_bounds__(kResThreads, 1)
resident_sweep_kernel(uint32_t *__restrict__ state, const uint64_t *__restrict__ seeds,
                      const uint32_t t0, const uint32_t n_sweeps, const int cycle)
{
    constexpr int L = 64 * WPR;
    constexpr int GPP = L * WPR / 4;              // 128-bit groups per plane
    constexpr int PPI = kResThreads / GPP > 0 ? kResThreads / GPP : 1;   // planes per iteration
    static_assert(GPP <= kResThreads, "a plane must fit one pass of the block");
    extern __shared__ __align__(16) uint4 res_smem[];

    cg::cluster_group cluster = cg::this_cluster();
    const int CS = (int)cluster.num_blocks();
    const int rank = (int)cluster.block_rank();
    const int PZ = L / CS;
    const int z0 = rank * PZ;
    const int rep = blockIdx.y;
    const int tid = threadIdx.x;
    const size_t GPC = (size_t)L * GPP;           // groups per colour
    uint4 *gstate = reinterpret_cast<uint4 *>(state) + (size_t)rep * 2 * GPC;

    // slot s of colour c = plane z0 - 1 + s  (s = 0 lower halo, 1..PZ own, PZ + 1 upper halo)

    // ---- load: own planes and halos of both colours from HBM ----
    for (int idx = tid; idx < 2 * (PZ + 2) * GPP; idx += kResThreads) {
        const int c = idx / ((PZ + 2) * GPP);
        const int rem = idx - c * (PZ + 2) * GPP;
        const int s = rem / GPP, g = rem - s * GPP;
        int z = z0 - 1 + s;
        z = z < 0 ? z + L : (z >= L ? z - L : z);
        res_smem[idx] = gstate[(size_t)c * GPC + (size_t)z * GPP + g];
    }

    // round keys of this replica (D5)
    const uint64_t seed = seeds[rep];
    PhiloxKeys keys;
    {
        uint32_t a = (uint32_t)seed, b = (uint32_t)(seed >> 32);
#pragma unroll
        for (int r = 0; r < 10; ++r) {
            keys.k0[r] = a;
            keys.k1[r] = b;
            a += kPhiloxW0;
            b += kPhiloxW1;
        }
    }

    // thread -> (plane offset inside an iteration, group inside the plane)
    const int pl = tid / GPP, g = tid - pl * GPP;
    const bool active = pl < PPI;
    const int g_prev = g == 0 ? GPP - 1 : g - 1, g_next = g == GPP - 1 ? 0 : g + 1;
    const int y0 = 4 * g / WPR;                   // first row of the group

    // halo slots of the neighbouring CTAs (distributed shared memory); colour c of a CTA starts
    // at res_smem + c * CSTRIDE
    const size_t CSTRIDE = (size_t)(PZ + 2) * GPP;
    const int rank_dn = rank == 0 ? CS - 1 : rank - 1, rank_up = rank == CS - 1 ? 0 : rank + 1;
    uint4 *peer_dn = cluster.map_shared_rank(res_smem, rank_dn);   // its slot PZ+1 <- my plane 0
    uint4 *peer_up = cluster.map_shared_rank(res_smem, rank_up);   // its slot 0    <- my plane PZ-1
    cluster.sync();                               // everybody loaded; peers' smem exists

    // one half-sweep of compile-time colour C (the compiler then folds the colour into the
    // smem offsets and the Philox counter)
    auto half_sweep = [&](auto colour, const uint32_t t, const int coarse) {
        constexpr int C = decltype(colour)::value;
        uint4 *own = res_smem + (size_t)C * CSTRIDE;
        const uint4 *oth = res_smem + (size_t)(1 - C) * CSTRIDE;
        if (active) {
            for (int zl = pl; zl < PZ; zl += PPI) {
                const int z = z0 + zl;
                const uint4 *pz = oth + (size_t)(zl + 1) * GPP;
                const uint4 sam = pz[g], prv = pz[g_prev], nxt = pz[g_next];
                const uint4 zm = pz[g - GPP], zp = pz[g + GPP];
                const uint4 o4 = own[(size_t)(zl + 1) * GPP + g];
                const uint32_t q = (uint32_t)z * GPP + g;
                const uint4 rho = philox4x32_10(q, t, (uint32_t)C, kTagTie, keys);
                const uint4 nw = res_update_group<WPR>(o4, prv, sam, nxt, zm, zp, rho, (y0 + z + C) & 1, y0, z, coarse);
                own[(size_t)(zl + 1) * GPP + g] = nw;
                if (zl == 0) peer_dn[(size_t)C * CSTRIDE + (size_t)(PZ + 1) * GPP + g] = nw;
                if (zl == PZ - 1) peer_up[(size_t)C * CSTRIDE + g] = nw;
            }
        }
        cluster.sync();
    };
    using Colour0 = std::integral_constant<int, 0>;
    using Colour1 = std::integral_constant<int, 1>;

    for (uint32_t it = 0; it < n_sweeps; ++it) {
        const uint32_t t = t0 + it;
        // 01 cycle: colour 0 first (D7); mixed cycle: the first colour is drawn per sweep (D10)
        if (cycle == 2) {                 // double checkerboard: red blocks (dark, light), then blue
            half_sweep(Colour0{}, t, 0);
            half_sweep(Colour1{}, t, 0);
            half_sweep(Colour0{}, t, 1);
            half_sweep(Colour1{}, t, 1);
        } else if (cycle == 1 && first_colour(seed, t)) {
            half_sweep(Colour1{}, t, -1);
            half_sweep(Colour0{}, t, -1);
        } else {
            half_sweep(Colour0{}, t, -1);
            half_sweep(Colour1{}, t, -1);
        }
    }

    // ---- store the own planes back ----
    for (int idx = tid; idx < 2 * PZ * GPP; idx += kResThreads) {
        const int c = idx / (PZ * GPP);
        const int rem = idx - c * PZ * GPP;
        gstate[(size_t)c * GPC + (size_t)z0 * GPP + rem] = res_smem[(size_t)c * (PZ + 2) * GPP + GPP + rem];
    }
}

// ---------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------
inline bool resident_supported(int L) { return L == 64 || L == 128 || L == 256; }

struct ResidentPlan {
    int cs;            // cluster size (0 = cannot run)
    size_t smem;
};

inline size_t resident_smem_bytes(int L, int cs)
{
    return (size_t)2 * (L / cs + 2) * ((size_t)L * L / 16);
}

template <int WPR>
inline cudaError_t resident_try(int cs, int n_rep, size_t smem, int *clusters)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)cs, (unsigned)n_rep);
    cfg.blockDim = dim3(kResThreads);
    cfg.dynamicSmemBytes = smem;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = (unsigned)cs;
    at[0].val.clusterDim.y = 1;
    at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    return cudaOccupancyMaxActiveClusters(clusters, resident_sweep_kernel<WPR>, &cfg);
}

// Pick the cluster size: the smallest that fits shared memory, then grown while all replicas'
// clusters stay co-resident (more SMs per lattice = shorter sweeps).
template <int WPR>
inline ResidentPlan resident_plan_t(int n_rep, int sm_count)
{
    constexpr int L = 64 * WPR;
    ResidentPlan best = {0, 0};
    cudaFuncSetAttribute(resident_sweep_kernel<WPR>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
    cudaFuncSetAttribute(resident_sweep_kernel<WPR>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                         200 * 1024);
    for (int cs = 1; cs <= 16; cs *= 2) {
        const size_t smem = resident_smem_bytes(L, cs);
        if (smem > 200 * 1024 || L / cs < 2) continue;
        if (best.cs && (size_t)n_rep * cs > (size_t)sm_count) break;
        int clusters = 0;
        if (resident_try<WPR>(cs, n_rep, smem, &clusters) != cudaSuccess || clusters < 1) {
            cudaGetLastError();
            continue;
        }
        if (best.cs && clusters < n_rep) break;      // would not be co-resident any more
        best.cs = cs;
        best.smem = smem;
    }
    return best;
}

inline ResidentPlan resident_plan(int L, int n_rep, int sm_count)
{
    switch (L) {
        case 64:  return resident_plan_t<1>(n_rep, sm_count);
        case 128: return resident_plan_t<2>(n_rep, sm_count);
        case 256: return resident_plan_t<4>(n_rep, sm_count);
        default:  return ResidentPlan{0, 0};
    }
}

// can a cluster of `cs` CTAs be scheduled at all on the current device? (ising3d_set_cluster_size)
inline cudaError_t resident_try_size(int L, int cs, int n_rep, int *clusters)
{
    const size_t smem = resident_smem_bytes(L, cs);
    auto prep = [](auto kernel) {
        cudaFuncSetAttribute(kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
        cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    };
    switch (L) {
        case 64:  prep(resident_sweep_kernel<1>); return resident_try<1>(cs, n_rep, smem, clusters);
        case 128: prep(resident_sweep_kernel<2>); return resident_try<2>(cs, n_rep, smem, clusters);
        case 256: prep(resident_sweep_kernel<4>); return resident_try<4>(cs, n_rep, smem, clusters);
        default:  return cudaErrorInvalidValue;
    }
}

template <int WPR>
inline cudaError_t launch_resident_t(uint32_t *state, const uint64_t *d_seeds, int n_rep,
                                     const ResidentPlan &plan, uint32_t t0, uint32_t n_sweeps,
                                     int cycle, cudaStream_t stream)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)plan.cs, (unsigned)n_rep);
    cfg.blockDim = dim3(kResThreads);
    cfg.dynamicSmemBytes = plan.smem;
    cfg.stream = stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = (unsigned)plan.cs;
    at[0].val.clusterDim.y = 1;
    at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, resident_sweep_kernel<WPR>, state, d_seeds, t0, n_sweeps, cycle);
}

inline cudaError_t launch_resident(uint32_t *state, const uint64_t *d_seeds, int L, int n_rep,
                                   const ResidentPlan &plan, uint32_t t0, uint32_t n_sweeps,
                                   int cycle, cudaStream_t stream)
{
    switch (L) {
        case 64:  return launch_resident_t<1>(state, d_seeds, n_rep, plan, t0, n_sweeps, cycle, stream);
        case 128: return launch_resident_t<2>(state, d_seeds, n_rep, plan, t0, n_sweeps, cycle, stream);
        case 256: return launch_resident_t<4>(state, d_seeds, n_rep, plan, t0, n_sweeps, cycle, stream);
        default:  return cudaErrorInvalidValue;
    }
}

}  // namespace ising
