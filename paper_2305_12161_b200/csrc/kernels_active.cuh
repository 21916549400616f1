// Activity-driven half-sweep (a2/a3/a4 at late times), L in {256, 512, 1024, 2048, 4096}.
//
// eq. (6) PAPER.md:105-108 changes a site only if Delta E <= 0, i.e. if n >= 3 of its six
// neighbours are antiparallel (D2).  A 128-spin group none of whose sites has n >= 3 is left as
// it is by a half-sweep whatever its random bits are, and it stays so until one of the words it
// reads changes.  After a few thousand sweeps most groups are in that state (8 % of them hold a
// site with n >= 3 at t = 10^5, L = 2048), while a warp of the dense kernels -- 32 groups, whole
// x rows -- almost always (81 %) still holds one: skipping work under a warp vote does not pay, a
// list of the groups that can change does.
//
// One flag per group and colour ("awake", 1 bit; 4 MB per colour at L = 2048) with the invariant
//   when colour c is updated, every colour-c group holding a site with n >= 3 has its flag set.
// activity_flags_kernel establishes it from a state (flag = some site of the group has n >= 3).
// active_halfsweep_kernel keeps it: it evaluates the flagged groups of colour c only, in place
// (same-colour sites do not interact, so the order is free), leaves a group's flag
// set iff the group still holds a tie (n = 3: the next sweep's random bit can flip it; a site with
// n >= 4 has flipped and now has n <= 2), and sets the flag of the other-colour groups that read
// a word it changed (same group index, y+-1, z+-1, and the row neighbour that takes the edge bit) -- of
// those only that hold a neighbour of a flipped site which now differs from it: that neighbour's n went
// up, any other neighbour's n went down, and a sleeping group's sites all have n <= 2.
// The random bits are the same counter-based Philox4x32-10 bits (q, t, colour, 0) as everywhere
// (D5), drawn only for groups that hold a tie, so the trajectory is bit-identical to the dense
// kernels'.
//
// Work distribution: a CTA draws bricks of 2048 groups (32 rows x 8 planes x all x at L = 2048:
// compact in y and z, so that the y+-1 and z+-1 words of one evaluation are the same-position
// words of the evaluations around it and come from L1) from a ticket counter, compacts the set
// flag bits into a shared-memory list (one flag byte per thread, CTA-wide prefix sum) and its 256
// threads evaluate the listed groups.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "kernels_fused2.cuh"   // SweepConsts, philox_folded
#include "philox.cuh"

namespace ising {

inline bool active_supported(int L) { return L == 256 || L == 512 || L == 1024 || L == 2048 || L == 4096; }

struct ActiveGeom {
    int lgL;          // L = 1 << lgL
    int lgR4;         // 128-spin groups per row R4 = L / 256 = 1 << lgR4
    uint32_t G;       // groups per colour = L * L * R4
    // work item of active_halfsweep_kernel: a brick of 2048 groups = PB planes x RB rows x all R4 groups
    int lgRS;         // groups per plane strip RS = RB * R4, RB = 32 rows
    int lgPB;         // planes per brick PB = 2048 / RS
};

inline ActiveGeom make_active_geom(int L)
{
    ActiveGeom g;
    g.lgL = 0;
    while ((1 << g.lgL) < L) ++g.lgL;
    g.lgR4 = g.lgL - 8;
    g.G = (uint32_t)L * (uint32_t)L * (uint32_t)(L >> 8);
    g.lgRS = g.lgR4 + 5;
    g.lgPB = 11 - g.lgRS;
    return g;
}

// The six neighbour words of group g of colour c and the per-word masks of eq. (6):
// tie = sites with n = 3 (U = 3 up neighbours), det = [U + s >= 4] = the new spin where no tie.
struct GroupEval {
    uint4 s, tie, det;
};

__device__ __forceinline__ void rule_split(uint32_t s, uint32_t n1, uint32_t n2, uint32_t n3, uint32_t n4,
                                           uint32_t n5, uint32_t n6, uint32_t &tie, uint32_t &det)
{
    const uint32_t sa = n1 ^ n2 ^ n3, ca = maj3(n1, n2, n3);
    const uint32_t sb = n4 ^ n5 ^ n6, cb = maj3(n4, n5, n6);
    tie = (sa ^ sb) & (ca ^ cb);                 // U = (sa + sb) + 2 (ca + cb) = 3
    det = maj3(ca, cb, maj3(sa, sb, s));         // [U + s >= 4]; equals s on the tie sites
}

struct GroupNbr {
    uint32_t gyp, gym, gzp, gzm, gprev, gnext;   // group indices (periodic)
    int o;                                       // in-row direction of the colour being updated
};

__device__ __forceinline__ GroupNbr group_neighbours(uint32_t g, int c, const ActiveGeom &geo)
{
    const uint32_t R4 = 1u << geo.lgR4, L = 1u << geo.lgL, GP = L << geo.lgR4;
    const uint32_t x4 = g & (R4 - 1), row = g >> geo.lgR4;
    const uint32_t y = row & (L - 1), z = row >> geo.lgL;
    GroupNbr n;
    n.gyp = (y + 1 == L) ? g - (L - 1) * R4 : g + R4;
    n.gym = (y == 0) ? g + (L - 1) * R4 : g - R4;
    n.gzp = (z + 1 == L) ? g - (L - 1) * GP : g + GP;
    n.gzm = (z == 0) ? g + (L - 1) * GP : g - GP;
    n.gprev = (x4 == 0) ? g + R4 - 1 : g - 1;
    n.gnext = (x4 == R4 - 1) ? g + 1 - R4 : g + 1;
    n.o = (int)((y + z + (uint32_t)c) & 1u);
    return n;
}

__device__ __forceinline__ GroupEval eval_group(const uint4 *__restrict__ own, const uint4 *__restrict__ oth,
                                                uint32_t g, const GroupNbr &n)
{
    GroupEval e;
    e.s = own[g];
    const uint4 a = __ldg(oth + g);
    const uint4 yp = __ldg(oth + n.gyp), ym = __ldg(oth + n.gym);
    const uint4 zp = __ldg(oth + n.gzp), zm = __ldg(oth + n.gzm);
    // D4: o = 0 -> neighbour k-1 (edge = word 3 of the previous group), o = 1 -> k+1 (word 0 of the next)
    const uint32_t *othw = reinterpret_cast<const uint32_t *>(oth);
    const uint32_t edge = __ldg(othw + (n.o ? 4 * (size_t)n.gnext : 4 * (size_t)n.gprev + 3));
    const uint4 x = xshift(a, n.o, edge);
    rule_split(e.s.x, a.x, x.x, yp.x, ym.x, zp.x, zm.x, e.tie.x, e.det.x);
    rule_split(e.s.y, a.y, x.y, yp.y, ym.y, zp.y, zm.y, e.tie.y, e.det.y);
    rule_split(e.s.z, a.z, x.z, yp.z, ym.z, zp.z, zm.z, e.tie.z, e.det.z);
    rule_split(e.s.w, a.w, x.w, yp.w, ym.w, zp.w, zm.w, e.tie.w, e.det.w);
    return e;
}

// Flags from a state: bit g of awake[c] = group g of colour c holds a site with n >= 3
// (Delta E <= 0, eq. (6)).  One thread per group, blockIdx.y = colour; count[c] += set flags.
__global__ void __launch_bounds__(256)
activity_flags_kernel(const uint32_t *__restrict__ state, uint32_t *__restrict__ awake,
                      unsigned long long *__restrict__ count, const ActiveGeom geo)
{
    const uint32_t g = blockIdx.x * 256u + threadIdx.x;          // G is a multiple of 1024
    const int c = blockIdx.y;
    const uint4 *base = reinterpret_cast<const uint4 *>(state);
    const uint4 *own = base + (size_t)c * geo.G, *oth = base + (size_t)(1 - c) * geo.G;
    const GroupNbr n = group_neighbours(g, c, geo);
    const GroupEval e = eval_group(own, oth, g, n);
    // a site changes or may change iff it is a tie or det differs from s (n >= 4)
    const uint32_t act = e.tie.x | e.tie.y | e.tie.z | e.tie.w | (e.det.x ^ e.s.x) | (e.det.y ^ e.s.y) |
                         (e.det.z ^ e.s.z) | (e.det.w ^ e.s.w);
    const uint32_t b = __ballot_sync(0xffffffffu, act != 0u);
    __shared__ unsigned int cta_count;
    if (threadIdx.x == 0) cta_count = 0;
    __syncthreads();
    if ((threadIdx.x & 31) == 0) {
        awake[(size_t)c * (geo.G >> 5) + (g >> 5)] = b;
        if (b) atomicAdd(&cta_count, (unsigned)__popc(b));
    }
    __syncthreads();
    if (threadIdx.x == 0 && cta_count) atomicAdd(count + c, (unsigned long long)cta_count);
}

// A second read of words eval_group has just read (they sit in L1).  volatile: the compiler must not merge
// it with the first read and keep 21 more registers alive across the Philox call for a branch few groups take.
__device__ __forceinline__ uint4 ldg_again(const uint4 *p)
{
    uint4 v;
    asm volatile("ld.global.nc.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ uint32_t ldg_again(const uint32_t *p)
{
    uint32_t v;
    asm volatile("ld.global.nc.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

constexpr int kActiveThreads = 256;
constexpr int kActiveChunk = 2048;       // groups per work item: 64 flag words = 256 flag bytes, one per thread

// ROLE = 0 / 1: first / second colour of the sweep (c = first ^ ROLE; keys.c1[ROLE] carries c).
// stat[0] += groups evaluated, stat[1] += groups changed, stat[2] += groups that held a site with
// Delta E <= 0 when they were evaluated (what activity_flags_kernel counts, taken at the colour's update).
// Work items (bricks of 2048 groups) are handed out through a ticket counter that is
// never reset: this launch owns tickets base .. base + n_chunks - 1 (mod 2^32), and every CTA draws
// exactly one ticket beyond them before it stops, so the next launch starts at
// base + n_chunks + gridDim.x (the host keeps count).
// Four CTAs per SM (64 registers, no spills; ptxas takes 80 unasked, which leaves room for three): the kernel
// waits for scattered sectors, so resident warps are what it needs (two CTAs per SM: 60 % slower).
template <int ROLE>
__global__ void __launch_bounds__(kActiveThreads, 4)
active_halfsweep_kernel(uint32_t *__restrict__ state, uint32_t *__restrict__ awake, const int c,
                        unsigned long long *__restrict__ stat, unsigned int *__restrict__ tickets,
                        const uint32_t base_ticket, const ActiveGeom geo,
                        const __grid_constant__ SweepConsts keys)
{
    __shared__ uint16_t list[kActiveChunk];
    __shared__ uint32_t keep[kActiveChunk / 32];
    __shared__ uint32_t wtot[kActiveThreads / 32];
    __shared__ uint32_t ticket[2];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    uint4 *basep = reinterpret_cast<uint4 *>(state);
    uint4 *own = basep + (size_t)c * geo.G;
    const uint4 *oth = basep + (size_t)(1 - c) * geo.G;
    uint32_t *aw_own = awake + (size_t)c * (geo.G >> 5);
    uint32_t *aw_oth = awake + (size_t)(1 - c) * (geo.G >> 5);
    const uint32_t n_chunks = geo.G / kActiveChunk;
    uint32_t evaluated = 0, changed = 0, held = 0;
    const uint8_t *flag_bytes = reinterpret_cast<const uint8_t *>(aw_own);
    // brick `chunk` = strip by (RB rows) of slab bz (PB planes); its groups are, plane by plane, RS
    // consecutive group indices from brick_base(chunk) + j * GP
    const uint32_t RS = 1u << geo.lgRS, GP = 1u << (geo.lgL + geo.lgR4);
    const int lg_ny = geo.lgL + geo.lgR4 - geo.lgRS;                  // strips per plane = L / RB
    auto brick_base = [&](uint32_t chunk) -> uint32_t {
        const uint32_t by = chunk & ((1u << lg_ny) - 1u), bz = chunk >> lg_ny;
        return ((bz << geo.lgPB) * GP) + (by << geo.lgRS);
    };
    // one flag byte (8 groups) per thread: plane fj of the brick, byte fb of its strip
    const uint32_t fj = (uint32_t)tid >> (geo.lgRS - 3), fb = (uint32_t)tid & ((RS >> 3) - 1u);
    auto flag_byte = [&](uint32_t chunk) -> uint32_t {
        return chunk < n_chunks ? flag_bytes[((size_t)brick_base(chunk) + (size_t)fj * GP) / 8 + fb] : 0u;
    };
    if (tid == 0) ticket[0] = atomicAdd(tickets, 1u) - base_ticket;
    __syncthreads();
    // the next brick's byte is fetched while this brick is evaluated
    uint32_t f_next = flag_byte(ticket[0]);
    for (int par = 0;; par ^= 1) {
        const uint32_t chunk = ticket[par];
        if (chunk >= n_chunks) break;
        if (tid == 0) ticket[par ^ 1] = atomicAdd(tickets, 1u) - base_ticket;   // read after the barrier below
        const uint32_t f = f_next;
        uint32_t incl = __popc(f);
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const uint32_t v = __shfl_up_sync(0xffffffffu, incl, d);
            if (lane >= d) incl += v;
        }
        if (lane == 31) wtot[warp] = incl;
        if (tid < kActiveChunk / 32) keep[tid] = 0u;
        __syncthreads();
        f_next = flag_byte(ticket[par ^ 1]);
        const uint32_t base = brick_base(chunk);
        uint32_t p = incl - __popc(f), total = 0;
#pragma unroll
        for (int w = 0; w < kActiveThreads / 32; ++w) {
            if (w < warp) p += wtot[w];
            total += wtot[w];
        }
        if (total == 0) {                      // nothing awake here (uniform: every thread sees the same total)
            __syncthreads();                   // wtot / ticket are rewritten in the next round
            continue;
        }
        for (uint32_t ff = f; ff; ff &= ff - 1) list[p++] = (uint16_t)(tid * 8 + (__ffs(ff) - 1));
        __syncthreads();
        for (uint32_t i = tid; i < total; i += kActiveThreads) {
            const uint32_t li = list[i];                     // plane (li >> lgRS) of the brick, group li & (RS - 1) of its strip
            const uint32_t g = base + (li >> geo.lgRS) * GP + (li & (RS - 1u));
            const GroupNbr n = group_neighbours(g, c, geo);
            const GroupEval e = eval_group(own, oth, g, n);
            uint4 nw = e.det;
            const uint32_t anytie = e.tie.x | e.tie.y | e.tie.z | e.tie.w;
            if (anytie) {
                // eq. (6), Delta E = 0: flip iff the site's random bit is 1 (D2, D5)
                const uint4 rho = philox_folded<ROLE>(g, keys);
                nw.x ^= e.tie.x & rho.x;
                nw.y ^= e.tie.y & rho.y;
                nw.z ^= e.tie.z & rho.z;
                nw.w ^= e.tie.w & rho.w;
                atomicOr(&keep[li >> 5], 1u << (li & 31));
            }
            // a site with n >= 4 shows as det != s, one with n = 3 as a tie
            if (anytie | (e.det.x ^ e.s.x) | (e.det.y ^ e.s.y) | (e.det.z ^ e.s.z) | (e.det.w ^ e.s.w)) ++held;
            const uint4 d = make_uint4(nw.x ^ e.s.x, nw.y ^ e.s.y, nw.z ^ e.s.z, nw.w ^ e.s.w);
            if (d.x | d.y | d.z | d.w) {
                own[g] = nw;
                ++changed;
                // Wake other-colour groups (D4).  A flip moves the antiparallel count n of each of its six
                // neighbours by one: up if the neighbour differs from the new spin, down if it equals it.  A
                // sleeping group has n <= 2 on all its sites, and only a step up can bring one to n >= 3,
                // so a group is woken only if it holds a neighbour, of a flipped site, that differs from the
                // new spin.  The neighbour words are the ones eval_group just read (L1).
                auto up = [&](const uint4 &v) -> uint32_t {
                    return (d.x & (nw.x ^ v.x)) | (d.y & (nw.y ^ v.y)) | (d.z & (nw.z ^ v.z)) | (d.w & (nw.w ^ v.w));
                };
                // one neighbour word at a time (few registers live): y+-1, z+-1
                if (up(ldg_again(oth + n.gyp))) atomicOr(aw_oth + (n.gyp >> 5), 1u << (n.gyp & 31));
                if (up(ldg_again(oth + n.gym))) atomicOr(aw_oth + (n.gym >> 5), 1u << (n.gym & 31));
                if (up(ldg_again(oth + n.gzp))) atomicOr(aw_oth + (n.gzp >> 5), 1u << (n.gzp & 31));
                if (up(ldg_again(oth + n.gzm))) atomicOr(aw_oth + (n.gzm >> 5), 1u << (n.gzm & 31));
                // in-row neighbours: bit k of the same-index group and the bit beside it; the one bit of x
                // that came from `edge` (bit 127 with o = 1, bit 0 with o = 0) lies in the next / previous group
                const uint4 a = ldg_again(oth + g);
                const uint32_t *othw = reinterpret_cast<const uint32_t *>(oth);
                const uint32_t edge = ldg_again(othw + (n.o ? 4 * (size_t)n.gnext : 4 * (size_t)n.gprev + 3));
                const uint4 x = xshift(a, n.o, edge);
                uint4 ux = make_uint4(d.x & (nw.x ^ x.x), d.y & (nw.y ^ x.y), d.z & (nw.z ^ x.z), d.w & (nw.w ^ x.w));
                const uint32_t up_edge = n.o ? (ux.w >> 31) : (ux.x & 1u);
                if (n.o) ux.w &= 0x7fffffffu;
                else ux.x &= ~1u;
                if (up(a) | ux.x | ux.y | ux.z | ux.w) atomicOr(aw_oth + (g >> 5), 1u << (g & 31));
                if (up_edge) {
                    const uint32_t ge = n.o ? n.gnext : n.gprev;
                    atomicOr(aw_oth + (ge >> 5), 1u << (ge & 31));
                }
            }
        }
        __syncthreads();
        if (tid < kActiveChunk / 32) {
            const uint32_t bit0 = 32u * (uint32_t)tid;        // first list index of this flag word
            aw_own[(base + (bit0 >> geo.lgRS) * GP + (bit0 & (RS - 1u))) >> 5] = keep[tid];
        }
        if (tid == 0) evaluated += total;
    }
    for (int d = 16; d; d >>= 1) {
        changed += __shfl_xor_sync(0xffffffffu, changed, d);
        held += __shfl_xor_sync(0xffffffffu, held, d);
    }
    if (lane == 0 && (evaluated | changed | held)) {
        if (evaluated) atomicAdd(stat, (unsigned long long)evaluated);
        if (changed) atomicAdd(stat + 1, (unsigned long long)changed);
        if (held) atomicAdd(stat + 2, (unsigned long long)held);
    }
}

inline cudaError_t launch_activity_flags(const uint32_t *state, uint32_t *awake, unsigned long long *count,
                                         int L, cudaStream_t stream)
{
    const ActiveGeom geo = make_active_geom(L);
    activity_flags_kernel<<<dim3(geo.G / 256u, 2u), 256, 0, stream>>>(state, awake, count, geo);
    return cudaGetLastError();
}

struct ActivePlan {
    unsigned grid = 0;            // resident CTAs: the ticket queue balances the chunks over them
    uint32_t next_ticket = 0;     // first ticket of the next launch (the counter itself is never reset)
    bool ready = false;
};

inline cudaError_t plan_active(ActivePlan &plan, int L, int sm_count)
{
    int occ = 0;
    cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, active_halfsweep_kernel<0>,
                                                                  kActiveThreads, 0);
    if (e != cudaSuccess) return e;
    if (occ < 1) occ = 1;
    const ActiveGeom geo = make_active_geom(L);
    plan.grid = (unsigned)(sm_count * occ);
    const unsigned n_chunks = geo.G / kActiveChunk;
    if (plan.grid > n_chunks) plan.grid = n_chunks;
    plan.ready = true;
    return cudaSuccess;
}

// One sweep = the two half-sweeps in the order (first, 1 - first) (D7, D10).  `tickets` is the
// handle's ticket counter (zero when the plan was made); one counter per stream-ordered sequence.
inline cudaError_t launch_active_sweep(uint32_t *state, uint32_t *awake, unsigned long long *stat,
                                       unsigned int *tickets, ActivePlan &plan, int L, uint32_t t,
                                       uint64_t seed, int first, cudaStream_t stream)
{
    const ActiveGeom geo = make_active_geom(L);
    const SweepConsts keys = make_sweep_consts(seed, t, first);
    const uint32_t per_launch = geo.G / kActiveChunk + plan.grid;
    // the host's ticket count follows the device counter only for launches that were accepted: after a
    // refused launch the caller resets both (reset_active_tickets)
    active_halfsweep_kernel<0><<<plan.grid, kActiveThreads, 0, stream>>>(state, awake, first, stat, tickets,
                                                                       plan.next_ticket, geo, keys);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    plan.next_ticket += per_launch;
    active_halfsweep_kernel<1><<<plan.grid, kActiveThreads, 0, stream>>>(state, awake, 1 - first, stat, tickets,
                                                                       plan.next_ticket, geo, keys);
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    plan.next_ticket += per_launch;
    return cudaSuccess;
}

// After a failed launch: device counter and host count back to zero, in stream order.
inline cudaError_t reset_active_tickets(unsigned int *tickets, ActivePlan &plan, cudaStream_t stream)
{
    plan.next_ticket = 0;
    return cudaMemsetAsync(tickets, 0, sizeof(unsigned int), stream);
}

}  // namespace ising
