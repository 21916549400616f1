// Tensor-core formulation of the pair counts a8 (D8) for large lattices (L a multiple of 512).
//
// Along one axis the lattice is a 0/1 matrix X[pos][line], pos = 0..L-1 the coordinate along
// the axis, line = one of the L^2 lattice lines (1 <=> s = +1).  With the Gram matrix
//     G[a][b] = sum_line X[a][line] * X[b][line]                     (a dense contraction, K = L^2)
// the antiparallel-pair count of D8 is
//     A(r) = sum_a sum_line [X[a] != X[a+r]] = 2 N_up - 2 sum_a G[a][(a + r) mod L],
// exactly, in integers.  G is computed on the 5th-generation tensor cores: tcgen05.mma
// kind::i8 (u8 x u8 -> s32 accumulators in tensor memory; |G| <= L^2 < 2^31), issued by one
// thread, 128 x 128 x 32 per instruction.  The operands do not exist in memory as bytes: the
// line bits are expanded to bytes by the CUDA cores straight into the 128-byte-swizzled K-major
// shared-memory tiles the MMA reads (one LOP3 per 4 bytes, see expand_row).
//
// Three kernels:
//   gather_lines_kernel<AX>  packed state (D3) -> Xw[pos][L^2/32] line words (bit = one line), in
//                            the handle's spare ping-pong buffer: plane/row copies for z and y
//                            (a site keeps its bit under a y/z shift and alternates colour), a
//                            32x32 warp bit-transpose for x.
//   gram_kernel              persistent CTAs, dynamic task queue; task = (128 positions a) x
//                            (up to 3 units of 128 positions b = a0 + 128 u ...) x (a slice of K).
//                            8 expander warps fill a 4-stage ring (full/empty mbarriers): the B
//                            tiles go to shared memory (generic -> async proxy fence), the A tile
//                            to tensor memory (tcgen05.st, so the tensor core reads only B from
//                            shared memory); warp 8 issues the MMAs (A from TMEM) and commits; the
//                            expander warps read the accumulators back (tcgen05.ld) and add
//                            G[a][b] to a shared-memory histogram over r = b - a.
//   gram_finalize_kernel     A_mu(r) = 2 N_up - 2 Gsum_mu(r).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "kernels_fused.cuh"     // smem_u32, mbar_init, mbar_wait
#include "kernels_measure.cuh"   // warp_transpose32

namespace ising {

constexpr int kGramExpWarps = 8;                       // expander / epilogue warps
constexpr int kGramRowsPerThread = (128 * (1 + 3) + kGramExpWarps * 32 - 1) / (kGramExpWarps * 32);
constexpr int kGramThreads = (kGramExpWarps + 1) * 32;   // + the MMA warp
constexpr int kGramMaxStages = 4;
constexpr int kGramMaxUnits = 3;                       // 3 x 128 accumulator columns; the rest of TMEM holds A
constexpr uint32_t kGramTmemA = 128u * kGramMaxUnits;  // first TMEM column of the A stages (32 columns each)
constexpr int kGramTile = 128 * 128;                   // bytes of one 128-row operand tile (K = 128)

inline bool gram_supported(int L) { return L >= 512 && (L % 512) == 0; }

// ---- gather: packed state -> line words Xw[pos][RW], RW = L*L/32 ------------------------------
// z: Xw[z][p*PW + i]          = W[(z+p)&1][z][i],            PW = L*L/64 plane words, i = y*WPR+wi
// y: Xw[y][(p*L + z)*WPR + wi] = W[(y+p)&1][z][y][wi]
template <int AX>
__global__ void __launch_bounds__(256)
gather_lines_yz_kernel(const uint32_t *__restrict__ state, uint32_t *__restrict__ xw, const int L)
{
    const int WPR = L >> 6;
    const size_t PW = (size_t)L * WPR, WPC = PW * L, RW = 2 * PW;
    const size_t n4 = (size_t)L * RW / 4;
    for (size_t i4 = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i4 < n4;
         i4 += (size_t)gridDim.x * blockDim.x) {
        const size_t o = i4 * 4;
        const size_t pos = o / RW, lw = o - pos * RW;
        size_t src;
        if (AX == 2) {
            const size_t p = lw / PW, i = lw - p * PW;
            src = ((pos + p) & 1) * WPC + pos * PW + i;
        } else {
            const size_t p = lw / PW, rem = lw - p * PW;
            const size_t z = rem / WPR, wi = rem - z * WPR;
            src = ((pos + p) & 1) * WPC + (z * L + pos) * WPR + wi;
        }
        *reinterpret_cast<uint4 *>(xw + o) = *reinterpret_cast<const uint4 *>(state + src);
    }
}

// x: Xw[x][z*(L/32) + yb] bit i = spin (x, 32 yb + i, z).  One block = (z, NWB consecutive words
// of the rows = 64 NWB x-positions, all y); the transposed words go through shared memory so
// that the stores are runs of L/32 consecutive line words.
__global__ void __launch_bounds__(256)
gather_lines_x_kernel(const uint32_t *__restrict__ state, uint32_t *__restrict__ xw, const int L,
                      const int NWB)
{
    extern __shared__ uint32_t gx_smem[];              // out [64 NWB x][L/32 + 1], raw [2][256][NWB + 1]
    const int WPR = L >> 6, YB = L >> 5, LD = YB + 1, RD = NWB + 1;
    const size_t PW = (size_t)L * WPR, WPC = PW * L, RW = 2 * PW;
    const int z = blockIdx.x / (WPR / NWB), wi0 = (blockIdx.x % (WPR / NWB)) * NWB;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    uint32_t *raw = gx_smem + (size_t)64 * NWB * LD;
    for (int y0 = 0; y0 < L; y0 += 256) {
        // both colours of rows y0..y0+255, words wi0..wi0+NWB-1: runs of NWB words (coalesced)
        for (int idx = threadIdx.x; idx < 2 * 256 * NWB; idx += 256) {
            const int w = idx % NWB, yl = (idx / NWB) & 255, col = idx / (NWB * 256);
            raw[(col * 256 + yl) * RD + w] =
                state[(size_t)col * WPC + ((size_t)z * L + y0 + yl) * WPR + wi0 + w];
        }
        __syncthreads();
        // job = (yb in the batch, w, eo): lane = row 32 yb + lane; even-x sites sit in colour (y+z)&1
        for (int job = warp; job < 8 * 2 * NWB; job += 8) {
            const int eo = job & 1, w = (job >> 1) % NWB, ybl = job / (2 * NWB);
            const int yl = 32 * ybl + lane;
            const int col = (y0 + yl + z + eo) & 1;
            const uint32_t t = warp_transpose32(raw[(col * 256 + yl) * RD + w], lane);
            gx_smem[(2 * (32 * w + lane) + eo) * LD + (y0 >> 5) + ybl] = t;   // lane j: k = 32 w + j
        }
        __syncthreads();
    }
    for (int idx = threadIdx.x; idx < 64 * NWB * YB; idx += 256) {
        const int xl = idx / YB, yb = idx - xl * YB;
        xw[(size_t)(64 * wi0 + xl) * RW + (size_t)z * YB + yb] = gx_smem[xl * LD + yb];
    }
}

// ---- tcgen05 helpers ---------------------------------------------------------------------------
// shared-memory matrix descriptor: K-major, SWIZZLE_128B (8 rows x 128 B atoms, 1024 B apart)
__device__ __forceinline__ uint64_t umma_desc_k128(uint32_t saddr)
{
    uint64_t d = 0;
    d |= (uint64_t)((saddr & 0x3FFFF) >> 4);   // start address >> 4, bits [0,14)
    d |= (uint64_t)1 << 16;                    // leading byte offset (unused for one K atom)
    d |= (uint64_t)(1024 >> 4) << 32;          // stride byte offset: 8 rows x 128 B
    d |= (uint64_t)1 << 46;                    // descriptor version (sm_100)
    d |= (uint64_t)2 << 61;                    // SWIZZLE_128B
    return d;
}

// instruction descriptor, kind::i8: D = s32, A = B = u8, both K-major, M = 128, N = 128
constexpr uint32_t kGramIdesc = (2u << 4) | ((128u >> 3) << 17) | ((128u >> 4) << 24);
constexpr uint32_t kGramIdesc256 = (2u << 4) | ((256u >> 3) << 17) | ((128u >> 4) << 24);   // N = 256

// D[tmem] (+)= A[tmem] * B[smem]: A in tensor memory (lane = row, 4 K-bytes per 32-bit column)
__device__ __forceinline__ void umma_i8_ts(uint32_t tmem_d, uint32_t tmem_a, uint64_t db, uint32_t idesc,
                                           uint32_t accumulate)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::i8 [%0], [%1], %2, %3, p;\n\t}\n"
        ::"r"(tmem_d), "r"(tmem_a), "l"(db), "r"(idesc), "r"(accumulate)
        : "memory");
}

__device__ __forceinline__ void umma_commit(uint32_t bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar)
                 : "memory");
}

__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}

// One row of a tile: 128 line bits (4 words) -> 128 bytes, 16-byte piece c stored at c ^ (row & 7).
// The contraction index may be permuted freely as long as A and B agree, and the byte VALUES may
// differ between A and B as long as every product of two set bytes is the same constant.  So:
//   A row: byte-swapped word & (0x01010101 << j)        -> bytes in {0, 2^j}
//   B row: bit-reversed word  & (0x01010101 << (7 - j)) -> bytes in {0, 2^(7-j)}, same line per byte
// for j = 0..7: one PRMT or BREV plus eight LOP3 per 32 lines, no shifts, no multiplies, and every
// product is 2^7: the accumulators hold 128 * G exactly (per task 128 * 128 * K_slice < 2^31).
template <bool IS_B>
__device__ __forceinline__ void expand_row(uint8_t *tile, const int row, const uint4 w)
{
    const uint32_t in[4] = {w.x, w.y, w.z, w.w};
    uint8_t *base = tile + row * 128;
    const int sw = row & 7;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const uint32_t v = IS_B ? __brev(in[i]) : __byte_perm(in[i], 0u, 0x0123u);
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            uint4 o;
            o.x = v & (0x01010101u << (IS_B ? 7 - (4 * h + 0) : 4 * h + 0));
            o.y = v & (0x01010101u << (IS_B ? 7 - (4 * h + 1) : 4 * h + 1));
            o.z = v & (0x01010101u << (IS_B ? 7 - (4 * h + 2) : 4 * h + 2));
            o.w = v & (0x01010101u << (IS_B ? 7 - (4 * h + 3) : 4 * h + 3));
            *reinterpret_cast<uint4 *>(base + (((2 * i + h) ^ sw) << 4)) = o;
        }
    }
}
// An A row goes to tensor memory instead: the warp stores its 32 rows (lane = row) as 32 columns,
// column 8 i + j = the four K-bytes of bit j of the bytes of line word i (the order expand_row<true>
// gives the B rows in shared memory).  Halves the shared-memory traffic of the kernel: the tensor
// core then reads only B from shared memory.
__device__ __forceinline__ void expand_row_tmem(const uint32_t taddr, const uint4 w)
{
    const uint32_t in[4] = {w.x, w.y, w.z, w.w};
    uint32_t a[32];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const uint32_t v = __byte_perm(in[i], 0u, 0x0123u);
#pragma unroll
        for (int j = 0; j < 8; ++j) a[8 * i + j] = v & (0x01010101u << j);
    }
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,"
        "%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31,%32};"
        ::"r"(taddr), "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(a[4]), "r"(a[5]), "r"(a[6]), "r"(a[7]),
          "r"(a[8]), "r"(a[9]), "r"(a[10]), "r"(a[11]), "r"(a[12]), "r"(a[13]), "r"(a[14]), "r"(a[15]),
          "r"(a[16]), "r"(a[17]), "r"(a[18]), "r"(a[19]), "r"(a[20]), "r"(a[21]), "r"(a[22]), "r"(a[23]),
          "r"(a[24]), "r"(a[25]), "r"(a[26]), "r"(a[27]), "r"(a[28]), "r"(a[29]), "r"(a[30]), "r"(a[31])
        : "memory");
}
constexpr int kGramProductShift = 7;       // accumulators = G << 7

struct GramPlan {
    int n_groups;            // column groups per row block
    int units[8];            // units (of 128 columns) per group
    int ustart[8];           // first unit of each group
    int max_units;           // largest group: a stage is (1 + max_units) tiles
    int n_stages;            // ring depth (4: B tiles in shared memory, A tiles in tensor memory)
    int n_slices;            // K slices
    int n_tasks;             // n_slices * (L/128) * n_groups
};

inline GramPlan make_gram_plan(int L, int sm_count)
{
    GramPlan p = {};
    const int U = L / 256 + 1;                       // units covering b - a in [0, L/2 + 127]
    p.n_groups = (U + kGramMaxUnits - 1) / kGramMaxUnits;
    int u = 0;
    for (int g = 0; g < p.n_groups; ++g) {
        p.units[g] = U / p.n_groups + (g < U % p.n_groups ? 1 : 0);
        p.ustart[g] = u;
        u += p.units[g];
    }
    p.max_units = p.units[0];
    p.n_stages = kGramMaxStages;
    const int tiles = (L / 128) * p.n_groups;
    p.n_slices = (sm_count * 12 + tiles - 1) / tiles;
    // the s32 accumulators hold 128 * G, G <= lines per slice: keep 128 * K_slice < 2^31 on any device
    const long long kmax = (1ll << 31) / 128 - 1;
    const int min_slices = (int)(((long long)L * L + kmax - 1) / kmax);
    if (p.n_slices < min_slices) p.n_slices = min_slices;
    p.n_tasks = p.n_slices * tiles;
    return p;
}

inline size_t gram_smem_bytes(int L, const GramPlan &p)
{
    return (size_t)p.n_stages * p.max_units * kGramTile + (size_t)(L / 2 + 1) * 4 + 1024 + 256;
}

// ---- the Gram kernel ---------------------------------------------------------------------------
// xw: line words Xw[pos][RW]; gsum[r] += sum_a G[a][(a+r) mod L] for r = 1..L/2 (64-bit);
// queue: task counter (zeroed by the host before the launch).
__global__ void __launch_bounds__(kGramThreads, 1)
gram_kernel(const uint32_t *__restrict__ xw, unsigned long long *__restrict__ gsum,
            unsigned int *__restrict__ queue, const int L, const __grid_constant__ GramPlan plan)
{
    extern __shared__ __align__(1024) uint8_t gram_raw[];
    uint8_t *smem = gram_raw + ((1024u - (smem_u32(gram_raw) & 1023u)) & 1023u);
    // stage s: max_units B tiles in shared memory + 32 TMEM columns of A
    uint8_t *tiles = smem;
    const int NS = plan.n_stages;
    const size_t stage_bytes = (size_t)plan.max_units * kGramTile;   // B tiles only; A lives in TMEM
    uint32_t *hist = reinterpret_cast<uint32_t *>(smem + (size_t)NS * stage_bytes);
    __shared__ uint64_t full_bar[kGramMaxStages], empty_bar[kGramMaxStages], acc_full, acc_empty;
    __shared__ uint32_t tmem_base_s;
    __shared__ int task_s[2];

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const size_t RW = (size_t)L * L / 32;
    const int n_chunks = (int)(RW / 4);
    const int half = L >> 1;
    const int row_blocks = L / 128;
    const int tiles_per_slice = row_blocks * plan.n_groups;

    for (int r = tid; r <= half; r += kGramThreads) hist[r] = 0;
    if (warp == kGramExpWarps) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(
                         smem_u32(&tmem_base_s)), "r"(512));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    if (tid == 0) {
        for (int s = 0; s < NS; ++s) {
            mbar_init(smem_u32(&full_bar[s]), kGramExpWarps);
            mbar_init(smem_u32(&empty_bar[s]), 1);
        }
        mbar_init(smem_u32(&acc_full), 1);
        mbar_init(smem_u32(&acc_empty), kGramExpWarps);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        task_s[0] = (int)atomicAdd(queue, 1u);
    }
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;");
    const uint32_t tmem_base = tmem_base_s;

    uint32_t it = 0;                                   // chunk counter over all tasks
    int rs = 0;                                        // ring position: stage rs, wrap parity rp
    uint32_t rp = 0;
    int n_done = 0;                                    // tasks finished by this CTA
    // hist[] is 32-bit: a task adds at most 128 pairs * 128 lines per chunk to one r.  `hist_bound`
    // (CTA-uniform) bounds what one entry may hold; the histogram is flushed to the 64-bit global
    // sums before another task could pass 2^32, whatever the SM count or the queue balance.
    unsigned long long hist_bound = 0;
    const unsigned long long task_max =
        128ull * 128ull * (unsigned long long)((n_chunks + plan.n_slices - 1) / plan.n_slices + 1);
    for (int task = task_s[0]; task < plan.n_tasks; ++n_done) {
        // decode: slice-major so that concurrently running CTAs read the same K range (L2 reuse)
        const int slice = task / tiles_per_slice, tl = task - slice * tiles_per_slice;
        const int rb = tl / plan.n_groups, grp = tl - rb * plan.n_groups;
        const int a0 = rb * 128, nu = plan.units[grp], us = plan.ustart[grp];
        const int b0 = a0 + 128 * us;
        const int c_begin = (int)((long long)n_chunks * slice / plan.n_slices);
        const int c_end = (int)((long long)n_chunks * (slice + 1) / plan.n_slices);
        const int n_rows = 128 + 128 * nu;             // A rows, then the B rows of the nu units

        if (warp < kGramExpWarps) {
            // ------------------------------------------------ expanders
            // this thread's rows (at most kGramRowsPerThread of up to 640): tile, row inside the tile, source row
            constexpr int RPT = kGramRowsPerThread;
            uint8_t *t_tile[RPT];
            int t_row[RPT];
            const uint32_t *t_src[RPT];
            bool t_ok[RPT];
#pragma unroll
            for (int i = 0; i < RPT; ++i) {
                const int row = tid + i * kGramExpWarps * 32;
                t_ok[i] = row < n_rows;
                // rows 0..127: A (positions a0 + row); then the B units (positions b0 + ...)
                int pos, ub = -1;
                if (row < 128) {
                    pos = a0 + row;
                } else {
                    ub = (row >> 7) - 1;                                   // unit inside the group
                    pos = b0 + 128 * ub + (row & 127);
                }
                if (pos >= L) pos -= L;
                if (pos >= L) pos -= L;                                    // rows past n_rows: harmless
                t_tile[i] = tiles + (size_t)(ub < 0 ? 0 : ub) * kGramTile;   // B unit u = slot u (A rows: unused)
                t_row[i] = row & 127;
                t_src[i] = xw + (size_t)pos * RW;
            }
            uint4 wn[RPT];                                                   // prefetched line words
#pragma unroll
            for (int i = 0; i < RPT; ++i)
                if (t_ok[i]) wn[i] = *reinterpret_cast<const uint4 *>(t_src[i] + 4 * (size_t)c_begin);
            for (int c = c_begin; c < c_end; ++c, ++it) {
                uint4 wc[RPT];
#pragma unroll
                for (int i = 0; i < RPT; ++i) wc[i] = wn[i];
                if (c + 1 < c_end) {
#pragma unroll
                    for (int i = 0; i < RPT; ++i)
                        if (t_ok[i]) wn[i] = *reinterpret_cast<const uint4 *>(t_src[i] + 4 * (size_t)(c + 1));
                }
                mbar_wait(smem_u32(&empty_bar[rs]), rp ^ 1);
                const size_t soff = (size_t)rs * stage_bytes;
#pragma unroll
                for (int i = 0; i < RPT; ++i)
                    if (t_ok[i]) {
                        if (tid + i * kGramExpWarps * 32 < 128)        // warps 0..3, i = 0: the A rows
                            expand_row_tmem(tmem_base + kGramTmemA + 32u * (uint32_t)rs +
                                                ((uint32_t)(32 * warp) << 16), wc[i]);
                        else
                            expand_row<true>(t_tile[i] + soff, t_row[i], wc[i]);
                    }
                if (warp < 4) asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
                asm volatile("tcgen05.fence::before_thread_sync;");
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                __syncwarp();
                if (lane == 0) mbar_arrive(smem_u32(&full_bar[rs]));
                if (++rs == NS) { rs = 0; rp ^= 1; }
            }
            // ------------------------------------------------ epilogue: G[a][b] -> hist[b - a]
            mbar_wait(smem_u32(&acc_full), (uint32_t)(n_done & 1));
            asm volatile("tcgen05.fence::after_thread_sync;");
            {
                const int lrow = 32 * (warp & 3) + lane;           // TMEM lane = row of the tile
                const int ncol = 128 * nu, chalf = ncol / (kGramExpWarps / 4);
                const int cbeg = (warp >> 2) * chalf;
                for (int c0 = cbeg; c0 < cbeg + chalf; c0 += 16) {
                    uint32_t v[16];
                    const uint32_t taddr = tmem_base + ((uint32_t)(32 * (warp & 3)) << 16) + (uint32_t)c0;
                    asm volatile(
                        "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
                        "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]),
                          "=r"(v[7]), "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]),
                          "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
                        : "r"(taddr));
                    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
                    for (int j = 0; j < 16; ++j) {
                        const int r = 128 * us + c0 + j - lrow;    // b - a (before the periodic wrap)
                        if (r >= 1 && r <= half) atomicAdd(&hist[r], v[j] >> kGramProductShift);
                    }
                }
            }
            asm volatile("tcgen05.fence::before_thread_sync;");
            __syncwarp();
            if (lane == 0) mbar_arrive(smem_u32(&acc_empty));
        } else {
            // ------------------------------------------------ MMA issuer (one thread)
            if (lane == 0) {
                if (n_done > 0) {
                    mbar_wait(smem_u32(&acc_empty), (uint32_t)((n_done - 1) & 1));
                    asm volatile("tcgen05.fence::after_thread_sync;");
                }
                int ms = rs;
                uint32_t mp = rp;
                for (int c = c_begin; c < c_end; ++c) {
                    const int s = ms;
                    mbar_wait(smem_u32(&full_bar[s]), mp);
                    if (++ms == NS) { ms = 0; mp ^= 1; }
                    asm volatile("tcgen05.fence::after_thread_sync;");
                    const uint32_t sbase = smem_u32(tiles + (size_t)s * stage_bytes);
                    const uint32_t ta = tmem_base + kGramTmemA + 32u * (uint32_t)s;   // A: 8 columns per K = 32
                    for (int u = 0; u < nu; u += 2) {          // two units (N = 256) per instruction where possible
                        const uint64_t db = umma_desc_k128(sbase + (uint32_t)u * kGramTile);
                        const uint32_t idesc = (u + 1 < nu) ? kGramIdesc256 : kGramIdesc;
#pragma unroll
                        for (int ks = 0; ks < 4; ++ks)         // K = 32 per instruction: +32 B in the atom
                            umma_i8_ts(tmem_base + (uint32_t)(128 * u), ta + (uint32_t)(8 * ks),
                                       db + (uint64_t)(2 * ks), idesc, (c > c_begin || ks > 0) ? 1u : 0u);
                    }
                    umma_commit(smem_u32(&empty_bar[s]));      // frees the stage when the MMAs have read it
                }
                umma_commit(smem_u32(&acc_full));              // accumulators of this task complete
            }
            // all lanes of the MMA warp advance the ring position like the expanders did
            {
                const int adv = c_end - c_begin;
                it += (uint32_t)adv;
                const int tot = rs + adv;
                if ((tot / NS) & 1) rp ^= 1;
                rs = tot % NS;
            }
            __syncwarp();
        }
        // next task (one fetch per CTA, broadcast through shared memory)
        if (tid == 0) task_s[(n_done + 1) & 1] = (int)atomicAdd(queue, 1u);
        __syncthreads();
        task = task_s[(n_done + 1) & 1];
        hist_bound += task_max;
        if (hist_bound + task_max > 0xFFFFFFFFull) {
            for (int r = 1 + tid; r <= half; r += kGramThreads) {
                if (hist[r]) atomicAdd(&gsum[r], (unsigned long long)hist[r]);
                hist[r] = 0;
            }
            hist_bound = 0;
            __syncthreads();
        }
    }

    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    for (int r = 1 + tid; r <= half; r += kGramThreads)
        if (hist[r]) atomicAdd(&gsum[r], (unsigned long long)hist[r]);
    if (warp == kGramExpWarps)
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(512));
}

// A_mu(r) = 2 N_up - 2 Gsum_mu(r) for r = 1..L/2 (counts layout of kernels_measure.cuh)
__global__ void gram_finalize_kernel(unsigned long long *__restrict__ counts,
                                     const unsigned long long *__restrict__ gsum, const int nr)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= 3 * nr) return;
    const int r = i % nr;
    counts[1 + i] = r == 0 ? 0ull : 2ull * counts[0] - 2ull * gsum[i];
}

}  // namespace ising
