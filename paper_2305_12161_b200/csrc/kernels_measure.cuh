// Measurement reductions a6-a8 (D8): N_up and the antiparallel-pair counts
//   A_mu(r) = #{sites i : s_i != s_{i + r e_mu}},  mu = x,y,z,  r = 1..L/2, periodic
// (eq. (2) PAPER.md:43 reduced to integer counts; the axis-averaged estimator is
// BASELINE.json's, the paper itself goes through an FFT).
//
// All three axes are brought to ONE problem: "line words".  A line word sequence S[0..L)
// holds 32 independent lattice lines running along the measured axis, one per bit:
// bit j of S[a] = spin at position a of line j.  Then
//   A_mu(r) = sum over sequences, sum_a popc(S[a] ^ S[(a + r) mod L]).
// How the packed layout D3 yields such sequences (derived from D3/D4):
//   z axis: position (y, wi) of a plane and a class p in {0,1}:  S[z] = W[(z+p)&1][z][y][wi]
//           (a site keeps its bit (k = x>>1) under a z shift and changes colour iff r is odd).
//   y axis: position (z, wi), class p:                            S[y] = W[(y+p)&1][z][y][wi].
//   x axis: 32 consecutive rows (y0..y0+31, z); the row words of the colour holding the even-x
//           sites (colour (y+z)&1) and of the other colour are bit-transposed 32x32 with warp
//           shuffles, S[2k] = even-x word k, S[2k+1] = odd-x word k: S[x] = the 32 rows at x.
// L^2/32 sequences per axis, each L*(L/2) word pairs: 2.7e11 pairs per axis at L = 2048, far
// more ALU work than memory traffic (the lattice is read once per axis).
//
// Kernel: persistent CTAs; a tile of C sequences (C*L = 32768 words, 128 KiB) sits in shared
// memory; a thread owns (sequence, 8 consecutive displacements r = 8j..8j+7), keeps a sliding
// window of the sequence in registers (8 x-words, 16 y-words: 64 pairs per 4 LDS.128) and adds
// the 8 XOR words of each displacement into a carry-save counter stack (Harley-Seal: ones,
// twos, fours; one POPC per 8 words on the overflow): 22 LOP3 + 1 POPC + 1 IADD per 8 word
// pairs instead of 8 x (XOR + POPC + IADD + 2 LDS).  Counts go to shared-memory u32 counters
// (one per r) and leave the CTA once, as 64-bit atomics.
//
// counts layout per replica: [0] = N_up, [1 + mu*(L/2+1) + r] = A_mu(r), mu = 0,1,2 = x,y,z.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace ising {

// ---- N_up -----------------------------------------------------------------
__global__ void __launch_bounds__(256)
count_up_kernel(const uint32_t *__restrict__ state, unsigned long long *__restrict__ counts,
                size_t words_per_replica, int counts_per_replica)
{
    const int rep = blockIdx.y;
    const uint4 *p = reinterpret_cast<const uint4 *>(state + (size_t)rep * words_per_replica);
    const size_t n4 = words_per_replica / 4;
    unsigned long long acc = 0;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4;
         i += (size_t)gridDim.x * blockDim.x) {
        const uint4 v = p[i];
        acc += __popc(v.x) + __popc(v.y) + __popc(v.z) + __popc(v.w);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    __shared__ unsigned long long sh[8];
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long s = 0;
        for (int i = 0; i < (int)(blockDim.x >> 5); ++i) s += sh[i];
        atomicAdd(&counts[(size_t)rep * counts_per_replica], s);
    }
}

// ---- A_mu(r) ----------------------------------------------------------------
constexpr int kAcThreads = 512;
constexpr int kAcPad = 4;        // words of padding per sequence: conflict-free LDS.128 across sequences

// 32x32 bit transpose across the lanes of a warp: on return, bit i of lane j's word is bit j
// of lane i's input word.
__device__ __forceinline__ uint32_t warp_transpose32(uint32_t a, const int lane)
{
#pragma unroll
    for (int s = 16; s >= 1; s >>= 1) {
        const uint32_t m = s == 16 ? 0x0000FFFFu : s == 8 ? 0x00FF00FFu : s == 4 ? 0x0F0F0F0Fu
                         : s == 2 ? 0x33333333u : 0x55555555u;
        const uint32_t o = __shfl_xor_sync(0xffffffffu, a, s);
        a = (lane & s) ? (((o >> s) & m) | (a & ~m)) : ((a & m) | ((o & m) << s));
    }
    return a;
}

// carry-save adder: (h, l) = a + b + c per bit, as exactly two LOP3 (written as PTX lop3 so that
// the compiler does not re-associate the XORs of fresh inputs into extra instructions)
__device__ __forceinline__ uint32_t lop3_xor3(uint32_t a, uint32_t b, uint32_t c)
{
    uint32_t r;
    asm("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(r) : "r"(a), "r"(b), "r"(c));
    return r;
}
__device__ __forceinline__ uint32_t lop3_maj3(uint32_t a, uint32_t b, uint32_t c)
{
    uint32_t r;
    asm("lop3.b32 %0, %1, %2, %3, 0xE8;" : "=r"(r) : "r"(a), "r"(b), "r"(c));
    return r;
}
__device__ __forceinline__ uint32_t lop_xor2(uint32_t a, uint32_t b)
{
    uint32_t r;
    asm("xor.b32 %0, %1, %2;" : "=r"(r) : "r"(a), "r"(b));
    return r;
}
#define ISING_CSA(h, l, a, b, c)                       \
    {                                                  \
        const uint32_t a__ = (a), b__ = (b), c__ = (c); \
        (h) = lop3_maj3(a__, b__, c__);                \
        (l) = lop3_xor3(a__, b__, c__);                \
    }

struct AcStack {                 // bit-sliced counter of one displacement
    uint32_t ones, twos, fours, eights_count;
};

// word k of the 16-word window (lo, hi), k compile-time
template <int K>
__device__ __forceinline__ uint32_t ac_win(const uint32_t (&lo)[8], const uint32_t (&hi)[8])
{
    return K < 8 ? lo[K & 7] : hi[K & 7];
}

// add the 8 words x[k] ^ y[k + I], k = 0..7, y = (lo, hi), to the stack
template <int I>
__device__ __forceinline__ void ac_add8(AcStack &s, const uint32_t (&x)[8],
                                        const uint32_t (&lo)[8], const uint32_t (&hi)[8])
{
    uint32_t t0, t1, t2, t3, f0, f1, e;
    ISING_CSA(t0, s.ones, s.ones, lop_xor2(x[0], ac_win<0 + I>(lo, hi)), lop_xor2(x[1], ac_win<1 + I>(lo, hi)));
    ISING_CSA(t1, s.ones, s.ones, lop_xor2(x[2], ac_win<2 + I>(lo, hi)), lop_xor2(x[3], ac_win<3 + I>(lo, hi)));
    ISING_CSA(f0, s.twos, s.twos, t0, t1);
    ISING_CSA(t2, s.ones, s.ones, lop_xor2(x[4], ac_win<4 + I>(lo, hi)), lop_xor2(x[5], ac_win<5 + I>(lo, hi)));
    ISING_CSA(t3, s.ones, s.ones, lop_xor2(x[6], ac_win<6 + I>(lo, hi)), lop_xor2(x[7], ac_win<7 + I>(lo, hi)));
    ISING_CSA(f1, s.twos, s.twos, t2, t3);
    ISING_CSA(e, s.fours, s.fours, f0, f1);
    s.eights_count += __popc(e);
}

__device__ __forceinline__ void ac_add64(AcStack (&st)[8], const uint32_t (&x)[8],
                                         const uint32_t (&lo)[8], const uint32_t (&hi)[8])
{
    ac_add8<0>(st[0], x, lo, hi);
    ac_add8<1>(st[1], x, lo, hi);
    ac_add8<2>(st[2], x, lo, hi);
    ac_add8<3>(st[3], x, lo, hi);
    ac_add8<4>(st[4], x, lo, hi);
    ac_add8<5>(st[5], x, lo, hi);
    ac_add8<6>(st[6], x, lo, hi);
    ac_add8<7>(st[7], x, lo, hi);
}

__device__ __forceinline__ uint32_t ac_total(const AcStack &s)
{
    return 8u * s.eights_count + 4u * __popc(s.fours) + 2u * __popc(s.twos) + __popc(s.ones);
}

__device__ __forceinline__ void ld8(uint32_t *dst, const uint32_t *src)
{
    const uint4 a = *reinterpret_cast<const uint4 *>(src);
    const uint4 b = *reinterpret_cast<const uint4 *>(src + 4);
    dst[0] = a.x; dst[1] = a.y; dst[2] = a.z; dst[3] = a.w;
    dst[4] = b.x; dst[5] = b.y; dst[6] = b.z; dst[7] = b.w;
}

// AX = 0 (x), 1 (y), 2 (z).  Grid: (persistent CTAs, replicas).  C = sequences per tile
// (a power of two, >= 8, dividing L^2/32), shared memory = C*(L+pad) + (L/2+1) words.
template <int AX>
__global__ void __launch_bounds__(kAcThreads, 1)
autocorr_kernel(const uint32_t *__restrict__ state, unsigned long long *__restrict__ counts,
                const int L, const int C, const int n_tiles, const int counts_per_replica)
{
    extern __shared__ __align__(16) uint32_t ac_smem[];
    const int LP = L + kAcPad;
    uint32_t *S = ac_smem;                   // [C][LP]
    uint32_t *cnt = ac_smem + (size_t)C * LP;   // [L/2 + 1]
    const int WPR = L >> 6;
    const size_t WPC = (size_t)L * L * WPR;
    const int rep = blockIdx.y;
    const uint32_t *base = state + (size_t)rep * 2 * WPC;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nr = L / 2 + 1;

    for (int r = tid; r < nr; r += kAcThreads) cnt[r] = 0;
    // cnt[] is 32-bit: one tile adds at most 32 * C * L (= 2^20 for full tiles) to an entry, so it is
    // flushed to the 64-bit global counters every `flush_every` tiles, whatever the grid size
    const int flush_every = (int)(0xFFFFFFFFull / (32ull * (unsigned long long)C * (unsigned long long)L));
    int since_flush = 0;

    for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        __syncthreads();                     // previous tile fully consumed, cnt zeroed
        // ------------------------------------------------------------ load the tile
        if (AX == 0) {
            // sequence c = rows (tile*C + c)*32 .. +31; warp job = (c, wi, eo)
            const int jobs = C * WPR * 2;
            for (int job0 = warp * 4; job0 < jobs; job0 += (kAcThreads / 32) * 4) {
                uint32_t w[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int job = job0 + u;            // jobs is a multiple of 4
                    const int eo = job & 1, wi = (job >> 1) % WPR, c = (job >> 1) / WPR;
                    const size_t row = ((size_t)tile * C + c) * 32 + lane;
                    const int y = (int)(row % L), z = (int)(row / L);
                    const int col = (y + z + eo) & 1;
                    w[u] = __ldg(base + (size_t)col * WPC + row * WPR + wi);
                }
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int job = job0 + u;
                    const int eo = job & 1, wi = (job >> 1) % WPR, c = (job >> 1) / WPR;
                    const uint32_t t = warp_transpose32(w[u], lane);
                    S[(size_t)c * LP + 2 * (32 * wi + lane) + eo] = t;
                }
            }
        } else {
            // C/2 consecutive positions (pos = y*WPR+wi for z, z*WPR+wi for y), two classes each
            const int H = C >> 1;
            const size_t pos0 = (size_t)tile * H;
            const int total = 2 * L * H;
            for (int idx = tid; idx < total; idx += kAcThreads) {
                const int pi = idx % H;
                const int rest = idx / H;
                const int col = rest & 1, a = rest >> 1;     // colour, position along the axis
                const size_t pos = pos0 + pi;
                size_t off;
                if (AX == 2) {
                    off = (size_t)a * L * WPR + pos;
                } else {
                    const size_t z = pos / WPR, wi = pos % WPR;
                    off = (z * L + a) * WPR + wi;
                }
                const int p = (col + a) & 1;
                S[(size_t)(2 * pi + p) * LP + a] = __ldg(base + (size_t)col * WPC + off);
            }
        }
        __syncthreads();
        // ------------------------------------------------------------ r = 1 .. L/2 - 1 (and r = 0)
        const int n_tasks = C * (L >> 4);
        for (int task = tid; task < n_tasks; task += kAcThreads) {
            const int c = task & (C - 1), j = task / C;     // C is a power of two
            const uint32_t *col = S + (size_t)c * LP;
            AcStack st[8];
#pragma unroll
            for (int i = 0; i < 8; ++i) st[i] = AcStack{0u, 0u, 0u, 0u};
            uint32_t x[8], ya[8], yb[8];      // window = (ya, yb), then (yb, ya): no moves
            int b = 8 * j;
            ld8(ya, col + b);
#pragma unroll 1
            for (int a0 = 0; a0 < L; a0 += 16) {     // L is a multiple of 64
                b += 8;
                if (b >= L) b -= L;
                ld8(yb, col + b);
                ld8(x, col + a0);
                ac_add64(st, x, ya, yb);
                b += 8;
                if (b >= L) b -= L;
                ld8(ya, col + b);
                ld8(x, col + a0 + 8);
                ac_add64(st, x, yb, ya);
            }
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const int r = 8 * j + i;
                if (r >= 1) atomicAdd(&cnt[r], ac_total(st[i]));
            }
        }
        // ------------------------------------------------------------ r = L/2
        {
            uint32_t acc = 0;
            const int half = L >> 1;
            for (int idx = tid; idx < C * L; idx += kAcThreads) {
                const int c = idx / L, a = idx - c * L;
                int b = a + half;
                if (b >= L) b -= L;
                acc += __popc(S[(size_t)c * LP + a] ^ S[(size_t)c * LP + b]);
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
            if (lane == 0) atomicAdd(&cnt[half], acc);
        }
        if (++since_flush >= flush_every) {
            __syncthreads();
            for (int r = 1 + tid; r < nr; r += kAcThreads) {
                if (cnt[r])
                    atomicAdd(&counts[(size_t)rep * counts_per_replica + 1 + AX * nr + r],
                              (unsigned long long)cnt[r]);
                cnt[r] = 0;
            }
            since_flush = 0;
        }
    }
    __syncthreads();
    for (int r = 1 + tid; r < nr; r += kAcThreads)
        if (cnt[r])
            atomicAdd(&counts[(size_t)rep * counts_per_replica + 1 + AX * nr + r],
                      (unsigned long long)cnt[r]);
}

#undef ISING_CSA

// sequences per tile: C * L = 32768 words where possible
inline int autocorr_tile_sequences(int L)
{
    int c = 1;
    while (2 * c * L <= 32768) c *= 2;
    const int n_seq = L * L / 32;
    if (c > n_seq) c = n_seq;
    if (c < 8) c = 8;
    return c;
}

inline size_t autocorr_smem_bytes(int L, int C)
{
    return ((size_t)C * (L + kAcPad) + (size_t)(L / 2 + 1)) * 4;
}

}  // namespace ising
