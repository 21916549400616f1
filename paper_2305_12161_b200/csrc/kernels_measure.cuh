// Measurement reductions a6-a8 (D8): N_up and the antiparallel-pair counts
//   A_mu(r) = #{sites i : s_i != s_{i + r e_mu}},  mu = x,y,z,  r = 1..L/2, periodic
// (eq. (2) PAPER.md:43 reduced to integer counts; the axis-averaged estimator is
// BASELINE.json's, the paper itself goes through an FFT).
// Everything is XOR + popcount on the packed words, reduced with warp shuffles and one
// 64-bit atomic per (warp, r).
//
// Which packed bit is the partner of a site (derived from D3):
//   y or z displacement r: same word position in row y+r (plane z+r); same colour array if
//     r is even, the other colour if r is odd.
//   x displacement r: same row; r even: same colour, k' = k + r/2;
//     r odd: other colour, k' = k + (r-1)/2 + o, o = (y+z+c)&1 of the origin site's colour c.
//     k' is taken mod L/2, i.e. a rotation of the row's L/2 bits.
//
// counts layout per replica: [0] = N_up, [1 + mu*(L/2+1) + r] = A_mu(r).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace ising {

__device__ __forceinline__ uint32_t warp_sum(uint32_t v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

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

// ---- A_y(r), A_z(r) --------------------------------------------------------
// One block = one "column tile": a fixed z (AX = 1) or fixed y (AX = 2), WX consecutive
// words of the row (WX a power of two, ragged tail zero-padded), all L positions along the
// measured axis, both colours: T[2][L][WX] in shared memory.  Warp w takes the
// displacements r = 1+w, 1+w+nw, ...; its lanes stride over the tile.
template <int AX>
__global__ void __launch_bounds__(512)
measure_yz_kernel(const uint32_t *__restrict__ state, unsigned long long *__restrict__ counts,
                  int L, int WX, int tiles_per_row, int counts_per_replica)
{
    extern __shared__ uint32_t T[];
    const int WPR = L >> 6;
    const size_t WPC = (size_t)L * L * WPR;
    const int rep = blockIdx.y;
    const int fixed = blockIdx.x / tiles_per_row;
    const int wi0 = (blockIdx.x % tiles_per_row) * WX;
    const int LW = L * WX;
    const uint32_t *base = state + (size_t)rep * 2 * WPC;
    for (int idx = threadIdx.x; idx < 2 * LW; idx += blockDim.x) {
        const int c = idx / LW;
        const int rem = idx - c * LW;
        const int a = rem / WX;
        const int j = rem - a * WX;
        const size_t row = (AX == 1) ? (size_t)fixed * L + a : (size_t)a * L + fixed;
        T[idx] = (wi0 + j < WPR) ? base[(size_t)c * WPC + row * WPR + wi0 + j] : 0u;
    }
    __syncthreads();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nw = blockDim.x >> 5;
    const int nr = L / 2 + 1;
    for (int r = 1 + warp; r <= L / 2; r += nw) {
        uint32_t acc = 0;
        const int shift = r * WX;
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            const uint32_t *own = T + c * LW;
            const uint32_t *par = T + ((c ^ (r & 1)) * LW);
            for (int idx = lane; idx < LW; idx += 32) {
                int q = idx + shift;
                if (q >= LW) q -= LW;
                acc += __popc(own[idx] ^ par[q]);
            }
        }
        acc = warp_sum(acc);
        if (lane == 0)
            atomicAdd(&counts[(size_t)rep * counts_per_replica + 1 + AX * nr + r],
                      (unsigned long long)acc);
    }
}

// ---- A_x(r) ---------------------------------------------------------------
// One block = RX consecutive rows (row = z*L + y), both colours: T[2][RX][WPR].
__global__ void __launch_bounds__(512)
measure_x_kernel(const uint32_t *__restrict__ state, unsigned long long *__restrict__ counts,
                 int L, int RX, int counts_per_replica)
{
    extern __shared__ uint32_t T[];
    const int WPR = L >> 6;
    const size_t WPC = (size_t)L * L * WPR;
    const int rep = blockIdx.y;
    const size_t row0 = (size_t)blockIdx.x * RX;
    const int RW = RX * WPR;
    const uint32_t *base = state + (size_t)rep * 2 * WPC;
    for (int idx = threadIdx.x; idx < 2 * RW; idx += blockDim.x) {
        const int c = idx / RW;
        const int rem = idx - c * RW;
        T[idx] = base[(size_t)c * WPC + row0 * WPR + rem];
    }
    __syncthreads();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nw = blockDim.x >> 5;
    const int nr = L / 2 + 1;
    for (int r = 1 + warp; r <= L / 2; r += nw) {
        uint32_t acc = 0;
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            const int src = (r & 1) ? 1 - c : c;
            for (int idx = lane; idx < RW; idx += 32) {
                const int rr = idx / WPR;
                const int wi = idx - rr * WPR;
                int s;
                if (r & 1) {
                    const size_t rowg = row0 + rr;
                    const int y = (int)(rowg % L), z = (int)(rowg / L);
                    s = (r - 1) / 2 + ((y + z + c) & 1);
                } else {
                    s = r / 2;
                }
                int a = wi + (s >> 5);
                if (a >= WPR) a -= WPR;
                int b = a + 1;
                if (b >= WPR) b -= WPR;
                const uint32_t *srow = T + src * RW + rr * WPR;
                const uint32_t v = __funnelshift_r(srow[a], srow[b], s & 31);
                acc += __popc(T[c * RW + idx] ^ v);
            }
        }
        acc = warp_sum(acc);
        if (lane == 0)
            atomicAdd(&counts[(size_t)rep * counts_per_replica + 1 + 0 * nr + r],
                      (unsigned long long)acc);
    }
}

}  // namespace ising
