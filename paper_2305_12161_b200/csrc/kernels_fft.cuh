// The paper's own correlation estimator: eq. (7) PAPER.md:128,
//     mean_i s_i s_{i+k} = [F^-1(|F s|^2)]_k,
// with the 3-D real-to-complex transform in place ("in-place real-data DFT ... eight bytes per
// site"), then the radial average "over the three-dimensional correlation matrix"
// and the structure factor S(k) = |F s|^2 / N.
//
// The two transforms are cuFFT library calls (fp64 D2Z / Z2D, in place); everything around them
// is here:
//   unpack_real_kernel   packed bits (D3) -> +-1.0 in the padded in-place layout [z][y][L+2]
//   power_kernel         |F s|^2 in place, and its radial sums over |k| bins (S(k))
//   radial_kernel        P(d) = llrint(F^-1(...)[d] / N): the transform of +-1 data is an integer
//                        up to round-off (< 1e-3 at L = 2048), so the correlation matrix is
//                        recovered EXACTLY and its radial sums are integer sums
// Radial bins (reading D12): minimal image, bin b = nearest integer to |d|, decided in integers:
// (2b-1)^2 <= 4|d|^2 < (2b+1)^2; bins 0..L/2.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace ising {

__device__ __forceinline__ int radial_bin_dev(const int L, int dx, int dy, int dz)
{
    const int h = L >> 1;
    if (dx > h) dx -= L;
    if (dy > h) dy -= L;
    if (dz > h) dz -= L;
    const long long n4 = 4ll * ((long long)dx * dx + (long long)dy * dy + (long long)dz * dz);
    long long b = (long long)((sqrt((double)n4) + 1.0) * 0.5);       // guess, then exact fix-up
    while ((2 * b + 1) * (2 * b + 1) <= n4) ++b;
    while (b > 0 && (2 * b - 1) * (2 * b - 1) > n4) --b;
    return (int)b;
}

// one warp = one (z, y, wi): lane j writes the sites x = 2k, 2k+1 (k = 32 wi + j) as a double2
__global__ void __launch_bounds__(256)
unpack_real_kernel(const uint32_t *__restrict__ state, double *__restrict__ buf, const int L)
{
    const int WPR = L >> 6, LP = L + 2;
    const size_t WPC = (size_t)L * L * WPR;
    const int lane = threadIdx.x & 31;
    const size_t n_warps = WPC;                              // one per word position of a colour
    for (size_t w = ((size_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5; w < n_warps;
         w += ((size_t)gridDim.x * blockDim.x) >> 5) {
        const int wi = (int)(w % WPR);
        const size_t row = w / WPR;
        const int y = (int)(row % L), z = (int)(row / L);
        const uint32_t w0 = state[w], w1 = state[WPC + w];   // colour 0 / colour 1 word
        // colour c holds x = 2k + ((y+z+c)&1): the even-x sites are in colour (y+z)&1
        const uint32_t we = ((y + z) & 1) ? w1 : w0, wo = ((y + z) & 1) ? w0 : w1;
        double2 v;
        v.x = ((we >> lane) & 1u) ? 1.0 : -1.0;
        v.y = ((wo >> lane) & 1u) ? 1.0 : -1.0;
        *reinterpret_cast<double2 *>(buf + row * LP + 2 * (32 * wi + lane)) = v;
    }
}

// in-place: (re, im) -> (re^2 + im^2, 0); radial sums of the power over the k bins, with weight 2
// for the half-spectrum elements whose Hermitian partner is not stored (0 < kx < L/2)
__global__ void __launch_bounds__(256)
power_kernel(double2 *__restrict__ buf, double *__restrict__ s_sum, const int L)
{
    extern __shared__ double pw_smem[];                      // [L/2 + 1]
    const int H = L / 2 + 1;
    for (int b = threadIdx.x; b < H; b += blockDim.x) pw_smem[b] = 0.0;
    __syncthreads();
    const size_t n = (size_t)L * L * H;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n;
         i += (size_t)gridDim.x * blockDim.x) {
        const int kx = (int)(i % H);
        const size_t r = i / H;
        const int ky = (int)(r % L), kz = (int)(r / L);
        const double2 c = buf[i];
        const double p = c.x * c.x + c.y * c.y;
        buf[i] = make_double2(p, 0.0);
        const int b = radial_bin_dev(L, kx, ky, kz);
        if (b < H) atomicAdd(&pw_smem[b], (kx == 0 || kx == L / 2) ? p : 2.0 * p);
    }
    __syncthreads();
    for (int b = threadIdx.x; b < H; b += blockDim.x)
        if (pw_smem[b] != 0.0) atomicAdd(&s_sum[b], pw_smem[b]);
}

// radial sums of the integer correlation matrix P(d) = llrint(buf[d] / N) and the bin populations
__global__ void __launch_bounds__(256)
radial_kernel(const double *__restrict__ buf, unsigned long long *__restrict__ p_sum,
              unsigned long long *__restrict__ shell, unsigned long long *__restrict__ max_dev_bits, const int L)
{
    extern __shared__ unsigned long long rd_smem[];          // [2][L/2 + 1]
    const int H = L / 2 + 1, LP = L + 2;
    for (int b = threadIdx.x; b < 2 * H; b += blockDim.x) rd_smem[b] = 0ull;
    __syncthreads();
    const double inv_n = 1.0 / ((double)L * (double)L * (double)L);
    const size_t n = (size_t)L * L * L;
    double dev = 0.0;                                        // exactness margin of D12: max |v/N - P|
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n;
         i += (size_t)gridDim.x * blockDim.x) {
        const int dx = (int)(i % L);
        const size_t r = i / L;
        const int dy = (int)(r % L), dz = (int)(r / L);
        const int b = radial_bin_dev(L, dx, dy, dz);
        if (b < H) {
            const double v = buf[r * LP + dx] * inv_n;
            const long long P = llrint(v);
            dev = fmax(dev, fabs(v - (double)P));
            atomicAdd(&rd_smem[b], (unsigned long long)P);   // two's complement: sums of signed values
            atomicAdd(&rd_smem[H + b], 1ull);
        }
    }
    __syncthreads();
    for (int b = threadIdx.x; b < H; b += blockDim.x) {
        if (rd_smem[b]) atomicAdd(&p_sum[b], rd_smem[b]);
        if (rd_smem[H + b]) atomicAdd(&shell[b], rd_smem[H + b]);
    }
    for (int o = 16; o; o >>= 1) dev = fmax(dev, __shfl_xor_sync(0xffffffffu, dev, o));
    // non-negative doubles order like their bit patterns
    if ((threadIdx.x & 31) == 0 && dev > 0.0) atomicMax(max_dev_bits, (unsigned long long)__double_as_longlong(dev));
}

}  // namespace ising
