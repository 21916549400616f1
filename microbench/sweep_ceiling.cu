// Microbenchmark: what the arithmetic of one fused2 step costs on its own, and what each other
// ingredient of the step adds.  Per iteration a thread does what f2_step does for its two rows and two
// colours -- 4 philox_folded calls, 4 rule_group calls, 4 x-neighbour shifts (the device functions of
// csrc/kernels_fused2.cuh) -- on register data, at the kernel's occupancy (256 threads, 2 CTAs per SM).
// Modes add, one at a time: the block barrier per step; the step's shared-memory traffic (8 LDS.128 +
// 2 STS.128 per thread); its global stores (4 STG.128 per thread, streaming or L2-resident); the same
// stores through shared memory and cp.async.bulk.  No bulk loads, no HBM reads.
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -std=c++17 -o /tmp/sweep_ceiling \
//        paper_2305_12161_b200/sweep_ceiling.cu && /tmp/sweep_ceiling
// Results: profiles/r1h_sweep_ceiling.md.
#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>
#include "csrc/kernels_fused2.cuh"
using namespace ising;

template <int MODE>
__global__ void __launch_bounds__(256, 2) k(uint4 *out, int iters, const __grid_constant__ SweepConsts keys)
{
    extern __shared__ __align__(128) uint4 dsm[];
    uint4 (*sm)[512] = reinterpret_cast<uint4 (*)[512]>(dsm);
    uint4 (*ws)[512] = reinterpret_cast<uint4 (*)[512]>(dsm + 4 * 512);
    const int tid = threadIdx.x, lane = tid & 31;
    const int lp = (lane & ~7) | ((lane - 1) & 7), ln = (lane & ~7) | ((lane + 1) & 7);
    uint4 W[3][2], B[3][2];
    for (int i = 0; i < 3; ++i) for (int r = 0; r < 2; ++r) {
        W[i][r] = make_uint4(tid * 7 + i, tid ^ 0x55, i + r, blockIdx.x);
        B[i][r] = make_uint4(tid * 3 + i, tid ^ 0xAA, i * r, blockIdx.x + 1);
    }
    if (MODE >= 2) { for (int i = tid; i < 4 * 512; i += 256) (&sm[0][0])[i] = make_uint4(i, i * 3, i * 5, i * 7); __syncthreads(); }
    uint32_t q = blockIdx.x * 1000003u + tid;
#pragma unroll 1
    for (int it = 0; it < iters; it += 2) {
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            uint4 Wym, Wyp, Bo0, Bo1, Bym, Byp;
            if (MODE >= 2) {
                const uint4 *p = sm[(it + u) & 3];
                W[2][0] = p[tid]; W[2][1] = p[tid + 256]; Bo0 = p[(tid + 8) & 511]; Bo1 = p[(tid + 264) & 511];
                Wym = p[(tid + 504) & 511]; Wyp = p[(tid + 16) & 511];
            } else { Wym = W[0][1]; Wyp = W[2][0]; Bo0 = B[0][0]; Bo1 = B[0][1]; }
            const uint4 r0 = philox_folded<0>(q, keys), r1 = philox_folded<0>(q + 8, keys);
            const uint4 x0 = u ? xneigh<1>(W[1][0], lp, ln) : xneigh<0>(W[1][0], lp, ln);
            const uint4 x1 = u ? xneigh<0>(W[1][1], lp, ln) : xneigh<1>(W[1][1], lp, ln);
            B[2][0] = rule_group(Bo0, r0, W[1][0], x0, Wym, W[1][1], W[0][0], W[2][0]);
            B[2][1] = rule_group(Bo1, r1, W[1][1], x1, W[1][0], Wyp, W[0][1], W[2][1]);
            if (MODE >= 2) { uint4 *p = sm[(it + u + 2) & 3]; p[tid] = B[2][0]; p[tid + 256] = B[2][1];
                             const uint4 *pr = sm[(it + u + 1) & 3]; Bym = pr[(tid + 504) & 511]; Byp = pr[(tid + 16) & 511]; }
            else { Bym = B[0][1]; Byp = B[2][0]; }
            const uint4 s0 = philox_folded<1>(q + 1, keys), s1 = philox_folded<1>(q + 9, keys);
            const uint4 y0 = u ? xneigh<1>(B[1][0], lp, ln) : xneigh<0>(B[1][0], lp, ln);
            const uint4 y1 = u ? xneigh<0>(B[1][1], lp, ln) : xneigh<1>(B[1][1], lp, ln);
            const uint4 n0 = rule_group(W[0][0], s0, B[1][0], y0, Bym, B[1][1], B[0][0], B[2][0]);
            const uint4 n1 = rule_group(W[0][1], s1, B[1][1], y1, B[1][0], Byp, B[0][1], B[2][1]);
            if (MODE == 5) {
                uint4 *p = ws[(it + u) & 3]; p[tid] = n0; p[tid + 256] = n1;
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            } else
            if (MODE >= 3) { uint4 *d = out + ((size_t)blockIdx.x * 256 + tid) * 4 + (size_t)((it + u) & (MODE == 4 ? 3 : 255)) * gridDim.x * 1024;
                             d[0] = B[2][0]; d[1] = B[2][1]; d[2] = n0; d[3] = n1; }
            // rotate windows (values stay data dependent)
            W[0][0] = W[1][0]; W[0][1] = W[1][1]; W[1][0] = MODE >= 2 ? W[2][0] : n0; W[1][1] = MODE >= 2 ? W[2][1] : n1;
            if (MODE < 2) { W[2][0] = n1; W[2][1] = n0; }
            else { W[1][0].x ^= n0.x ^ n0.y; W[1][0].z ^= n0.z ^ n0.w; W[1][1].y ^= n1.y ^ n1.x; W[1][1].w ^= n1.z ^ n1.w; }
            B[0][0] = B[1][0]; B[0][1] = B[1][1]; B[1][0] = B[2][0]; B[1][1] = B[2][1];
            q += 4096;
            if (MODE >= 1) __syncthreads();
            if (MODE == 5 && tid == 0) {
                uint4 *d = out + (size_t)blockIdx.x * 1024 + (size_t)((it + u) & 255) * gridDim.x * 1024;
                asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(d), "r"(smem_u32(sm[(it + u + 2) & 3])), "r"(8192) : "memory");
                asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(d + 512), "r"(smem_u32(ws[(it + u) & 3])), "r"(8192) : "memory");
                asm volatile("cp.async.bulk.commit_group;" ::: "memory");
                asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory");
            }
        }
    }
    uint4 r = W[0][0];
    r.x ^= W[1][1].y ^ B[1][0].z ^ B[0][1].w ^ W[2][0].x;
    if (MODE == 5 && tid == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
    if (r.x == 0x12345678u) out[tid] = r;
}

template <int MODE> void run(const char *name, uint4 *out, int ctas, int iters)
{
    SweepConsts keys = make_sweep_consts(12345, 7, 0);
    cudaFuncSetAttribute(k<MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, 65536);
    k<MODE><<<ctas, 256, 65536>>>(out, 16, keys);
    cudaEvent_t a, b; cudaEventCreate(&a); cudaEventCreate(&b);
    cudaEventRecord(a);
    k<MODE><<<ctas, 256, 65536>>>(out, iters, keys);
    cudaEventRecord(b); cudaEventSynchronize(b);
    float ms; cudaEventElapsedTime(&ms, a, b);
    const double sites = (double)ctas * 256 * iters * 512.0;     // 4 groups x 128 sites per thread-iteration
    printf("%-34s %8.3f ms  %9.0f site-updates/ns  (%s)\n", name, ms, sites / (ms * 1e6), cudaGetErrorString(cudaGetLastError()));
}

int main()
{
    uint4 *out; cudaMalloc(&out, (size_t)296 * 1024 * 1024 * 16 + (1 << 20));
    for (int ctas : {296, 592}) {
        printf("CTAs %d (256 threads, 2 resident per SM)\n", ctas);
        run<0>("arithmetic only", out, ctas, 2000);
        run<1>("+ __syncthreads per step", out, ctas, 2000);
        run<2>("+ shared-memory loads/stores", out, ctas, 2000);
        run<3>("+ global stores (64 B/thread/step)", out, ctas, 2000);
        run<4>("  same stores, L2-resident target", out, ctas, 2000);
        run<5>("  stores via smem + bulk async copy", out, ctas, 2000);
    }
    return 0;
}
