// Cost of one barrier across the CTAs that would share ONE small lattice (configs 1-2):
// a half-sweep of an L = 256 lattice on more than the 16 SMs of one thread-block cluster needs a
// barrier over all its CTAs twice per sweep (colour 1 sees the updated colour 0).
//   * cluster barrier (barrier.cluster arrive/wait, hardware) for cluster sizes 2..16,
//   * grid barrier (cooperative groups grid.sync(), through L2) for 16..148 CTAs,
// each timed over many rounds with nothing else in the loop: ns per barrier.
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -std=c++17 -rdc=true -o /tmp/grid_barrier microbench/grid_barrier.cu
//   /tmp/grid_barrier
#include <cooperative_groups.h>
#include <cstdio>
#include <cuda_runtime.h>

namespace cg = cooperative_groups;

constexpr int kRounds = 20000;

__global__ void __launch_bounds__(256) grid_sync_kernel(int *sink)
{
    cg::grid_group grid = cg::this_grid();
    int acc = threadIdx.x;
    for (int i = 0; i < kRounds; ++i) {
        grid.sync();
        acc += i;
    }
    if (acc == -1) *sink = acc;
}

__global__ void __launch_bounds__(256) cluster_sync_kernel(int *sink)
{
    int acc = threadIdx.x;
    for (int i = 0; i < kRounds; ++i) {
        asm volatile("barrier.cluster.arrive.release.aligned;\nbarrier.cluster.wait.acquire.aligned;\n" ::: "memory");
        acc += i;
    }
    if (acc == -1) *sink = acc;
}

__global__ void __launch_bounds__(256) block_sync_kernel(int *sink)
{
    int acc = threadIdx.x;
    for (int i = 0; i < kRounds; ++i) {
        __syncthreads();
        acc += i;
    }
    if (acc == -1) *sink = acc;
}

static float time_launch(cudaLaunchConfig_t &cfg, void *fn, int *sink, bool coop)
{
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    void *args[] = {&sink};
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {
        cudaEventRecord(e0, 0);
        cudaError_t e = coop ? cudaLaunchCooperativeKernel(fn, cfg.gridDim, cfg.blockDim, args, 0, 0)
                             : cudaLaunchKernelExC(&cfg, fn, args);
        cudaEventRecord(e1, 0);
        if (e != cudaSuccess || cudaEventSynchronize(e1) != cudaSuccess) {
            printf("  launch failed: %s\n", cudaGetErrorString(e != cudaSuccess ? e : cudaGetLastError()));
            cudaGetLastError();
            return -1.f;
        }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best) best = ms;
    }
    return best;
}

int main()
{
    int *sink = nullptr;
    cudaMalloc(&sink, 4);
    cudaDeviceProp prop;
    cudaGetDeviceProperties(&prop, 0);
    printf("%s, %d SMs\n", prop.name, prop.multiProcessorCount);
    {
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(prop.multiProcessorCount);
        cfg.blockDim = dim3(256);
        const float ms = time_launch(cfg, (void *)block_sync_kernel, sink, false);
        printf("__syncthreads, 256 threads           : %8.1f ns per barrier\n", ms * 1e6f / kRounds);
    }
    cudaFuncSetAttribute(cluster_sync_kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
    for (int cs = 2; cs <= 16; cs *= 2) {
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(cs);
        cfg.blockDim = dim3(256);
        cudaLaunchAttribute at;
        at.id = cudaLaunchAttributeClusterDimension;
        at.val.clusterDim.x = cs;
        at.val.clusterDim.y = 1;
        at.val.clusterDim.z = 1;
        cfg.attrs = &at;
        cfg.numAttrs = 1;
        const float ms = time_launch(cfg, (void *)cluster_sync_kernel, sink, false);
        printf("cluster barrier, %2d CTAs (1 cluster)  : %8.1f ns per barrier\n", cs, ms * 1e6f / kRounds);
    }
    for (int n : {16, 32, 64, 128, 148}) {
        if (n > prop.multiProcessorCount) continue;
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(n);
        cfg.blockDim = dim3(256);
        const float ms = time_launch(cfg, (void *)grid_sync_kernel, sink, true);
        printf("grid.sync(), %3d CTAs (one per SM)    : %8.1f ns per barrier\n", n, ms * 1e6f / kRounds);
    }
    cudaFree(sink);
    return 0;
}
