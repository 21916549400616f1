// Issue-rate microbenchmarks of the integer pipes the sweep and measurement kernels live on
// (LOP3, SHF, IMAD.WIDE, POPC, IADD, IMAD.LO, legacy IMMA u8): the denominators of the ALU
// roofline in DESIGN.md 5.1 / 5.5 are measured with this program on the GPU box, not assumed.
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o /tmp/pipe_rates paper_2305_12161_b200/pipe_rates.cu
//   /tmp/pipe_rates
// 64 resident warps per SM, 8 independent chains per thread; rates are thread-ops per second
// from CUDA events, and per clock per SM at the SM clock the driver reports as maximum.
#include <cstdint>
#include <cstdio>
#include <cuda_runtime.h>

#define ITER 4096
#define NCH 8

template <int OP>
__global__ void __launch_bounds__(256) k(uint32_t *out, uint32_t seed, long long *cyc)
{
    uint32_t v[NCH];
#pragma unroll
    for (int i = 0; i < NCH; ++i) v[i] = seed + threadIdx.x * 977u + i * 131u + blockIdx.x;
    uint32_t a = seed * 3 + threadIdx.x, b = seed * 7 + 1;
    
#pragma unroll 1
    for (int it = 0; it < ITER; ++it) {
#pragma unroll
        for (int i = 0; i < NCH; ++i) {
            if (OP == 0) {   // LOP3 (maj-like, not foldable)
                asm volatile("lop3.b32 %0, %0, %1, %2, 0xE8;" : "+r"(v[i]) : "r"(a), "r"(b));
            } else if (OP == 1) {   // SHF
                asm volatile("shf.l.wrap.b32 %0, %0, %1, 1;" : "+r"(v[i]) : "r"(a));
            } else if (OP == 2) {   // IMAD.WIDE: 32x32->64, use hi^lo
                unsigned long long p;
                asm volatile("mul.wide.u32 %0, %1, %2;" : "=l"(p) : "r"(v[i]), "r"(0xD2511F53u));
                v[i] = (uint32_t)(p >> 32);   // only the multiply chain
                if ((uint32_t)p == 0x12345u) a ^= 1;
            } else if (OP == 3) {   // POPC
                asm volatile("popc.b32 %0, %0;" : "+r"(v[i]));
                v[i] += a;   // keep it non-trivial (adds one IADD per popc)
            } else if (OP == 4) {   // IADD3
                asm volatile("add.u32 %0, %0, %1;" : "+r"(v[i]) : "r"(a));
            } else if (OP == 5) {   // pure POPC chain
                asm volatile("popc.b32 %0, %0;" : "+r"(v[i]));
            } else if (OP == 6) {   // mixed LOP3 + IMAD.WIDE (philox-like round)
                unsigned long long p;
                asm volatile("mul.wide.u32 %0, %1, %2;" : "=l"(p) : "r"(v[i]), "r"(0xD2511F53u));
                asm volatile("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(v[i]) : "r"((uint32_t)(p >> 32)), "r"((uint32_t)p), "r"(b));
            } else if (OP == 7) {   // IMAD (32-bit mad.lo)
                asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(v[i]) : "r"(a), "r"(b));
            }
        }
    }
    
    uint32_t s = a;
#pragma unroll
    for (int i = 0; i < NCH; ++i) s ^= v[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
    (void)cyc;
}

// legacy IMMA m16n8k32 u8: 4 independent accumulator sets per warp
__global__ void __launch_bounds__(256) k_imma(int *out, uint32_t seed, long long *cyc)
{
    uint32_t a0 = seed + threadIdx.x, a1 = a0 * 3, a2 = a0 * 5, a3 = a0 * 7, b0 = a0 * 11, b1 = a0 * 13;
    int d[8][4];
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) d[i][j] = 0;
    
#pragma unroll 1
    for (int it = 0; it < ITER; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i)
            asm volatile(
                "mma.sync.aligned.m16n8k32.row.col.s32.u8.u8.s32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                : "+r"(d[i][0]), "+r"(d[i][1]), "+r"(d[i][2]), "+r"(d[i][3])
                : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
    }
    
    int s = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) s += d[i][j];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
    (void)cyc;
}

template <typename F>
void run(const char *name, F launch, double ops_per_thread_iter, int blocks)
{
    uint32_t *out;
    long long *cyc, hc = 0;
    cudaMalloc(&out, (size_t)blocks * 256 * 4);
    cudaMalloc(&cyc, 8);
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    launch(out, cyc);
    cudaDeviceSynchronize();
    cudaEventRecord(e0);
    launch(out, cyc);
    cudaEventRecord(e1);
    cudaDeviceSynchronize();
    float ms;
    cudaEventElapsedTime(&ms, e0, e1);
    (void)hc;
    int khz = 0, sms = 0;
    cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, 0);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, 0);
    double total = ops_per_thread_iter * ITER * 256.0 * blocks;
    double per_s = total / (ms * 1e-3);
    printf("%-28s %8.3f ms  %10.3e thread-ops/s  %7.1f thread-ops/clk/SM at %d MHz x %d SMs  err=%s\n",
           name, ms, per_s, per_s / (khz * 1e3 * sms), khz / 1000, sms, cudaGetErrorString(cudaGetLastError()));
    cudaFree(out);
    cudaFree(cyc);
}

int main()
{
    const int blocks = 148 * 8;   // 8 CTAs x 256 thr = 64 warps per SM
#define RUN(OP, NAME) run(NAME, [&](uint32_t *o, long long *c) { k<OP><<<blocks, 256>>>(o, 12345u, c); }, NCH, blocks)
    RUN(0, "LOP3");
    RUN(1, "SHF");
    RUN(2, "IMAD.WIDE (+xor lo)");
    RUN(3, "POPC + IADD");
    RUN(4, "IADD");
    RUN(5, "POPC");
    RUN(6, "IMAD.WIDE + LOP3 pair");
    RUN(7, "IMAD.LO");
    run("IMMA.16832.U8 legacy (MACs)", [&](uint32_t *o, long long *c) { k_imma<<<blocks, 256>>>((int *)o, 12345u, c); },
        8.0 * 16 * 8 * 32 / 32.0, blocks);
    return 0;
}
