// fma_pipe.cu -- measurement tool, not part of libhg: FP32 pipe rates behind DESIGN.md's "alu" roofline
// (FFMA vs packed FFMA2 in its operand forms, and FFMA2 interleaved with ALU-pipe and LDS.128 instructions).
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -std=c++17 paper_2402_18008_b200/csrc/microbench/fma_pipe.cu -o /tmp/fma_pipe && /tmp/fma_pipe
// Output of one run on the B200 box: profiles/r01c_microbench.md.
#include <cstdio>
#include <cuda_runtime.h>
// MODE 0: FFMA2 vec*vec+vec ; 1: FFMA2 scalar-broadcast*vec+vec ; 2: scalar FFMA ; 3: FFMA2 + interleaved LEA.HI every 4; 4: FFMA2 + LDS.128 broadcast every 6
template <int MODE, int ACC>
__global__ void __launch_bounds__(512, 2) k(float* out, int iters, long long* cyc)
{
    __shared__ float4 sm[64];
    if (threadIdx.x < 64) sm[threadIdx.x] = make_float4(threadIdx.x, 1, 2, 3);
    __syncthreads();
    float2 a[ACC]; float s[ACC]; 
    for (int i = 0; i < ACC; ++i) { a[i] = make_float2(threadIdx.x * 1e-3f + i, i * 0.5f); s[i] = a[i].x; }
    float2 m = make_float2(1.0001f, 0.9999f); float ms = 1.0001f; float2 c = make_float2(1e-3f, 2e-3f);
    unsigned cnt = 0;
    long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < ACC; ++i) {
            if (MODE == 0) a[i] = __ffma2_rn(a[i], m, c);
            else if (MODE == 1) a[i] = __ffma2_rn(make_float2(ms, ms), a[i], c);
            else if (MODE == 2) { s[i] = fmaf(s[i], ms, 1e-3f); }
            else if (MODE == 3) { a[i] = __ffma2_rn(a[i], m, c); if ((i & 3) == 3) cnt += __float_as_uint(a[i].x) >> 31; }
            else if (MODE == 4) { a[i] = __ffma2_rn(a[i], m, c); if ((i % 6) == 5) { float4 v = sm[(it + i) & 63]; c.x = v.x; } }
            else if (MODE == 5) { a[i] = __ffma2_rn(a[i], m, c); if ((i & 1) == 1) cnt += __float_as_uint(a[i].x) >> 31; }
        }
    }
    long long t1 = clock64();
    float r = 0; for (int i = 0; i < ACC; ++i) r += a[i].x + a[i].y + s[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = r + cnt;
    if (threadIdx.x == 0 && blockIdx.x == 0) *cyc = t1 - t0;
}
template <int MODE, int ACC> void run(const char* name, float* out, long long* cyc)
{
    const int iters = 65536;
    k<MODE, ACC><<<148 * 2, 512>>>(out, iters, cyc);
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    cudaEventRecord(e0);
    k<MODE, ACC><<<148 * 2, 512>>>(out, iters, cyc);
    cudaEventRecord(e1); cudaEventSynchronize(e1);
    float ms; cudaEventElapsedTime(&ms, e0, e1);
    long long c; cudaMemcpy(&c, cyc, 8, cudaMemcpyDeviceToHost);
    double fma_per_thread = double(iters) * ACC * (MODE == 2 ? 1 : 2);
    double per_clk_sm = fma_per_thread * 1024 / double(c);
    printf("%-34s ACC=%2d  %.3f ms  lanes/clk/SM@1965MHz = %.1f (clock64: %.1f, %.0f MHz)\n", name, ACC, ms, fma_per_thread * 1024 / (ms * 1e-3 * 1.965e9), per_clk_sm, c / (ms * 1e3));
}
int main()
{
    float* out; long long* cyc; cudaMalloc(&out, 148 * 2 * 512 * 4); cudaMalloc(&cyc, 8);
    run<0, 8>("FFMA2 vec", out, cyc); run<0, 16>("FFMA2 vec", out, cyc);
    run<1, 8>("FFMA2 scalar-bcast", out, cyc); run<1, 16>("FFMA2 scalar-bcast", out, cyc);
    run<2, 8>("FFMA", out, cyc); run<2, 16>("FFMA", out, cyc);
    run<3, 16>("FFMA2 + LEA.HI 1:4", out, cyc);
    run<5, 16>("FFMA2 + LEA.HI 1:2", out, cyc);
    run<4, 12>("FFMA2 + LDS.128 1:6", out, cyc);
    return 0;
}
