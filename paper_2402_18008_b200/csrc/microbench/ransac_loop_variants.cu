// ransac_loop_variants.cu -- measurement tool, not part of libhg: the hot loop of ransac_score_kernel
// (hg_ransac.cu) in isolation, with pieces removed (no classification, no shared-memory loads, scalar FFMA,
// other group sizes / block shapes), to separate FMA-pipe, dispatch and LDS limits.
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -std=c++17 paper_2402_18008_b200/csrc/microbench/ransac_loop_variants.cu -o /tmp/rlv && /tmp/rlv
// Output of one run on the B200 box: profiles/r01c_microbench.md.
#include <cstdio>
#include <cuda_runtime.h>
#include <stdint.h>
__device__ __forceinline__ float2 f2(float v) { return make_float2(v, v); }
__device__ __forceinline__ float2 neg2(float2 a) { return make_float2(-a.x, -a.y); }
struct HC { float h[9]; float Bc; unsigned thr; };
__device__ __forceinline__ float2 score2(const HC& c, float2 sx, float2 sy, float2 ndx, float2 ndy)
{
    const float2 X = __ffma2_rn(f2(c.h[0]), sx, __ffma2_rn(f2(c.h[1]), sy, f2(c.h[2])));
    const float2 Y = __ffma2_rn(f2(c.h[3]), sx, __ffma2_rn(f2(c.h[4]), sy, f2(c.h[5])));
    const float2 W = __ffma2_rn(f2(c.h[6]), sx, __ffma2_rn(f2(c.h[7]), sy, f2(c.h[8])));
    const float2 ex = __ffma2_rn(ndx, W, X);
    const float2 ey = __ffma2_rn(ndy, W, Y);
    const float2 w2 = __ffma2_rn(W, W, f2(-c.Bc));
    const float2 p  = __ffma2_rn(ex, ex, neg2(w2));
    return __ffma2_rn(ey, ey, p);
}
__device__ __forceinline__ float score1(const HC& c, float sx, float sy, float ndx, float ndy)
{
    const float X = fmaf(c.h[0], sx, fmaf(c.h[1], sy, c.h[2]));
    const float Y = fmaf(c.h[3], sx, fmaf(c.h[4], sy, c.h[5]));
    const float W = fmaf(c.h[6], sx, fmaf(c.h[7], sy, c.h[8]));
    const float ex = fmaf(ndx, W, X), ey = fmaf(ndy, W, Y);
    const float w2 = fmaf(W, W, -c.Bc);
    return fmaf(ey, ey, fmaf(ex, ex, -w2));
}
// MODE 0: full (LDS + ffma2 + count + classify); 1: no classify; 2: no LDS (entries loaded once per 4);
// 3: scalar FFMA version full; 4: pure ffma2 (no lds, no count)
template <int MODE, int G, int BLOCK, int MINB>
__global__ void __launch_bounds__(BLOCK, MINB) k(const float4* __restrict__ table, int n_entries, int reps, const float* __restrict__ hyp, int* out)
{
    extern __shared__ float4 tb[];
    for (int i = threadIdx.x; i < 2 * n_entries; i += BLOCK) tb[i] = table[i];
    __syncthreads();
    HC c;
    const int t = blockIdx.x * BLOCK + threadIdx.x;
    for (int i = 0; i < 9; ++i) c.h[i] = hyp[t * 12 + i];
    c.Bc = hyp[t * 12 + 9]; c.thr = __float_as_uint(2.f * c.Bc);
    unsigned n_in = 0, namb = 0;
    for (int r = 0; r < reps; ++r) {
#pragma unroll 1
        for (int k0 = 0; k0 < n_entries; k0 += G) {
            float2 a[G];
            bool amb = false;
            float4 A0, B0;
            if (MODE == 2 || MODE == 4) { A0 = tb[2 * k0]; B0 = tb[2 * k0 + 1]; }
#pragma unroll
            for (int g = 0; g < G; ++g) {
                float4 A, B;
                if (MODE == 2 || MODE == 4) { A = A0; B = B0; A0.x += 1.f; B0.y += 1.f;}
                else { A = tb[2 * (k0 + g)]; B = tb[2 * (k0 + g) + 1]; }
                if (MODE == 3) {
                    a[g].x = score1(c, A.x, A.z, B.x, B.z);
                    a[g].y = score1(c, A.y, A.w, B.y, B.w);
                } else
                    a[g] = score2(c, make_float2(A.x, A.y), make_float2(A.z, A.w), make_float2(B.x, B.y), make_float2(B.z, B.w));
                if (MODE != 4) {
                    n_in += (__float_as_uint(a[g].x) >> 31) + (__float_as_uint(a[g].y) >> 31);
                } else { n_in += __float_as_uint(a[g].x) & __float_as_uint(a[g].y); if (g != G-1) continue; }
                if (MODE == 0 || MODE == 2 || MODE == 3) amb |= (__float_as_uint(a[g].x) <= c.thr) | (__float_as_uint(a[g].y) <= c.thr);
            }
            if (amb) ++namb;
        }
    }
    out[t] = n_in + (namb << 16);
}
template <int MODE, int G, int BLOCK, int MINB>
void run(const char* name, float4* table, float* hyp, int* out, int n_entries, int reps)
{
    const int nthreads = 148 * BLOCK * MINB * 4;
    size_t smem = size_t(n_entries) * 32;
    cudaFuncSetAttribute(k<MODE, G, BLOCK, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    k<MODE, G, BLOCK, MINB><<<nthreads / BLOCK, BLOCK, smem>>>(table, n_entries, reps, hyp, out);
    cudaEventRecord(e0);
    k<MODE, G, BLOCK, MINB><<<nthreads / BLOCK, BLOCK, smem>>>(table, n_entries, reps, hyp, out);
    cudaEventRecord(e1); cudaEventSynchronize(e1);
    float ms; cudaEventElapsedTime(&ms, e0, e1);
    double pairs = double(nthreads) * n_entries * 2 * reps;
    double fma_rate = pairs * 11 / (ms * 1e-3) / (148.0 * 128 * 1.965e9);
    printf("%-28s G=%d block=%d x%d : %.3f ms  %.4g pairs/s  fma-pipe frac %.3f  (%s)\n", name, G, BLOCK, MINB, ms, pairs / ms * 1e3, fma_rate, cudaGetErrorString(cudaGetLastError()));
}
int main()
{
    const int n_entries = 1024, reps = 8;
    float4* table; float* hyp; int* out;
    cudaMalloc(&table, n_entries * 32); cudaMalloc(&hyp, 148 * 1024 * 4 * 12 * 4 * 2); cudaMalloc(&out, 148 * 1024 * 4 * 4 * 2);
    float* ht = new float[n_entries * 8]; for (int i = 0; i < n_entries * 8; ++i) ht[i] = (i * 37 % 640) * 1.f;
    cudaMemcpy(table, ht, n_entries * 32, cudaMemcpyHostToDevice);
    float* hh = new float[148 * 1024 * 4 * 12 * 2]; for (int i = 0; i < 148 * 1024 * 4 * 12 * 2; ++i) hh[i] = ((i * 2654435761u) >> 8) * 1e-9f;
    cudaMemcpy(hyp, hh, 148 * 1024 * 4 * 12 * 4 * 2, cudaMemcpyHostToDevice);
    run<0, 4, 512, 2>("full", table, hyp, out, n_entries, reps);
    run<0, 8, 512, 2>("full", table, hyp, out, n_entries, reps);
    run<0, 2, 512, 2>("full", table, hyp, out, n_entries, reps);
    run<1, 4, 512, 2>("no classify", table, hyp, out, n_entries, reps);
    run<2, 4, 512, 2>("no LDS", table, hyp, out, n_entries, reps);
    run<4, 4, 512, 2>("pure ffma2", table, hyp, out, n_entries, reps);
    run<4, 8, 512, 2>("pure ffma2", table, hyp, out, n_entries, reps);
    run<3, 4, 512, 2>("scalar ffma full", table, hyp, out, n_entries, reps);
    run<3, 2, 512, 2>("scalar ffma full", table, hyp, out, n_entries, reps);
    run<0, 4, 256, 4>("full", table, hyp, out, n_entries, reps);
    run<0, 4, 384, 3>("full 56regs", table, hyp, out, n_entries, reps);
    run<0, 4, 512, 1>("full 1cta", table, hyp, out, n_entries, reps);
    run<0, 8, 512, 1>("full 1cta", table, hyp, out, n_entries, reps);
    run<0, 4, 256, 1>("full 8 warps", table, hyp, out, n_entries, reps);
    return 0;
}
