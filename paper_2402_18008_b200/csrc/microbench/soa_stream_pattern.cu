// soa_stream_pattern.cu -- measurement tool, not part of libhg: the memory pattern of solve_soa_kernel without its
// arithmetic (16 input planes read, 9 output planes written, 128-bit accesses, 2^26 elements per plane), against
// variants of the pattern, to tell what part of the gap to the datasheet bandwidth belongs to the pattern.
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -std=c++17 paper_2402_18008_b200/csrc/microbench/soa_stream_pattern.cu -o /tmp/ssp && /tmp/ssp
// Output of one run on the B200 box: profiles/r01c_microbench.md.
#include <cstdio>
#include <cuda_runtime.h>
#include <stdint.h>

// TILES consecutive 4 KB tiles per plane and CTA (TILES = 1 is the production pattern).
template <int NIN, int NOUT, int TILES>
__global__ void __launch_bounds__(256) pattern(const float4* __restrict__ in, float4* __restrict__ out, int64_t nvec)
{
    for (int t = 0; t < TILES; ++t) {
        const int64_t i = (static_cast<int64_t>(blockIdx.x) * TILES + t) * 256 + threadIdx.x;
        if (i >= nvec) return;
        float4 v[NIN];
#pragma unroll
        for (int k = 0; k < NIN; ++k) v[k] = __ldcs(in + k * nvec + i);
        float4 acc = v[0];
#pragma unroll
        for (int k = 1; k < NIN; ++k) { acc.x += v[k].x; acc.y += v[k].y; acc.z += v[k].z; acc.w += v[k].w; }
#pragma unroll
        for (int k = 0; k < NOUT; ++k) { acc.x += 1.f; __stcs(out + k * nvec + i, acc); }
    }
}

template <int NIN, int NOUT, int TILES>
void run(const char* name, const float4* in, float4* out, int64_t nvec)
{
    const int64_t blocks = (nvec + 256 * TILES - 1) / (256 * TILES);
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    for (int w = 0; w < 3; ++w) pattern<NIN, NOUT, TILES><<<(unsigned)blocks, 256>>>(in, out, nvec);
    cudaEventRecord(e0);
    for (int r = 0; r < 10; ++r) pattern<NIN, NOUT, TILES><<<(unsigned)blocks, 256>>>(in, out, nvec);
    cudaEventRecord(e1); cudaEventSynchronize(e1);
    float ms; cudaEventElapsedTime(&ms, e0, e1); ms /= 10;
    printf("%-44s %.4f ms  %.1f GB/s  (%s)\n", name, ms, double(nvec) * 16 * (NIN + NOUT) / ms / 1e6, cudaGetErrorString(cudaGetLastError()));
}

int main()
{
    const int64_t n = int64_t(1) << 26, nvec = n / 4;
    float4 *in, *out;
    cudaMalloc(&in, size_t(n) * 4 * 16); cudaMalloc(&out, size_t(n) * 4 * 16);
    cudaMemset(in, 0, size_t(n) * 4 * 16);
    run<16, 9, 1>("16 planes in, 9 out (production pattern)", in, out, nvec);
    run<16, 9, 4>("16 in, 9 out, 4 tiles per CTA", in, out, nvec);
    run<8, 9, 1>("8 in, 9 out (rect / SK pattern)", in, out, nvec);
    run<16, 0, 1>("16 in, read only", in, out, nvec);
    run<1, 9, 1>("1 in, 9 out (write heavy)", in, out, nvec);
    run<1, 1, 1>("1 in, 1 out (copy)", in, out, nvec);
    run<4, 4, 1>("4 in, 4 out", in, out, nvec);
    run<12, 13, 1>("12 in, 13 out", in, out, nvec);
    return 0;
}
