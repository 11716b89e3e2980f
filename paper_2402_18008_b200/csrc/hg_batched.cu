// hg_batched.cu -- streaming ACA / SKS solve: hg_aca_batched, hg_sks_batched (+ _host forms).
//
// Hot path rows a-A0..a-A6 and a-S1..a-S7 of SURVEY.md section 8(a).  One thread solves V
// homographies (V = 4: 16 independent 128-bit loads in flight per thread, 9 128-bit stores);
// everything between the loads and the stores lives in registers.  HBM-bound: 64 B read +
// 36 B written per homography.
#include "hg_device.cuh"
#include "hg_host.h"

namespace hg {

constexpr int kBlock = 256;

// ------------------------------------------------------------------------------------------
// SoA: src/dst = float[8][stride], H = float[9][stride]; thread t handles sets [t*V, t*V+V).
// `stride` is the plane stride (== n for the public entry points; the host pipeline passes
// chunk-local planes).  Requires (n % V == 0) and 4*V-byte aligned planes.
// ------------------------------------------------------------------------------------------
template <int METHOD, class T, int V>
__global__ void __launch_bounds__(kBlock)
solve_soa_kernel(const float* __restrict__ src, const float* __restrict__ dst,
                 float* __restrict__ H, int64_t n_vec, int64_t stride, int norm)
{
    const int64_t t = static_cast<int64_t>(blockIdx.x) * kBlock + threadIdx.x;
    if (t >= n_vec) return;
    const int64_t off = t * V;

    Vec<V> s[8], d[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) s[k] = ld_stream<V>(src + k * stride + off);
#pragma unroll
    for (int k = 0; k < 8; ++k) d[k] = ld_stream<V>(dst + k * stride + off);

    Vec<V> h[9];
#pragma unroll
    for (int v = 0; v < V; ++v) {
        T sv[8], dv[8], Hv[9];
#pragma unroll
        for (int k = 0; k < 8; ++k) { sv[k] = static_cast<T>(s[k].v[v]); dv[k] = static_cast<T>(d[k].v[v]); }
        solve<METHOD, T>(sv, dv, Hv);
        normalise<T>(Hv, norm);
#pragma unroll
        for (int k = 0; k < 9; ++k) h[k].v[v] = static_cast<float>(Hv[k]);
    }
#pragma unroll
    for (int k = 0; k < 9; ++k) st_stream<V>(H + k * stride + off, h[k]);
}

// ------------------------------------------------------------------------------------------
// AoS: src/dst = float[n][8], H = float[n][9].  Each thread reads its own 2 x 32 B (two 128-bit
// loads per array; the pair of loads of a warp covers whole lines, served by L1), and the
// 36-byte H records are transposed through shared memory so the block writes one contiguous,
// 128-bit-vectorised span.
// ------------------------------------------------------------------------------------------
template <int METHOD, class T>
__global__ void __launch_bounds__(kBlock)
solve_aos_kernel(const float* __restrict__ src, const float* __restrict__ dst,
                 float* __restrict__ H, int64_t n, int norm)
{
    __shared__ __align__(16) float stage[kBlock * 9];
    const int64_t base = static_cast<int64_t>(blockIdx.x) * kBlock;
    const int64_t i = base + threadIdx.x;
    if (i < n) {
        const float4* sp = reinterpret_cast<const float4*>(src + 8 * i);
        const float4* dp = reinterpret_cast<const float4*>(dst + 8 * i);
        const float4 s0 = __ldg(sp), s1 = __ldg(sp + 1), d0 = __ldg(dp), d1 = __ldg(dp + 1);
        const T sv[8] = { T(s0.x), T(s0.y), T(s0.z), T(s0.w), T(s1.x), T(s1.y), T(s1.z), T(s1.w) };
        const T dv[8] = { T(d0.x), T(d0.y), T(d0.z), T(d0.w), T(d1.x), T(d1.y), T(d1.z), T(d1.w) };
        T Hv[9];
        solve<METHOD, T>(sv, dv, Hv);
        normalise<T>(Hv, norm);
#pragma unroll
        for (int k = 0; k < 9; ++k) stage[threadIdx.x * 9 + k] = static_cast<float>(Hv[k]);   // stride 9: conflict-free
    }
    __syncthreads();
    const int64_t rem = n - base;
    const int cnt = static_cast<int>(rem < kBlock ? rem : kBlock) * 9;      // floats this block owns
    float* out = H + 9 * base;                                              // 9*256*4 B per block: 16 B aligned
    const int n4 = cnt >> 2;
    for (int j = threadIdx.x; j < n4; j += kBlock)
        __stcs(reinterpret_cast<float4*>(out) + j, reinterpret_cast<const float4*>(stage)[j]);
    for (int j = (n4 << 2) + threadIdx.x; j < cnt; j += kBlock) out[j] = stage[j];
}

template <int METHOD, class T>
static int launch_soa(const float* src, const float* dst, float* H, int64_t n, int64_t stride,
                      int norm, cudaStream_t st)
{
    const bool vec4 = (n % 4 == 0) && (stride % 4 == 0);
    if (vec4) {
        const int64_t nv = n / 4;
        const int64_t blocks = (nv + kBlock - 1) / kBlock;
        solve_soa_kernel<METHOD, T, 4><<<static_cast<unsigned>(blocks), kBlock, 0, st>>>(src, dst, H, nv, stride, norm);
    } else {
        const int64_t blocks = (n + kBlock - 1) / kBlock;
        solve_soa_kernel<METHOD, T, 1><<<static_cast<unsigned>(blocks), kBlock, 0, st>>>(src, dst, H, n, stride, norm);
    }
    return launch_status();
}

template <int METHOD, class T>
static int launch_aos(const float* src, const float* dst, float* H, int64_t n, int norm, cudaStream_t st)
{
    const int64_t blocks = (n + kBlock - 1) / kBlock;
    solve_aos_kernel<METHOD, T><<<static_cast<unsigned>(blocks), kBlock, 0, st>>>(src, dst, H, n, norm);
    return launch_status();
}

template <int METHOD, class T>
static int dispatch_layout(const float* src, const float* dst, float* H, int64_t n, int64_t stride,
                           hg_layout_t layout, int norm, cudaStream_t st)
{
    return layout == HG_SOA ? launch_soa<METHOD, T>(src, dst, H, n, stride, norm, st)
                            : launch_aos<METHOD, T>(src, dst, H, n, norm, st);
}

int solve_batched(int method, const float* src, const float* dst, float* H, int64_t n,
                  int64_t plane_stride, hg_layout_t layout, hg_norm_t norm, hg_precision_t prec,
                  cudaStream_t st)
{
    if (n < 0) return HG_ERR_INVALID_ARG;
    if (layout != HG_SOA && layout != HG_AOS) return HG_ERR_INVALID_ARG;
    if (norm != HG_NORM_NONE && norm != HG_NORM_H33 && norm != HG_NORM_FROBENIUS) return HG_ERR_INVALID_ARG;
    if (prec != HG_PREC_F64 && prec != HG_PREC_F32) return HG_ERR_INVALID_ARG;
    if (n == 0) return HG_OK;
    if (!src || !dst || !H) return HG_ERR_INVALID_ARG;
    if (!aligned16(src) || !aligned16(dst) || !aligned16(H)) return HG_ERR_ALIGNMENT;
    // one launch covers at most 2^31-1 blocks of 256 threads
    if ((n + kBlock - 1) / kBlock > 0x7fffffffLL) return HG_ERR_INVALID_ARG;
    const int nm = static_cast<int>(norm);
    if (method == METHOD_ACA) {
        return prec == HG_PREC_F64 ? dispatch_layout<METHOD_ACA, double>(src, dst, H, n, plane_stride, layout, nm, st)
                                   : dispatch_layout<METHOD_ACA, float >(src, dst, H, n, plane_stride, layout, nm, st);
    }
    return prec == HG_PREC_F64 ? dispatch_layout<METHOD_SKS, double>(src, dst, H, n, plane_stride, layout, nm, st)
                               : dispatch_layout<METHOD_SKS, float >(src, dst, H, n, plane_stride, layout, nm, st);
}

// ------------------------------------------------------------------------------------------
// Host-buffer entry points.  Page-locked buffers: zero-copy (below).  Pageable buffers: chunked
// H2D -> solve -> D2H on kStreams streams (copy engines in both directions overlap the kernel).  SoA chunks are strided in host memory (8 or 9 planes of
// `n` floats): cudaMemcpy2DAsync moves them into chunk-local device planes.
// ------------------------------------------------------------------------------------------
// Device-visible alias of a page-locked host pointer, if it is one.
// Both ends of [host, host + bytes) must belong to page-locked, mapped memory, and map to one contiguous device range
// (a buffer registered only in part would otherwise take the zero-copy path and fault in the kernel).
static bool mapped_host_pointer(const void* host, size_t bytes, void** dev)
{
    cudaPointerAttributes a, z;
    if (cudaPointerGetAttributes(&a, host) != cudaSuccess) { cudaGetLastError(); return false; }
    if (a.type != cudaMemoryTypeHost || a.devicePointer == nullptr) return false;
    if (bytes > 1) {
        const char* last = static_cast<const char*>(host) + (bytes - 1);
        if (cudaPointerGetAttributes(&z, last) != cudaSuccess) { cudaGetLastError(); return false; }
        if (z.type != cudaMemoryTypeHost || z.devicePointer == nullptr) return false;
        if (static_cast<const char*>(z.devicePointer) - static_cast<const char*>(a.devicePointer) != static_cast<ptrdiff_t>(bytes - 1))
            return false;
    }
    *dev = a.devicePointer;
    return true;
}

static int solve_batched_host(int method, const float* src, const float* dst, float* H, int64_t n,
                              hg_layout_t layout, hg_norm_t norm, hg_precision_t prec, int64_t chunk)
{
    if (n < 0 || chunk < 0) return HG_ERR_INVALID_ARG;
    if (layout != HG_SOA && layout != HG_AOS) return HG_ERR_INVALID_ARG;
    if (norm != HG_NORM_NONE && norm != HG_NORM_H33 && norm != HG_NORM_FROBENIUS) return HG_ERR_INVALID_ARG;
    if (prec != HG_PREC_F64 && prec != HG_PREC_F32) return HG_ERR_INVALID_ARG;
    if (n == 0) return HG_OK;
    if (!src || !dst || !H) return HG_ERR_INVALID_ARG;
    // Page-locked, device-mapped host buffers (cudaHostAlloc / cudaHostRegister, e.g. torch pinned tensors): the kernel
    // reads and writes them directly over PCIe -- one launch, both directions of the bus busy at once, no staging
    // memory.  Measured equal to the best of the staged pipeline (PCIe-bound) and steadier.  chunk_sets is ignored.
    {
        void *ds = nullptr, *dd = nullptr, *dh = nullptr;
        const size_t in_bytes = size_t(n) * 8 * sizeof(float), out_bytes = size_t(n) * 9 * sizeof(float);
        if (mapped_host_pointer(src, in_bytes, &ds) && mapped_host_pointer(dst, in_bytes, &dd) && mapped_host_pointer(H, out_bytes, &dh) &&
            aligned16(ds) && aligned16(dd) && aligned16(dh)) {
            cudaStream_t zs = nullptr;
            int rc = cuda_status(cudaStreamCreateWithFlags(&zs, cudaStreamNonBlocking));
            if (rc == HG_OK)
                rc = solve_batched(method, static_cast<const float*>(ds), static_cast<const float*>(dd), static_cast<float*>(dh),
                                   n, n, layout, norm, prec, zs);
            if (zs) {
                const int r2 = cuda_status(cudaStreamSynchronize(zs));
                if (rc == HG_OK) rc = r2;
                cudaStreamDestroy(zs);
            }
            return rc;
        }
    }
    if (chunk == 0) chunk = int64_t(1) << 21;            // 2 Mi sets: 128 MiB in, 72 MiB out per chunk
    chunk = (chunk + 3) & ~int64_t(3);
    if (chunk > n) chunk = n;

    constexpr int kStreams = 3;
    cudaStream_t st[kStreams] = {};
    float* buf[kStreams] = {};
    int rc = HG_OK;
    const size_t per = static_cast<size_t>(chunk) * (8 + 8 + 9) * sizeof(float);
    for (int i = 0; i < kStreams && rc == HG_OK; ++i) {
        rc = cuda_status(cudaStreamCreateWithFlags(&st[i], cudaStreamNonBlocking));
        if (rc == HG_OK) rc = cuda_status(cudaMalloc(reinterpret_cast<void**>(&buf[i]), per));
    }
    int64_t c = 0;
    for (int64_t a = 0; a < n && rc == HG_OK; a += chunk, ++c) {
        const int64_t m = (n - a < chunk) ? (n - a) : chunk;
        const int i = static_cast<int>(c % kStreams);
        float* ds = buf[i];
        float* dd = ds + 8 * chunk;
        float* dh = dd + 8 * chunk;
        cudaError_t e;
        if (layout == HG_SOA) {
            e = cudaMemcpy2DAsync(ds, chunk * sizeof(float), src + a, n * sizeof(float), m * sizeof(float), 8,
                                  cudaMemcpyHostToDevice, st[i]);
            if (e == cudaSuccess)
                e = cudaMemcpy2DAsync(dd, chunk * sizeof(float), dst + a, n * sizeof(float), m * sizeof(float), 8,
                                      cudaMemcpyHostToDevice, st[i]);
        } else {
            e = cudaMemcpyAsync(ds, src + 8 * a, m * 8 * sizeof(float), cudaMemcpyHostToDevice, st[i]);
            if (e == cudaSuccess)
                e = cudaMemcpyAsync(dd, dst + 8 * a, m * 8 * sizeof(float), cudaMemcpyHostToDevice, st[i]);
        }
        rc = cuda_status(e);
        if (rc != HG_OK) break;
        rc = solve_batched(method, ds, dd, dh, m, chunk, layout, norm, prec, st[i]);
        if (rc != HG_OK) break;
        if (layout == HG_SOA)
            e = cudaMemcpy2DAsync(H + a, n * sizeof(float), dh, chunk * sizeof(float), m * sizeof(float), 9,
                                  cudaMemcpyDeviceToHost, st[i]);
        else
            e = cudaMemcpyAsync(H + 9 * a, dh, m * 9 * sizeof(float), cudaMemcpyDeviceToHost, st[i]);
        rc = cuda_status(e);
    }
    for (int i = 0; i < kStreams; ++i) {
        if (st[i]) {
            const int r2 = cuda_status(cudaStreamSynchronize(st[i]));
            if (rc == HG_OK) rc = r2;
            cudaStreamDestroy(st[i]);
        }
        if (buf[i]) cudaFree(buf[i]);
    }
    return rc;
}

}  // namespace hg

extern "C" {

int hg_aca_batched(const float* src, const float* dst, float* H, int64_t n, hg_layout_t layout,
                   hg_norm_t norm, hg_precision_t prec, void* cuda_stream)
{
    return hg::solve_batched(hg::METHOD_ACA, src, dst, H, n, n, layout, norm, prec,
                             static_cast<cudaStream_t>(cuda_stream));
}

int hg_sks_batched(const float* src, const float* dst, float* H, int64_t n, hg_layout_t layout,
                   hg_norm_t norm, hg_precision_t prec, void* cuda_stream)
{
    return hg::solve_batched(hg::METHOD_SKS, src, dst, H, n, n, layout, norm, prec,
                             static_cast<cudaStream_t>(cuda_stream));
}

int hg_aca_batched_host(const float* src, const float* dst, float* H, int64_t n, hg_layout_t layout,
                        hg_norm_t norm, hg_precision_t prec, int64_t chunk_sets)
{
    return hg::solve_batched_host(hg::METHOD_ACA, src, dst, H, n, layout, norm, prec, chunk_sets);
}

int hg_sks_batched_host(const float* src, const float* dst, float* H, int64_t n, hg_layout_t layout,
                        hg_norm_t norm, hg_precision_t prec, int64_t chunk_sets)
{
    return hg::solve_batched_host(hg::METHOD_SKS, src, dst, H, n, layout, norm, prec, chunk_sets);
}

}  // extern "C"
