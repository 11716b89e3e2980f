// hg_grid.cu -- hg_offsets_to_grid: 4-point offsets -> H (ACA) -> dense sampling grid, fused.
//
// Rows a-G0..a-G2 of SURVEY.md section 8(a).  The deep-homography parameterisation (P:25, P:131,
// P:540-544): the network predicts the offsets of the four corners of a fixed source rectangle;
// the module turns them into H; the pipeline then warps with H.  One CTA per item: warp 0 solves
// the item's H once in fp64, folds the pixel lattice into it, broadcasts 9 fp32 numbers through
// shared memory, and all warps sweep the patch with 128-bit streaming stores.
// HBM-write-bound: 8 B per pixel.
#include "hg_device.cuh"
#include "hg_host.h"

namespace hg {

constexpr int kGridBlock = 256;

struct RectParams {
    double x0, y0, w, h;      // source rectangle
    double step_x, step_y;    // lattice pitch: w/(grid_w-1), h/(grid_h-1) (0 when the extent is 1)
};

// Corners TL,TR,BR,BL + offsets -> (s, d) in the M,N,P,Q roles of the general solver (R11).
__device__ __forceinline__ void corners_from_offsets(const RectParams& rp, const float4 o0, const float4 o1,
                                                     double s[8], double d[8])
{
    s[0] = rp.x0;        s[1] = rp.y0;
    s[2] = rp.x0 + rp.w; s[3] = rp.y0;
    s[4] = rp.x0 + rp.w; s[5] = rp.y0 + rp.h;
    s[6] = rp.x0;        s[7] = rp.y0 + rp.h;
    d[0] = s[0] + double(o0.x); d[1] = s[1] + double(o0.y);
    d[2] = s[2] + double(o0.z); d[3] = s[3] + double(o0.w);
    d[4] = s[4] + double(o1.x); d[5] = s[5] + double(o1.y);
    d[6] = s[6] + double(o1.z); d[7] = s[7] + double(o1.w);
}

// PIX = 2: grid_w even, one 128-bit store covers two pixels; PIX = 1: 64-bit store per pixel.
template <int PIX>
__global__ void __launch_bounds__(kGridBlock)
offsets_to_grid_kernel(const float* __restrict__ offsets, RectParams rp, int grid_w, int grid_h,
                       int tx_count, float* __restrict__ H_out, float* __restrict__ grid, int norm)
{
    __shared__ float hs[9];
    const int64_t b = blockIdx.x;
    if (threadIdx.x < 32) {
        const float4* op = reinterpret_cast<const float4*>(offsets + 8 * b);
        const float4 o0 = __ldg(op), o1 = __ldg(op + 1);
        double s[8], d[8], Hd[9];
        corners_from_offsets(rp, o0, o1, s, d);
        aca_solve<double>(s, d, Hd);
        // overflow-safe common scale for the fp32 sweep (projective: any scale gives the same grid)
        double m = 0.0;
#pragma unroll
        for (int k = 0; k < 9; ++k) m = fmax(m, fabs(Hd[k]));
        const double r = K<double>::rcp(m);
        if (H_out != nullptr) {
            double Hn[9];
#pragma unroll
            for (int k = 0; k < 9; ++k) Hn[k] = Hd[k] * r;
            normalise<double>(Hn, norm);
            if (norm == 0) {
#pragma unroll
                for (int k = 0; k < 9; ++k) Hn[k] = Hd[k];
            }
            if (threadIdx.x == 0) {
#pragma unroll
                for (int k = 0; k < 9; ++k) H_out[9 * b + k] = static_cast<float>(Hn[k]);
            }
        }
        // fold the lattice x = x0 + i*step_x, y = y0 + j*step_y into H: L = H * [sx 0 x0; 0 sy y0; 0 0 1]
        if (threadIdx.x == 0) {
#pragma unroll
            for (int row = 0; row < 3; ++row) {
                const double a = Hd[3 * row] * r, bb = Hd[3 * row + 1] * r, c = Hd[3 * row + 2] * r;
                hs[3 * row]     = static_cast<float>(a * rp.step_x);
                hs[3 * row + 1] = static_cast<float>(bb * rp.step_y);
                hs[3 * row + 2] = static_cast<float>(fma(a, rp.x0, fma(bb, rp.y0, c)));
            }
        }
    }
    __syncthreads();
    const float l11 = hs[0], l12 = hs[1], l13 = hs[2];
    const float l21 = hs[3], l22 = hs[4], l23 = hs[5];
    const float l31 = hs[6], l32 = hs[7], l33 = hs[8];

    const int tx = threadIdx.x & (tx_count - 1);
    const int ty = threadIdx.x / tx_count;
    const int rows_per_pass = kGridBlock / tx_count;
    float* g = grid + static_cast<int64_t>(2) * grid_w * grid_h * b;

    for (int j = ty; j < grid_h; j += rows_per_pass) {
        const float fj = static_cast<float>(j);
        const float rx = fmaf(l12, fj, l13), ry = fmaf(l22, fj, l23), rw = fmaf(l32, fj, l33);
        float* row = g + static_cast<int64_t>(2) * grid_w * j;
        for (int i = tx * PIX; i < grid_w; i += tx_count * PIX) {
            const float fi = static_cast<float>(i);
            const float X0 = fmaf(l11, fi, rx), Y0 = fmaf(l21, fi, ry), W0 = fmaf(l31, fi, rw);
            const float q0 = __frcp_rn(W0);
            if (PIX == 2) {
                const float X1 = X0 + l11, Y1 = Y0 + l21, W1 = W0 + l31;
                const float q1 = __frcp_rn(W1);
                __stcs(reinterpret_cast<float4*>(row + 2 * i), make_float4(X0 * q0, Y0 * q0, X1 * q1, Y1 * q1));
            } else {
                __stcs(reinterpret_cast<float2*>(row + 2 * i), make_float2(X0 * q0, Y0 * q0));
            }
        }
    }
}

// H only (C1: the latency-bound deep-pipeline call): one thread per item, 36-byte records
// transposed through shared memory for contiguous stores.
__global__ void __launch_bounds__(kGridBlock)
offsets_to_h_kernel(const float* __restrict__ offsets, RectParams rp, float* __restrict__ H_out,
                    int64_t n, int norm)
{
    __shared__ float stage[kGridBlock * 9];
    const int64_t base = static_cast<int64_t>(blockIdx.x) * kGridBlock;
    const int64_t b = base + threadIdx.x;
    if (b < n) {
        const float4* op = reinterpret_cast<const float4*>(offsets + 8 * b);
        const float4 o0 = __ldg(op), o1 = __ldg(op + 1);
        double s[8], d[8], Hd[9];
        corners_from_offsets(rp, o0, o1, s, d);
        aca_solve<double>(s, d, Hd);
        normalise<double>(Hd, norm);
#pragma unroll
        for (int k = 0; k < 9; ++k) stage[threadIdx.x * 9 + k] = static_cast<float>(Hd[k]);
    }
    __syncthreads();
    const int64_t rem = n - base;
    const int cnt = static_cast<int>(rem < kGridBlock ? rem : kGridBlock) * 9;
    float* out = H_out + 9 * base;
    for (int j = threadIdx.x; j < cnt; j += kGridBlock) out[j] = stage[j];
}

static int pow2_at_least(int v) { int p = 1; while (p < v) p <<= 1; return p; }

}  // namespace hg

extern "C" int hg_offsets_to_grid(const float* offsets, float x0, float y0, float w, float h,
                                  int32_t grid_w, int32_t grid_h, float* H, float* grid, int64_t n,
                                  hg_norm_t norm, void* cuda_stream)
{
    using namespace hg;
    if (n < 0) return HG_ERR_INVALID_ARG;
    if (norm != HG_NORM_NONE && norm != HG_NORM_H33 && norm != HG_NORM_FROBENIUS) return HG_ERR_INVALID_ARG;
    if (!(w != 0.0f) || !(h != 0.0f)) return HG_ERR_INVALID_ARG;
    if (grid != nullptr && (grid_w < 1 || grid_h < 1)) return HG_ERR_INVALID_ARG;
    if (n == 0 || (H == nullptr && grid == nullptr)) return HG_OK;
    if (offsets == nullptr) return HG_ERR_INVALID_ARG;
    if (!aligned16(offsets) || (grid != nullptr && !aligned16(grid)) || (H != nullptr && !aligned4(H)))
        return HG_ERR_ALIGNMENT;
    if (n > 0x7fffffffLL) return HG_ERR_INVALID_ARG;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    RectParams rp;
    rp.x0 = x0; rp.y0 = y0; rp.w = w; rp.h = h;
    rp.step_x = (grid_w > 1) ? double(w) / double(grid_w - 1) : 0.0;
    rp.step_y = (grid_h > 1) ? double(h) / double(grid_h - 1) : 0.0;
    if (grid == nullptr) {
        const int64_t blocks = (n + kGridBlock - 1) / kGridBlock;
        offsets_to_h_kernel<<<static_cast<unsigned>(blocks), kGridBlock, 0, st>>>(offsets, rp, H, n, int(norm));
        return launch_status();
    }
    // 128-bit stores need every row (and item) to start 16-byte aligned: grid_w even.
    const bool pairs = (grid_w % 2 == 0);
    const int per_row = pairs ? grid_w / 2 : grid_w;
    int tx_count = pow2_at_least(per_row);
    if (tx_count > kGridBlock) tx_count = kGridBlock;
    if (pairs)
        offsets_to_grid_kernel<2><<<static_cast<unsigned>(n), kGridBlock, 0, st>>>(offsets, rp, grid_w, grid_h, tx_count, H, grid, int(norm));
    else
        offsets_to_grid_kernel<1><<<static_cast<unsigned>(n), kGridBlock, 0, st>>>(offsets, rp, grid_w, grid_h, tx_count, H, grid, int(norm));
    return launch_status();
}
