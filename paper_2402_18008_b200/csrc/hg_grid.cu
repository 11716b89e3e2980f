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
constexpr size_t kWarpStageBytes = 110 * 1024;   // staged image per CTA: two CTAs per SM

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

// ------------------------------------------------------------------------------------------
// Offsets -> H -> warped image ("warp image with H"; reading R17): the
// sampling grid never reaches HBM.  Lanes map to adjacent pixels of a row, so the four bilinear taps
// of a warp fall into one or two lines each and every store instruction writes a full line.
// Zero padding: a tap outside the image contributes 0; a non-finite position gives 0.
// Per pixel and channel: 4 B read + 4 B written.  Two kernels: the gather form below for image planes too large
// for shared memory, and the staged form (offsets_to_warp_plane_kernel) for everything else.
// ------------------------------------------------------------------------------------------
struct WarpGeom { int out_w, out_h, img_w, img_h, channels, rows_per_band; };

// The four taps of one sampling position: element offsets into an image plane (always inside the plane)
// and weights (zero for a tap that lies outside the image).  Branch-free: the position is first clamped to
// [-1, size], where every tap is either valid or carries weight zero -- this also sends NaN to -1.
struct Taps { int o00, o01, o10, o11; float w00, w01, w10, w11; };

__device__ __forceinline__ Taps make_taps(float u, float v, int img_w, int img_h)
{
    const float uc = fminf(fmaxf(u, -1.f), static_cast<float>(img_w));
    const float vc = fminf(fmaxf(v, -1.f), static_cast<float>(img_h));
    const float u0 = floorf(uc), v0 = floorf(vc);
    const float fu = uc - u0, fv = vc - v0;                                   // exact
    const int iu = static_cast<int>(u0), iv = static_cast<int>(v0);           // [-1, img_w], [-1, img_h]
    const float wx0 = (static_cast<unsigned>(iu) < static_cast<unsigned>(img_w)) ? 1.f - fu : 0.f;
    const float wx1 = (static_cast<unsigned>(iu + 1) < static_cast<unsigned>(img_w)) ? fu : 0.f;
    const float wy0 = (static_cast<unsigned>(iv) < static_cast<unsigned>(img_h)) ? 1.f - fv : 0.f;
    const float wy1 = (static_cast<unsigned>(iv + 1) < static_cast<unsigned>(img_h)) ? fv : 0.f;
    const int cx0 = min(max(iu, 0), img_w - 1), cx1 = min(iu + 1, img_w - 1);
    const int r0 = min(max(iv, 0), img_h - 1) * img_w, r1 = min(iv + 1, img_h - 1) * img_w;
    Taps t;
    t.o00 = r0 + cx0; t.o01 = r0 + cx1; t.o10 = r1 + cx0; t.o11 = r1 + cx1;
    t.w00 = wy0 * wx0; t.w01 = wy0 * wx1; t.w10 = wy1 * wx0; t.w11 = wy1 * wx1;
    return t;
}

// Gather form (images too large to stage): taps read from global memory through the read-only path / L1.
__device__ __forceinline__ float gather(const float* __restrict__ img, const Taps& t)
{
    return fmaf(t.w11, __ldg(img + t.o11), fmaf(t.w10, __ldg(img + t.o10),
           fmaf(t.w01, __ldg(img + t.o01), t.w00 * __ldg(img + t.o00))));
}

// All four taps inside the image, `p` points at tap (0,0).  Nested lerps: the same bilinear form as gather() up to rounding.
__device__ __forceinline__ float lerp2(float a, float b, float c, float d, float fu, float fv)
{
    const float top = fmaf(fu, b - a, a), bot = fmaf(fu, d - c, c);
    return fmaf(fv, bot - top, top);
}

__device__ __forceinline__ float lds_f32(uint32_t addr)
{ float v; asm("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr)); return v; }

__device__ __forceinline__ float gather_interior_gmem(const float* __restrict__ p, int img_w, float fu, float fv)
{
    return lerp2(__ldg(p), __ldg(p + 1), __ldg(p + img_w), __ldg(p + img_w + 1), fu, fv);
}

__device__ __forceinline__ float rcp_approx(float x)
{ float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }

// CH = compile-time channel count (0: read it from the geometry).  blockIdx.x = item, blockIdx.y = band of rows.
template <int CH>
__global__ void __launch_bounds__(kGridBlock, CH == 0 ? 2 : 4)
offsets_to_warp_kernel(const float* __restrict__ offsets, RectParams rp, WarpGeom g, int tx_count,
                       const float* __restrict__ image, float* __restrict__ warped, float* __restrict__ H_out, int norm)
{
    __shared__ float hs[9];
    const int64_t b = blockIdx.x;
    if (threadIdx.x < 32) {
        const float4* op = reinterpret_cast<const float4*>(offsets + 8 * b);
        const float4 o0 = __ldg(op), o1 = __ldg(op + 1);
        double s[8], d[8], Hd[9];
        corners_from_offsets(rp, o0, o1, s, d);
        aca_solve<double>(s, d, Hd);
        double m = 0.0;
#pragma unroll
        for (int k = 0; k < 9; ++k) m = fmax(m, fabs(Hd[k]));
        const double r = K<double>::rcp(m);
        if (H_out != nullptr && blockIdx.y == 0) {
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
    const int channels = CH > 0 ? CH : g.channels;
    const int img_w = g.img_w, img_h = g.img_h, out_w = g.out_w;
    const int img_plane = img_w * img_h;
    const int out_plane = out_w * g.out_h;
    const float wm1 = static_cast<float>(img_w - 1), hm1 = static_cast<float>(img_h - 1);
    const float* img_b = image + b * channels * static_cast<int64_t>(img_plane);
    float* out_b = warped + b * channels * static_cast<int64_t>(out_plane);
    const int j_begin = blockIdx.y * g.rows_per_band;
    const int j_end = min(g.out_h, j_begin + g.rows_per_band);
    const int64_t out_step = static_cast<int64_t>(rows_per_pass) * out_w;

    for (int i = tx; i < out_w; i += tx_count) {
        const float fi = static_cast<float>(i);
        const float cx = fmaf(l11, fi, l13), cy = fmaf(l21, fi, l23), cw = fmaf(l31, fi, l33);
        float* op_row = out_b + i + static_cast<int64_t>(j_begin + ty) * out_w;
        float fj = static_cast<float>(j_begin + ty);
        const float fstep = static_cast<float>(rows_per_pass);
#pragma unroll 2
        for (int j = j_begin + ty; j < j_end; j += rows_per_pass, op_row += out_step, fj += fstep) {
            const float X = fmaf(l12, fj, cx), Y = fmaf(l22, fj, cy), Wv = fmaf(l32, fj, cw);
            const float q = rcp_approx(Wv);
            const float u = X * q, v = Y * q;
            float* op = op_row;
            // Interior fast path, decided per warp: all four taps of every lane inside the image -- no clamping,
            // no weight selection, one address.  NaN fails the comparisons and takes the general path.
            const bool interior = (u >= 0.f) && (u < wm1) && (v >= 0.f) && (v < hm1);
            if (__all_sync(0xffffffffu, interior)) {
                // floor without the conversion pipe: (u - 1/2) + 1.5 * 2^23 rounds to an integer k in the low mantissa
                // bits, k = floor(u) except k = u - 1 for some integral u, where fu = 1 gives the same sample.
                const float tu = __fadd_rn(__fadd_rn(u, -0.5f), 12582912.f), tv = __fadd_rn(__fadd_rn(v, -0.5f), 12582912.f);
                const float fu = u - __fadd_rn(tu, -12582912.f), fv = v - __fadd_rn(tv, -12582912.f);
                const int e = (__float_as_int(tv) - 0x4B400000) * img_w + (__float_as_int(tu) - 0x4B400000);
                const float* p = img_b + e;
                if (CH > 0) {
#pragma unroll
                    for (int c = 0; c < CH; ++c) { __stcs(op, gather_interior_gmem(p, img_w, fu, fv)); p += img_plane; op += out_plane; }
                } else {
                    for (int c = 0; c < channels; ++c) { __stcs(op, gather_interior_gmem(p, img_w, fu, fv)); p += img_plane; op += out_plane; }
                }
            } else {
                const Taps t = make_taps(u, v, img_w, img_h);
                const float* ip = img_b;
                if (CH > 0) {
#pragma unroll
                    for (int c = 0; c < CH; ++c) { __stcs(op, gather(ip, t)); ip += img_plane; op += out_plane; }
                } else {
                    for (int c = 0; c < channels; ++c) { __stcs(op, gather(ip, t)); ip += img_plane; op += out_plane; }
                }
            }
        }
    }
}

// ------------------------------------------------------------------------------------------
// The staged form of the same operation: one CTA per (item, channel[, band of rows]).  The image plane is staged in
// shared memory inside a frame of zeros (2 rows above, 3 below, >= 4 columns left and right), and the pixel position
// is produced already normalised to that frame, so that one saturating multiply clamps it and the zero frame IS the
// zero padding of reading R17: no interior test, no tap selection, no branch in the pixel loop.
//   rows of H:  U = (u + 2) / (img_w + 3), V = (v + 2) / (img_h + 3) are folded into rows 1-2 in fp64
//   per pixel:  (X', Y') = FFMA2,  W = FFMA,  q = rcp(W),  U, V = sat(X' q), sat(Y' q)      -- u in [-2, w + 1]
//               (k + M)  = FFMA2.RM(UV, scale, M - 2)     round-down: k = floor(u) exactly, in the low mantissa bits
//               (k + 2)  = FADD2 (exact),   (fu, fv) = FFMA2(UV, scale, -(k + 2))           -- fu in [0, 1]
//               address = IMAD + LEA,  4 x LDS,  lerp = FADD2 + FFMA2 + FADD + FFMA,  STG
// about 24 issued instructions per pixel against 63 for the gather form above (profiles/r02_summary.md).
// Non-finite positions saturate to 0 (NaN) or to a frame corner (inf): zero, as R17 asks.
// ------------------------------------------------------------------------------------------
struct PlaneGeom {
    int out_w, out_h, img_w, img_h, channels, bands, rows_per_band;
    int stride;            // floats per staged row: 4 + img_w + right pad, a multiple of 4
    int bulk;              // 1: rows are copied by cp.async.bulk (16-byte rules hold), 0: by plain loads
};

constexpr int kFrameTop = 2, kFrameBottom = 3, kFrameLeft = 4;
constexpr float kFloorMagic = 12582912.f;      // 1.5 * 2^23

__global__ void __launch_bounds__(kGridBlock, 3)
offsets_to_warp_plane_kernel(const float* __restrict__ offsets, RectParams rp, PlaneGeom g, int tx_count,
                             const float* __restrict__ image, float* __restrict__ warped, float* __restrict__ H_out, int norm)
{
    __shared__ float hs[9];
    __shared__ uint64_t img_bar;
    extern __shared__ __align__(128) float img_s[];
    const int64_t b = blockIdx.x;
    const int c = blockIdx.y / g.bands, band = blockIdx.y - c * g.bands;
    const int stride = g.stride, img_w = g.img_w, img_h = g.img_h;
    const float* plane = image + (b * g.channels + c) * static_cast<int64_t>(img_w) * img_h;
    const uint32_t row_bytes = 4u * static_cast<uint32_t>(img_w);

    if (threadIdx.x == 0 && g.bulk) {
        mbar_init(&img_bar, 1);
        fence_barrier_init();
        mbar_arrive_expect_tx(&img_bar, row_bytes * static_cast<uint32_t>(img_h));
    }
    // the zero frame: whole rows above and below, pads left and right of every image row
    for (int r = threadIdx.x; r < (kFrameTop + kFrameBottom) * (stride >> 2); r += kGridBlock) {
        const int fr = r / (stride >> 2), q4 = r - fr * (stride >> 2);
        const int row = fr < kFrameTop ? fr : img_h + fr;              // 0, 1, img_h + 2, img_h + 3, img_h + 4
        reinterpret_cast<float4*>(img_s + row * stride)[q4] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    const int right = stride - kFrameLeft - img_w;                     // >= 4
    for (int r = threadIdx.x; r < img_h * (kFrameLeft + right); r += kGridBlock) {
        const int y = r / (kFrameLeft + right), k = r - y * (kFrameLeft + right);
        img_s[(y + kFrameTop) * stride + (k < kFrameLeft ? k : img_w + k)] = 0.f;
    }
    __syncthreads();
    if (g.bulk) {
        for (int y = threadIdx.x; y < img_h; y += kGridBlock)
            bulk_copy_g2s(img_s + (y + kFrameTop) * stride + kFrameLeft, plane + static_cast<int64_t>(y) * img_w, row_bytes, &img_bar);
    } else {
        for (int e = threadIdx.x; e < img_w * img_h; e += kGridBlock) {
            const int y = e / img_w, x = e - y * img_w;
            img_s[(y + kFrameTop) * stride + kFrameLeft + x] = __ldg(plane + e);
        }
    }
    if (threadIdx.x < 32) {
        const float4* op = reinterpret_cast<const float4*>(offsets + 8 * b);
        const float4 o0 = __ldg(op), o1 = __ldg(op + 1);
        double s[8], d[8], Hd[9];
        corners_from_offsets(rp, o0, o1, s, d);
        aca_solve<double>(s, d, Hd);
        double m = 0.0;
#pragma unroll
        for (int k = 0; k < 9; ++k) m = fmax(m, fabs(Hd[k]));
        const double r = K<double>::rcp(m);
        if (H_out != nullptr && blockIdx.y == 0) {
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
        if (threadIdx.x == 0) {
            // L = H * [sx 0 x0; 0 sy y0; 0 0 1] (the lattice), then rows 1-2 -> frame-normalised coordinates
            double L[9];
#pragma unroll
            for (int row = 0; row < 3; ++row) {
                const double a = Hd[3 * row] * r, bb = Hd[3 * row + 1] * r, cc = Hd[3 * row + 2] * r;
                L[3 * row] = a * rp.step_x; L[3 * row + 1] = bb * rp.step_y; L[3 * row + 2] = fma(a, rp.x0, fma(bb, rp.y0, cc));
            }
            const double iu = 1.0 / (img_w + 3.0), iv = 1.0 / (img_h + 3.0);
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                hs[k]     = static_cast<float>((L[k] + 2.0 * L[6 + k]) * iu);
                hs[3 + k] = static_cast<float>((L[3 + k] + 2.0 * L[6 + k]) * iv);
                hs[6 + k] = static_cast<float>(L[6 + k]);
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
    const int out_w = g.out_w;
    float* out_p = warped + (b * g.channels + c) * static_cast<int64_t>(out_w) * g.out_h;
    const int j_begin = band * g.rows_per_band;
    const int j_end = min(g.out_h, j_begin + g.rows_per_band);
    const float2 scale = make_float2(static_cast<float>(img_w + 3), static_cast<float>(img_h + 3));
    const float2 L2 = make_float2(l12, l22);
    // frame element of sample index (ku, kv): (kv + 2) * stride + (ku + 4); the floor trick leaves k + 0x4B400000
    const uint32_t base = smem_u32(img_s) + 4u * static_cast<uint32_t>(kFrameTop * stride + kFrameLeft)
                          - 4u * (0x4B400000u * static_cast<uint32_t>(stride) + 0x4B400000u);
    const uint32_t sbytes = 4u * static_cast<uint32_t>(stride);
    if (g.bulk) mbar_wait(&img_bar, 0);
    else        __syncthreads();

    for (int i = tx; i < out_w; i += tx_count) {
        const float fi = static_cast<float>(i);
        const float2 C2 = make_float2(fmaf(l11, fi, l13), fmaf(l21, fi, l23));
        const float cw = fmaf(l31, fi, l33);
        float* op = out_p + i + static_cast<int64_t>(j_begin + ty) * out_w;
        const int64_t out_step = static_cast<int64_t>(rows_per_pass) * out_w;
        float fj = static_cast<float>(j_begin + ty);
        const float fstep = static_cast<float>(rows_per_pass);
#pragma unroll 4
        for (int j = j_begin + ty; j < j_end; j += rows_per_pass, op += out_step, fj += fstep) {
            const float2 P = __ffma2_rn(L2, make_float2(fj, fj), C2);
            const float Wv = fmaf(l32, fj, cw);
            const float q = rcp_approx(Wv);
            float2 UV;
            asm("mul.rn.sat.f32 %0, %1, %2;" : "=f"(UV.x) : "f"(P.x), "f"(q));
            asm("mul.rn.sat.f32 %0, %1, %2;" : "=f"(UV.y) : "f"(P.y), "f"(q));
            const float2 T = __ffma2_rd(UV, scale, make_float2(kFloorMagic - 2.f, kFloorMagic - 2.f));
            const float2 R = __fadd2_rn(T, make_float2(2.f - kFloorMagic, 2.f - kFloorMagic));
            const float2 F = __ffma2_rn(UV, scale, make_float2(-R.x, -R.y));
            const uint32_t at = base + 4u * (__float_as_uint(T.y) * static_cast<uint32_t>(stride) + __float_as_uint(T.x));
            const float2 ac = make_float2(lds_f32(at), lds_f32(at + sbytes));
            const float2 bd = make_float2(lds_f32(at + 4u), lds_f32(at + sbytes + 4u));
            const float2 D = __fadd2_rn(bd, make_float2(-ac.x, -ac.y));
            const float2 TB = __ffma2_rn(make_float2(F.x, F.x), D, ac);              // (top, bottom)
            __stcs(op, fmaf(F.y, TB.y - TB.x, TB.x));
        }
    }
}

template <int CH>
static int launch_warp(dim3 grid, cudaStream_t st, const float* offsets, const RectParams& rp, const WarpGeom& g,
                       int tx_count, const float* image, float* warped, float* H, int norm)
{
    offsets_to_warp_kernel<CH><<<grid, kGridBlock, 0, st>>>(offsets, rp, g, tx_count, image, warped, H, norm);
    return launch_status();
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

extern "C" int hg_offsets_to_warp(const float* offsets, float x0, float y0, float w, float h,
                                  int32_t out_w, int32_t out_h, const float* image, int32_t channels,
                                  int32_t img_w, int32_t img_h, float* warped, float* H, int64_t n,
                                  hg_norm_t norm, void* cuda_stream)
{
    using namespace hg;
    if (n < 0) return HG_ERR_INVALID_ARG;
    if (norm != HG_NORM_NONE && norm != HG_NORM_H33 && norm != HG_NORM_FROBENIUS) return HG_ERR_INVALID_ARG;
    if (!(w != 0.0f) || !(h != 0.0f)) return HG_ERR_INVALID_ARG;
    if (out_w < 1 || out_h < 1 || img_w < 1 || img_h < 1 || channels < 1) return HG_ERR_INVALID_ARG;
    if (int64_t(img_w) * img_h > 0x3fffffffLL || int64_t(out_w) * out_h > 0x3fffffffLL) return HG_ERR_INVALID_ARG;
    if (n == 0) return HG_OK;
    if (!offsets || !image || !warped) return HG_ERR_INVALID_ARG;
    if (!aligned16(offsets) || !aligned4(warped) || !aligned4(image) || (H != nullptr && !aligned4(H))) return HG_ERR_ALIGNMENT;
    if (n > 0x7fffffffLL) return HG_ERR_INVALID_ARG;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    RectParams rp;
    rp.x0 = x0; rp.y0 = y0; rp.w = w; rp.h = h;
    rp.step_x = (out_w > 1) ? double(w) / double(out_w - 1) : 0.0;
    rp.step_y = (out_h > 1) ? double(h) / double(out_h - 1) : 0.0;
    int tx_count = pow2_at_least(out_w < 32 ? 32 : out_w);
    if (tx_count > kGridBlock) tx_count = kGridBlock;
    // enough CTAs to fill the machine when the batch is small: split the rows into bands
    int bands = 1;
    const int rows_per_pass = kGridBlock / tx_count;
    while (n * bands < 4 * 148 && (out_h + bands - 1) / bands > rows_per_pass) bands *= 2;
    WarpGeom g;
    g.out_w = out_w; g.out_h = out_h; g.img_w = img_w; g.img_h = img_h; g.channels = channels;
    g.rows_per_band = (out_h + bands - 1) / bands;
    bands = (out_h + g.rows_per_band - 1) / g.rows_per_band;
    const dim3 grid(static_cast<unsigned>(n), static_cast<unsigned>(bands));
    // Staged form: one image plane per CTA inside a zero frame, when at least two such CTAs fit on an SM.
    {
        int stride = kFrameLeft + ((img_w + 3) & ~3) + 4;
        if (stride % 32 == 0) stride += 4;                              // rows must not start in the same bank
        const size_t plane_bytes = size_t(img_h + kFrameTop + kFrameBottom) * stride * sizeof(float);
        if (plane_bytes <= kWarpStageBytes && int64_t(channels) * out_h <= 65535) {
            PlaneGeom pg;
            pg.out_w = out_w; pg.out_h = out_h; pg.img_w = img_w; pg.img_h = img_h; pg.channels = channels;
            // rows are split into bands only while the batch alone cannot fill the machine
            int pb = 1;
            while (n * channels * pb < 3 * 148 && (out_h + pb - 1) / pb > rows_per_pass) pb *= 2;
            pg.rows_per_band = (out_h + pb - 1) / pb;
            pg.bands = (out_h + pg.rows_per_band - 1) / pg.rows_per_band;
            pg.stride = stride;
            pg.bulk = (img_w % 4 == 0 && aligned16(image)) ? 1 : 0;
            if (cudaFuncSetAttribute(offsets_to_warp_plane_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                     int(kWarpStageBytes)) != cudaSuccess) return HG_ERR_CUDA;
            const dim3 pgrid(static_cast<unsigned>(n), static_cast<unsigned>(channels * pg.bands));
            offsets_to_warp_plane_kernel<<<pgrid, kGridBlock, plane_bytes, st>>>(offsets, rp, pg, tx_count, image, warped, H, int(norm));
            return launch_status();
        }
    }
    const int nm = int(norm);
    if (channels == 1) return launch_warp<1>(grid, st, offsets, rp, g, tx_count, image, warped, H, nm);
    if (channels == 3) return launch_warp<3>(grid, st, offsets, rp, g, tx_count, image, warped, H, nm);
    return launch_warp<0>(grid, st, offsets, rp, g, tx_count, image, warped, H, nm);
}
