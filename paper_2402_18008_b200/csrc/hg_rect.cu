// hg_rect.cu -- hg_aca_rect_batched: TensorACA for a rectangular source.
//
// Deep-homography pipelines predict the offsets of the four corners of a FIXED source rectangle
// (P:25).  For a rectangle H_A1 is trivial and Q3 = (1,1,1) (Eq. 42-43),
// so H follows from the target quadrangle alone (Eq. 44-45; Algorithm 1):
// 47 FLOPs, and only the 8 offsets are read -- 32 B in + 36 B out = 68 B per homography instead of
// the general solver's 100 B.  Same streaming skeleton as hg_batched.cu; fp64 registers, fp32 I/O.
#include <type_traits>

#include "hg_device.cuh"
#include "hg_host.h"

namespace hg {

constexpr int kRectBlock = 256;

struct RectSrc {            // the source rectangle {M1.x, M1.y, w_rec, r_rec} of P:544 plus its height
    double x0, y0, w, h, r; // r = w / h  (reading R6)
};

// Eq. 45 evaluated column by column, as Algorithm 1 does:
//   col1 = Q4.x * n2 + t2 * m2,   col2 = r_rec * (Q4.y * p2 + t2 * m2),
//   col3 = -M1.x * col1 - M1.y * col2 - w_rec * t2 * m2          (m2, n2, p2 homogeneous, weight 1)
// with Q4 = f_A2-scaled fourth point of the target quadrangle in its affine frame (Eq. 28) and
// t2 = f_A2 - Q4.x - Q4.y (Eq. 30).  Corner order of `o` is TL,TR,BR,BL; roles M=TL, N=TR, Q=BR, P=BL.
// The scale is Eq. 45's (the negative of Algorithm 1's printed cross-product convention, R6).
template <class T>
__device__ __forceinline__ void aca_rect_solve(const RectSrc& rs, const T o[8], T H[9])
{
    const T x0 = T(rs.x0), y0 = T(rs.y0), w = T(rs.w), h = T(rs.h), r = T(rs.r);
    const T m2x = x0 + o[0],     m2y = y0 + o[1];
    const T n2x = x0 + w + o[2], n2y = y0 + o[3];
    const T q2x = x0 + w + o[4], q2y = y0 + h + o[5];
    const T p2x = x0 + o[6],     p2y = y0 + h + o[7];
    const T ax = n2x - m2x, ay = n2y - m2y;            // M2N2
    const T bx = p2x - m2x, by = p2y - m2y;            // M2P2
    const T qx = q2x - m2x, qy = q2y - m2y;            // M2Q2
    const T fA2 = det2(ax, ay, bx, by);
    const T Q4x = det2(qx, qy, bx, by);
    const T Q4y = det2(ax, ay, qx, qy);
    const T t2 = fA2 - Q4x - Q4y;
    const T bx3 = t2 * m2x, by3 = t2 * m2y;            // b = t2 * m2 (Algorithm 1 step 3)
    const T h11 = K<T>::fma(Q4x, n2x, bx3), h21 = K<T>::fma(Q4x, n2y, by3), h31 = Q4x + t2;
    const T h12 = r * K<T>::fma(Q4y, p2x, bx3), h22 = r * K<T>::fma(Q4y, p2y, by3), h32 = r * (Q4y + t2);
    H[0] = h11; H[1] = h12; H[2] = -K<T>::fma(x0, h11, K<T>::fma(y0, h12, w * bx3));
    H[3] = h21; H[4] = h22; H[5] = -K<T>::fma(x0, h21, K<T>::fma(y0, h22, w * by3));
    H[6] = h31; H[7] = h32; H[8] = -K<T>::fma(x0, h31, K<T>::fma(y0, h32, w * t2));
}

// SoA: offsets = float[8][n] planes (TL.x, TL.y, TR.x, ..., BL.y), H = float[9][n]; thread per V items.
template <class T, int V>
__global__ void __launch_bounds__(kRectBlock)
rect_soa_kernel(const float* __restrict__ offsets, RectSrc rs, float* __restrict__ H, int64_t n_vec, int64_t stride, int norm)
{
    const int64_t t = static_cast<int64_t>(blockIdx.x) * kRectBlock + threadIdx.x;
    if (t >= n_vec) return;
    const int64_t off = t * V;
    Vec<V> o[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) o[k] = ld_stream<V>(offsets + k * stride + off);
    Vec<V> hv[9];
#pragma unroll
    for (int v = 0; v < V; ++v) {
        T ov[8], Hv[9];
#pragma unroll
        for (int k = 0; k < 8; ++k) ov[k] = static_cast<T>(o[k].v[v]);
        aca_rect_solve<T>(rs, ov, Hv);
        normalise<T>(Hv, norm);
#pragma unroll
        for (int k = 0; k < 9; ++k) hv[k].v[v] = static_cast<float>(Hv[k]);
    }
#pragma unroll
    for (int k = 0; k < 9; ++k) st_stream<V>(H + k * stride + off, hv[k]);
}

// AoS: offsets = float[n][4][2] (what a regression head emits), H = float[n][3][3].  A thread reads its
// own 32 B record with two 128-bit loads; the 36-byte H records go through shared memory so the block
// writes one contiguous 128-bit-vectorised span.
template <class T>
__global__ void __launch_bounds__(kRectBlock)
rect_aos_kernel(const float* __restrict__ offsets, RectSrc rs, float* __restrict__ H, int64_t n, int norm)
{
    // Two items per thread (i and i + kRectBlock): four independent 128-bit loads in flight per thread, which a
    // 32-byte-per-item stream needs to cover the HBM latency.
    constexpr int ITEMS = 2;
    __shared__ __align__(16) float stage[ITEMS * kRectBlock * 9];
    const int64_t base = static_cast<int64_t>(blockIdx.x) * (ITEMS * kRectBlock);
    float4 o[ITEMS][2];
#pragma unroll
    for (int k = 0; k < ITEMS; ++k) {
        const int64_t i = base + k * kRectBlock + threadIdx.x;
        if (i < n) {
            const float4* op = reinterpret_cast<const float4*>(offsets + 8 * i);
            o[k][0] = __ldcs(op); o[k][1] = __ldcs(op + 1);
        }
    }
#pragma unroll
    for (int k = 0; k < ITEMS; ++k) {
        const int64_t i = base + k * kRectBlock + threadIdx.x;
        if (i < n) {
            const T ov[8] = { T(o[k][0].x), T(o[k][0].y), T(o[k][0].z), T(o[k][0].w), T(o[k][1].x), T(o[k][1].y), T(o[k][1].z), T(o[k][1].w) };
            T Hv[9];
            aca_rect_solve<T>(rs, ov, Hv);
            normalise<T>(Hv, norm);
#pragma unroll
            for (int q = 0; q < 9; ++q) stage[(k * kRectBlock + threadIdx.x) * 9 + q] = static_cast<float>(Hv[q]);
        }
    }
    __syncthreads();
    const int64_t rem = n - base;
    const int cnt = static_cast<int>(rem < ITEMS * kRectBlock ? rem : ITEMS * kRectBlock) * 9;
    float* out = H + 9 * base;
    const int n4 = cnt >> 2;
    for (int j = threadIdx.x; j < n4; j += kRectBlock)
        __stcs(reinterpret_cast<float4*>(out) + j, reinterpret_cast<const float4*>(stage)[j]);
    for (int j = (n4 << 2) + threadIdx.x; j < cnt; j += kRectBlock) out[j] = stage[j];
}

// ------------------------------------------------------------------------------------------
// Backward of G(offsets) = H / h33 ("naturally differential"): reverse mode
// through aca_rect_solve and the h33 normalisation, by hand, in fp64.  g[9] = dL/dG (g[8] ignored:
// G33 == 1), go[8] = dL/d offsets.  ~130 FLOPs.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void aca_rect_backward(const RectSrc& rs, const double o[8], const double g[9], double go[8])
{
    const double x0 = rs.x0, y0 = rs.y0, w = rs.w, h = rs.h, r = rs.r;
    // forward (same steps as aca_rect_solve)
    const double m2x = x0 + o[0],     m2y = y0 + o[1];
    const double n2x = x0 + w + o[2], n2y = y0 + o[3];
    const double q2x = x0 + w + o[4], q2y = y0 + h + o[5];
    const double p2x = x0 + o[6],     p2y = y0 + h + o[7];
    const double ax = n2x - m2x, ay = n2y - m2y, bx = p2x - m2x, by = p2y - m2y, qx = q2x - m2x, qy = q2y - m2y;
    const double fA2 = det2(ax, ay, bx, by), Q4x = det2(qx, qy, bx, by), Q4y = det2(ax, ay, qx, qy);
    const double t2 = fA2 - Q4x - Q4y;
    const double Bx = t2 * m2x, By = t2 * m2y;
    const double h11 = fma(Q4x, n2x, Bx), h21 = fma(Q4x, n2y, By), h31 = Q4x + t2;
    const double u12 = fma(Q4y, p2x, Bx), u22 = fma(Q4y, p2y, By), u32 = Q4y + t2;
    const double h12 = r * u12, h22 = r * u22, h32 = r * u32;
    const double h13 = -fma(x0, h11, fma(y0, h12, w * Bx));
    const double h23 = -fma(x0, h21, fma(y0, h22, w * By));
    const double h33 = -fma(x0, h31, fma(y0, h32, w * t2));
    // G = H / h33:  dL/dh_ij = g_ij / h33 (ij != 33),  dL/dh33 = -sum g_ij h_ij / h33^2
    const double inv = K<double>::rcp(h33);
    double g11 = g[0] * inv, g12 = g[1] * inv, g13 = g[2] * inv;
    double g21 = g[3] * inv, g22 = g[4] * inv, g23 = g[5] * inv;
    double g31 = g[6] * inv, g32 = g[7] * inv;
    const double dot = fma(g11, h11, fma(g12, h12, fma(g13, h13, fma(g21, h21, fma(g22, h22, fma(g23, h23, fma(g31, h31, g32 * h32)))))));
    const double g33 = -dot * inv;
    // third column: h_i3 = -(x0 h_i1 + y0 h_i2 + w {Bx, By, t2})
    g11 = fma(-x0, g13, g11); g12 = fma(-y0, g13, g12);
    g21 = fma(-x0, g23, g21); g22 = fma(-y0, g23, g22);
    g31 = fma(-x0, g33, g31); g32 = fma(-y0, g33, g32);
    double gBx = -w * g13, gBy = -w * g23, gt2 = -w * g33;
    // second column: h_i2 = r * u_i2, u = Q4y * p2 + B
    const double gu12 = r * g12, gu22 = r * g22, gu32 = r * g32;
    double gQ4y = fma(gu12, p2x, fma(gu22, p2y, gu32));
    double gp2x = gu12 * Q4y, gp2y = gu22 * Q4y;
    gBx += gu12; gBy += gu22; gt2 += gu32;
    // first column: h_i1 = Q4x * n2 + B
    double gQ4x = fma(g11, n2x, fma(g21, n2y, g31));
    double gn2x = g11 * Q4x, gn2y = g21 * Q4x;
    gBx += g11; gBy += g21; gt2 += g31;
    // B = t2 * m2
    gt2 = fma(gBx, m2x, fma(gBy, m2y, gt2));
    double gm2x = gBx * t2, gm2y = gBy * t2;
    // t2 = fA2 - Q4x - Q4y
    const double gfA2 = gt2;
    gQ4x -= gt2; gQ4y -= gt2;
    // the three determinants
    double gax = fma(gQ4y, qy, gfA2 * by),  gay = -fma(gQ4y, qx, gfA2 * bx);
    double gbx = -fma(gQ4x, qy, gfA2 * ay), gby = fma(gQ4x, qx, gfA2 * ax);
    double gqx = fma(gQ4x, by, -gQ4y * ay), gqy = fma(gQ4y, ax, -gQ4x * bx);
    // a = n2 - m2, b = p2 - m2, q = q2 - m2
    gn2x += gax; gn2y += gay; gp2x += gbx; gp2y += gby;
    gm2x -= gax + gbx + gqx; gm2y -= gay + gby + gqy;
    go[0] = gm2x; go[1] = gm2y; go[2] = gn2x; go[3] = gn2y; go[4] = gqx; go[5] = gqy; go[6] = gp2x; go[7] = gp2y;
}

// offsets float[n][4][2], grad_G float[n][3][3], grad_off float[n][4][2].
// The SoA skeleton plus a transpose inside the warp: a warp owns a tile of 128 consecutive items (4 per lane).  Its
// 4 KB of offsets and 4.5 KB of gradient records are contiguous, so the lanes fetch them with 17 fully coalesced
// 128-bit loads each (all issued before the first use), park them in the warp's own slice of shared memory, and after
// a __syncwarp every lane picks up the records of its four items; results travel back the same way and leave with 8
// coalesced 128-bit stores per lane.  No CTA barrier, four independent fp64 chains per thread.  16-byte chunks of the
// 32-byte records are XOR-swizzled by their row so that both directions are bank-conflict free (36-byte records
// advance by 9 chunks per lane: conflict free as they are).  The first version (two items per thread, load -> CTA
// barrier -> compute) reached 0.89 of the HBM roofline; a lane reading its own 128 B directly from global memory 0.65.
constexpr int kBwdItems = 4;                              // items per lane
constexpr int kBwdTile = 32 * kBwdItems;                  // items per warp
constexpr int kBwdWarpFloats = kBwdTile * (8 + 9);        // floats of shared memory per warp

__device__ __forceinline__ int swz(int chunk) { return chunk ^ ((chunk >> 3) & 7); }     // 16-byte chunks, 8 per 128-byte row

__global__ void __launch_bounds__(kRectBlock, 2)
rect_backward_kernel(const float* __restrict__ offsets, RectSrc rs, const float* __restrict__ grad_G,
                     float* __restrict__ grad_off, int64_t n)
{
    extern __shared__ __align__(128) float bwd_smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t tile0 = (static_cast<int64_t>(blockIdx.x) * (kRectBlock / 32) + warp) * kBwdTile;
    if (tile0 >= n) return;
    if (tile0 + kBwdTile <= n) {
        float4* so = reinterpret_cast<float4*>(bwd_smem + warp * kBwdWarpFloats);       // 256 chunks: offsets, later results
        float4* sg = so + 2 * kBwdTile;                                                   // 288 chunks: gradient records
        const float4* op = reinterpret_cast<const float4*>(offsets + 8 * tile0);
        const float4* gp = reinterpret_cast<const float4*>(grad_G + 9 * tile0);
        float4 lo[8], lg[9];
#pragma unroll
        for (int k = 0; k < 8; ++k) lo[k] = __ldcs(op + 32 * k + lane);
#pragma unroll
        for (int k = 0; k < 9; ++k) lg[k] = __ldcs(gp + 32 * k + lane);
#pragma unroll
        for (int k = 0; k < 8; ++k) so[swz(32 * k + lane)] = lo[k];
#pragma unroll
        for (int k = 0; k < 9; ++k) sg[32 * k + lane] = lg[k];
        __syncwarp();
        float4 mo[8], mg[9];                                  // this lane's four items: chunks 8*lane.. and 9*lane..
#pragma unroll
        for (int k = 0; k < 8; ++k) mo[k] = so[swz(8 * lane + k)];
#pragma unroll
        for (int k = 0; k < 9; ++k) mg[k] = sg[9 * lane + k];
        __syncwarp();                                         // the offsets area is rewritten with results below
        const float* of = reinterpret_cast<const float*>(mo);
        const float* gf = reinterpret_cast<const float*>(mg);
#pragma unroll
        for (int v = 0; v < kBwdItems; ++v) {
            double o[8], g[9], go[8];
#pragma unroll
            for (int q = 0; q < 8; ++q) o[q] = static_cast<double>(of[8 * v + q]);
#pragma unroll
            for (int q = 0; q < 9; ++q) g[q] = static_cast<double>(gf[9 * v + q]);
            aca_rect_backward(rs, o, g, go);
            so[swz(8 * lane + 2 * v)]     = make_float4(float(go[0]), float(go[1]), float(go[2]), float(go[3]));
            so[swz(8 * lane + 2 * v + 1)] = make_float4(float(go[4]), float(go[5]), float(go[6]), float(go[7]));
        }
        __syncwarp();
        float4* out = reinterpret_cast<float4*>(grad_off + 8 * tile0);
#pragma unroll
        for (int k = 0; k < 8; ++k) __stcs(out + 32 * k + lane, so[swz(32 * k + lane)]);
    } else {                                                  // the last, partial tile: item by item
        for (int64_t i = tile0 + lane; i < n; i += 32) {
            double o[8], g[9], go[8];
#pragma unroll
            for (int q = 0; q < 8; ++q) o[q] = static_cast<double>(__ldcs(offsets + 8 * i + q));
#pragma unroll
            for (int q = 0; q < 9; ++q) g[q] = static_cast<double>(__ldcs(grad_G + 9 * i + q));
            aca_rect_backward(rs, o, g, go);
#pragma unroll
            for (int q = 0; q < 8; ++q) __stcs(grad_off + 8 * i + q, static_cast<float>(go[q]));
        }
    }
}

// SoA form of the backward: offsets = float[8][n] planes, grad_G = float[9][n] planes, grad_off = float[8][n] planes.
// The forward streaming skeleton: thread per V items, 17 independent 128-bit loads, V fp64 chains, 8 stores.
template <int V>
__global__ void __launch_bounds__(kRectBlock, 2)
rect_backward_soa_kernel(const float* __restrict__ offsets, RectSrc rs, const float* __restrict__ grad_G,
                         float* __restrict__ grad_off, int64_t n_vec, int64_t stride)
{
    const int64_t t = static_cast<int64_t>(blockIdx.x) * kRectBlock + threadIdx.x;
    if (t >= n_vec) return;
    const int64_t off = t * V;
    Vec<V> o[8], g[9];
#pragma unroll
    for (int k = 0; k < 8; ++k) o[k] = ld_stream<V>(offsets + k * stride + off);
#pragma unroll
    for (int k = 0; k < 9; ++k) g[k] = ld_stream<V>(grad_G + k * stride + off);
    Vec<V> r[8];
#pragma unroll
    for (int v = 0; v < V; ++v) {
        double ov[8], gv[9], go[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) ov[k] = static_cast<double>(o[k].v[v]);
#pragma unroll
        for (int k = 0; k < 9; ++k) gv[k] = static_cast<double>(g[k].v[v]);
        aca_rect_backward(rs, ov, gv, go);
#pragma unroll
        for (int k = 0; k < 8; ++k) r[k].v[v] = static_cast<float>(go[k]);
    }
#pragma unroll
    for (int k = 0; k < 8; ++k) st_stream<V>(grad_off + k * stride + off, r[k]);
}

template <class T>
static int rect_dispatch(const float* offsets, const RectSrc& rs, float* H, int64_t n, hg_layout_t layout, int norm, cudaStream_t st)
{
    if (layout == HG_SOA) {
        if (n % 4 == 0) {
            const int64_t nv = n / 4, blocks = (nv + kRectBlock - 1) / kRectBlock;
            rect_soa_kernel<T, 4><<<static_cast<unsigned>(blocks), kRectBlock, 0, st>>>(offsets, rs, H, nv, n, norm);
        } else {
            const int64_t blocks = (n + kRectBlock - 1) / kRectBlock;
            rect_soa_kernel<T, 1><<<static_cast<unsigned>(blocks), kRectBlock, 0, st>>>(offsets, rs, H, n, n, norm);
        }
    } else {
        const int64_t blocks = (n + 2 * kRectBlock - 1) / (2 * kRectBlock);
        rect_aos_kernel<T><<<static_cast<unsigned>(blocks), kRectBlock, 0, st>>>(offsets, rs, H, n, norm);
    }
    return launch_status();
}

// ------------------------------------------------------------------------------------------
// Backward through the grid (second half): dL/d offsets of
//   grid[b][j][i] = pi(G_b (x_i, y_j, 1)),  G = H / h33,  H from the offsets (Algorithm 1)
// given dL/d grid.  One CTA per item, the shape of the forward kernel run in reverse: warp 0 solves H in fp64 and folds
// the lattice into it (so the sweep uses integer pixel indices), every thread streams its share of the item's gradient
// (8 B per pixel, 128-bit loads, four in flight) and accumulates, in fp32, the nine sums
//   S_r = sum over pixels of coef_r * (i, j, 1),  coef = (g_u / W,  g_v / W,  -(g_u u + g_v v) / W)
// (the projection's own partials, quotient rule); the CTA reduces them in fp64 and one thread unfolds the lattice
// (dL/dG_r = L S_r) and leaves dL/dG -- its eight used entries in the item's grad_offsets record, all nine in grad_G
// when that is asked for.  A second, thread-per-item kernel then runs the hand-written reverse mode of Algorithm 1 above
// in place.  (Done at the end of the streaming kernel by one thread, those ~130 dependent fp64 operations held the CTA's
// slot for 2 of its 11 microseconds and cost 80 registers: 0.77 of the copy rate; split: see DESIGN.md.)
// Read-bound: 8 B per pixel in, 32 B per item out.
// ------------------------------------------------------------------------------------------
constexpr int kGridBwdDepth = 3;             // batches of four units in flight per thread (asynchronous copies)
__device__ __forceinline__ float rcp_approx(float x) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }

// One pixel.  Packed fp32 throughout: rows 1 and 2 of L as the halves of one register pair, so that (X, Y), (u, v), the
// coefficients (g_u, g_v) / W and their three accumulators are FFMA2 / FMUL2 / FADD2 -- 14 issued instructions per pixel
// instead of 25 (the kernel was issue-bound before: 0.86 of the copy rate).
//   acc[0] = sum (a, b) i,  acc[1] = sum (a, b) j,  acc[2] = sum (a, b),  acc[3] = sum c' (i, j),  c0 = sum c',   c' = a u + b v
__device__ __forceinline__ void grid_bwd_pixel(const float2 l01, const float2 l02, const float2 l03, float l6, float l7, float l8,
                                               float fi, float fj, float2 g, float2 acc[4], float& c0)
{
    const float2 I = make_float2(fi, fi), J = make_float2(fj, fj);
    const float2 XY = __ffma2_rn(l01, I, __ffma2_rn(l02, J, l03));
    const float W = fmaf(l6, fi, fmaf(l7, fj, l8));
    const float q = rcp_approx(W);
    const float2 Q = make_float2(q, q);
    const float2 uv = __fmul2_rn(XY, Q), ab = __fmul2_rn(g, Q);
    const float2 p = __fmul2_rn(ab, uv);
    const float c = p.x + p.y;
    acc[0] = __ffma2_rn(ab, I, acc[0]);
    acc[1] = __ffma2_rn(ab, J, acc[1]);
    acc[2] = __fadd2_rn(acc[2], ab);
    acc[3] = __ffma2_rn(make_float2(c, c), make_float2(fi, fj), acc[3]);
    c0 += c;
}

template <int PIX>   // 2: grid_w even, one 128-bit load covers two pixels of a row; 1: 64-bit load per pixel
__global__ void __launch_bounds__(kRectBlock)
grid_backward_kernel(const float* __restrict__ offsets, RectSrc rs, int grid_w, int grid_h, double step_x, double step_y,
                     const float* __restrict__ grad_grid, float* __restrict__ grad_offsets, float* __restrict__ grad_G)
{
    __shared__ float lh[9];
    __shared__ double red[kRectBlock / 32][9];
    const int64_t b = blockIdx.x;
    const int per_row = grid_w / PIX;
    const int total = per_row * grid_h;
    const float* g_item = grad_grid + static_cast<int64_t>(2) * grid_w * grid_h * b;
    const int d_row = kRectBlock / per_row, d_col = kRectBlock - d_row * per_row;
    const int row0 = threadIdx.x / per_row;
    float frow = static_cast<float>(row0), fcol = static_cast<float>(PIX * (static_cast<int>(threadIdx.x) - row0 * per_row));   // lattice indices, exact in fp32
    const float f_drow = static_cast<float>(d_row), f_dcol = static_cast<float>(PIX * d_col), f_width = static_cast<float>(PIX * per_row);
    constexpr int kUnitBytes = 8 * PIX;
    constexpr int kDepth = kGridBwdDepth;
    extern __shared__ __align__(16) unsigned char stage_raw[];
    unsigned char (*stage)[4][kRectBlock][kUnitBytes] = reinterpret_cast<unsigned char (*)[4][kRectBlock][kUnitBytes]>(stage_raw);
    auto issue = [&](int batch, int slot) {
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int qc = min((batch * 4 + u) * kRectBlock + static_cast<int>(threadIdx.x), total - 1);   // past the end: read again, zeroed below
            const uint32_t dst = smem_u32(&stage[slot][u][threadIdx.x][0]);
            const void* src = reinterpret_cast<const unsigned char*>(g_item) + static_cast<size_t>(qc) * kUnitBytes;
            if (PIX == 2) asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" :: "r"(dst), "l"(src) : "memory");
            else          asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" :: "r"(dst), "l"(src) : "memory");
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    const int n_batches = (total + 4 * kRectBlock - 1) / (4 * kRectBlock);
    issue(0, 0);                                 // in flight while warp 0 solves
    if (n_batches > 1) issue(1, 1);
    else asm volatile("cp.async.commit_group;" ::: "memory");
    if (threadIdx.x < 32) {
        const float4* op = reinterpret_cast<const float4*>(offsets + 8 * b);
        const float4 o0 = __ldg(op), o1 = __ldg(op + 1);
        const double ov[8] = { o0.x, o0.y, o0.z, o0.w, o1.x, o1.y, o1.z, o1.w };
        double Hd[9];
        aca_rect_solve<double>(rs, ov, Hd);
        const double r = K<double>::rcp(Hd[8]);
        if (threadIdx.x == 0) {
#pragma unroll
            for (int r3 = 0; r3 < 3; ++r3) {              // L = G * [sx 0 x0; 0 sy y0; 0 0 1]
                const double a = Hd[3 * r3] * r, bb = Hd[3 * r3 + 1] * r, c = Hd[3 * r3 + 2] * r;
                lh[3 * r3]     = static_cast<float>(a * step_x);
                lh[3 * r3 + 1] = static_cast<float>(bb * step_y);
                lh[3 * r3 + 2] = static_cast<float>(fma(a, rs.x0, fma(bb, rs.y0, c)));
            }
        }
    }
    __syncthreads();
    const float2 l01 = make_float2(lh[0], lh[3]), l02 = make_float2(lh[1], lh[4]), l03 = make_float2(lh[2], lh[5]);
    const float l6 = lh[6], l7 = lh[7], l8 = lh[8];
    float2 acc[4];
    float c0 = 0.f;
#pragma unroll
    for (int k = 0; k < 4; ++k) acc[k] = make_float2(0.f, 0.f);

    // units of PIX pixels, row-major; this thread takes units tid, tid + 256, ...; (col, row) advance without a division.
    // The gradient comes through per-thread asynchronous copies (LDGSTS, L1 bypassed) into the thread's own slots of shared
    // memory, three batches of four 16-byte units in flight per thread: bytes in flight do not cost registers (with plain
    // loads ptxas kept two of the four in flight at 54 registers and the kernel ran at 0.62 of the copy rate), and since a
    // thread reads back only what it copied itself, no barrier is needed -- cp.async.wait_group orders it.
    // one batch = four units of this thread from slot `slot`; RAGGED: units past the end of the item count as a zero gradient
    auto batch = [&](int k, int slot, auto ragged) {
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            float4 g4;
            if (PIX == 2) g4 = *reinterpret_cast<const float4*>(&stage[slot][u][threadIdx.x][0]);
            else { const float2 t = *reinterpret_cast<const float2*>(&stage[slot][u][threadIdx.x][0]); g4 = make_float4(t.x, t.y, 0.f, 0.f); }
            float fi = fcol, fj = frow;
            if (decltype(ragged)::value && (k * 4 + u) * kRectBlock + static_cast<int>(threadIdx.x) >= total) {
                g4 = make_float4(0.f, 0.f, 0.f, 0.f); fi = 0.f; fj = 0.f;                 // lattice point (0, 0): a finite W
            }
            grid_bwd_pixel(l01, l02, l03, l6, l7, l8, fi, fj, make_float2(g4.x, g4.y), acc, c0);
            if (PIX == 2) grid_bwd_pixel(l01, l02, l03, l6, l7, l8, fi + 1.f, fj, make_float2(g4.z, g4.w), acc, c0);
            fcol += f_dcol; frow += f_drow;
            if (fcol >= f_width) { fcol -= f_width; frow += 1.f; }
        }
    };
    int slot = 0;
    for (int k = 0; k < n_batches; ++k) {
        const int next = slot + 2 >= kDepth ? slot + 2 - kDepth : slot + 2;
        if (k + 2 < n_batches) issue(k + 2, next);
        else asm volatile("cp.async.commit_group;" ::: "memory");
        asm volatile("cp.async.wait_group 2;" ::: "memory");
        if ((k + 1) * 4 * kRectBlock <= total) batch(k, slot, std::false_type());       // CTA-uniform: only the last batch can be ragged
        else batch(k, slot, std::true_type());
        slot = slot + 1 == kDepth ? 0 : slot + 1;
    }
    // S_1 = (a i, a j, a), S_2 = (b i, b j, b), S_3 = -(c' i, c' j, c')
    const float s[9] = { acc[0].x, acc[1].x, acc[2].x, acc[0].y, acc[1].y, acc[2].y, -acc[3].x, -acc[3].y, -c0 };

    // CTA reduction: fp32 across the lanes of a warp (a 5-level tree on 32 partial sums), fp64 across warps
    double sd[9];
#pragma unroll
    for (int k = 0; k < 9; ++k) {
        float t = s[k];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
        sd[k] = static_cast<double>(t);
    }
    if ((threadIdx.x & 31) == 0) {
#pragma unroll
        for (int k = 0; k < 9; ++k) red[threadIdx.x >> 5][k] = sd[k];
    }
    __syncthreads();
    if (threadIdx.x != 0) return;
    double S[9], dG[9];
#pragma unroll
    for (int k = 0; k < 9; ++k) {
        double t = 0.0;
#pragma unroll
        for (int w = 0; w < kRectBlock / 32; ++w) t += red[w][k];
        S[k] = t;
    }
#pragma unroll
    for (int row3 = 0; row3 < 3; ++row3) {               // dL/dG_r = L S_r
        dG[3 * row3]     = fma(step_x, S[3 * row3], rs.x0 * S[3 * row3 + 2]);
        dG[3 * row3 + 1] = fma(step_y, S[3 * row3 + 1], rs.y0 * S[3 * row3 + 2]);
        dG[3 * row3 + 2] = S[3 * row3 + 2];
    }
    float4* out = reinterpret_cast<float4*>(grad_offsets + 8 * b);       // dL/dG[0..7], finished in place by the kernel below
    out[0] = make_float4(static_cast<float>(dG[0]), static_cast<float>(dG[1]), static_cast<float>(dG[2]), static_cast<float>(dG[3]));
    out[1] = make_float4(static_cast<float>(dG[4]), static_cast<float>(dG[5]), static_cast<float>(dG[6]), static_cast<float>(dG[7]));
    if (grad_G != nullptr) {
#pragma unroll
        for (int k = 0; k < 9; ++k) grad_G[9 * b + k] = static_cast<float>(dG[k]);
    }
}

// grad_offsets[b] holds dL/dG[0..7] (fp32) on entry and dL/d offsets on exit: the reverse mode of Algorithm 1, thread per item.
__global__ void __launch_bounds__(kRectBlock)
grid_backward_finish_kernel(const float* __restrict__ offsets, RectSrc rs, float* __restrict__ grad_offsets, int64_t n)
{
    const int64_t b = static_cast<int64_t>(blockIdx.x) * kRectBlock + threadIdx.x;
    if (b >= n) return;
    const float4* op = reinterpret_cast<const float4*>(offsets + 8 * b);
    float4* gp = reinterpret_cast<float4*>(grad_offsets + 8 * b);
    const float4 o0 = __ldg(op), o1 = __ldg(op + 1), g0 = gp[0], g1 = gp[1];
    const double ov[8] = { o0.x, o0.y, o0.z, o0.w, o1.x, o1.y, o1.z, o1.w };
    const double dG[9] = { g0.x, g0.y, g0.z, g0.w, g1.x, g1.y, g1.z, g1.w, 0.0 };
    double go[8];
    aca_rect_backward(rs, ov, dG, go);
    gp[0] = make_float4(static_cast<float>(go[0]), static_cast<float>(go[1]), static_cast<float>(go[2]), static_cast<float>(go[3]));
    gp[1] = make_float4(static_cast<float>(go[4]), static_cast<float>(go[5]), static_cast<float>(go[6]), static_cast<float>(go[7]));
}

}  // namespace hg

extern "C" int hg_aca_rect_batched(const float* offsets, float x0, float y0, float w, float h, float* H, int64_t n,
                                   hg_layout_t layout, hg_norm_t norm, hg_precision_t prec, void* cuda_stream)
{
    using namespace hg;
    if (n < 0) return HG_ERR_INVALID_ARG;
    if (layout != HG_SOA && layout != HG_AOS) return HG_ERR_INVALID_ARG;
    if (norm != HG_NORM_NONE && norm != HG_NORM_H33 && norm != HG_NORM_FROBENIUS) return HG_ERR_INVALID_ARG;
    if (prec != HG_PREC_F64 && prec != HG_PREC_F32) return HG_ERR_INVALID_ARG;
    if (!(w != 0.0f) || !(h != 0.0f) || !(w == w) || !(h == h)) return HG_ERR_INVALID_ARG;
    if (n == 0) return HG_OK;
    if (!offsets || !H) return HG_ERR_INVALID_ARG;
    if (!aligned16(offsets) || !aligned16(H)) return HG_ERR_ALIGNMENT;
    if ((n + kRectBlock - 1) / kRectBlock > 0x7fffffffLL) return HG_ERR_INVALID_ARG;
    RectSrc rs;
    rs.x0 = x0; rs.y0 = y0; rs.w = w; rs.h = h; rs.r = double(w) / double(h);
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    return prec == HG_PREC_F64 ? rect_dispatch<double>(offsets, rs, H, n, layout, int(norm), st)
                               : rect_dispatch<float>(offsets, rs, H, n, layout, int(norm), st);
}

extern "C" int hg_aca_rect_backward_soa(const float* offsets, float x0, float y0, float w, float h, const float* grad_H,
                                        float* grad_offsets, int64_t n, void* cuda_stream)
{
    using namespace hg;
    if (n < 0) return HG_ERR_INVALID_ARG;
    if (!(w != 0.0f) || !(h != 0.0f) || !(w == w) || !(h == h)) return HG_ERR_INVALID_ARG;
    if (n == 0) return HG_OK;
    if (!offsets || !grad_H || !grad_offsets) return HG_ERR_INVALID_ARG;
    if (!aligned16(offsets) || !aligned16(grad_H) || !aligned16(grad_offsets)) return HG_ERR_ALIGNMENT;
    if ((n + kRectBlock - 1) / kRectBlock > 0x7fffffffLL) return HG_ERR_INVALID_ARG;
    RectSrc rs;
    rs.x0 = x0; rs.y0 = y0; rs.w = w; rs.h = h; rs.r = double(w) / double(h);
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    if (n % 4 == 0) {
        const int64_t nv = n / 4, blocks = (nv + kRectBlock - 1) / kRectBlock;
        rect_backward_soa_kernel<4><<<static_cast<unsigned>(blocks), kRectBlock, 0, st>>>(offsets, rs, grad_H, grad_offsets, nv, n);
    } else {
        const int64_t blocks = (n + kRectBlock - 1) / kRectBlock;
        rect_backward_soa_kernel<1><<<static_cast<unsigned>(blocks), kRectBlock, 0, st>>>(offsets, rs, grad_H, grad_offsets, n, n);
    }
    return launch_status();
}

extern "C" int hg_aca_rect_backward(const float* offsets, float x0, float y0, float w, float h, const float* grad_H,
                                    float* grad_offsets, int64_t n, void* cuda_stream)
{
    using namespace hg;
    if (n < 0) return HG_ERR_INVALID_ARG;
    if (!(w != 0.0f) || !(h != 0.0f) || !(w == w) || !(h == h)) return HG_ERR_INVALID_ARG;
    if (n == 0) return HG_OK;
    if (!offsets || !grad_H || !grad_offsets) return HG_ERR_INVALID_ARG;
    if (!aligned16(offsets) || !aligned16(grad_H) || !aligned16(grad_offsets)) return HG_ERR_ALIGNMENT;
    if ((n + kRectBlock - 1) / kRectBlock > 0x7fffffffLL) return HG_ERR_INVALID_ARG;
    RectSrc rs;
    rs.x0 = x0; rs.y0 = y0; rs.w = w; rs.h = h; rs.r = double(w) / double(h);
    const int64_t per_block = int64_t(kRectBlock / 32) * kBwdTile;
    const int64_t blocks = (n + per_block - 1) / per_block;
    const size_t smem = size_t(kRectBlock / 32) * kBwdWarpFloats * sizeof(float);
    if (cudaFuncSetAttribute(rect_backward_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, int(smem)) != cudaSuccess)
        return HG_ERR_CUDA;
    rect_backward_kernel<<<static_cast<unsigned>(blocks), kRectBlock, smem, static_cast<cudaStream_t>(cuda_stream)>>>(
        offsets, rs, grad_H, grad_offsets, n);
    return launch_status();
}

extern "C" int hg_offsets_to_grid_backward(const float* offsets, float x0, float y0, float w, float h, int32_t grid_w, int32_t grid_h,
                                           const float* grad_grid, float* grad_offsets, float* grad_G, int64_t n, void* cuda_stream)
{
    using namespace hg;
    if (n < 0 || grid_w < 1 || grid_h < 1) return HG_ERR_INVALID_ARG;
    if (grid_w > (1 << 24) || grid_h > (1 << 24) || static_cast<int64_t>(grid_w) * grid_h > 0x3fffffffLL)
        return HG_ERR_INVALID_ARG;                      // lattice indices are carried in fp32 (exact below 2^24)
    if (!(w != 0.0f) || !(h != 0.0f) || !(w == w) || !(h == h)) return HG_ERR_INVALID_ARG;
    if (n == 0) return HG_OK;
    if (!offsets || !grad_grid || !grad_offsets) return HG_ERR_INVALID_ARG;
    if (!aligned16(offsets) || !aligned16(grad_grid) || !aligned16(grad_offsets) || (grad_G && !aligned4(grad_G))) return HG_ERR_ALIGNMENT;
    if (n > 0x7fffffffLL) return HG_ERR_INVALID_ARG;
    RectSrc rs;
    rs.x0 = x0; rs.y0 = y0; rs.w = w; rs.h = h; rs.r = double(w) / double(h);
    const double step_x = (grid_w > 1) ? double(w) / double(grid_w - 1) : 0.0;
    const double step_y = (grid_h > 1) ? double(h) / double(grid_h - 1) : 0.0;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const size_t smem = size_t(kGridBwdDepth) * 4 * kRectBlock * (grid_w % 2 == 0 ? 16 : 8);
    if (cudaFuncSetAttribute(grid_backward_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(size_t(kGridBwdDepth) * 4 * kRectBlock * 16)) != cudaSuccess)
        return HG_ERR_CUDA;
    if (grid_w % 2 == 0)
        grid_backward_kernel<2><<<static_cast<unsigned>(n), kRectBlock, smem, st>>>(offsets, rs, grid_w, grid_h, step_x, step_y, grad_grid,
                                                                               grad_offsets, grad_G);
    else
        grid_backward_kernel<1><<<static_cast<unsigned>(n), kRectBlock, smem, st>>>(offsets, rs, grid_w, grid_h, step_x, step_y, grad_grid,
                                                                               grad_offsets, grad_G);
    if (launch_status() != HG_OK) return HG_ERR_CUDA;
    grid_backward_finish_kernel<<<static_cast<unsigned>((n + kRectBlock - 1) / kRectBlock), kRectBlock, 0, st>>>(offsets, rs, grad_offsets, n);
    return launch_status();
}
