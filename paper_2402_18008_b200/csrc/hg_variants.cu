// hg_variants.cu -- solver variants of SURVEY.md 8(f) rows 3-4 on the streaming skeleton:
//   hg_affine_batched      affine H_A = H_A2^-1 * H_A1 from three correspondences (Eq. 41)
//   hg_sk_batched          simplified SK, Hbar = H_S2^-1 * H_K for a fixed object pattern (Eq. 17)
//   hg_aca_batched_f64 / hg_sks_batched_f64   the general solvers with fp64 storage, the precision of
//                          the paper's own GPU experiment ("double-precision floating-point")
// One generic kernel pair (SoA / AoS) parameterised by the per-set operation and the storage type; every
// access is a 128-bit (or, for 24-byte records, 64-bit) streaming load/store.  All HBM-bound.
#include "hg_device.cuh"
#include "hg_host.h"

namespace hg {

constexpr int kVarBlock = 256;

// ---- per-set operations ------------------------------------------------------------------------
// Each Op declares NA / NB = scalars read per set from the first / second input array and
// apply(x, H): x[0..NA) from the first array, x[NA..NA+NB) from the second.

// Eq. 41 first row: H_A = H_A2^-1 * H_A1, H_A1 = [b1y -b1x 0; -a1y a1x 0; 0 0 fA1] * T(-M1) (Eq. 23, R2),
// H_A2^-1 = [M2N2 M2P2 M2; 0 0 1] (Eq. 25, R1).  33 FLOPs, no division; h31 = h32 = 0, h33 = f_A1.
struct AffineOp {
    static constexpr int NA = 6, NB = 6;
    template <class T> __device__ __forceinline__ void apply(const T* x, T H[9]) const
    {
        const T* s = x; const T* d = x + 6;
        const T a1x = s[2] - s[0], a1y = s[3] - s[1], b1x = s[4] - s[0], b1y = s[5] - s[1];
        const T a2x = d[2] - d[0], a2y = d[3] - d[1], b2x = d[4] - d[0], b2y = d[5] - d[1];
        const T fA1 = det2(a1x, a1y, b1x, b1y);
        const T h11 = det2(a2x, b2x, a1y, b1y);            // a2x*b1y - b2x*a1y
        const T h12 = det2(b2x, a2x, b1x, a1x);            // b2x*a1x - a2x*b1x
        const T h21 = det2(a2y, b2y, a1y, b1y);
        const T h22 = det2(b2y, a2y, b1x, a1x);
        H[0] = h11; H[1] = h12; H[2] = K<T>::fma(-h12, s[1], K<T>::fma(-h11, s[0], fA1 * d[0]));
        H[3] = h21; H[4] = h22; H[5] = K<T>::fma(-h22, s[1], K<T>::fma(-h21, s[0], fA1 * d[1]));
        H[6] = T(0); H[7] = T(0); H[8] = fA1;
    }
};

// Eq. 17: Hbar = H_S2^-1 * H_K.  The object pattern is fixed for the call: P5, Q7 and the reciprocal of
// Eq. 14's determinant are call constants (Table 3 row "SK": zero per-image cost); per image the
// target-side half of SKS remains: two reciprocals.
struct SkOp {
    static constexpr int NA = 8, NB = 0;
    double P5x, P5y, Q7x, Q7y, rden;
    template <class T> __device__ __forceinline__ void apply(const T* d, T H[9]) const
    {
        const T half = T(0.5);
        const T p5x = T(P5x), p5y = T(P5y), q7x = T(Q7x), q7y = T(Q7y), rd = T(rden);
        const T O2x = half * (d[0] + d[2]), O2y = half * (d[1] + d[3]);
        const T v2x = d[2] - O2x, v2y = d[3] - O2y;
        const T f2 = K<T>::fma(v2x, v2x, v2y * v2y);
        T ex = d[4] - O2x, ey = d[5] - O2y;
        const T P4x = K<T>::fma(v2x, ex, v2y * ey), P4y = det2(v2x, v2y, ex, ey);
        ex = d[6] - O2x; ey = d[7] - O2y;
        const T Q4x = K<T>::fma(v2x, ex, v2y * ey), Q4y = det2(v2x, v2y, ex, ey);
        T r = K<T>::rcp(P4y); const T P6x = P4x * r, P6y = f2 * r;
        r = K<T>::rcp(Q4y);   const T Q6x = Q4x * r, Q6y = f2 * r;
        const T Q8x = Q6x - P6x, Q8y = Q6y - P6y;
        const T aK = det2(Q8x, Q8y, q7y, q7x) * rd;          // (Q8x*Q7x - Q8y*Q7y) / den
        const T bK = det2(Q8y, Q8x, q7y, q7x) * rd;
        const T uK = K<T>::fma(-bK, p5y, K<T>::fma(-aK, p5x, P6x));
        const T vK = K<T>::fma(-aK, p5y, K<T>::fma(-bK, p5x, P6y));
        H[0] = K<T>::fma(v2x, aK, O2x * bK);
        H[1] = K<T>::fma(v2x, uK, K<T>::fma(O2x, vK, -v2y));
        H[2] = K<T>::fma(v2x, bK, O2x * aK);
        H[3] = K<T>::fma(v2y, aK, O2y * bK);
        H[4] = K<T>::fma(v2y, uK, K<T>::fma(O2y, vK, v2x));
        H[5] = K<T>::fma(v2y, bK, O2y * aK);
        H[6] = bK; H[7] = vK; H[8] = aK;
    }
};

template <int METHOD>
struct GeneralOp {
    static constexpr int NA = 8, NB = 8;
    template <class T> __device__ __forceinline__ void apply(const T* x, T H[9]) const { solve<METHOD, T>(x, x + 8, H); }
};

// ---- 16-byte streaming vectors of the storage type ---------------------------------------------
template <class IO> struct IoVec;
template <> struct IoVec<float> {
    static constexpr int V = 4;
    float v[4];
    static __device__ __forceinline__ IoVec ld(const float* p)
    { const float4 t = __ldcs(reinterpret_cast<const float4*>(p)); IoVec r; r.v[0] = t.x; r.v[1] = t.y; r.v[2] = t.z; r.v[3] = t.w; return r; }
    __device__ __forceinline__ void st(float* p) const { __stcs(reinterpret_cast<float4*>(p), make_float4(v[0], v[1], v[2], v[3])); }
};
template <> struct IoVec<double> {
    static constexpr int V = 2;
    double v[2];
    static __device__ __forceinline__ IoVec ld(const double* p)
    { const double2 t = __ldcs(reinterpret_cast<const double2*>(p)); IoVec r; r.v[0] = t.x; r.v[1] = t.y; return r; }
    __device__ __forceinline__ void st(double* p) const { __stcs(reinterpret_cast<double2*>(p), make_double2(v[0], v[1])); }
};

// SoA: a = IO[NA][stride], b = IO[NB][stride], H = IO[9][stride].  VEC = true: thread per 16 bytes of each plane.
template <class Op, class IO, class T, bool VEC>
__global__ void __launch_bounds__(kVarBlock)
variant_soa_kernel(const IO* __restrict__ a, const IO* __restrict__ b, IO* __restrict__ H, int64_t n_thr, int64_t stride,
                   int norm, Op op)
{
    constexpr int V = VEC ? IoVec<IO>::V : 1;
    constexpr int NA = Op::NA, NB = Op::NB;
    const int64_t t = static_cast<int64_t>(blockIdx.x) * kVarBlock + threadIdx.x;
    if (t >= n_thr) return;
    const int64_t off = t * V;
    IO in[NA + NB][V];
#pragma unroll
    for (int k = 0; k < NA + NB; ++k) {
        const IO* p = (k < NA ? a + k * stride : b + (k - NA) * stride) + off;
        if (VEC) { const IoVec<IO> x = IoVec<IO>::ld(p);
#pragma unroll
                   for (int v = 0; v < V; ++v) in[k][v] = x.v[v]; }
        else in[k][0] = __ldcs(p);
    }
    IO out[9][V];
#pragma unroll
    for (int v = 0; v < V; ++v) {
        T x[NA + NB], Hv[9];
#pragma unroll
        for (int k = 0; k < NA + NB; ++k) x[k] = static_cast<T>(in[k][v]);
        op.template apply<T>(x, Hv);
        normalise<T>(Hv, norm);
#pragma unroll
        for (int k = 0; k < 9; ++k) out[k][v] = static_cast<IO>(Hv[k]);
    }
#pragma unroll
    for (int k = 0; k < 9; ++k) {
        IO* p = H + k * stride + off;
        if (VEC) { IoVec<IO> x;
#pragma unroll
                   for (int v = 0; v < V; ++v) x.v[v] = out[k][v];
                   x.st(p); }
        else __stcs(p, out[k][0]);
    }
}

// One AoS record of N scalars, read with the widest aligned vector loads its size allows.
template <class IO, int N>
__device__ __forceinline__ void load_record(const IO* __restrict__ p, IO x[N])
{
    constexpr int bytes = N * int(sizeof(IO));
    if (bytes % 16 == 0) {
        const int4* q = reinterpret_cast<const int4*>(p);
#pragma unroll
        for (int j = 0; j < bytes / 16; ++j) { const int4 t = __ldcs(q + j); reinterpret_cast<int4*>(x)[j] = t; }
    } else {
        const int2* q = reinterpret_cast<const int2*>(p);
#pragma unroll
        for (int j = 0; j < bytes / 8; ++j) { const int2 t = __ldcs(q + j); reinterpret_cast<int2*>(x)[j] = t; }
    }
}

// AoS: a = IO[n][NA], b = IO[n][NB], H = IO[n][9] (records transposed through shared memory for contiguous stores).
// ITEMS records per thread (i, i + kVarBlock, ...), all loads issued before the first use: a thin input stream
// (32 B per set) needs two to keep enough bytes in flight.
template <class Op, class IO, class T, int ITEMS>
__global__ void __launch_bounds__(kVarBlock)
variant_aos_kernel(const IO* __restrict__ a, const IO* __restrict__ b, IO* __restrict__ H, int64_t n, int norm, Op op)
{
    constexpr int NA = Op::NA, NB = Op::NB;
    __shared__ __align__(16) IO stage[ITEMS * kVarBlock * 9];
    const int64_t base = static_cast<int64_t>(blockIdx.x) * (ITEMS * kVarBlock);
    __align__(16) IO xa[ITEMS][NA];
    __align__(16) IO xb[ITEMS][NB > 0 ? NB : 2];
#pragma unroll
    for (int it = 0; it < ITEMS; ++it) {
        const int64_t i = base + it * kVarBlock + threadIdx.x;
        if (i < n) {
            load_record<IO, NA>(a + NA * i, xa[it]);
            if constexpr (NB > 0) load_record<IO, NB>(b + NB * i, xb[it]);
        }
    }
#pragma unroll
    for (int it = 0; it < ITEMS; ++it) {
        const int64_t i = base + it * kVarBlock + threadIdx.x;
        if (i < n) {
            T x[NA + NB], Hv[9];
#pragma unroll
            for (int k = 0; k < NA; ++k) x[k] = static_cast<T>(xa[it][k]);
            if constexpr (NB > 0) {
#pragma unroll
                for (int k = 0; k < NB; ++k) x[NA + k] = static_cast<T>(xb[it][k]);
            }
            op.template apply<T>(x, Hv);
            normalise<T>(Hv, norm);
#pragma unroll
            for (int k = 0; k < 9; ++k) stage[(it * kVarBlock + threadIdx.x) * 9 + k] = static_cast<IO>(Hv[k]);
        }
    }
    __syncthreads();
    const int64_t rem = n - base;
    const int cnt = static_cast<int>(rem < ITEMS * kVarBlock ? rem : ITEMS * kVarBlock) * 9;
    IO* out = H + 9 * base;
    constexpr int PER = 16 / int(sizeof(IO));
    const int nv = cnt / PER;
    for (int j = threadIdx.x; j < nv; j += kVarBlock)
        __stcs(reinterpret_cast<int4*>(out) + j, reinterpret_cast<const int4*>(stage)[j]);
    for (int j = nv * PER + threadIdx.x; j < cnt; j += kVarBlock) out[j] = stage[j];
}

template <class Op, class IO, class T>
static int variant_launch(const IO* a, const IO* b, IO* H, int64_t n, hg_layout_t layout, int norm, const Op& op, cudaStream_t st)
{
    if (layout == HG_SOA) {
        constexpr int V = IoVec<IO>::V;
        if (n % V == 0) {
            const int64_t nt = n / V, blocks = (nt + kVarBlock - 1) / kVarBlock;
            variant_soa_kernel<Op, IO, T, true><<<static_cast<unsigned>(blocks), kVarBlock, 0, st>>>(a, b, H, nt, n, norm, op);
        } else {
            const int64_t blocks = (n + kVarBlock - 1) / kVarBlock;
            variant_soa_kernel<Op, IO, T, false><<<static_cast<unsigned>(blocks), kVarBlock, 0, st>>>(a, b, H, n, n, norm, op);
        }
    } else {
        constexpr int ITEMS = ((Op::NA + Op::NB) * int(sizeof(IO)) <= 32) ? 2 : 1;
        const int64_t blocks = (n + ITEMS * kVarBlock - 1) / (ITEMS * kVarBlock);
        variant_aos_kernel<Op, IO, T, ITEMS><<<static_cast<unsigned>(blocks), kVarBlock, 0, st>>>(a, b, H, n, norm, op);
    }
    return launch_status();
}

static int check_common(int64_t n, hg_layout_t layout, hg_norm_t norm)
{
    if (n < 0) return HG_ERR_INVALID_ARG;
    if (layout != HG_SOA && layout != HG_AOS) return HG_ERR_INVALID_ARG;
    if (norm != HG_NORM_NONE && norm != HG_NORM_H33 && norm != HG_NORM_FROBENIUS) return HG_ERR_INVALID_ARG;
    if ((n + kVarBlock - 1) / kVarBlock > 0x7fffffffLL) return HG_ERR_INVALID_ARG;
    return HG_OK;
}

}  // namespace hg

extern "C" {

int hg_affine_batched(const float* src3, const float* dst3, float* H, int64_t n, hg_layout_t layout,
                      hg_norm_t norm, hg_precision_t prec, void* cuda_stream)
{
    using namespace hg;
    const int rc = check_common(n, layout, norm);
    if (rc != HG_OK) return rc;
    if (prec != HG_PREC_F64 && prec != HG_PREC_F32) return HG_ERR_INVALID_ARG;
    if (n == 0) return HG_OK;
    if (!src3 || !dst3 || !H) return HG_ERR_INVALID_ARG;
    if (!aligned16(src3) || !aligned16(dst3) || !aligned16(H)) return HG_ERR_ALIGNMENT;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    return prec == HG_PREC_F64 ? variant_launch<AffineOp, float, double>(src3, dst3, H, n, layout, int(norm), AffineOp(), st)
                               : variant_launch<AffineOp, float, float>(src3, dst3, H, n, layout, int(norm), AffineOp(), st);
}

int hg_sk_batched(double P3x, double P3y, double Q3x, double Q3y, const float* dst, float* H, int64_t n,
                  hg_layout_t layout, hg_norm_t norm, hg_precision_t prec, void* cuda_stream)
{
    using namespace hg;
    const int rc = check_common(n, layout, norm);
    if (rc != HG_OK) return rc;
    if (prec != HG_PREC_F64 && prec != HG_PREC_F32) return HG_ERR_INVALID_ARG;
    if (!(P3x == P3x) || !(P3y == P3y) || !(Q3x == Q3x) || !(Q3y == Q3y)) return HG_ERR_INVALID_ARG;
    if (n == 0) return HG_OK;
    if (!dst || !H) return HG_ERR_INVALID_ARG;
    if (!aligned16(dst) || !aligned16(H)) return HG_ERR_ALIGNMENT;
    // pattern constants (Eq. 12-14 with f_S1 = 1), once per call on the host
    SkOp op;
    const double rP3 = 1.0 / P3y, rQ3 = 1.0 / Q3y;
    op.P5x = P3x * rP3; op.P5y = rP3;
    op.Q7x = Q3x * rQ3 - op.P5x; op.Q7y = rQ3 - op.P5y;
    op.rden = 1.0 / (op.Q7x * op.Q7x - op.Q7y * op.Q7y);
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    return prec == HG_PREC_F64 ? variant_launch<SkOp, float, double>(dst, nullptr, H, n, layout, int(norm), op, st)
                               : variant_launch<SkOp, float, float>(dst, nullptr, H, n, layout, int(norm), op, st);
}

static int solve_f64(int method, const double* src, const double* dst, double* H, int64_t n, hg_layout_t layout,
                     hg_norm_t norm, void* cuda_stream)
{
    using namespace hg;
    const int rc = check_common(n, layout, norm);
    if (rc != HG_OK) return rc;
    if (n == 0) return HG_OK;
    if (!src || !dst || !H) return HG_ERR_INVALID_ARG;
    if (!aligned16(src) || !aligned16(dst) || !aligned16(H)) return HG_ERR_ALIGNMENT;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    return method == METHOD_ACA
        ? variant_launch<GeneralOp<METHOD_ACA>, double, double>(src, dst, H, n, layout, int(norm), GeneralOp<METHOD_ACA>(), st)
        : variant_launch<GeneralOp<METHOD_SKS>, double, double>(src, dst, H, n, layout, int(norm), GeneralOp<METHOD_SKS>(), st);
}

int hg_aca_batched_f64(const double* src, const double* dst, double* H, int64_t n, hg_layout_t layout,
                       hg_norm_t norm, void* cuda_stream)
{ return solve_f64(hg::METHOD_ACA, src, dst, H, n, layout, norm, cuda_stream); }

int hg_sks_batched_f64(const double* src, const double* dst, double* H, int64_t n, hg_layout_t layout,
                       hg_norm_t norm, void* cuda_stream)
{ return solve_f64(hg::METHOD_SKS, src, dst, H, n, layout, norm, cuda_stream); }

}  // extern "C"
