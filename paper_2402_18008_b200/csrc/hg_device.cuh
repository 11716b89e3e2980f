// hg_device.cuh -- device-side building blocks of libhg (sm_100a).
//
// Scalar arithmetic of the two minimal 4-point solvers of arXiv 2402.18008, restated from the
// paper ("P:<line>" = /root/reference/PAPER.md) for a register-resident, FMA-contracted
// evaluation, plus the streaming load/store helpers.  Templated on the working type T
// (double = HG_PREC_F64, float = HG_PREC_F32).  This file shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace hg {

// ------------------------------------------------------------------------------------------
// Small arithmetic kit per working type.
// ------------------------------------------------------------------------------------------
template <class T> struct K;

template <> struct K<float> {
    static __device__ __forceinline__ float fma(float a, float b, float c) { return __fmaf_rn(a, b, c); }
    static __device__ __forceinline__ float rcp(float x) { return __frcp_rn(x); }
    static __device__ __forceinline__ float abs(float x) { return fabsf(x); }
    static __device__ __forceinline__ float max(float a, float b) { return fmaxf(a, b); }
    // 1 / sqrt(sum h^2) without overflow: the raw ACA scale (~1e23 at 640x480) squares past
    // fp32, so pre-scale by the power of two that brings max|h| to [1,2).
    static __device__ __forceinline__ float frob_scale(const float h[9])
    {
        float m = 0.f;
#pragma unroll
        for (int i = 0; i < 9; ++i) m = fmaxf(m, fabsf(h[i]));
        // 2^-e with e = exponent(m), built from the bits (m == 0, inf, NaN fall through as-is)
        const uint32_t eb = (__float_as_uint(m) >> 23) & 0xffu;
        const float p = __uint_as_float(((254u - eb) & 0xffu) << 23);   // 2^(127-eb)
        float ss = 0.f;
#pragma unroll
        for (int i = 0; i < 9; ++i) { const float v = h[i] * p; ss = __fmaf_rn(v, v, ss); }
        return p * rsqrtf(ss);
    }
};

template <> struct K<double> {
    static __device__ __forceinline__ double fma(double a, double b, double c) { return __fma_rn(a, b, c); }
    // Reciprocal: MUFU.RCP64H seed (>= 20 bits) + two Newton steps (4 DFMA) -> ~1 ulp.
    // x == 0 or non-finite gives a non-finite result (degenerate set, reading R8).
    static __device__ __forceinline__ double rcp(double x)
    {
        double r;
        asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
        double e = __fma_rn(-x, r, 1.0);
        r = __fma_rn(r, e, r);
        e = __fma_rn(-x, r, 1.0);
        r = __fma_rn(r, e, r);
        return r;
    }
    static __device__ __forceinline__ double abs(double x) { return fabs(x); }
    static __device__ __forceinline__ double max(double a, double b) { return fmax(a, b); }
    // fp64 range (1e308) holds the square of any raw H whose fp32 rounding is finite.
    static __device__ __forceinline__ double frob_scale(const double h[9])
    {
        double ss = 0.0;
#pragma unroll
        for (int i = 0; i < 9; ++i) ss = __fma_rn(h[i], h[i], ss);
        double y;
        asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(ss));
        // two Newton steps: y <- y + y * (0.5 - 0.5 * ss * y^2)
#pragma unroll
        for (int it = 0; it < 2; ++it) {
            const double hy = 0.5 * y;
            const double e = __fma_rn(-ss * y, hy, 0.5);
            y = __fma_rn(y, e, y);
        }
        return y;
    }
};

// a*d - b*c with one rounding on the second product (exact in fp64 for fp32-difference inputs).
template <class T>
__device__ __forceinline__ T det2(T a, T b, T c, T d) { return K<T>::fma(a, d, -(b * c)); }

// ------------------------------------------------------------------------------------------
// ACA: H = H_A2^-1 * H_C * H_A1  (Eq. 27).  No division.
//   s = (M1,N1,P1,Q1), d = (M2,N2,P2,Q2), each x0,y0,...,x3,y3.
// ------------------------------------------------------------------------------------------
template <class T>
__device__ __forceinline__ void aca_solve(const T s[8], const T d[8], T H[9])
{
    // H_A1 / H_A2: edge vectors from the first anchor and the affine scale f_A (Eq. 23-24).
    const T a1x = s[2] - s[0], a1y = s[3] - s[1];      // M1N1
    const T b1x = s[4] - s[0], b1y = s[5] - s[1];      // M1P1
    const T q1x = s[6] - s[0], q1y = s[7] - s[1];      // M1Q1
    const T a2x = d[2] - d[0], a2y = d[3] - d[1];      // M2N2
    const T b2x = d[4] - d[0], b2y = d[5] - d[1];      // M2P2
    const T q2x = d[6] - d[0], q2y = d[7] - d[1];      // M2Q2
    const T fA1 = det2(a1x, a1y, b1x, b1y);
    const T fA2 = det2(a2x, a2y, b2x, b2y);
    // Fourth point in the affine frames, scaled by f_A (Eq. 28).
    const T Q3x = det2(q1x, q1y, b1x, b1y);
    const T Q3y = det2(a1x, a1y, q1x, q1y);
    const T Q4x = det2(q2x, q2y, b2x, b2y);
    const T Q4y = det2(a2x, a2y, q2x, q2y);
    // Core transformation up to scale (Eq. 30-32).
    const T t1 = fA1 - Q3x - Q3y;
    const T t2 = fA2 - Q4x - Q4y;
    const T c11 = t1 * Q3y * Q4x;
    const T c22 = t1 * Q3x * Q4y;
    const T c33 = t2 * Q3x * Q3y;
    // G = H_A2^-1 * H_C with H_A2^-1 = [M2N2 M2P2 M2; 0 0 1] (Eq. 25 is lost in the extraction,
    // reading R1), H_C = [c11 0 0; 0 c22 0; c11-c33 c22-c33 c33] (Eq. 31):
    //   G[:,0] = c11*n2 - c33*m2,  G[:,1] = c22*p2 - c33*m2,  G[:,2] = c33*m2   (homogeneous).
    const T g13 = c33 * d[0], g23 = c33 * d[1];
    const T g11 = K<T>::fma(c11, d[2], -g13), g21 = K<T>::fma(c11, d[3], -g23), g31 = c11 - c33;
    const T g12 = K<T>::fma(c22, d[4], -g13), g22 = K<T>::fma(c22, d[5], -g23), g32 = c22 - c33;
    // H = G * H_A1, H_A1 = [b1y -b1x 0; -a1y a1x 0; 0 0 fA1] * T(-M1)  (Eq. 23, reading R2).
    const T h11 = det2(g11, g12, a1y, b1y);            // g11*b1y - g12*a1y
    const T h21 = det2(g21, g22, a1y, b1y);
    const T h31 = det2(g31, g32, a1y, b1y);
    const T h12 = det2(g12, g11, b1x, a1x);            // g12*a1x - g11*b1x
    const T h22 = det2(g22, g21, b1x, a1x);
    const T h32 = det2(g32, g31, b1x, a1x);
    H[0] = h11; H[1] = h12; H[2] = K<T>::fma(-h12, s[1], K<T>::fma(-h11, s[0], g13 * fA1));
    H[3] = h21; H[4] = h22; H[5] = K<T>::fma(-h22, s[1], K<T>::fma(-h21, s[0], g23 * fA1));
    H[6] = h31; H[7] = h32; H[8] = K<T>::fma(-h32, s[1], K<T>::fma(-h31, s[0], c33 * fA1));
}

// ------------------------------------------------------------------------------------------
// SKS: H = H_S2^-1 * H_K * H_S1,  H_K = H_E^-1 * H_S' * H_E  (Eq. 16).  5 reciprocals.
// ------------------------------------------------------------------------------------------
template <class T>
__device__ __forceinline__ void sks_solve(const T s[8], const T d[8], T H[9])
{
    const T half = T(0.5);
    // Similarity of each plane from its two anchors: midpoint O, half-vector v = ON, f_S = |v|^2
    // (Eq. 6, 7, 9).
    const T O1x = half * (s[0] + s[2]), O1y = half * (s[1] + s[3]);
    const T v1x = s[2] - O1x, v1y = s[3] - O1y;
    const T f1 = K<T>::fma(v1x, v1x, v1y * v1y);
    const T O2x = half * (d[0] + d[2]), O2y = half * (d[1] + d[3]);
    const T v2x = d[2] - O2x, v2y = d[3] - O2y;
    const T f2 = K<T>::fma(v2x, v2x, v2y * v2y);
    // P, Q in the similarity frames, homogeneous weight f_S (Eq. 8; layout per R2).
    T ex, ey;
    ex = s[4] - O1x; ey = s[5] - O1y;
    const T P3x = K<T>::fma(v1x, ex, v1y * ey), P3y = det2(v1x, v1y, ex, ey);
    ex = s[6] - O1x; ey = s[7] - O1y;
    const T Q3x = K<T>::fma(v1x, ex, v1y * ey), Q3y = det2(v1x, v1y, ex, ey);
    ex = d[4] - O2x; ey = d[5] - O2y;
    const T P4x = K<T>::fma(v2x, ex, v2y * ey), P4y = det2(v2x, v2y, ex, ey);
    ex = d[6] - O2x; ey = d[7] - O2y;
    const T Q4x = K<T>::fma(v2x, ex, v2y * ey), Q4y = det2(v2x, v2y, ex, ey);
    // H_E exchanges the 2nd and 3rd homogeneous coordinates (Eq. 12); dehomogenise:
    // X5 = (X3.x / X3.y, f_S / X3.y).  Reciprocals 1-4.
    T r;
    r = K<T>::rcp(P3y); const T P5x = P3x * r, P5y = f1 * r;
    r = K<T>::rcp(Q3y); const T Q5x = Q3x * r, Q5y = f1 * r;
    r = K<T>::rcp(P4y); const T P6x = P4x * r, P6y = f2 * r;
    r = K<T>::rcp(Q4y); const T Q6x = Q4x * r, Q6y = f2 * r;
    // Translate P5, P6 to the origin (Eq. 13; readings R3, R4).
    const T Q7x = Q5x - P5x, Q7y = Q5y - P5y;
    const T Q8x = Q6x - P6x, Q8y = Q6y - P6y;
    // Hyperbolic rotation + scale: the 2x2 system of Eq. 14.  Reciprocal 5.
    r = K<T>::rcp(K<T>::fma(Q7x, Q7x, -(Q7y * Q7y)));
    const T aK = det2(Q8x, Q8y, Q7y, Q7x) * r;          // (Q8x*Q7x - Q8y*Q7y) / den
    const T bK = det2(Q8y, Q8x, Q7y, Q7x) * r;          // (Q8y*Q7x - Q8x*Q7y) / den
    // Kernel transformation H_K = [aK uK bK; 0 1 0; bK vK aK] (Eq. 11, 15).
    const T uK = K<T>::fma(-bK, P5y, K<T>::fma(-aK, P5x, P6x));
    const T vK = K<T>::fma(-aK, P5y, K<T>::fma(-bK, P5x, P6y));
    // J = H_S2^-1 * H_K,  H_S2^-1 = [v2x -v2y O2x; v2y v2x O2y; 0 0 1]  (Eq. 10).
    const T j11 = K<T>::fma(v2x, aK, O2x * bK);
    const T j12 = K<T>::fma(v2x, uK, K<T>::fma(O2x, vK, -v2y));
    const T j13 = K<T>::fma(v2x, bK, O2x * aK);
    const T j21 = K<T>::fma(v2y, aK, O2y * bK);
    const T j22 = K<T>::fma(v2y, uK, K<T>::fma(O2y, vK, v2x));
    const T j23 = K<T>::fma(v2y, bK, O2y * aK);
    // H = J * H_S1,  H_S1 = [v1x v1y 0; -v1y v1x 0; 0 0 f1] * T(-O1)  (Eq. 8).
    const T s13 = -K<T>::fma(v1x, O1x, v1y * O1y);
    const T s23 = det2(v1y, v1x, O1y, O1x);             // v1y*O1x - v1x*O1y
    H[0] = det2(j11, j12, v1y, v1x);                    // j11*v1x - j12*v1y
    H[1] = K<T>::fma(j11, v1y, j12 * v1x);
    H[2] = K<T>::fma(j11, s13, K<T>::fma(j12, s23, j13 * f1));
    H[3] = det2(j21, j22, v1y, v1x);
    H[4] = K<T>::fma(j21, v1y, j22 * v1x);
    H[5] = K<T>::fma(j21, s13, K<T>::fma(j22, s23, j23 * f1));
    H[6] = det2(bK, vK, v1y, v1x);
    H[7] = K<T>::fma(bK, v1y, vK * v1x);
    H[8] = K<T>::fma(bK, s13, K<T>::fma(vK, s23, aK * f1));
}

enum { METHOD_ACA = 0, METHOD_SKS = 1 };

template <int METHOD, class T>
__device__ __forceinline__ void solve(const T s[8], const T d[8], T H[9])
{
    if (METHOD == METHOD_ACA) aca_solve<T>(s, d, H);
    else                      sks_solve<T>(s, d, H);
}

// Scale H in place per hg_norm_t (0 none, 1 h33, 2 Frobenius).
template <class T>
__device__ __forceinline__ void normalise(T H[9], int norm)
{
    if (norm == 1) {
        const T r = K<T>::rcp(H[8]);
#pragma unroll
        for (int i = 0; i < 8; ++i) H[i] *= r;
        H[8] = H[8] * r;                                // 1, or NaN when h33 is 0 / non-finite
    } else if (norm == 2) {
        const T r = K<T>::frob_scale(H);
#pragma unroll
        for (int i = 0; i < 9; ++i) H[i] *= r;
    }
}

// ------------------------------------------------------------------------------------------
// Streaming (touch-once) global accesses: evict-first in L1/L2 so 6.7 GB does not thrash L2.
// ------------------------------------------------------------------------------------------
template <int V> struct Vec;
template <> struct Vec<1> { float v[1]; };
template <> struct __align__(8)  Vec<2> { float v[2]; };
template <> struct __align__(16) Vec<4> { float v[4]; };

template <int V> __device__ __forceinline__ Vec<V> ld_stream(const float* p);
template <> __device__ __forceinline__ Vec<1> ld_stream<1>(const float* p)
{ Vec<1> r; r.v[0] = __ldcs(p); return r; }
template <> __device__ __forceinline__ Vec<2> ld_stream<2>(const float* p)
{ const float2 t = __ldcs(reinterpret_cast<const float2*>(p)); Vec<2> r; r.v[0] = t.x; r.v[1] = t.y; return r; }
template <> __device__ __forceinline__ Vec<4> ld_stream<4>(const float* p)
{ const float4 t = __ldcs(reinterpret_cast<const float4*>(p)); Vec<4> r; r.v[0] = t.x; r.v[1] = t.y; r.v[2] = t.z; r.v[3] = t.w; return r; }

template <int V> __device__ __forceinline__ void st_stream(float* p, const Vec<V>& x);
template <> __device__ __forceinline__ void st_stream<1>(float* p, const Vec<1>& x) { __stcs(p, x.v[0]); }
template <> __device__ __forceinline__ void st_stream<2>(float* p, const Vec<2>& x)
{ __stcs(reinterpret_cast<float2*>(p), make_float2(x.v[0], x.v[1])); }
template <> __device__ __forceinline__ void st_stream<4>(float* p, const Vec<4>& x)
{ __stcs(reinterpret_cast<float4*>(p), make_float4(x.v[0], x.v[1], x.v[2], x.v[3])); }

// ------------------------------------------------------------------------------------------
// mbarrier + 1-D bulk-async copy (TMA): global -> shared memory staging with byte-count completion.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return static_cast<uint32_t>(__cvta_generic_to_shared(p)); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count)
{ asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(smem_u32(bar)), "r"(count) : "memory"); }
__device__ __forceinline__ void fence_barrier_init()
{ asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes)
{ asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(smem_u32(bar)), "r"(bytes) : "memory"); }
__device__ __forceinline__ void bulk_copy_g2s(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 :: "r"(smem_u32(dst_smem)), "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra DONE;\n"
        "bra LAB_WAIT;\n"
        "DONE:\n"
        "}" :: "r"(smem_u32(bar)), "r"(parity) : "memory");
}

}  // namespace hg
