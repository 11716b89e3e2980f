// hg_ransac.cu -- hg_ransac_hypothesize_score / hg_ransac_adaptive: RANSAC hypothesis generation fused
// with inlier scoring (rows a-R0..a-R5 of SURVEY.md section 8(a)).
//
// Launches on the caller's stream, no host synchronisation:
//   1. prep     : correspondence table -> packed, threshold-folded fp32 table in the workspace
//                 (+ coordinate bounds for the error band)
//   2. score    : one thread per hypothesis: gather 4 correspondences, fp64 ACA solve, fold the
//                 threshold into H, then sweep the whole table with packed FFMA2 arithmetic, two points
//                 per instruction.  One value per pair, a = (ex^2 + ey^2 - W^2) + Bc, against a rigorous
//                 per-hypothesis fp32 error band Bc: a < 0 is a
//                 sure inlier, a > 2 Bc a sure outlier; the rare pair in between is decided on the
//                 spot in fp64 by the definition (reading R9) from the fp64 H kept in shared memory.
//                 Where the table comes from ("operand paths"):
//                   - tables of <= 4096 points: the packed table is copied into the
//                     64 KB constant bank; the sweep reads it through the uniform datapath (LDCU.64 ->
//                     uniform-register FFMA2 operands), which costs no register-file bandwidth -- the
//                     limiter of a three-operand FFMA2 stream on this part;
//                   - everything else: the table is staged in shared memory by bulk-async copies /
//                     mbarrier (32 KB stages) and read with broadcast LDS.128.
//   3. finalize : decode the packed (count, index) maximum, re-solve that hypothesis, emit best_H.
// Compute-bound on the FP32 pipe: 11 packed instructions per two (hypothesis, point) pairs.
#include <memory>
#include <mutex>

#include "hg_device.cuh"
#include "hg_host.h"

namespace hg {

constexpr int kRBlock     = 512;    // threads (= hypotheses) per scoring CTA
constexpr int kChunkPairs = 1024;   // point pairs per shared-memory stage: 1024 * 32 B = 32 KB
constexpr int kStages     = 2;
constexpr size_t kHeaderBytes = 128;
constexpr int kConstPairs = 2048;   // table entries (point pairs) the constant bank holds: 2048 * 32 B = 64 KB

struct RansacHeader {               // first 128 bytes of the workspace
    unsigned long long best_key;    // (count << 32) | (0xFFFFFFFF - hypothesis index)
    unsigned long long n_fixup;     // hypotheses with at least one pair decided in fp64
    unsigned long long n_pairs_f64; // (hypothesis, point) pairs decided in fp64
    unsigned long long n_evaluated; // adaptive mode: hypotheses scored when the run stopped
    unsigned long long n_rejected;  // HG_RANSAC_REJECT_DEGENERATE: hypotheses rejected by the sample check (R20)
    unsigned long long n_band;      // pairs inside the table-wide band (re-tested against the per-pair band)
    unsigned long long reserved[2];
    unsigned int bound_bits[4];     // float bits of max|sx|, max|sy|, max|dx/t|, max|dy/t|
    unsigned int stop;              // adaptive mode: set by the round kernel, later rounds return at once
    unsigned int blocks_done;       // tiny-call kernel: CTAs whose counts and candidate are complete
    unsigned int pad[10];
};
static_assert(sizeof(RansacHeader) == kHeaderBytes, "header layout");

// The packed table of a call with <= 4096 points, in the constant bank: the sweep's point operands then come
// through the uniform datapath.  One per device context; calls that use it are ordered by ConstTableGuard.
__constant__ float4 c_table[2 * kConstPairs];

// Per-hypothesis constants of the fp32 sweep.
struct HypConst {
    float h[9];     // rows 1,2 of H scaled by 1/(t*max|h|), row 3 by 1/max|h|
    float Bc;       // band: |computed - exact| of (ex^2 + ey^2 - W^2) < Bc for every table point whenever it matters
    unsigned thr;   // float bits of 2*Bc
    float K, K0;    // per-pair band K|W| + K0 <= Bc, used only by the cold path
};

// ---- packed fp32 helpers -------------------------------------------------------------------
__device__ __forceinline__ float2 f2(float v) { return make_float2(v, v); }
__device__ __forceinline__ float2 neg2(float2 a) { return make_float2(-a.x, -a.y); }

// Two points against one hypothesis: a = (ex^2 + ey^2 - W^2) + Bc, 11 packed FP32 instructions.
//   a < 0         <=> surely inlier;   a > 2*Bc  <=> surely outlier;   0 <= a <= 2*Bc: decide in fp64.
// ndx, ndy hold -d/t.
__device__ __forceinline__ float2 score2(const HypConst& c, float2 sx, float2 sy, float2 ndx, float2 ndy)
{
    const float2 X = __ffma2_rn(f2(c.h[0]), sx, __ffma2_rn(f2(c.h[1]), sy, f2(c.h[2])));
    const float2 Y = __ffma2_rn(f2(c.h[3]), sx, __ffma2_rn(f2(c.h[4]), sy, f2(c.h[5])));
    const float2 W = __ffma2_rn(f2(c.h[6]), sx, __ffma2_rn(f2(c.h[7]), sy, f2(c.h[8])));
    const float2 ex = __ffma2_rn(ndx, W, X);                     // X/t - (dx/t) W
    const float2 ey = __ffma2_rn(ndy, W, Y);
    const float2 w2 = __ffma2_rn(W, W, f2(-c.Bc));               // W^2 - Bc
    const float2 p  = __ffma2_rn(ex, ex, neg2(w2));
    return __ffma2_rn(ey, ey, p);                                // ex^2 + ey^2 - W^2 + Bc
}

__device__ __forceinline__ unsigned sign_bit(float v) { return __float_as_uint(v) >> 31; }

// ---- hypothesis set-up (shared by score and finalize) --------------------------------
__device__ __forceinline__ void gather_sets(const float2* __restrict__ src_xy, const float2* __restrict__ dst_xy,
                                            const int4 id, double s[8], double d[8])
{
    const int ids[4] = { id.x, id.y, id.z, id.w };
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const float2 sp = __ldg(src_xy + ids[k]);
        const float2 dq = __ldg(dst_xy + ids[k]);
        s[2 * k] = sp.x; s[2 * k + 1] = sp.y;
        d[2 * k] = dq.x; d[2 * k + 1] = dq.y;
    }
}

// ---- sample check (reading R20; degenerate configurations P:786) ---------------------------------
// Twice the signed area of triangle (i, j, k); one IEEE operation per difference, product and subtraction (no FMA
// contraction): the comparison below is a decision, taken in the same arithmetic as the oracle's.
__device__ __forceinline__ double signed_area2(const double p[8], int i, int j, int k)
{
    const double ux = __dsub_rn(p[2 * j], p[2 * i]), uy = __dsub_rn(p[2 * j + 1], p[2 * i + 1]);
    const double vx = __dsub_rn(p[2 * k], p[2 * i]), vy = __dsub_rn(p[2 * k + 1], p[2 * i + 1]);
    return __dsub_rn(__dmul_rn(ux, vy), __dmul_rn(uy, vx));
}

// true: reject.  Some triangle of the source or target quadruple has area <= min_area (lim2 = 2 * min_area), or a
// triangle's orientation differs between the planes.
__device__ __forceinline__ bool sample_rejected(const double s[8], const double d[8], double lim2)
{
    bool rej = false;
#pragma unroll
    for (int t = 0; t < 4; ++t) {
        const int i = t == 3 ? 1 : 0, j = t < 2 ? 1 : 2, k = t == 0 ? 2 : 3;           // (0,1,2) (0,1,3) (0,2,3) (1,2,3)
        const double a1 = signed_area2(s, i, j, k), a2 = signed_area2(d, i, j, k);
        rej = rej || !(fabs(a1) > lim2) || !(fabs(a2) > lim2) || ((a1 > 0.0) != (a2 > 0.0));
    }
    return rej;
}

// ---- where the hypotheses of a launch come from ----------------------------------------------
struct HypSource {
    const int4* idx;            // caller-supplied indices [n_hyp][4], or nullptr: sample on the device
    int4* idx_out;              // sampling mode, nullable: the sampled indices are written here
    unsigned long long seed;    // sampling mode
    long long h0, h1;           // this launch scores hypotheses [h0, h1)
    unsigned flags;             // HG_RANSAC_* option bits
    double reject_lim2;         // HG_RANSAC_REJECT_DEGENERATE: 2 * min_area_px2
    int check_stop;             // 1: return at once when hdr->stop is set (adaptive termination)
    int part_entries;           // table entries per blockIdx.y part (a multiple of 8); >= n_pairs: no split
    int* acc;                   // split mode: partial counts are added here (zeroed before the launch)
};

// Philox4x32-10 (Salmon et al., SC'11), the counter-based generator of reading R19: 10 rounds of
// (c0,c1,c2,c3) <- (hi(M1 c2) ^ c1 ^ k0, lo(M1 c2), hi(M0 c0) ^ c3 ^ k1, lo(M0 c0)), k += (W0, W1).
__device__ __forceinline__ uint4 philox4x32_10(uint4 c, uint2 k)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const unsigned hi0 = __umulhi(0xD2511F53u, c.x), lo0 = 0xD2511F53u * c.x;
        const unsigned hi1 = __umulhi(0xCD9E8D57u, c.z), lo1 = 0xCD9E8D57u * c.z;
        c = make_uint4(hi1 ^ c.y ^ k.x, lo1, hi0 ^ c.w ^ k.y, lo0);
        k.x += 0x9E3779B9u; k.y += 0xBB67AE85u;
    }
    return c;
}

// The 4 indices of hypothesis h: attempt a draws Philox(counter = (lo(h), hi(h), a, 0), key = seed), index =
// floor(word * n_pts / 2^32); first attempt with pairwise distinct indices wins; after 32 failures
// i, i+1, i+2, i+3 (mod n_pts) with i = attempt 0's first index.
__device__ __forceinline__ int4 sample4(unsigned long long seed, unsigned long long h, int n_pts)
{
    const uint2 key = make_uint2(static_cast<unsigned>(seed), static_cast<unsigned>(seed >> 32));
    int first = 0;
    for (unsigned a = 0; a < 32u; ++a) {
        const uint4 r = philox4x32_10(make_uint4(static_cast<unsigned>(h), static_cast<unsigned>(h >> 32), a, 0u), key);
        const int4 id = make_int4(static_cast<int>(__umulhi(r.x, static_cast<unsigned>(n_pts))),
                                  static_cast<int>(__umulhi(r.y, static_cast<unsigned>(n_pts))),
                                  static_cast<int>(__umulhi(r.z, static_cast<unsigned>(n_pts))),
                                  static_cast<int>(__umulhi(r.w, static_cast<unsigned>(n_pts))));
        if (a == 0) first = id.x;
        if (id.x != id.y && id.x != id.z && id.x != id.w && id.y != id.z && id.y != id.w && id.z != id.w) return id;
    }
    return make_int4(first % n_pts, (first + 1) % n_pts, (first + 2) % n_pts, (first + 3) % n_pts);
}

__device__ __forceinline__ int4 hypothesis_indices(const HypSource& hs, long long hidx, int n_pts)
{
    return hs.idx ? __ldg(hs.idx + hidx) : sample4(hs.seed, static_cast<unsigned long long>(hidx), n_pts);
}

// fp64 ACA solve (raw scale in H), max-abs normalisation (Hn) and threshold folding (c.h).
// Returns false for an unusable H (all zero or non-finite): such a hypothesis scores 0 (R9: W == 0).
__device__ __forceinline__ bool solve_for_sweep(const double s[8], const double d[8], double inv_t, double H[9], double Hn[9],
                                                HypConst& c)
{
    aca_solve<double>(s, d, H);
    double m = 0.0;
#pragma unroll
    for (int k = 0; k < 9; ++k) m = fmax(m, fabs(H[k]));
    const bool ok = (m > 0.0) && (m < 1.0e300);                  // false for 0, inf, NaN
    const double r = ok ? K<double>::rcp(m) : 0.0;
#pragma unroll
    for (int k = 0; k < 9; ++k) Hn[k] = H[k] * r;
    const double rt = inv_t;
#pragma unroll
    for (int k = 0; k < 6; ++k) c.h[k] = static_cast<float>(Hn[k] * rt);
#pragma unroll
    for (int k = 6; k < 9; ++k) c.h[k] = static_cast<float>(Hn[k]);
    return ok;
}

// The error band of the fp32 sweep for the folded H in c.h and the coordinate bounds of the table.
__device__ __forceinline__ void error_band(const float bounds[4], bool ok, HypConst& c)
{
    // Error band, u = 2^-24:
    //   A_r = |h_r1| Sx + |h_r2| Sy + |h_r3|;  c1 = u (3 A1 + 4 Dx A3), c2 = u (3 A2 + 4 Dy A3), eW = 3 u A3
    //   C = c1 + c2 + eW;  K = 4 C + 16 u A3;  K0 = 32 C^2      (evaluated in fp64, rounded up)
    const double u = 5.9604644775390625e-08;
    const double Sx = bounds[0], Sy = bounds[1], Dx = bounds[2], Dy = bounds[3];
    const double A1 = fabs(double(c.h[0])) * Sx + fabs(double(c.h[1])) * Sy + fabs(double(c.h[2]));
    const double A2 = fabs(double(c.h[3])) * Sx + fabs(double(c.h[4])) * Sy + fabs(double(c.h[5]));
    const double A3 = fabs(double(c.h[6])) * Sx + fabs(double(c.h[7])) * Sy + fabs(double(c.h[8]));
    const double C = u * (3.0 * A1 + 4.0 * Dx * A3) + u * (3.0 * A2 + 4.0 * Dy * A3) + 3.0 * u * A3;
    const double Kd = (4.0 * C + 16.0 * u * A3) * 1.000001;
    const double K0d = 32.0 * C * C * 1.000001;
    // One band for the whole table: |W^| <= A3 (1 + 3u) for every point, so Bc >= K |W^| + K0.
    c.K = __double2float_ru(Kd);
    c.K0 = __double2float_ru(K0d);
    c.Bc = __double2float_ru(Kd * A3 * 1.000001 + K0d);
    c.thr = __float_as_uint(2.0f * c.Bc);
    if (!ok) {                          // unusable H: every point a sure outlier (X = 1, W = 0 => a = 1 > 0)
#pragma unroll
        for (int k = 0; k < 9; ++k) c.h[k] = 0.f;
        c.h[2] = 1.f; c.Bc = 0.f; c.thr = 0u;
    }
}

__device__ __forceinline__ bool make_hypothesis(const double s[8], const double d[8], double inv_t,
                                                const float bounds[4], double Hn[9], HypConst& c)
{
    double H[9];
    const bool ok = solve_for_sweep(s, d, inv_t, H, Hn, c);
    error_band(bounds, ok, c);
    return ok;
}

// The definition, in fp64 (reading R9): ||pi(H s) - d||_2 <= t, W == 0 -> outlier.
__device__ __forceinline__ bool inlier_f64(const double H[9], double sx, double sy, double dx, double dy, double t)
{
    const double X = fma(H[0], sx, fma(H[1], sy, H[2]));
    const double Y = fma(H[3], sx, fma(H[4], sy, H[5]));
    const double W = fma(H[6], sx, fma(H[7], sy, H[8]));
    if (W == 0.0) return false;
    const double ex = X / W - dx, ey = Y / W - dy;
    return sqrt(fma(ex, ex, ey * ey)) <= t;
}

// The definition (reading R9: ||pi(H s) - d||_2 <= t, W == 0 -> outlier) in fp64, multiplied through by W^2 so that it
// needs no division and no square root:  (X - dx W)^2 + (Y - dy W)^2 <= (t W)^2.  Same decision as the quotient form
// except within a few fp64 ulps of the threshold; ~12 dependent fp64 operations instead of two divisions and a root,
// which is what a warp waits for when one of its lanes has a pair inside the band.
__device__ __forceinline__ bool inlier_f64_nodiv(const double H[9], double sx, double sy, double dx, double dy, double t)
{
    const double X = fma(H[0], sx, fma(H[1], sy, H[2]));
    const double Y = fma(H[3], sx, fma(H[4], sy, H[5]));
    const double W = fma(H[6], sx, fma(H[7], sy, H[8]));
    if (W == 0.0) return false;
    const double ex = fma(-dx, W, X), ey = fma(-dy, W, Y), tw = t * W;
    return fma(ex, ex, ey * ey) <= tw * tw;
}

// ---- 1. prep ---------------------------------------------------------------------------------
// Table entry of point pair k (points 2k, 2k+1; an odd tail point is duplicated):
//   float4 (sx0, sx1, sy0, sy1), float4 (-dx0/t, -dx1/t, -dy0/t, -dy1/t)
__global__ void __launch_bounds__(256)
ransac_prep_kernel(const float2* __restrict__ src_xy, const float2* __restrict__ dst_xy, int n_pts,
                   int n_pairs, double inv_t, float4* __restrict__ table, RansacHeader* __restrict__ hdr)
{
    float m0 = 0.f, m1 = 0.f, m2 = 0.f, m3 = 0.f;
    for (int k = blockIdx.x * blockDim.x + threadIdx.x; k < n_pairs; k += gridDim.x * blockDim.x) {
        const int i0 = 2 * k, i1 = (2 * k + 1 < n_pts) ? 2 * k + 1 : 2 * k;
        const float2 s0 = __ldg(src_xy + i0), s1 = __ldg(src_xy + i1);
        const float2 d0 = __ldg(dst_xy + i0), d1 = __ldg(dst_xy + i1);
        const float4 A = make_float4(s0.x, s1.x, s0.y, s1.y);
        const float4 B = make_float4(static_cast<float>(-double(d0.x) * inv_t), static_cast<float>(-double(d1.x) * inv_t),
                                     static_cast<float>(-double(d0.y) * inv_t), static_cast<float>(-double(d1.y) * inv_t));
        table[2 * k] = A;
        table[2 * k + 1] = B;
        m0 = fmaxf(m0, fmaxf(fabsf(A.x), fabsf(A.y)));
        m1 = fmaxf(m1, fmaxf(fabsf(A.z), fabsf(A.w)));
        m2 = fmaxf(m2, fmaxf(fabsf(B.x), fabsf(B.y)));
        m3 = fmaxf(m3, fmaxf(fabsf(B.z), fabsf(B.w)));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        m0 = fmaxf(m0, __shfl_xor_sync(0xffffffffu, m0, o));
        m1 = fmaxf(m1, __shfl_xor_sync(0xffffffffu, m1, o));
        m2 = fmaxf(m2, __shfl_xor_sync(0xffffffffu, m2, o));
        m3 = fmaxf(m3, __shfl_xor_sync(0xffffffffu, m3, o));
    }
    if ((threadIdx.x & 31) == 0) {       // non-negative floats order like their bit patterns
        atomicMax(&hdr->bound_bits[0], __float_as_uint(m0));
        atomicMax(&hdr->bound_bits[1], __float_as_uint(m1));
        atomicMax(&hdr->bound_bits[2], __float_as_uint(m2));
        atomicMax(&hdr->bound_bits[3], __float_as_uint(m3));
    }
}

// ---- 2. score --------------------------------------------------------------------------------
__device__ __forceinline__ unsigned long long pack_key(unsigned count, unsigned index)
{ return (static_cast<unsigned long long>(count) << 32) | static_cast<unsigned long long>(0xFFFFFFFFu - index); }

__device__ __forceinline__ unsigned long long warp_max_u64(unsigned long long v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const unsigned long long w = __shfl_xor_sync(0xffffffffu, v, o);
        v = (w > v) ? w : v;
    }
    return v;
}

// ---- the cold path: pairs whose fp32 value fell inside the table-wide band --------------------------------
// Inside the sweep such a pair is only re-tested against the tighter per-pair band (same fp32 arithmetic, a few dozen
// instructions, no memory traffic beyond the constant/shared table).  What is still undecided -- 6e-5 of the pairs of
// C4 -- needs the definition in fp64 (global loads, two divisions, a square root): the sweep appends the point index to
// a small per-thread queue in shared memory, and after the sweep `drain_queue` decides the queued pairs, all lanes of
// the warp at once, so the loads and the fp64 arithmetic of different hypotheses overlap and the warps of a CTA stay
// together while they walk the table.
constexpr int kQueueCap = 8;            // queued pairs per thread (C4: 0.3 per hypothesis on average)


struct SlowCtx {
    const float2* src_xy;
    const float2* dst_xy;
    const float4* table;     // packed table in global memory (the sweep's fp32 operands, bit for bit)
    int4 id;                 // the hypothesis' four correspondences
    double inv_t, t;
    float bounds[4];
    unsigned* queue;         // this thread's queue in shared memory, stride kRBlock
    unsigned n64;            // out: pairs decided in fp64
};

// A queued pair is first tested against the tighter per-pair band K|W| + K0 with the same fp32 arithmetic (bit-identical
// X, Y, W, ex, ey: same operands and FMA nesting as score2).  Returns 1 = surely inlier, 0 = surely outlier, 2 = undecided.
__device__ __forceinline__ unsigned recheck_f32(const HypConst& c, float sx, float sy, float ndx, float ndy)
{
    const float X = __fmaf_rn(c.h[0], sx, __fmaf_rn(c.h[1], sy, c.h[2]));
    const float Y = __fmaf_rn(c.h[3], sx, __fmaf_rn(c.h[4], sy, c.h[5]));
    const float W = __fmaf_rn(c.h[6], sx, __fmaf_rn(c.h[7], sy, c.h[8]));
    const float ex = __fmaf_rn(ndx, W, X), ey = __fmaf_rn(ndy, W, Y);
    const float w2 = __fmaf_rn(W, W, -c.K0);
    const float dp = __fmaf_rn(ey, ey, __fmaf_rn(ex, ex, -w2));          // diff + K0
    const float aw = fabsf(W);
    if (__fmaf_rn(c.K, aw, dp) < 0.f) return 1u;                          // diff + (K|W| + K0) < 0
    if (__fmaf_rn(c.K, aw, 2.0f * c.K0) - dp < 0.f) return 0u;            // (K|W| + K0) - diff < 0
    return 2u;
}

// Decide the `qn` queued pairs of this thread by the definition in fp64 (reading R9): re-derive the hypothesis (the same
// deterministic fp64 solve as the set-up, so H is bit-identical).  Returns the number of inliers among them.
__device__ __noinline__ unsigned drain_queue(SlowCtx& cx, unsigned qn)
{
    double s[8], d[8], Hn[9];
    HypConst hc;
    gather_sets(cx.src_xy, cx.dst_xy, cx.id, s, d);
    make_hypothesis(s, d, cx.inv_t, cx.bounds, Hn, hc);
    unsigned n = 0;
    for (unsigned j = 0; j < qn; ++j) {
        const int pt = static_cast<int>(cx.queue[j * kRBlock]);
        const float2 sp = __ldg(cx.src_xy + pt), dq = __ldg(cx.dst_xy + pt);
        n += inlier_f64(Hn, sp.x, sp.y, dq.x, dq.y, cx.t) ? 1u : 0u;
        ++cx.n64;
    }
    return n;
}

// Verification mode (HG_RANSAC_DECIDE_ALL_F64): every pair of points [p0, p1) by the fp64 definition.
__device__ __noinline__ unsigned count_all_f64(SlowCtx& cx, int p0, int p1)
{
    double s[8], d[8], Hn[9];
    HypConst hc;
    gather_sets(cx.src_xy, cx.dst_xy, cx.id, s, d);
    make_hypothesis(s, d, cx.inv_t, cx.bounds, Hn, hc);
    unsigned c = 0;
    for (int pt = p0; pt < p1; ++pt) {
        const float2 sp = __ldg(cx.src_xy + pt), dq = __ldg(cx.dst_xy + pt);
        c += inlier_f64(Hn, sp.x, sp.y, dq.x, dq.y, cx.t) ? 1u : 0u;
    }
    cx.n64 += static_cast<unsigned>(p1 - p0);
    return c;
}

// Queue overflow (more than kQueueCap undecided pairs for one hypothesis: a horizon line through the table, or data
// sitting exactly on the threshold): the whole warp recounts lane L's hypothesis over points [p0, p1) -- every lane
// re-derives that hypothesis (deterministic, so identical), takes every 32nd point, applies the per-pair band to the
// sweep's own fp32 arithmetic and the fp64 definition to what stays undecided.  Returns the count (same on all lanes).
__device__ __noinline__ unsigned recount_warp(SlowCtx& cx, int L, int p0, int p1)
{
    const int4 id = make_int4(__shfl_sync(0xffffffffu, cx.id.x, L), __shfl_sync(0xffffffffu, cx.id.y, L),
                              __shfl_sync(0xffffffffu, cx.id.z, L), __shfl_sync(0xffffffffu, cx.id.w, L));
    double s[8], d[8], Hn[9];
    HypConst hc;
    gather_sets(cx.src_xy, cx.dst_xy, id, s, d);
    make_hypothesis(s, d, cx.inv_t, cx.bounds, Hn, hc);
    const int lane = threadIdx.x & 31;
    unsigned c = 0, n64 = 0;
    for (int pt = p0 + lane; pt < p1; pt += 32) {
        const float4 A = __ldg(cx.table + 2 * (pt >> 1)), B = __ldg(cx.table + 2 * (pt >> 1) + 1);
        const bool hi = pt & 1;
        unsigned r = recheck_f32(hc, hi ? A.y : A.x, hi ? A.w : A.z, hi ? B.y : B.x, hi ? B.w : B.z);
        if (r == 2u) {
            const float2 sp = __ldg(cx.src_xy + pt), dq = __ldg(cx.dst_xy + pt);
            r = inlier_f64(Hn, sp.x, sp.y, dq.x, dq.y, cx.t) ? 1u : 0u;
            ++n64;
        }
        c += r;
    }
    c = __reduce_add_sync(0xffffffffu, c);
    n64 = __reduce_add_sync(0xffffffffu, n64);
    if (lane == L) cx.n64 += n64;
    return c;
}

// Entry e of the table as the sweep sees it: CONST -> c_table (absolute float4 index), else shared memory.
template <bool CONST>
__device__ __forceinline__ float4 table_at(const float4* __restrict__ tb, int i) { return CONST ? c_table[i] : tb[i]; }

// G consecutive table entries (2G points) against one hypothesis; the entries are float4 [i0, i0 + 2G) of the
// table (`tb` in shared memory, or c_table when CONST).  `pt0` = index of the first point.
// Fast path: 11 FFMA2 + 2 sign-bit adds + one 3-input unsigned min per entry; the cold branch (queue the pair) is
// taken by a warp only when one of its lanes has a pair inside the band.
template <int G, bool ONLY_X, bool CONST>
__device__ __forceinline__ void sweep_group(const HypConst& hc, const float4* __restrict__ tb, int i0, int pt0,
                                            SlowCtx& cx, unsigned& n_in, unsigned& qn, unsigned& n_band)
{
    float2 a[G];
    bool amb = false;
#pragma unroll
    for (int g = 0; g < G; ++g) {
        const float4 A = table_at<CONST>(tb, i0 + 2 * g), B = table_at<CONST>(tb, i0 + 2 * g + 1);
        a[g] = score2(hc, make_float2(A.x, A.y), make_float2(A.z, A.w), make_float2(B.x, B.y), make_float2(B.z, B.w));
        n_in += sign_bit(a[g].x);
        amb |= (__float_as_uint(a[g].x) <= hc.thr);
        if (!ONLY_X) {
            n_in += sign_bit(a[g].y);
            amb |= (__float_as_uint(a[g].y) <= hc.thr);
        }
    }
    if (amb) {
        unsigned mask = 0u;                                   // bit 2g + j: lane j of entry g is in the band
#pragma unroll
        for (int g = 0; g < G; ++g) {
            mask |= (__float_as_uint(a[g].x) <= hc.thr) ? (1u << (2 * g)) : 0u;
            if (!ONLY_X) mask |= (__float_as_uint(a[g].y) <= hc.thr) ? (2u << (2 * g)) : 0u;
        }
#pragma unroll 1
        while (mask) {
            const int i = __ffs(mask) - 1;
            mask &= mask - 1u;
            // entry g = i >> 1 lives at float4 i0 + 2g, i0 + 2g + 1 (a per-lane index: a plain LDC in CONST mode)
            const float4 A = table_at<CONST>(tb, i0 + (i & ~1)), B = table_at<CONST>(tb, i0 + (i | 1));
            const bool hi = i & 1;
            const unsigned r = recheck_f32(hc, hi ? A.y : A.x, hi ? A.w : A.z, hi ? B.y : B.x, hi ? B.w : B.z);
            ++n_band;
            if (r == 2u) {
                if (qn < kQueueCap) cx.queue[qn * kRBlock] = static_cast<unsigned>(pt0 + i);
                ++qn;                                         // qn > kQueueCap: overflow, see the end of the sweep
            } else {
                n_in += r;
            }
        }
    }
}

constexpr int kSyncEntries = 512;   // constant-bank path: table entries between CTA barriers (a multiple of kGroup)
constexpr int kGroup = 8;     // table entries per cold-path check (8: +2 % over 4 on C4, measured)

// CONST: the table is c_table (no staging, no table in shared memory); else it is staged from `table` (global).
template <bool CONST>
__global__ void __launch_bounds__(kRBlock, 2)
ransac_score_kernel(const float2* __restrict__ src_xy, const float2* __restrict__ dst_xy, int n_pts,
                    const float4* __restrict__ table, int n_pairs, HypSource hs,
                    double inv_t, double t, int* __restrict__ counts, RansacHeader* __restrict__ hdr)
{
    if (hs.check_stop && hdr->stop) return;                 // uniform: written by an earlier launch on this stream
    extern __shared__ __align__(128) unsigned char smem_raw[];
    constexpr size_t kStageBytes = CONST ? 0 : size_t(kStages) * kChunkPairs * 32;
    float4* stage_buf = reinterpret_cast<float4*>(smem_raw);                       // kStages * kChunkPairs * 2 float4
    unsigned* queue = reinterpret_cast<unsigned*>(smem_raw + kStageBytes);         // [kQueueCap][kRBlock]
    uint64_t* full = reinterpret_cast<uint64_t*>(queue + kQueueCap * kRBlock);

    // Small hypothesis batches are split over the table as well (blockIdx.y = part), so that a call with a few
    // thousand hypotheses still fills the machine; this CTA sweeps entries [e_begin, e_end).
    const int e_begin = blockIdx.y * hs.part_entries;
    const int e_end = min(n_pairs, e_begin + hs.part_entries);
    const bool split = gridDim.y > 1;
    const int n_chunks = (e_end - e_begin + kChunkPairs - 1) / kChunkPairs;
    if (!CONST) {
        if (threadIdx.x == 0) {
            for (int s = 0; s < kStages; ++s) mbar_init(&full[s], 1);
            fence_barrier_init();
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            for (int c = 0; c < kStages && c < n_chunks; ++c) {
                const int first = e_begin + c * kChunkPairs;
                const int pairs = min(kChunkPairs, e_end - first);
                mbar_arrive_expect_tx(&full[c], pairs * 32u);
                bulk_copy_g2s(stage_buf + size_t(c) * kChunkPairs * 2, table + size_t(first) * 2, pairs * 32u, &full[c]);
            }
        }
    }

    // hypothesis set-up (overlaps the first table copies)
    long long hidx = hs.h0 + static_cast<long long>(blockIdx.x) * kRBlock + threadIdx.x;
    bool active = hidx < hs.h1;
    HypConst hc;
    SlowCtx cx;
    bool ok = false;
    {
        cx.bounds[0] = __uint_as_float(hdr->bound_bits[0]); cx.bounds[1] = __uint_as_float(hdr->bound_bits[1]);
        cx.bounds[2] = __uint_as_float(hdr->bound_bits[2]); cx.bounds[3] = __uint_as_float(hdr->bound_bits[3]);
        double s[8], d[8], Hn[9];
        cx.id = active ? hypothesis_indices(hs, hidx, n_pts) : make_int4(0, 0, 0, 0);   // inactive: degenerate => sure outliers
        if (active && hs.idx_out && blockIdx.y == 0) hs.idx_out[hidx] = cx.id;
        gather_sets(src_xy, dst_xy, cx.id, s, d);
        if (hs.flags & HG_RANSAC_REJECT_DEGENERATE) {
            // Reading R20.  A rejected hypothesis scores 0 at once; the accepted ones are compacted onto the first threads
            // of the CTA, so that whole warps fall idle and skip the sweep (the queue area is free until the sweep starts).
            __shared__ unsigned warp_accepted[kRBlock / 32];
            int4* ids = reinterpret_cast<int4*>(queue);                                   // [kRBlock]
            unsigned* owners = queue + 4 * kRBlock;                                       // [kRBlock]
            const bool accept = active && !sample_rejected(s, d, hs.reject_lim2);
            const unsigned lane = threadIdx.x & 31u, wid = threadIdx.x >> 5;
            const unsigned bal = __ballot_sync(0xffffffffu, accept);
            if (active && !accept) {
                if (!split && counts) counts[hidx] = 0;
            }
            {   // rejected hypotheses still take part in the argmax with count 0; statistics
                unsigned long long key = (active && !accept && !split) ? pack_key(0u, static_cast<unsigned>(hidx)) : 0ull;
                key = warp_max_u64(key);
                const unsigned nrej = __popc(__ballot_sync(0xffffffffu, active && !accept));
                if (lane == 0) {
                    if (key != 0ull) atomicMax(&hdr->best_key, key);
                    if (nrej && blockIdx.y == 0) atomicAdd(&hdr->n_rejected, static_cast<unsigned long long>(nrej));
                    warp_accepted[wid] = __popc(bal);
                }
            }
            __syncthreads();
            unsigned before = 0, total = 0;
#pragma unroll
            for (unsigned w = 0; w < kRBlock / 32; ++w) { const unsigned c = warp_accepted[w]; before += (w < wid) ? c : 0u; total += c; }
            if (accept) {
                const unsigned rank = before + __popc(bal & ((1u << lane) - 1u));
                ids[rank] = cx.id;
                owners[rank] = threadIdx.x;
            }
            __syncthreads();
            active = threadIdx.x < total;
            if (active) {
                cx.id = ids[threadIdx.x];
                hidx = hs.h0 + static_cast<long long>(blockIdx.x) * kRBlock + owners[threadIdx.x];
            } else {
                cx.id = make_int4(0, 0, 0, 0);
            }
            __syncthreads();                                                              // the queue area is reused by the sweep
            gather_sets(src_xy, dst_xy, cx.id, s, d);
        }
        ok = make_hypothesis(s, d, inv_t, cx.bounds, Hn, hc) && active;
    }
    const bool warp_live = __any_sync(0xffffffffu, active);    // a warp without hypotheses skips the sweep (not the barriers)
    cx.src_xy = src_xy; cx.dst_xy = dst_xy; cx.table = table; cx.inv_t = inv_t; cx.t = t;
    cx.queue = queue + threadIdx.x; cx.n64 = 0u;

    unsigned n_in = 0, qn = 0, n_band = 0;
    const int full_pairs = n_pts >> 1;                     // entries holding two distinct points
    if (hs.flags & HG_RANSAC_DECIDE_ALL_F64) {
        // verification mode: no fp32 sweep, every pair of this part by the definition in fp64
        const int p0 = 2 * e_begin, p1 = min(n_pts, 2 * e_end);
        if (active) n_in = count_all_f64(cx, p0, p1);
    } else if (CONST) {
        const int e_two = min(e_end, full_pairs);          // entries [e_begin, e_two) hold two distinct points
        int k = e_begin;
        // Windows of kSyncEntries entries with a CTA barrier in between: the warps of a CTA drift apart (cold-path
        // excursions), and the constant cache serves the uniform loads well only while they walk the table together
        // (C4: 1.68 ms without the barriers, 1.62 ms with a window of 512 or 1024 entries, 1.63 ms with 256).
#pragma unroll 1
        for (int w_end = e_begin; k + kGroup <= e_two; ) {
            w_end = min(e_two, w_end + kSyncEntries);
            if (warp_live) {
#pragma unroll 1
                for (; k + kGroup <= w_end; k += kGroup)
                    sweep_group<kGroup, false, true>(hc, nullptr, 2 * k, 2 * k, cx, n_in, qn, n_band);
            } else {
                k += (w_end - k) / kGroup * kGroup;
            }
            if (w_end < e_two) __syncthreads();
            else break;
        }
        if (warp_live) {
#pragma unroll 1
            for (; k < e_two; ++k)
                sweep_group<1, false, true>(hc, nullptr, 2 * k, 2 * k, cx, n_in, qn, n_band);
            if ((n_pts & 1) && full_pairs >= e_begin && full_pairs < e_end)     // odd tail point: counts once
                sweep_group<1, true, true>(hc, nullptr, 2 * full_pairs, 2 * full_pairs, cx, n_in, qn, n_band);
        }
    } else {
        for (int c = 0; c < n_chunks; ++c) {
            const int st = c % kStages;
            mbar_wait(&full[st], (c / kStages) & 1);
            const float4* tb = stage_buf + size_t(st) * kChunkPairs * 2;
            const int first = e_begin + c * kChunkPairs;
            const int pairs = min(min(kChunkPairs, e_end - first), full_pairs - first);   // may be <= 0 in a tail-only chunk
            if (warp_live) {
                int k = 0;
#pragma unroll 1
                for (; k + kGroup <= pairs; k += kGroup)
                    sweep_group<kGroup, false, false>(hc, tb, 2 * k, 2 * (first + k), cx, n_in, qn, n_band);
#pragma unroll 1
                for (; k < pairs; ++k)
                    sweep_group<1, false, false>(hc, tb, 2 * k, 2 * (first + k), cx, n_in, qn, n_band);
                // odd tail point: the duplicated entry counts once
                if ((n_pts & 1) && full_pairs >= first && full_pairs < min(first + kChunkPairs, e_end))
                    sweep_group<1, true, false>(hc, tb, 2 * (full_pairs - first), 2 * full_pairs, cx, n_in, qn, n_band);
            }
            if (c + kStages < n_chunks) {                      // refill this stage (uniform branch)
                __syncthreads();
                if (threadIdx.x == 0) {
                    const int fn = e_begin + (c + kStages) * kChunkPairs;
                    const int pn = min(kChunkPairs, e_end - fn);
                    mbar_arrive_expect_tx(&full[st], pn * 32u);
                    bulk_copy_g2s(stage_buf + size_t(st) * kChunkPairs * 2, table + size_t(fn) * 2, pn * 32u, &full[st]);
                }
            }
        }
    }

    // The queued pairs, all lanes of the warp together.  A hypothesis with more than kQueueCap undecided pairs is instead
    // recounted from scratch by the whole warp.
    if (__any_sync(0xffffffffu, qn != 0u)) {
        unsigned ovf = __ballot_sync(0xffffffffu, qn > kQueueCap);
        if (qn != 0u && qn <= kQueueCap) n_in += drain_queue(cx, qn);
        while (ovf) {                                       // warp-uniform
            const int L = __ffs(ovf) - 1;
            ovf &= ovf - 1u;
            const unsigned c = recount_warp(cx, L, 2 * e_begin, min(n_pts, 2 * e_end));
            if ((threadIdx.x & 31) == L) n_in = c;
        }
    }
    const unsigned n64 = active ? cx.n64 : 0u;
    const unsigned count = ok ? n_in : 0u;
    if (split) {                                            // partial count; ransac_best_kernel finishes the job
        if (active && count) atomicAdd(hs.acc + hidx, static_cast<int>(count));
    } else {
        unsigned long long key = 0ull;
        if (active) {
            if (counts) counts[hidx] = static_cast<int>(count);
            key = pack_key(count, static_cast<unsigned>(hidx));
        }
        key = warp_max_u64(key);
        if ((threadIdx.x & 31) == 0 && key != 0ull) atomicMax(&hdr->best_key, key);
    }
    // statistics: hypotheses that needed fp64 decisions, and how many pairs
    const unsigned amb_mask = __ballot_sync(0xffffffffu, n64 != 0u);
    const unsigned band_tot = __reduce_add_sync(0xffffffffu, active ? n_band : 0u);
    if (amb_mask) {
        const unsigned tot = __reduce_add_sync(0xffffffffu, n64);
        if ((threadIdx.x & 31) == 0) {
            atomicAdd(&hdr->n_fixup, static_cast<unsigned long long>(__popc(amb_mask)));
            atomicAdd(&hdr->n_pairs_f64, static_cast<unsigned long long>(tot));
        }
    }
    if (band_tot && (threadIdx.x & 31) == 0) atomicAdd(&hdr->n_band, static_cast<unsigned long long>(band_tot));
}

// ---- 2a. tiny calls (the regime of the paper's Table 6) --------------------------------------------------
// A call of a few thousand hypotheses on a table that fits shared memory is latency-, not throughput-bound: what it costs
// is the number of dependent round trips to L2 (~450 ns each at this clock), barriers and launches on its critical path,
// not its arithmetic.  The call is two launches that overlap: a one-CTA kernel that zeroes the header and the slots and
// releases its dependent at once (programmatic dependent launch), and this kernel, which touches them only after
// `griddepcontrol.wait` -- its whole set-up and sweep run meanwhile.  (A memset node instead costs 3 us in a graph.)
// Decomposition: blockIdx.x = a group of 32 hypotheses (lane = hypothesis), blockIdx.y = a part of the table; the CTAs
// of one group form a thread-block cluster (1 x P x 1, P <= 8, chosen so that the call covers the machine).  Critical path:
//   1. one round trip: the hypothesis indices and the whole table (every CTA packs all of it into shared memory; the
//      sampled correspondences are then gathered from there instead of by a second, dependent round trip);
//   2. every warp derives the 32 hypotheses itself (fp64 solve: latency, not throughput, at one warp per scheduler -- no
//      exchange is cheaper than recomputing) and sweeps a quarter of its CTA's part; pairs inside the band are only noted
//      and decided after the sweep, all lanes side by side;
//   3. partial counts reach the cluster's rank-0 CTA by st.async into its shared memory, completing on its mbarrier (no
//      cluster-wide barrier: ~400 cycles instead of ~1900);
//   4. that CTA emits counts[] and publishes the group's best (count, index) with -- from its own registers -- the
//      unit-Frobenius H of that hypothesis in a slot of stamped words, taking a global ticket in the same breath (no fence);
//   5. the last group reads the slots (one more round trip) and writes the winner.
constexpr int kTinyHyp = 32;                      // hypotheses per group
constexpr int kTinyThreads = 128;
constexpr int kTinyWarps = kTinyThreads / 32;     // warps of a CTA = quarters of its part of the table
constexpr int kTinyMaxParts = 8;                  // portable cluster size

__device__ __forceinline__ void grid_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void grid_dependency_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void cluster_arrive_release() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait_acquire() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }

// Zeroes the first `n16` 16-byte words of the workspace; its dependent launch may start at once.
__global__ void __launch_bounds__(256) ransac_zero_kernel(uint4* __restrict__ p, int n16)
{
    grid_launch_dependents();
    for (int i = blockIdx.x * 256 + threadIdx.x; i < n16; i += gridDim.x * 256) p[i] = make_uint4(0u, 0u, 0u, 0u);
}

// What a group leaves for the final step: its best (count, index) and that hypothesis' unit-Frobenius H.
// Every 64-bit word carries its own stamp (high half) beside 32 bits of payload: key low, key high, h[0..8].  A relaxed
// 64-bit store or load is single-copy atomic, so a word whose stamp reads kSlotStamp is this call's (the zero kernel
// cleared the slots) -- the final step can therefore take its ticket WITHOUT first waiting for the slot stores to be
// acknowledged (no fence: one round trip to L2 instead of two), and the last group simply re-reads a word whose stamp has
// not landed yet.  The stores were issued before the ticket, so they land whatever the issuing CTA does next: the wait is
// bounded by a memory latency and depends on no other CTA being scheduled.
constexpr int kSlotWords = 11;
constexpr unsigned kSlotStamp = 0x5EED0001u;
struct __align__(16) TinySlot { unsigned long long w[kSlotWords + 1]; };
static_assert(sizeof(TinySlot) == 96, "slot layout");
__device__ __forceinline__ void st_relaxed_gpu_u64(unsigned long long* p, unsigned long long v)
{ asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" :: "l"(p), "l"(v) : "memory"); }
__device__ __forceinline__ unsigned long long ld_relaxed_gpu_u64(const unsigned long long* p)
{ unsigned long long v; asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory"); return v; }
__device__ __forceinline__ unsigned long long stamped(unsigned payload) { return (static_cast<unsigned long long>(kSlotStamp) << 32) | payload; }

// Table entry of the tiny kernel: the two float4 of the packed table plus the raw targets (dx0, dx1, dy0, dy1), so that a
// pair inside the band is decided by the definition from shared memory and the fp64 H the thread still holds, and the
// sampled correspondences are gathered from it.
constexpr int kTinyEntry = 3;                     // float4 per entry

// One 32-bit word into the shared memory of CTA `rank` of this cluster, counted (4 bytes) on that CTA's mbarrier when it has
// landed: the consumer waits on its own mbarrier and then reads its own shared memory -- no cluster-wide barrier.
__device__ __forceinline__ void st_async_cluster_u32(const void* local_data, const uint64_t* local_bar, unsigned rank, unsigned v)
{
    unsigned rd, rb;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(rd) : "r"(smem_u32(local_data)), "r"(rank));
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(rb) : "r"(smem_u32(local_bar)), "r"(rank));
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.u32 [%0], %1, [%2];" :: "r"(rd), "r"(v), "r"(rb) : "memory");
}

// Point `hi` of table entry `e` by the definition in fp64 (reading R9); the entry holds the raw coordinates.
__device__ __forceinline__ unsigned tiny_inlier_f64(const double Hn[9], double t, const float4* __restrict__ e, unsigned hi)
{
    const float4 A = e[0], D = e[2];
    return inlier_f64_nodiv(Hn, hi ? A.y : A.x, hi ? A.w : A.z, hi ? D.y : D.x, hi ? D.w : D.z, t) ? 1u : 0u;
}

// The noted pairs of this thread (queue items: first entry of the group << 16 | 16 flags, bit 2g + j = point j of entry
// k0 + g) by the definition in fp64; returns the number of inliers among them.  Out of line and with H by value: one copy
// of the code, H stays in registers at the call sites.
__device__ __noinline__ unsigned tiny_drain(const float4* __restrict__ tb, const unsigned* __restrict__ queue, unsigned qn, double t,
                                            double h0, double h1, double h2, double h3, double h4, double h5, double h6, double h7, double h8)
{
    const double Hn[9] = { h0, h1, h2, h3, h4, h5, h6, h7, h8 };
    unsigned n = 0;
    for (unsigned j = 0; j < qn; ++j) {
        const unsigned item = queue[j * kTinyThreads];
        unsigned m = item & 0xffffu;
        while (m) {
            const int i = __ffs(m) - 1;
            m &= m - 1u;
            n += tiny_inlier_f64(Hn, t, tb + kTinyEntry * ((item >> 16) + (i >> 1)), i & 1);   // (a noted pair has a value >= 0: the sweep has not counted it)
        }
    }
    return n;
}

// G consecutive entries (2G points) from entry k0 of the table `tb`, against one hypothesis.  The fast path is the one of
// sweep_group.  When a pair of the group lies inside the table-wide band the thread only notes (k0, which of the 2G points)
// in its own queue -- branch-free flags and one store: what a lone warp per scheduler pays for a divergent excursion is
// its latency, not its instruction count -- and the warp decides the noted pairs after the sweep, all lanes side by side,
// straight by the definition in fp64 (cheap since it needs no division; the per-pair fp32 band of the big kernel would
// cost as much as it saves here).  A thread whose queue is full (a hypothesis with a horizon line through the table)
// drains it on the spot and goes on.  `n64` counts the pairs noted = decided in fp64.
template <int G, bool ONLY_X>
__device__ __forceinline__ void tiny_group(const HypConst& hc, const double Hn[9], double t, const float4* __restrict__ tb, int k0,
                                           unsigned* __restrict__ queue, unsigned& n_in, unsigned& qn, unsigned& n64)
{
    float2 a[G];
    bool amb = false;
#pragma unroll
    for (int g = 0; g < G; ++g) {
        const float4 A = tb[kTinyEntry * (k0 + g)], B = tb[kTinyEntry * (k0 + g) + 1];
        a[g] = score2(hc, make_float2(A.x, A.y), make_float2(A.z, A.w), make_float2(B.x, B.y), make_float2(B.z, B.w));
        n_in += sign_bit(a[g].x);
        amb |= (__float_as_uint(a[g].x) <= hc.thr);
        if (!ONLY_X) {
            n_in += sign_bit(a[g].y);
            amb |= (__float_as_uint(a[g].y) <= hc.thr);
        }
    }
    if (amb) {
        unsigned mask = 0u;                                   // bit 2g + j: point j of entry k0 + g is in the band
#pragma unroll
        for (int g = 0; g < G; ++g) {
            mask |= (__float_as_uint(a[g].x) <= hc.thr) ? (1u << (2 * g)) : 0u;
            if (!ONLY_X) mask |= (__float_as_uint(a[g].y) <= hc.thr) ? (2u << (2 * g)) : 0u;
        }
        if (qn == kQueueCap) {
            n_in += tiny_drain(tb, queue, qn, t, Hn[0], Hn[1], Hn[2], Hn[3], Hn[4], Hn[5], Hn[6], Hn[7], Hn[8]);
            qn = 0u;
        }
        queue[qn * kTinyThreads] = (static_cast<unsigned>(k0) << 16) | mask;
        ++qn;
        n64 += __popc(mask);
    }
}

// statistics words of one warp (the header is zero by now)
__device__ __forceinline__ void tiny_stats(RansacHeader* __restrict__ hdr, unsigned n64, unsigned n_band)
{
    const unsigned amb_mask = __ballot_sync(0xffffffffu, n64 != 0u);
    const unsigned tot = __reduce_add_sync(0xffffffffu, n64);
    const unsigned band_tot = __reduce_add_sync(0xffffffffu, n_band);
    if ((threadIdx.x & 31) == 0) {
        if (amb_mask) { atomicAdd(&hdr->n_fixup, static_cast<unsigned long long>(__popc(amb_mask)));
                        atomicAdd(&hdr->n_pairs_f64, static_cast<unsigned long long>(tot)); }
        if (band_tot) atomicAdd(&hdr->n_band, static_cast<unsigned long long>(band_tot));
    }
}

__global__ void __launch_bounds__(kTinyThreads)
ransac_tiny_kernel(const float2* __restrict__ src_xy, const float2* __restrict__ dst_xy, int n_pts, int n_pairs, HypSource hs,
                   double inv_t, double t, int* __restrict__ counts, RansacHeader* __restrict__ hdr, TinySlot* __restrict__ slots,
                   float* __restrict__ best_H, long long* __restrict__ best_index, int* __restrict__ best_count,
                   long long* __restrict__ n_evaluated)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float4* tb = reinterpret_cast<float4*>(smem_raw);                   // n_pairs * kTinyEntry float4: the whole table
    unsigned* queue = reinterpret_cast<unsigned*>(tb + size_t(n_pairs) * kTinyEntry) + threadIdx.x;   // [kQueueCap][kTinyThreads]
    __shared__ float red[4][kTinyWarps];
    __shared__ unsigned partial[kTinyWarps][kTinyHyp];
    __shared__ unsigned cl_partial[kTinyMaxParts][kTinyHyp];            // rank 0: the counts of the other parts land here
    __shared__ __align__(8) uint64_t cl_bar;                            // rank 0: completes when all of them have
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int part = blockIdx.y, parts = gridDim.y;                     // cluster = (1, parts, 1): rank = part
    if (parts > 1) {
        if (part == 0 && threadIdx.x == 0) {
            mbar_init(&cl_bar, 1);
            fence_barrier_init();
            mbar_arrive_expect_tx(&cl_bar, static_cast<uint32_t>(parts - 1) * kTinyHyp * 4u);
        }
        cluster_arrive_release();                   // waited for by the senders: rank 0 runs and its mbarrier is armed
    }

    // first loads: the hypothesis (lane = hypothesis, every warp its own copy) and the table
    const long long hidx = hs.h0 + static_cast<long long>(blockIdx.x) * kTinyHyp + lane;
    const bool active = hidx < hs.h1;
    int4 id = make_int4(0, 0, 0, 0);                                    // beyond the last hypothesis: a degenerate sample
    if (active) {                                                       // caller's indices, or sampled on the device (R19)
        id = hypothesis_indices(hs, hidx, n_pts);
        if (hs.idx_out && part == 0 && wid == 0) hs.idx_out[hidx] = id;
    }

    // One pass over the table: every CTA packs all of it into its shared memory (the sampled correspondences are gathered
    // from there, one memory latency earlier than a dependent global gather) and takes the coordinate bounds; it sweeps only
    // its part.  Two points per 128-bit load, four loads of each plane in flight per thread.
    const int e0 = min(n_pairs, part * hs.part_entries), e1 = min(n_pairs, e0 + hs.part_entries);
    const int full_pairs = n_pts >> 1;
    const float4* s4 = reinterpret_cast<const float4*>(src_xy);
    const float4* d4 = reinterpret_cast<const float4*>(dst_xy);
    float m0 = 0.f, m1 = 0.f, m2 = 0.f, m3 = 0.f;
    unsigned n_in = 0, n64 = 0, n_band = 0;
    for (int base = 0; base < n_pairs; base += 4 * kTinyThreads) {
        float4 sv[4], dv[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int k = base + u * kTinyThreads + threadIdx.x;
            if (k < full_pairs) { sv[u] = __ldg(s4 + k); dv[u] = __ldg(d4 + k); }
            else if (k < n_pairs) {                                                       // odd tail point, duplicated
                const float2 a = __ldg(src_xy + 2 * k), b = __ldg(dst_xy + 2 * k);
                sv[u] = make_float4(a.x, a.y, a.x, a.y); dv[u] = make_float4(b.x, b.y, b.x, b.y);
            } else { sv[u] = make_float4(0.f, 0.f, 0.f, 0.f); dv[u] = sv[u]; }
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int k = base + u * kTinyThreads + threadIdx.x;
            const float4 A = make_float4(sv[u].x, sv[u].z, sv[u].y, sv[u].w);
            const float4 B = make_float4(static_cast<float>(-double(dv[u].x) * inv_t), static_cast<float>(-double(dv[u].z) * inv_t),
                                         static_cast<float>(-double(dv[u].y) * inv_t), static_cast<float>(-double(dv[u].w) * inv_t));
            if (k < n_pairs) {
                float4* e = tb + kTinyEntry * k;
                e[0] = A; e[1] = B; e[2] = make_float4(dv[u].x, dv[u].z, dv[u].y, dv[u].w);
            }
            m0 = fmaxf(m0, fmaxf(fabsf(A.x), fabsf(A.y)));
            m1 = fmaxf(m1, fmaxf(fabsf(A.z), fabsf(A.w)));
            m2 = fmaxf(m2, fmaxf(fabsf(B.x), fabsf(B.y)));
            m3 = fmaxf(m3, fmaxf(fabsf(B.z), fabsf(B.w)));
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        m0 = fmaxf(m0, __shfl_xor_sync(0xffffffffu, m0, o));
        m1 = fmaxf(m1, __shfl_xor_sync(0xffffffffu, m1, o));
        m2 = fmaxf(m2, __shfl_xor_sync(0xffffffffu, m2, o));
        m3 = fmaxf(m3, __shfl_xor_sync(0xffffffffu, m3, o));
    }
    if (lane == 0) { red[0][wid] = m0; red[1][wid] = m1; red[2][wid] = m2; red[3][wid] = m3; }
    __syncthreads();

    // lane = hypothesis: gather from the table in shared memory, solve, sample check, band
    float bounds[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        float m = 0.f;
#pragma unroll
        for (int w = 0; w < kTinyWarps; ++w) m = fmaxf(m, red[q][w]);
        bounds[q] = m;
    }
    HypConst hc;
    double Hraw[9], Hn[9];
    bool usable, rejected = false;                   // usable: H finite and non-zero, sample not rejected
    {
        double s[8], d[8];
        const int ids[4] = { id.x, id.y, id.z, id.w };
#pragma unroll
        for (int k = 0; k < 4; ++k) {                // point p: entry p >> 1, half p & 1 of A = (sx0, sx1, sy0, sy1), D = (dx0, dx1, dy0, dy1)
            const float* e = reinterpret_cast<const float*>(tb + kTinyEntry * (ids[k] >> 1)) + (ids[k] & 1);
            s[2 * k] = e[0]; s[2 * k + 1] = e[2]; d[2 * k] = e[8]; d[2 * k + 1] = e[10];
        }
        usable = solve_for_sweep(s, d, inv_t, Hraw, Hn, hc);
        if ((hs.flags & HG_RANSAC_REJECT_DEGENERATE) && active && sample_rejected(s, d, hs.reject_lim2)) { usable = false; rejected = true; }
    }
    const bool ok = usable && active;
    error_band(bounds, usable, hc);                  // unusable: every point a sure outlier

    // quarter of this warp: whole groups of kGroup entries; the last non-empty quarter takes the remainder and the odd tail point
    const int per = ((e1 - e0 + kTinyWarps - 1) / kTinyWarps + kGroup - 1) / kGroup * kGroup;
    const int w0 = min(e1, e0 + wid * per), w1 = min(e1, w0 + per);
    unsigned qn = 0;
    if (hs.flags & HG_RANSAC_DECIDE_ALL_F64) {       // verification mode: every pair by the definition in fp64
        if (active) {
            for (int k = w0; k < w1; ++k) {
                const float4* e = tb + kTinyEntry * k;
                const float4 A = e[0], D = e[2];
                n_in += inlier_f64_nodiv(Hn, A.x, A.z, D.x, D.z, t) ? 1u : 0u;
                ++n64;
                if (2 * k + 1 < n_pts) { n_in += inlier_f64_nodiv(Hn, A.y, A.w, D.y, D.w, t) ? 1u : 0u; ++n64; }
            }
        }
    } else {
        const int e_two = min(w1, full_pairs);
        int k = w0;
#pragma unroll 1
        for (; k + kGroup <= e_two; k += kGroup)
            tiny_group<kGroup, false>(hc, Hn, t, tb, k, queue, n_in, qn, n64);
#pragma unroll 1
        for (; k < e_two; ++k)
            tiny_group<1, false>(hc, Hn, t, tb, k, queue, n_in, qn, n64);
        if ((n_pts & 1) && full_pairs >= w0 && full_pairs < w1)
            tiny_group<1, true>(hc, Hn, t, tb, full_pairs, queue, n_in, qn, n64);
        // the pairs noted during the sweep, all lanes of the warp side by side
        if (qn) n_in += tiny_drain(tb, queue, qn, t, Hn[0], Hn[1], Hn[2], Hn[3], Hn[4], Hn[5], Hn[6], Hn[7], Hn[8]);
        n_band = n64;
    }
    partial[wid][lane] = ok ? n_in : 0u;
    // the group's leader warp: every lane's candidate, the unit-Frobenius H (raw ACA scale normalised, as ransac_finalize_kernel does)
    float hcand[9];
    if (part == 0 && wid == 0) {
        normalise<double>(Hraw, 2);
#pragma unroll
        for (int k = 0; k < 9; ++k) hcand[k] = static_cast<float>(Hraw[k]);
    }
    grid_dependency_wait();                                   // the header is zero from here on
    __syncthreads();
    unsigned total = 0;
    if (wid == 0) {
#pragma unroll
        for (int w = 0; w < kTinyWarps; ++w) total += partial[w][lane];
    }
    if (parts > 1) {                                          // the parts of this group meet in the rank-0 CTA
        if (wid != 0) { tiny_stats(hdr, n64, n_band); return; }
        if (part != 0) {
            cluster_wait_acquire();
            st_async_cluster_u32(&cl_partial[part][lane], &cl_bar, 0u, total);
            tiny_stats(hdr, n64, n_band);
            return;
        }
        mbar_wait(&cl_bar, 0);
        for (int q = 1; q < parts; ++q) total += cl_partial[q][lane];
    }
    if (wid != 0) { tiny_stats(hdr, n64, n_band); return; }
    // The lane that holds the group's best hypothesis (largest count, lowest index = lowest lane) publishes the slot and, in
    // the same breath, takes the ticket (see TinySlot: stamped words, no fence in between).
    const unsigned cnt_max = __reduce_max_sync(0xffffffffu, active ? total : 0u);
    const int wl = __ffs(__ballot_sync(0xffffffffu, active && total == cnt_max)) - 1;
    unsigned ticket = 0;
    if (lane == wl) {
        const unsigned long long key = pack_key(total, static_cast<unsigned>(hidx));
        unsigned long long* sl = slots[blockIdx.x].w;
        st_relaxed_gpu_u64(sl + 0, stamped(static_cast<unsigned>(key)));
        st_relaxed_gpu_u64(sl + 1, stamped(static_cast<unsigned>(key >> 32)));
#pragma unroll
        for (int k = 0; k < 9; ++k) st_relaxed_gpu_u64(sl + 2 + k, stamped(__float_as_uint(hcand[k])));
        ticket = atomicAdd(&hdr->blocks_done, 1u);
    }
    if (active && counts) counts[hidx] = static_cast<int>(total);
    const unsigned nrej = __popc(__ballot_sync(0xffffffffu, rejected));
    if (lane == 0 && nrej) atomicAdd(&hdr->n_rejected, static_cast<unsigned long long>(nrej));
    tiny_stats(hdr, n64, n_band);
    ticket = __shfl_sync(0xffffffffu, ticket, wl);
    if (ticket != gridDim.x - 1) return;
    if (lane == 0) {                                          // a single round: every hypothesis was scored (adaptive entry point)
        hdr->n_evaluated = static_cast<unsigned long long>(hs.h1);
        if (n_evaluated) *n_evaluated = hs.h1;
    }
    // the last group: every group has issued its slot; the best slot of all
    const int n_groups = static_cast<int>(gridDim.x);
    if (n_groups <= 32) {                                     // one slot per lane, key and H in one round trip
        unsigned long long w[kSlotWords];
        unsigned long long bk = 0ull;
        if (lane < n_groups) {
            const unsigned long long* sl = slots[lane].w;
            bool all;
            do {
                all = true;
#pragma unroll
                for (int k = 0; k < kSlotWords; ++k) { w[k] = ld_relaxed_gpu_u64(sl + k); all = all && static_cast<unsigned>(w[k] >> 32) == kSlotStamp; }
            } while (!all);
            bk = (static_cast<unsigned long long>(static_cast<unsigned>(w[1])) << 32) | static_cast<unsigned>(w[0]);
        }
        const unsigned long long best = warp_max_u64(bk);
        if (bk == best && best != 0ull) {
            hdr->best_key = best;
            if (best_index) *best_index = static_cast<long long>(0xFFFFFFFFu - static_cast<unsigned>(best & 0xFFFFFFFFull));
            if (best_count) *best_count = static_cast<int>(best >> 32);
            if (best_H) {
#pragma unroll
                for (int k = 0; k < 9; ++k) best_H[k] = __uint_as_float(static_cast<unsigned>(w[2 + k]));
            }
        }
    } else {                                                  // keys first (four slots per lane in flight), then the winner's H
        unsigned long long bk = 0ull;
        int bg = 0;
        for (int base = 0; base < n_groups; base += 128) {
            unsigned long long lo[4], hi[4];
            bool all;
            do {
                all = true;
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int g = min(base + 32 * u + lane, n_groups - 1);
                    lo[u] = ld_relaxed_gpu_u64(slots[g].w); hi[u] = ld_relaxed_gpu_u64(slots[g].w + 1);
                    all = all && static_cast<unsigned>(lo[u] >> 32) == kSlotStamp && static_cast<unsigned>(hi[u] >> 32) == kSlotStamp;
                }
            } while (!all);
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const unsigned long long k64 = (static_cast<unsigned long long>(static_cast<unsigned>(hi[u])) << 32) | static_cast<unsigned>(lo[u]);
                if (k64 > bk) { bk = k64; bg = min(base + 32 * u + lane, n_groups - 1); }
            }
        }
        const unsigned long long best = warp_max_u64(bk);
        bg = __shfl_sync(0xffffffffu, bg, __ffs(__ballot_sync(0xffffffffu, bk == best)) - 1);
        if (lane < 9 && best_H) {
            unsigned long long w;
            do { w = ld_relaxed_gpu_u64(slots[bg].w + 2 + lane); } while (static_cast<unsigned>(w >> 32) != kSlotStamp);
            best_H[lane] = __uint_as_float(static_cast<unsigned>(w));
        }
        if (lane == 0) {
            hdr->best_key = best;
            if (best_index) *best_index = static_cast<long long>(0xFFFFFFFFu - static_cast<unsigned>(best & 0xFFFFFFFFull));
            if (best_count) *best_count = static_cast<int>(best >> 32);
        }
    }
}

// ---- 2b. best (split mode): total counts of hypotheses [h0, h1) -> counts[] and the packed maximum --------
__global__ void __launch_bounds__(256)
ransac_best_kernel(const int* __restrict__ acc, long long h0, long long h1, int* __restrict__ counts, RansacHeader* __restrict__ hdr,
                   int check_stop)
{
    if (check_stop && hdr->stop) return;
    const long long h = h0 + static_cast<long long>(blockIdx.x) * 256 + threadIdx.x;
    unsigned long long key = 0ull;
    if (h < h1) {
        const int c = acc[h];
        if (counts) counts[h] = c;
        key = pack_key(static_cast<unsigned>(c), static_cast<unsigned>(h));
    }
    key = warp_max_u64(key);
    if ((threadIdx.x & 31) == 0 && key != 0ull) atomicMax(&hdr->best_key, key);
}

// ---- 3. round (adaptive mode): the termination rule after `done` hypotheses ----------------------
// Reading R19: w = best_count / n_pts; stop iff done * log1p(-w^4) <= log1p(-confidence), i.e. once
// done >= log(1 - confidence) / log(1 - w^4); confidence <= 0 never stops early.
__global__ void ransac_round_kernel(RansacHeader* __restrict__ hdr, int n_pts, long long done, double confidence, int last)
{
    if (threadIdx.x != 0 || blockIdx.x != 0 || hdr->stop) return;
    bool stop = last != 0;
    if (confidence > 0.0) {
        const double w = static_cast<double>(hdr->best_key >> 32) / static_cast<double>(n_pts);
        const double q = w * w * w * w;
        stop = stop || (static_cast<double>(done) * log1p(-q) - log1p(-confidence) <= 0.0);
    }
    if (stop) { hdr->n_evaluated = static_cast<unsigned long long>(done); hdr->stop = 1u; }
}

// ---- 4. finalize -----------------------------------------------------------------------------
__global__ void ransac_finalize_kernel(const float2* __restrict__ src_xy, const float2* __restrict__ dst_xy, int n_pts,
                                       HypSource hs, const RansacHeader* __restrict__ hdr,
                                       float* __restrict__ best_H, long long* __restrict__ best_index,
                                       int* __restrict__ best_count, long long* __restrict__ n_evaluated)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    const unsigned long long key = hdr->best_key;
    const unsigned idx = 0xFFFFFFFFu - static_cast<unsigned>(key & 0xFFFFFFFFull);
    if (best_index) *best_index = static_cast<long long>(idx);
    if (best_count) *best_count = static_cast<int>(key >> 32);
    if (n_evaluated) *n_evaluated = static_cast<long long>(hdr->n_evaluated);
    if (best_H) {
        double s[8], d[8], H[9];
        gather_sets(src_xy, dst_xy, hypothesis_indices(hs, static_cast<long long>(idx), n_pts), s, d);
        aca_solve<double>(s, d, H);
        normalise<double>(H, 2);
#pragma unroll
        for (int k = 0; k < 9; ++k) best_H[k] = static_cast<float>(H[k]);
    }
}

static size_t align16(size_t v) { return (v + 15) & ~size_t(15); }
static size_t table_bytes(int32_t n_pts) { return size_t((n_pts + 1) / 2) * 32; }

// Launches with fewer hypothesis CTAs than half the machine also split the table over blockIdx.y.
constexpr int kSplitBelowCtas = 148;
constexpr int kMinPartEntries = 8;
constexpr int kFusedMaxPts = 4096;      // the one-kernel path packs the whole table in every CTA: tables that fit shared memory
constexpr int kTinyFillCtas = 128;       // tiny path: the table is split further while the call has fewer CTAs than this
constexpr int kTinyMaxGroups = 296;     // tiny path: at most two CTAs per SM's worth of 32-hypothesis groups ...
constexpr int kTinyMaxGroupsWide = 640; // ... and up to 20 480 hypotheses on tables of <= kTinyWidePts points, where it still beats the
constexpr int kTinyWidePts = 2048;      //     five launches of the generic path (16 384 x 2000: 30.6 vs 36.5 us; 37 888 x 2000: 56 vs 52)
constexpr size_t kTicketBytes = 128;    // so that the accumulator area of the smallest call still holds one TinySlot
// dynamic shared memory of the largest one-kernel call: the packed table of kFusedMaxPts points + the per-thread queues
constexpr size_t kTinyMaxSmem = size_t(kFusedMaxPts / 2) * kTinyEntry * sizeof(float4) + size_t(kQueueCap) * kTinyThreads * sizeof(unsigned);
static bool may_split(int64_t n_hyp) { return (n_hyp + kRBlock - 1) / kRBlock < kSplitBelowCtas; }

// Tiny path: CTAs (table parts) per group of 32 hypotheses -- a power of two <= 8 (the cluster size), doubled while the
// call does not yet cover the machine and every warp of the last part still gets table entries.
static int tiny_parts(int n_pairs, int64_t groups)
{
    int p = 1;
    while (p < kTinyMaxParts && groups * p < kTinyFillCtas && n_pairs > (2 * p - 1) * kTinyWarps * kGroup) p *= 2;
    return p;
}

// entries per part for a launch of n_hyp hypotheses (>= n_pairs: one part)
static int part_entries_for(int n_pairs, int64_t n_hyp, int ctas_per_sm = 2)
{
    const int64_t ctas = (n_hyp + kRBlock - 1) / kRBlock;
    if (ctas >= kSplitBelowCtas) return n_pairs;
    int64_t parts = (ctas_per_sm * kSplitBelowCtas) / ctas;                  // at most ctas_per_sm CTAs per SM: one wave, never a second,
    if (parts < 1) parts = 1;                                                // nearly empty one (16 384 hypotheses: 9 x 32 CTAs, not 10 x 32)
    const int64_t max_parts = n_pairs / kMinPartEntries > 0 ? n_pairs / kMinPartEntries : 1;
    if (parts > max_parts) parts = max_parts;
    if (parts <= 1) return n_pairs;
    int pe = static_cast<int>((n_pairs + parts - 1) / parts);
    pe = (pe + 7) & ~7;                                                     // whole groups of 8 entries
    return pe;
}

}  // namespace hg

extern "C" size_t hg_ransac_workspace_bytes(int32_t n_pts, int64_t n_hyp)
{
    if (n_pts < 0 || n_hyp < 0) return 0;
    // small batches accumulate partial counts (4 B per hypothesis) when the table is split over CTAs
    const size_t acc = hg::may_split(n_hyp) ? hg::align16(size_t(n_hyp) * sizeof(int)) + hg::kTicketBytes : 0;
    return hg::kHeaderBytes + hg::align16(hg::table_bytes(n_pts)) + acc;
}

namespace hg {

// The constant-bank copy of the table is the one piece of per-device state in the library.  Calls that use it are
// ordered against each other: a call makes its stream wait for the event the previous user recorded after its last
// scoring launch, then overwrites c_table.  Under stream capture no such cross-stream ordering can be recorded, so a
// call on a capturing stream never uses the constant bank (ransac_run takes the staged shared-memory operands
// instead): a captured call is self-contained and its replays may overlap any other RANSAC work.
class ConstTableGuard {
public:
    explicit ConstTableGuard(cudaStream_t st) : st_(st), lock_(mutex())
    {
        if (cudaGetDevice(&dev_) != cudaSuccess || dev_ < 0 || dev_ >= kMaxDevices) { status_ = HG_ERR_CUDA; return; }
        Slot& s = slots()[dev_];
        if (!s.ev && cudaEventCreateWithFlags(&s.ev, cudaEventDisableTiming) != cudaSuccess) { status_ = HG_ERR_CUDA; return; }
        if (s.used && cudaStreamWaitEvent(st, s.ev, 0) != cudaSuccess) status_ = HG_ERR_CUDA;
    }
    ~ConstTableGuard()
    {
        if (status_ != HG_OK) return;
        Slot& s = slots()[dev_];
        if (cudaEventRecord(s.ev, st_) == cudaSuccess) s.used = true;
    }
    int status() const { return status_; }

private:
    static constexpr int kMaxDevices = 64;
    struct Slot { cudaEvent_t ev = nullptr; bool used = false; };
    static std::mutex& mutex() { static std::mutex m; return m; }
    static Slot* slots() { static Slot s[kMaxDevices]; return s; }
    cudaStream_t st_;
    std::unique_lock<std::mutex> lock_;
    int dev_ = -1, status_ = HG_OK;
};

// Shared by the device entry points.  Sampling mode: hyp_idx == nullptr.  round_hyp == n_hyp and
// confidence <= 0 give the single-launch behaviour of hg_ransac_hypothesize_score.
static int ransac_run(const float* src_xy, const float* dst_xy, int32_t n_pts, const int32_t* hyp_idx, int32_t* hyp_idx_out,
                      unsigned long long seed, int64_t n_hyp, int64_t round_hyp, float threshold_px, double confidence,
                      bool adaptive, unsigned flags, double reject_lim2, int32_t* counts, float* best_H, int64_t* best_index, int32_t* best_count,
                      int64_t* n_evaluated, void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    unsigned char* ws = static_cast<unsigned char*>(workspace);
    RansacHeader* hdr = reinterpret_cast<RansacHeader*>(ws);
    // workspace layout: header | partial-count accumulator / tiny-call candidates (small calls only) | packed table
    const size_t acc_only = may_split(n_hyp) ? align16(size_t(n_hyp) * sizeof(int)) : 0;
    const size_t acc_bytes = acc_only ? acc_only + kTicketBytes : 0;
    float4* table = reinterpret_cast<float4*>(ws + kHeaderBytes + acc_bytes);
    const float2* s2 = reinterpret_cast<const float2*>(src_xy);
    const float2* d2 = reinterpret_cast<const float2*>(dst_xy);
    const int n_pairs = (n_pts + 1) / 2;
    const double t = static_cast<double>(threshold_px);
    const double inv_t = 1.0 / t;
    (void)workspace_bytes;

    const int64_t tiny_groups = (n_hyp + kTinyHyp - 1) / kTinyHyp;
    // (the adaptive entry point with a single round -- round_hyp >= max_hyp -- is the same call with on-device sampling)
    if ((!adaptive || round_hyp >= n_hyp) && acc_bytes && n_pts <= kFusedMaxPts && tiny_groups <= (n_pts <= kTinyWidePts ? kTinyMaxGroupsWide : kTinyMaxGroups) &&
        size_t(tiny_groups) * sizeof(TinySlot) <= acc_bytes) {
        // tiny call: a cluster of CTAs per 32 hypotheses, the table split over the cluster and over the warps of each
        // CTA; the accumulator area holds the candidates
        HypSource hs;
        hs.idx = reinterpret_cast<const int4*>(hyp_idx);
        hs.idx_out = reinterpret_cast<int4*>(hyp_idx_out);
        hs.seed = seed;
        hs.flags = flags;
        hs.reject_lim2 = reject_lim2;
        hs.check_stop = 0;
        hs.acc = nullptr;
        hs.h0 = 0; hs.h1 = n_hyp;
        const int parts = tiny_parts(n_pairs, tiny_groups);
        hs.part_entries = ((n_pairs + parts - 1) / parts + 7) & ~7;
        const size_t smem = size_t(n_pairs) * kTinyEntry * sizeof(float4) + size_t(kQueueCap) * kTinyThreads * sizeof(unsigned);
        // always the largest size the path can ask for: the attribute belongs to the function, not to the launch, so a per-call
        // value set by one host thread could be lowered by another between this call and the launch below
        if (cudaFuncSetAttribute(ransac_tiny_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, int(kTinyMaxSmem)) != cudaSuccess)
            return HG_ERR_CUDA;
        ransac_zero_kernel<<<1, 256, 0, st>>>(reinterpret_cast<uint4*>(hdr), int((kHeaderBytes + size_t(tiny_groups) * sizeof(TinySlot)) / 16));
        if (launch_status() != HG_OK) return HG_ERR_CUDA;
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(static_cast<unsigned>(tiny_groups), static_cast<unsigned>(parts), 1);
        cfg.blockDim = dim3(kTinyThreads, 1, 1);
        cfg.dynamicSmemBytes = smem;
        cfg.stream = st;
        cudaLaunchAttribute attrs[2];
        attrs[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;      // may start while the zero kernel runs
        attrs[0].val.programmaticStreamSerializationAllowed = 1;
        attrs[1].id = cudaLaunchAttributeClusterDimension;
        attrs[1].val.clusterDim.x = 1; attrs[1].val.clusterDim.y = static_cast<unsigned>(parts); attrs[1].val.clusterDim.z = 1;
        cfg.attrs = attrs;
        cfg.numAttrs = parts > 1 ? 2 : 1;
        TinySlot* cand = reinterpret_cast<TinySlot*>(ws + kHeaderBytes);
        if (cudaLaunchKernelEx(&cfg, ransac_tiny_kernel, s2, d2, n_pts, n_pairs, hs, inv_t, t, counts, hdr, cand, best_H,
                               reinterpret_cast<long long*>(best_index), best_count, reinterpret_cast<long long*>(n_evaluated)) != cudaSuccess) {
            (void)cudaGetLastError();
            return HG_ERR_CUDA;
        }
        return launch_status();
    }
    {   // header, accumulator: a kernel, not a memset (a memset node costs ~3 us inside a CUDA graph, this ~0.8 us)
        const int n16 = static_cast<int>((kHeaderBytes + acc_bytes) / 16);
        const int zb = n16 > 256 * 8 ? (n16 / (256 * 8) < 148 ? n16 / (256 * 8) : 148) : 1;
        ransac_zero_kernel<<<zb, 256, 0, st>>>(reinterpret_cast<uint4*>(hdr), n16);
        if (launch_status() != HG_OK) return HG_ERR_CUDA;
    }
    {
        int blocks = (n_pairs + 255) / 256;
        if (blocks > 1184) blocks = 1184;
        ransac_prep_kernel<<<blocks, 256, 0, st>>>(s2, d2, n_pts, n_pairs, inv_t, table, hdr);
        if (launch_status() != HG_OK) return HG_ERR_CUDA;
    }
    // Operand path: a table that fits the constant bank goes through the uniform datapath -- also when the launch is split
    // over table parts (mid-size calls: 7-10 % faster than the staged shared-memory sweep); the verification mode never
    // reads the table.
    // A call that is being captured into a CUDA graph stages its operands in shared memory: the constant bank is shared by
    // every stream of the device, and a replay cannot be ordered against the calls that will be running then.
    cudaStreamCaptureStatus capture = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(st, &capture) != cudaSuccess) { (void)cudaGetLastError(); return HG_ERR_CUDA; }
    const bool use_const = n_pairs <= kConstPairs && !(flags & HG_RANSAC_DECIDE_ALL_F64) && capture == cudaStreamCaptureStatusNone;
    const size_t stash = size_t(kQueueCap) * kRBlock * sizeof(unsigned) + kStages * sizeof(uint64_t);
    const size_t smem = (use_const ? 0 : size_t(kStages) * kChunkPairs * 32) + stash;
    auto* score = use_const ? ransac_score_kernel<true> : ransac_score_kernel<false>;
    // per call, not cached: the attribute belongs to the current device, and a process may drive several
    if (cudaFuncSetAttribute(score, cudaFuncAttributeMaxDynamicSharedMemorySize, int(smem)) != cudaSuccess) return HG_ERR_CUDA;
    std::unique_ptr<ConstTableGuard> guard;
    if (use_const) {
        guard.reset(new ConstTableGuard(st));
        if (guard->status() != HG_OK) return guard->status();
        if (cudaMemcpyToSymbolAsync(c_table, table, size_t(n_pairs) * 32, 0, cudaMemcpyDeviceToDevice, st) != cudaSuccess)
            return HG_ERR_CUDA;
    }
    HypSource hs;
    hs.idx = reinterpret_cast<const int4*>(hyp_idx);
    hs.idx_out = reinterpret_cast<int4*>(hyp_idx_out);
    hs.seed = seed;
    hs.flags = flags;
    hs.reject_lim2 = reject_lim2;
    hs.check_stop = adaptive ? 1 : 0;
    // split mode needs the accumulator, which the workspace holds only when the whole call is small (may_split(n_hyp))
    hs.acc = acc_bytes ? reinterpret_cast<int*>(ws + kHeaderBytes) : nullptr;
    for (int64_t h0 = 0; h0 < n_hyp; h0 += round_hyp) {
        const int64_t h1 = (h0 + round_hyp < n_hyp) ? h0 + round_hyp : n_hyp;
        hs.h0 = h0; hs.h1 = h1;
        hs.part_entries = hs.acc ? part_entries_for(n_pairs, h1 - h0) : n_pairs;
        const unsigned parts = static_cast<unsigned>((n_pairs + hs.part_entries - 1) / hs.part_entries);
        const dim3 grid(static_cast<unsigned>((h1 - h0 + kRBlock - 1) / kRBlock), parts);
        score<<<grid, kRBlock, smem, st>>>(s2, d2, n_pts, table, n_pairs, hs, inv_t, t, counts, hdr);
        if (launch_status() != HG_OK) return HG_ERR_CUDA;
        if (parts > 1) {
            const unsigned bb = static_cast<unsigned>((h1 - h0 + 255) / 256);
            ransac_best_kernel<<<bb, 256, 0, st>>>(hs.acc, hs.h0, hs.h1, counts, hdr, hs.check_stop);
            if (launch_status() != HG_OK) return HG_ERR_CUDA;
        }
        if (adaptive) {
            ransac_round_kernel<<<1, 32, 0, st>>>(hdr, n_pts, static_cast<long long>(h1), confidence, h1 == n_hyp ? 1 : 0);
            if (launch_status() != HG_OK) return HG_ERR_CUDA;
        }
    }
    guard.reset();                                         // records "table free" on the stream
    if (best_H || best_index || best_count || n_evaluated) {
        ransac_finalize_kernel<<<1, 32, 0, st>>>(s2, d2, n_pts, hs, hdr, best_H, reinterpret_cast<long long*>(best_index), best_count,
                                                 reinterpret_cast<long long*>(n_evaluated));
        if (launch_status() != HG_OK) return HG_ERR_CUDA;
    }
    return HG_OK;
}

static int check_options(const hg_ransac_options_t* o, unsigned* flags, double* reject_lim2)
{
    *flags = 0u;
    *reject_lim2 = 0.0;
    if (!o) return HG_OK;
    if (o->flags & ~(HG_RANSAC_REJECT_DEGENERATE | HG_RANSAC_DECIDE_ALL_F64)) return HG_ERR_INVALID_ARG;
    if (o->flags & HG_RANSAC_REJECT_DEGENERATE) {
        if (!(o->min_area_px2 >= 0.0f) || !(o->min_area_px2 < 3.0e38f)) return HG_ERR_INVALID_ARG;
        *reject_lim2 = 2.0 * static_cast<double>(o->min_area_px2);
    }
    *flags = o->flags;
    return HG_OK;
}

}  // namespace hg

extern "C" int hg_ransac_hypothesize_score_ex(const float* src_xy, const float* dst_xy, int32_t n_pts,
                                              const int32_t* hyp_idx, int64_t n_hyp, float threshold_px,
                                              const hg_ransac_options_t* options,
                                              int32_t* counts, float* best_H, int64_t* best_index,
                                              int32_t* best_count, void* workspace, size_t workspace_bytes,
                                              void* cuda_stream)
{
    using namespace hg;
    unsigned flags = 0u;
    double reject_lim2 = 0.0;
    if (n_hyp < 0 || n_hyp > 0x7fffffffLL) return HG_ERR_INVALID_ARG;
    if (n_pts < 4) return HG_ERR_INVALID_ARG;
    if (!(threshold_px > 0.0f) || !(threshold_px < 3.0e38f)) return HG_ERR_INVALID_ARG;
    if (check_options(options, &flags, &reject_lim2) != HG_OK) return HG_ERR_INVALID_ARG;
    if (n_hyp == 0) return HG_OK;
    if (!src_xy || !dst_xy || !hyp_idx || !workspace) return HG_ERR_INVALID_ARG;
    if (!aligned16(src_xy) || !aligned16(dst_xy) || !aligned16(hyp_idx) || !aligned16(workspace)) return HG_ERR_ALIGNMENT;
    if ((counts && !aligned4(counts)) || (best_H && !aligned4(best_H)) ||
        (best_index && (reinterpret_cast<uintptr_t>(best_index) & 7u)) || (best_count && !aligned4(best_count)))
        return HG_ERR_ALIGNMENT;
    if (workspace_bytes < hg_ransac_workspace_bytes(n_pts, n_hyp)) return HG_ERR_WORKSPACE;
    return ransac_run(src_xy, dst_xy, n_pts, hyp_idx, nullptr, 0ull, n_hyp, n_hyp, threshold_px, 0.0, false, flags, reject_lim2, counts, best_H,
                      best_index, best_count, nullptr, workspace, workspace_bytes, cuda_stream);
}

extern "C" int hg_ransac_hypothesize_score(const float* src_xy, const float* dst_xy, int32_t n_pts,
                                           const int32_t* hyp_idx, int64_t n_hyp, float threshold_px,
                                           int32_t* counts, float* best_H, int64_t* best_index,
                                           int32_t* best_count, void* workspace, size_t workspace_bytes,
                                           void* cuda_stream)
{
    return hg_ransac_hypothesize_score_ex(src_xy, dst_xy, n_pts, hyp_idx, n_hyp, threshold_px, nullptr, counts, best_H, best_index,
                                          best_count, workspace, workspace_bytes, cuda_stream);
}

extern "C" int hg_ransac_adaptive_ex(const float* src_xy, const float* dst_xy, int32_t n_pts, uint64_t seed, int64_t max_hyp,
                                     int64_t round_hyp, float threshold_px, float confidence,
                                     const hg_ransac_options_t* options, int32_t* counts,
                                     int32_t* hyp_idx_out, float* best_H, int64_t* best_index, int32_t* best_count,
                                     int64_t* n_evaluated, void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    using namespace hg;
    unsigned flags = 0u;
    double reject_lim2 = 0.0;
    if (max_hyp < 0 || max_hyp > 0x7fffffffLL || round_hyp < 1) return HG_ERR_INVALID_ARG;
    if (n_pts < 4) return HG_ERR_INVALID_ARG;
    if (!(threshold_px > 0.0f) || !(threshold_px < 3.0e38f)) return HG_ERR_INVALID_ARG;
    if (!(confidence < 1.0f) || !(confidence == confidence)) return HG_ERR_INVALID_ARG;
    if (check_options(options, &flags, &reject_lim2) != HG_OK) return HG_ERR_INVALID_ARG;
    if (max_hyp == 0) return HG_OK;
    if ((max_hyp + round_hyp - 1) / round_hyp > 65536) return HG_ERR_INVALID_ARG;          // launches per call
    if (!src_xy || !dst_xy || !workspace) return HG_ERR_INVALID_ARG;
    if (!aligned16(src_xy) || !aligned16(dst_xy) || !aligned16(workspace) || (hyp_idx_out && !aligned16(hyp_idx_out)))
        return HG_ERR_ALIGNMENT;
    if ((counts && !aligned4(counts)) || (best_H && !aligned4(best_H)) || (best_count && !aligned4(best_count)) ||
        (best_index && (reinterpret_cast<uintptr_t>(best_index) & 7u)) || (n_evaluated && (reinterpret_cast<uintptr_t>(n_evaluated) & 7u)))
        return HG_ERR_ALIGNMENT;
    if (workspace_bytes < hg_ransac_workspace_bytes(n_pts, max_hyp)) return HG_ERR_WORKSPACE;
    return ransac_run(src_xy, dst_xy, n_pts, nullptr, hyp_idx_out, seed, max_hyp, round_hyp, threshold_px,
                      static_cast<double>(confidence), true, flags, reject_lim2, counts, best_H, best_index, best_count, n_evaluated, workspace,
                      workspace_bytes, cuda_stream);
}

extern "C" int hg_ransac_adaptive(const float* src_xy, const float* dst_xy, int32_t n_pts, uint64_t seed, int64_t max_hyp,
                                  int64_t round_hyp, float threshold_px, float confidence, int32_t* counts,
                                  int32_t* hyp_idx_out, float* best_H, int64_t* best_index, int32_t* best_count,
                                  int64_t* n_evaluated, void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    return hg_ransac_adaptive_ex(src_xy, dst_xy, n_pts, seed, max_hyp, round_hyp, threshold_px, confidence, nullptr, counts,
                                 hyp_idx_out, best_H, best_index, best_count, n_evaluated, workspace, workspace_bytes, cuda_stream);
}

extern "C" int hg_ransac_hypothesize_score_host(const float* src_xy, const float* dst_xy, int32_t n_pts,
                                                const int32_t* hyp_idx, int64_t n_hyp, float threshold_px,
                                                int32_t* counts, float* best_H, int64_t* best_index,
                                                int32_t* best_count)
{
    using namespace hg;
    if (n_hyp < 0 || n_hyp > 0x7fffffffLL || n_pts < 4) return HG_ERR_INVALID_ARG;
    if (n_hyp == 0) return HG_OK;
    if (!src_xy || !dst_xy || !hyp_idx) return HG_ERR_INVALID_ARG;
    const size_t pts_b = size_t(n_pts) * 2 * sizeof(float);
    const size_t idx_b = size_t(n_hyp) * 4 * sizeof(int32_t);
    const size_t cnt_b = size_t(n_hyp) * sizeof(int32_t);
    const size_t ws_b = hg_ransac_workspace_bytes(n_pts, n_hyp);
    // one allocation: src | dst | idx | counts | best (64 B) | workspace, every part 256-byte aligned
    auto up = [](size_t v) { return (v + 255) & ~size_t(255); };
    const size_t o_src = 0, o_dst = o_src + up(pts_b), o_idx = o_dst + up(pts_b), o_cnt = o_idx + up(idx_b),
                 o_best = o_cnt + up(cnt_b), o_ws = o_best + 256, total = o_ws + up(ws_b);
    unsigned char* dev = nullptr;
    cudaStream_t st = nullptr;
    int rc = cuda_status(cudaMalloc(reinterpret_cast<void**>(&dev), total));
    if (rc == HG_OK) rc = cuda_status(cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking));
    if (rc == HG_OK) rc = cuda_status(cudaMemcpyAsync(dev + o_src, src_xy, pts_b, cudaMemcpyHostToDevice, st));
    if (rc == HG_OK) rc = cuda_status(cudaMemcpyAsync(dev + o_dst, dst_xy, pts_b, cudaMemcpyHostToDevice, st));
    if (rc == HG_OK) rc = cuda_status(cudaMemcpyAsync(dev + o_idx, hyp_idx, idx_b, cudaMemcpyHostToDevice, st));
    if (rc == HG_OK)
        rc = hg_ransac_hypothesize_score(reinterpret_cast<float*>(dev + o_src), reinterpret_cast<float*>(dev + o_dst), n_pts,
                                         reinterpret_cast<int32_t*>(dev + o_idx), n_hyp, threshold_px,
                                         reinterpret_cast<int32_t*>(dev + o_cnt), reinterpret_cast<float*>(dev + o_best),
                                         reinterpret_cast<int64_t*>(dev + o_best + 64),
                                         reinterpret_cast<int32_t*>(dev + o_best + 128), dev + o_ws, up(ws_b), st);
    if (rc == HG_OK && counts) rc = cuda_status(cudaMemcpyAsync(counts, dev + o_cnt, cnt_b, cudaMemcpyDeviceToHost, st));
    if (rc == HG_OK && best_H) rc = cuda_status(cudaMemcpyAsync(best_H, dev + o_best, 9 * sizeof(float), cudaMemcpyDeviceToHost, st));
    if (rc == HG_OK && best_index) rc = cuda_status(cudaMemcpyAsync(best_index, dev + o_best + 64, sizeof(int64_t), cudaMemcpyDeviceToHost, st));
    if (rc == HG_OK && best_count) rc = cuda_status(cudaMemcpyAsync(best_count, dev + o_best + 128, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    if (st) {
        const int r2 = cuda_status(cudaStreamSynchronize(st));
        if (rc == HG_OK) rc = r2;
        cudaStreamDestroy(st);
    }
    if (dev) cudaFree(dev);
    return rc;
}

// ---- the entry point that allocates nothing (include/hg.h: hg_ransac_hypothesize_score_noalloc) ----------------------
// For callers that cannot give the library a workspace because they cannot allocate one (see the header for who they
// are).  The one-kernel small-call path needs little scratch -- the header and one TinySlot per 32 hypotheses -- so
// that scratch is a fixed array in the library image.  The launch below repeats the tiny-call branch of ransac_run on
// purpose: the existing entry points are left exactly as they are.
namespace hg {

constexpr size_t kNoAllocScratchBytes = (kHeaderBytes + size_t(kTinyMaxGroups) * sizeof(TinySlot) + 255) & ~size_t(255);
static_assert(kNoAllocScratchBytes == HG_RANSAC_NOALLOC_SCRATCH_BYTES, "hg.h states the size of the array");
static_assert(HG_RANSAC_NOALLOC_MAX_HYP == kTinyMaxGroups * kTinyHyp, "hg.h states the hypothesis limit");
static_assert(HG_RANSAC_NOALLOC_MAX_PTS == kFusedMaxPts, "hg.h states the table limit");

// Device memory that exists on every GPU that loads this module, from load to process exit.  In HOST code this name is
// only a handle for the runtime's symbol calls -- it is not the device address and must never be passed to a kernel.
static __device__ __align__(256) unsigned char g_noalloc_scratch[kNoAllocScratchBytes];

// The device address of g_noalloc_scratch on the CURRENT device: asked from the runtime once per device (the array has a
// different address on each), under a lock, and cached.  No allocation: the array is part of the loaded module.
static int noalloc_scratch_address(unsigned char** out)
{
    constexpr int kMaxDevices = 64;
    static std::mutex m;
    static unsigned char* addr[kMaxDevices] = {};
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) { (void)cudaGetLastError(); return HG_ERR_CUDA; }
    std::lock_guard<std::mutex> lock(m);
    if (!addr[dev]) {
        void* p = nullptr;
        if (cudaGetSymbolAddress(&p, g_noalloc_scratch) != cudaSuccess || !p) { (void)cudaGetLastError(); return HG_ERR_CUDA; }
        if (!aligned16(p)) return HG_ERR_ALIGNMENT;           // cannot happen (__align__(256)); a wrong address must not get through
        addr[dev] = static_cast<unsigned char*>(p);
    }
    *out = addr[dev];
    return HG_OK;
}

}  // namespace hg

extern "C" int hg_ransac_hypothesize_score_noalloc(const float* src_xy, const float* dst_xy, int32_t n_pts,
                                                   const int32_t* hyp_idx, int64_t n_hyp, float threshold_px,
                                                   int32_t* counts, float* best_H, int64_t* best_index,
                                                   int32_t* best_count, void* cuda_stream)
{
    using namespace hg;
    if (n_hyp < 0 || n_pts < 4) return HG_ERR_INVALID_ARG;
    if (!(threshold_px > 0.0f) || !(threshold_px < 3.0e38f)) return HG_ERR_INVALID_ARG;
    if (n_hyp == 0) return HG_OK;
    if (!src_xy || !dst_xy || !hyp_idx) return HG_ERR_INVALID_ARG;
    if (!aligned16(src_xy) || !aligned16(dst_xy) || !aligned16(hyp_idx)) return HG_ERR_ALIGNMENT;
    if ((counts && !aligned4(counts)) || (best_H && !aligned4(best_H)) ||
        (best_index && (reinterpret_cast<uintptr_t>(best_index) & 7u)) || (best_count && !aligned4(best_count)))
        return HG_ERR_ALIGNMENT;
    // the fixed array holds the scratch of at most this much; nothing has been enqueued yet
    if (n_pts > HG_RANSAC_NOALLOC_MAX_PTS || n_hyp > HG_RANSAC_NOALLOC_MAX_HYP) return HG_ERR_TOO_LARGE;

    unsigned char* ws = nullptr;                               // device address of the array on the current device
    const int rc = noalloc_scratch_address(&ws);
    if (rc != HG_OK) return rc;

    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    RansacHeader* hdr = reinterpret_cast<RansacHeader*>(ws);
    TinySlot* cand = reinterpret_cast<TinySlot*>(ws + kHeaderBytes);
    const float2* s2 = reinterpret_cast<const float2*>(src_xy);
    const float2* d2 = reinterpret_cast<const float2*>(dst_xy);
    const int n_pairs = (n_pts + 1) / 2;
    const double t = static_cast<double>(threshold_px);
    const double inv_t = 1.0 / t;
    const int64_t groups = (n_hyp + kTinyHyp - 1) / kTinyHyp;
    if (kHeaderBytes + size_t(groups) * sizeof(TinySlot) > kNoAllocScratchBytes) return HG_ERR_TOO_LARGE;

    HypSource hs;
    hs.idx = reinterpret_cast<const int4*>(hyp_idx);
    hs.idx_out = nullptr;
    hs.seed = 0ull;
    hs.flags = 0u;
    hs.reject_lim2 = 0.0;
    hs.check_stop = 0;
    hs.acc = nullptr;
    hs.h0 = 0; hs.h1 = n_hyp;
    const int parts = tiny_parts(n_pairs, groups);
    hs.part_entries = ((n_pairs + parts - 1) / parts + 7) & ~7;
    const size_t smem = size_t(n_pairs) * kTinyEntry * sizeof(float4) + size_t(kQueueCap) * kTinyThreads * sizeof(unsigned);
    if (cudaFuncSetAttribute(ransac_tiny_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, int(kTinyMaxSmem)) != cudaSuccess) {
        (void)cudaGetLastError();
        return HG_ERR_CUDA;
    }
    // the array keeps the previous call's header, ticket and stamped slots: what this call reads starts at zero
    ransac_zero_kernel<<<1, 256, 0, st>>>(reinterpret_cast<uint4*>(hdr), int((kHeaderBytes + size_t(groups) * sizeof(TinySlot)) / 16));
    if (launch_status() != HG_OK) return HG_ERR_CUDA;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(static_cast<unsigned>(groups), static_cast<unsigned>(parts), 1);
    cfg.blockDim = dim3(kTinyThreads, 1, 1);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attrs[2];
    attrs[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attrs[0].val.programmaticStreamSerializationAllowed = 1;
    attrs[1].id = cudaLaunchAttributeClusterDimension;
    attrs[1].val.clusterDim.x = 1; attrs[1].val.clusterDim.y = static_cast<unsigned>(parts); attrs[1].val.clusterDim.z = 1;
    cfg.attrs = attrs;
    cfg.numAttrs = parts > 1 ? 2 : 1;
    if (cudaLaunchKernelEx(&cfg, ransac_tiny_kernel, s2, d2, n_pts, n_pairs, hs, inv_t, t, counts, hdr, cand, best_H,
                           reinterpret_cast<long long*>(best_index), best_count, static_cast<long long*>(nullptr)) != cudaSuccess) {
        (void)cudaGetLastError();
        return HG_ERR_CUDA;
    }
    return launch_status();
}
