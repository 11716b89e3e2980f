// ORACLE -- TEST INFRASTRUCTURE ONLY.
//
// Plain, slow, obviously-correct CPU evaluation (fp64 unless the scalar type T
// says otherwise) of what the hot path of arXiv 2402.18008 computes: one 3x3
// homography H (up to scale) from four point correspondences.  Written from
// /root/reference/PAPER.md ("P:<line>") in the paper's order and notation.
// Nothing here is blocked, fused or reordered beyond what the paper states.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
// --impl reference legs may build, load or call anything under oracle/.
// The CUDA path (paper_2402_18008_b200/) shares no code with this directory.
//
// Parity pins: every function below is pinned by tests/test_oracle_*.py
// (defining property, cross-method equality, closed forms, exact integer
// brute force, op counts, homogeneity degrees).  Nothing is "parity unpinned".
//
// Point roles (reading R11 of DESIGN.md): the four correspondences
// of a set are M, N, P, Q = points 0, 1, 2, 3.  s[] / d[] hold
// x0,y0,x1,y1,x2,y2,x3,y3 of the source (plane 1) / target (plane 2).
// H[] is row-major h11,h12,h13,h21,...,h33.
#pragma once
#include <cmath>
#include <cstdint>

namespace hgo {

// ---------------------------------------------------------------------------
// ACA: H = H_A2^-1 * H_C * H_A1  (Eq. 27).  85 FLOPs, no division
// (Table 4).  Returns the paper's raw scale (Eq. 31-32 convention).
// If `core` is non-null it receives c11, c22, c33 (Eq. 32).
// ---------------------------------------------------------------------------
template <class T>
void aca(const T s[8], const T d[8], T H[9], T* core = nullptr)
{
    const T M1x = s[0], M1y = s[1], N1x = s[2], N1y = s[3];
    const T P1x = s[4], P1y = s[5], Q1x = s[6], Q1y = s[7];
    const T M2x = d[0], M2y = d[1], N2x = d[2], N2y = d[3];
    const T P2x = d[4], P2y = d[5], Q2x = d[6], Q2y = d[7];

    // H_A1: Eq. 23-24.  7 FLOPs.
    const T MN1x = N1x - M1x, MN1y = N1y - M1y;
    const T MP1x = P1x - M1x, MP1y = P1y - M1y;
    const T fA1 = MN1x * MP1y - MN1y * MP1x;
    // H_A2 likewise.  7 FLOPs.
    const T MN2x = N2x - M2x, MN2y = N2y - M2y;
    const T MP2x = P2x - M2x, MP2y = P2y - M2y;
    const T fA2 = MN2x * MP2y - MN2y * MP2x;

    // Fourth correspondence relative to M (Table 4 columns 7-8, reading R7).  2+2 FLOPs.
    const T MQ1x = Q1x - M1x, MQ1y = Q1y - M1y;
    const T MQ2x = Q2x - M2x, MQ2y = Q2y - M2y;

    // Q3 = H_A1*Q1, Q4 = H_A2*Q2, both up to the scales fA1, fA2: Eq. 28.  6+6 FLOPs.
    const T Q3x = MQ1x * MP1y - MQ1y * MP1x;
    const T Q3y = MN1x * MQ1y - MN1y * MQ1x;
    const T Q4x = MQ2x * MP2y - MQ2y * MP2x;
    const T Q4y = MN2x * MQ2y - MN2y * MQ2x;

    // Eq. 30.  2+2 FLOPs.
    const T t1 = fA1 - Q3x - Q3y;
    const T t2 = fA2 - Q4x - Q4y;

    // H_C up to scale: Eq. 31-32.  8 FLOPs (6 products, 2 differences).
    const T c11 = t1 * Q3y * Q4x;
    const T c22 = t1 * Q3x * Q4y;
    const T c33 = t2 * Q3x * Q3y;
    const T c31 = c11 - c33;
    const T c32 = c22 - c33;
    if (core) { core[0] = c11; core[1] = c22; core[2] = c33; }

    // G = H_A2^-1 * H_C, with H_A2^-1 = [MN2 MP2 M2; 0 0 1] (Eq. 25, missing in the
    // extraction; reading R1): G = [c11*n2 - c33*m2, c22*p2 - c33*m2, c33*m2].  10 FLOPs.
    const T g13 = c33 * M2x;
    const T g23 = c33 * M2y;
    const T g11 = c11 * N2x - g13;
    const T g21 = c11 * N2y - g23;
    const T g12 = c22 * P2x - g13;
    const T g22 = c22 * P2y - g23;
    const T g31 = c31, g32 = c32, g33 = c33;

    // H = G * H_A1, H_A1 = [MP1y -MP1x 0; -MN1y MN1x 0; 0 0 fA1] * T(-M1) (Eq. 23, R2).  33 FLOPs.
    const T h11 = g11 * MP1y - g12 * MN1y;
    const T h21 = g21 * MP1y - g22 * MN1y;
    const T h31 = g31 * MP1y - g32 * MN1y;
    const T h12 = g12 * MN1x - g11 * MP1x;
    const T h22 = g22 * MN1x - g21 * MP1x;
    const T h32 = g32 * MN1x - g31 * MP1x;
    const T h13 = g13 * fA1 - h11 * M1x - h12 * M1y;
    const T h23 = g23 * fA1 - h21 * M1x - h22 * M1y;
    const T h33 = g33 * fA1 - h31 * M1x - h32 * M1y;

    H[0] = h11; H[1] = h12; H[2] = h13;
    H[3] = h21; H[4] = h22; H[5] = h23;
    H[6] = h31; H[7] = h32; H[8] = h33;
}

// ---------------------------------------------------------------------------
// SKS: H = H_S2^-1 * H_K * H_S1, H_K = H_E^-1 * H_S' * H_E  (Eq. 16).
// Anchors M, N -> (-1,0), (+1,0).  Five reciprocals.
// If `kern` is non-null it receives a_K, b_K, u_K, v_K (Eq. 15).
// ---------------------------------------------------------------------------
template <class T>
void sks(const T s[8], const T d[8], T H[9], T* kern = nullptr)
{
    const T half = T(0.5), one = T(1.0);
    const T M1x = s[0], M1y = s[1], N1x = s[2], N1y = s[3];
    const T P1x = s[4], P1y = s[5], Q1x = s[6], Q1y = s[7];
    const T M2x = d[0], M2y = d[1], N2x = d[2], N2y = d[3];
    const T P2x = d[4], P2y = d[5], Q2x = d[6], Q2y = d[7];

    // H_S1: Eq. 6, 7, 9.  6 + 3 FLOPs.
    const T O1x = half * (M1x + N1x), O1y = half * (M1y + N1y);
    const T v1x = N1x - O1x, v1y = N1y - O1y;
    const T fS1 = v1x * v1x + v1y * v1y;
    // H_S2 likewise.  6 + 3 FLOPs.
    const T O2x = half * (M2x + N2x), O2y = half * (M2y + N2y);
    const T v2x = N2x - O2x, v2y = N2y - O2y;
    const T fS2 = v2x * v2x + v2y * v2y;

    // P3 = H_S1*P1, Q3 = H_S1*Q1 (weight fS1); P4, Q4 under H_S2 (weight fS2):
    // Eq. 8 (layout per R2).  8 FLOPs each.
    const T eP1x = P1x - O1x, eP1y = P1y - O1y;
    const T P3x = v1x * eP1x + v1y * eP1y;
    const T P3y = v1x * eP1y - v1y * eP1x;
    const T eQ1x = Q1x - O1x, eQ1y = Q1y - O1y;
    const T Q3x = v1x * eQ1x + v1y * eQ1y;
    const T Q3y = v1x * eQ1y - v1y * eQ1x;
    const T eP2x = P2x - O2x, eP2y = P2y - O2y;
    const T P4x = v2x * eP2x + v2y * eP2y;
    const T P4y = v2x * eP2y - v2y * eP2x;
    const T eQ2x = Q2x - O2x, eQ2y = Q2y - O2y;
    const T Q4x = v2x * eQ2x + v2y * eQ2y;
    const T Q4y = v2x * eQ2y - v2y * eQ2x;

    // H_E swaps the 2nd and 3rd homogeneous coordinates (Eq. 12), then
    // dehomogenise: X5 = (X3.x / X3.y, f_S / X3.y).  One reciprocal + 2 products each.
    const T rP3 = one / P3y;
    const T P5x = P3x * rP3, P5y = fS1 * rP3;
    const T rQ3 = one / Q3y;
    const T Q5x = Q3x * rQ3, Q5y = fS1 * rQ3;
    const T rP4 = one / P4y;
    const T P6x = P4x * rP4, P6y = fS2 * rP4;
    const T rQ4 = one / Q4y;
    const T Q6x = Q4x * rQ4, Q6y = fS2 * rQ4;

    // Q7 = H_T1*H_E*Q3 = Q5 - P5 ; Q8 = H_T2*H_E*Q4 = Q6 - P6  (Eq. 13; R3, R4).
    const T Q7x = Q5x - P5x, Q7y = Q5y - P5y;
    const T Q8x = Q6x - P6x, Q8y = Q6y - P6y;

    // H_G: solve Eq. 14 for a_G, b_G.  Fifth reciprocal.
    const T rden = one / (Q7x * Q7x - Q7y * Q7y);
    const T aK = (Q8x * Q7x - Q8y * Q7y) * rden;
    const T bK = (Q8y * Q7x - Q8x * Q7y) * rden;

    // Eq. 15.  8 FLOPs.
    const T uK = P6x - aK * P5x - bK * P5y;
    const T vK = P6y - bK * P5x - aK * P5y;
    if (kern) { kern[0] = aK; kern[1] = bK; kern[2] = uK; kern[3] = vK; }

    // J = H_S2^-1 * H_K, H_S2^-1 per Eq. 10, H_K per Eq. 11.  20 FLOPs.
    const T j11 = v2x * aK + O2x * bK;
    const T j12 = v2x * uK - v2y + O2x * vK;
    const T j13 = v2x * bK + O2x * aK;
    const T j21 = v2y * aK + O2y * bK;
    const T j22 = v2y * uK + v2x + O2y * vK;
    const T j23 = v2y * bK + O2y * aK;
    const T j31 = bK, j32 = vK, j33 = aK;

    // H = J * H_S1, H_S1 = [v1x v1y s13; -v1y v1x s23; 0 0 fS1] (Eq. 8, R2).  6 + 33 = 39 FLOPs.
    const T s13 = -(v1x * O1x + v1y * O1y);
    const T s23 = v1y * O1x - v1x * O1y;
    H[0] = j11 * v1x - j12 * v1y;
    H[1] = j11 * v1y + j12 * v1x;
    H[2] = j11 * s13 + j12 * s23 + j13 * fS1;
    H[3] = j21 * v1x - j22 * v1y;
    H[4] = j21 * v1y + j22 * v1x;
    H[5] = j21 * s13 + j22 * s23 + j23 * fS1;
    H[6] = j31 * v1x - j32 * v1y;
    H[7] = j31 * v1y + j32 * v1x;
    H[8] = j31 * s13 + j32 * s23 + j33 * fS1;
}

// ---------------------------------------------------------------------------
// Simplified SK (object plane -> image, Eq. 17; Table 3 row "SK"):
//   Hbar = H * H_S1^-1 = H_S2^-1 * H_K.
// The object coordinates are expressed in the frame of the two anchors (M -> (-1,0), N -> (+1,0),
// so H_S1 = I and f_S1 = 1); everything that depends only on the known pattern -- P5, Q7 and the
// reciprocal of Eq. 14's determinant -- is computed once by sk_pattern() (zero per-image cost in
// Table 3), the per-image work is the target-side half of sks().  Hbar maps (-1,0), (1,0), P3, Q3
// to M2, N2, P2, Q2.
// ---------------------------------------------------------------------------
template <class T>
void sk_pattern(T P3x, T P3y, T Q3x, T Q3y, T pat[5])
{
    const T one = T(1.0);
    const T rP3 = one / P3y, rQ3 = one / Q3y;                  // Eq. 12 with f_S1 = 1
    const T P5x = P3x * rP3, P5y = rP3;
    const T Q5x = Q3x * rQ3, Q5y = rQ3;
    const T Q7x = Q5x - P5x, Q7y = Q5y - P5y;                  // Eq. 13 (R3, R4)
    pat[0] = P5x; pat[1] = P5y; pat[2] = Q7x; pat[3] = Q7y;
    pat[4] = one / (Q7x * Q7x - Q7y * Q7y);                    // determinant of Eq. 14
}

template <class T>
void sk(const T pat[5], const T d[8], T H[9])
{
    const T half = T(0.5), one = T(1.0);
    const T P5x = pat[0], P5y = pat[1], Q7x = pat[2], Q7y = pat[3], rden = pat[4];
    const T M2x = d[0], M2y = d[1], N2x = d[2], N2y = d[3];
    const T P2x = d[4], P2y = d[5], Q2x = d[6], Q2y = d[7];
    // H_S2: Eq. 6, 7, 9.  6 + 3 FLOPs.
    const T O2x = half * (M2x + N2x), O2y = half * (M2y + N2y);
    const T v2x = N2x - O2x, v2y = N2y - O2y;
    const T fS2 = v2x * v2x + v2y * v2y;
    // P4, Q4 (Eq. 8), then H_E and dehomogenisation (Eq. 12): P6, Q6.
    const T eP2x = P2x - O2x, eP2y = P2y - O2y;
    const T P4x = v2x * eP2x + v2y * eP2y;
    const T P4y = v2x * eP2y - v2y * eP2x;
    const T eQ2x = Q2x - O2x, eQ2y = Q2y - O2y;
    const T Q4x = v2x * eQ2x + v2y * eQ2y;
    const T Q4y = v2x * eQ2y - v2y * eQ2x;
    const T rP4 = one / P4y;
    const T P6x = P4x * rP4, P6y = fS2 * rP4;
    const T rQ4 = one / Q4y;
    const T Q6x = Q4x * rQ4, Q6y = fS2 * rQ4;
    const T Q8x = Q6x - P6x, Q8y = Q6y - P6y;
    // Eq. 14 with the pattern's determinant precomputed; Eq. 15.
    const T aK = (Q8x * Q7x - Q8y * Q7y) * rden;
    const T bK = (Q8y * Q7x - Q8x * Q7y) * rden;
    const T uK = P6x - aK * P5x - bK * P5y;
    const T vK = P6y - bK * P5x - aK * P5y;
    // Hbar = H_S2^-1 * H_K (Eq. 17; Eq. 10, 11).  20 FLOPs.
    H[0] = v2x * aK + O2x * bK;
    H[1] = v2x * uK - v2y + O2x * vK;
    H[2] = v2x * bK + O2x * aK;
    H[3] = v2y * aK + O2y * bK;
    H[4] = v2y * uK + v2x + O2y * vK;
    H[5] = v2y * bK + O2y * aK;
    H[6] = bK; H[7] = vK; H[8] = aK;
}

// ---------------------------------------------------------------------------
// Affine transformation from three correspondences (Sec. 5.2, Eq. 41 first row):
//   H_A = H_A2^-1 * H_A1   (the core transformation is the identity), 33 FLOPs.
// s[], d[] hold x,y of M, N, P.  H_A1 per Eq. 23 (R2), H_A2^-1 per Eq. 25 (R1).
// ---------------------------------------------------------------------------
template <class T>
void affine(const T s[6], const T d[6], T H[9])
{
    const T a1x = s[2] - s[0], a1y = s[3] - s[1];      // M1N1
    const T b1x = s[4] - s[0], b1y = s[5] - s[1];      // M1P1
    const T fA1 = a1x * b1y - a1y * b1x;
    const T a2x = d[2] - d[0], a2y = d[3] - d[1];      // M2N2
    const T b2x = d[4] - d[0], b2y = d[5] - d[1];      // M2P2
    // [M2N2 M2P2] * [b1y -b1x; -a1y a1x]
    const T h11 = a2x * b1y - b2x * a1y;
    const T h12 = b2x * a1x - a2x * b1x;
    const T h21 = a2y * b1y - b2y * a1y;
    const T h22 = b2y * a1x - a2y * b1x;
    // third column: f_A1 * M2 - L * M1
    H[0] = h11; H[1] = h12; H[2] = fA1 * d[0] - h11 * s[0] - h12 * s[1];
    H[3] = h21; H[4] = h22; H[5] = fA1 * d[1] - h21 * s[0] - h22 * s[1];
    H[6] = T(0.0); H[7] = T(0.0); H[8] = fA1;
}

// ---------------------------------------------------------------------------
// TensorACA for a rectangle: Algorithm 1, Eq. 42-45.
// Roles (reading R6): M1 = upper-left vertex, N1, Q1, P1 follow
// clockwise, i.e. M = TL, N = TR, Q = BR, P = BL; r_rec = w_rec / h_rec.
// m2, n2, p2, q2 are the projected corners in the target image.
// ---------------------------------------------------------------------------
template <class T>
void aca_rect(T M1x, T M1y, T w_rec, T r_rec,
              const T m2[2], const T n2[2], const T p2[2], const T q2[2], T H[9])
{
    // 1. difference vectors
    const T d1[3] = { n2[0] - m2[0], p2[0] - m2[0], q2[0] - m2[0] };
    const T d2[3] = { n2[1] - m2[1], p2[1] - m2[1], q2[1] - m2[1] };
    // 2. c = Cross(d1, d2).  (The standard cross product is the negative of the comment
    //    "[Q4.x; Q4.y; -fA2]" printed at P:581; every later step is linear in c, so only
    //    the global sign of H changes -- R6.)
    const T c[3] = { d1[1] * d2[2] - d1[2] * d2[1],
                     d1[2] * d2[0] - d1[0] * d2[2],
                     d1[0] * d2[1] - d1[1] * d2[0] };
    // 3. b = Sum(c) .* m2   (homogeneous m2 = [M2.x; M2.y; 1])
    const T sum = c[0] + c[1] + c[2];
    const T b[3] = { sum * m2[0], sum * m2[1], sum };
    // 4. first two columns
    const T h1[3] = { c[0] * n2[0] - b[0], c[0] * n2[1] - b[1], c[0] - b[2] };
    const T h2[3] = { r_rec * (c[1] * p2[0] - b[0]), r_rec * (c[1] * p2[1] - b[1]),
                      r_rec * (c[1] - b[2]) };
    // 5. last column
    const T h3[3] = { w_rec * b[0] - M1x * h1[0] - M1y * h2[0],
                      w_rec * b[1] - M1x * h1[1] - M1y * h2[1],
                      w_rec * b[2] - M1x * h1[2] - M1y * h2[2] };
    H[0] = h1[0]; H[1] = h2[0]; H[2] = h3[0];
    H[3] = h1[1]; H[4] = h2[1]; H[5] = h3[1];
    H[6] = h1[2]; H[7] = h2[2]; H[8] = h3[2];
}

// ---------------------------------------------------------------------------
// Polynomial closed form of H (Sec. 4.5, Eq. 33-35; the printed Eq. 33 is
// garbled -- reading R5):
//   H = c11 * n2 (p1 x m1)^T + c22 * p2 (m1 x n1)^T + c33 * m2 (n1 x p1)^T
// with homogeneous 3-vectors m1 = [M1.x, M1.y, 1] etc. and
//   c11 = |n1 p1 q1| |m1 n1 q1| |m2 q2 p2|,  c22 = |n1 p1 q1| |m1 q1 p1| |m2 n2 q2|,
//   c33 = |n2 p2 q2| |m1 q1 p1| |m1 n1 q1|.
// Evaluated with textbook 3x3 determinants and cross products (no step of aca()).
// ---------------------------------------------------------------------------
template <class T>
static T det3(const T a[3], const T b[3], const T c[3])
{
    return a[0] * (b[1] * c[2] - b[2] * c[1])
         - b[0] * (a[1] * c[2] - a[2] * c[1])
         + c[0] * (a[1] * b[2] - a[2] * b[1]);
}
template <class T>
static void cross3(const T a[3], const T b[3], T r[3])
{
    r[0] = a[1] * b[2] - a[2] * b[1];
    r[1] = a[2] * b[0] - a[0] * b[2];
    r[2] = a[0] * b[1] - a[1] * b[0];
}
template <class T>
void closed_form(const T s[8], const T d[8], T H[9])
{
    const T one = T(1.0);
    const T m1[3] = { s[0], s[1], one }, n1[3] = { s[2], s[3], one };
    const T p1[3] = { s[4], s[5], one }, q1[3] = { s[6], s[7], one };
    const T m2[3] = { d[0], d[1], one }, n2[3] = { d[2], d[3], one };
    const T p2[3] = { d[4], d[5], one }, q2[3] = { d[6], d[7], one };
    const T c11 = det3(n1, p1, q1) * det3(m1, n1, q1) * det3(m2, q2, p2);
    const T c22 = det3(n1, p1, q1) * det3(m1, q1, p1) * det3(m2, n2, q2);
    const T c33 = det3(n2, p2, q2) * det3(m1, q1, p1) * det3(m1, n1, q1);
    T r1[3], r2[3], r3[3];
    cross3(p1, m1, r1);
    cross3(m1, n1, r2);
    cross3(n1, p1, r3);
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j)
            H[3 * i + j] = c11 * n2[i] * r1[j] + c22 * p2[i] * r2[j] + c33 * m2[i] * r3[j];
}

// ---------------------------------------------------------------------------
// DLT / GPT-LU form: A(8x8) h = b with h33 = 1 (Eq. 1-3), solved by
// Gaussian elimination with partial pivoting.  Returns false if a pivot is 0.
// Row pair of correspondence (x,y)->(u,v):
//   [x y 1 0 0 0 -u*x -u*y | u]
//   [0 0 0 x y 1 -v*x -v*y | v]
// ---------------------------------------------------------------------------
inline bool dlt_ge(const double s[8], const double d[8], double H[9])
{
    double A[8][9];
    for (int k = 0; k < 4; ++k) {
        const double x = s[2 * k], y = s[2 * k + 1], u = d[2 * k], v = d[2 * k + 1];
        double* r0 = A[2 * k];
        double* r1 = A[2 * k + 1];
        r0[0] = x; r0[1] = y; r0[2] = 1; r0[3] = 0; r0[4] = 0; r0[5] = 0;
        r0[6] = -u * x; r0[7] = -u * y; r0[8] = u;
        r1[0] = 0; r1[1] = 0; r1[2] = 0; r1[3] = x; r1[4] = y; r1[5] = 1;
        r1[6] = -v * x; r1[7] = -v * y; r1[8] = v;
    }
    for (int col = 0; col < 8; ++col) {
        int piv = col;
        for (int r = col + 1; r < 8; ++r)
            if (std::fabs(A[r][col]) > std::fabs(A[piv][col])) piv = r;
        if (A[piv][col] == 0.0) return false;
        if (piv != col)
            for (int c = 0; c < 9; ++c) { double t = A[col][c]; A[col][c] = A[piv][c]; A[piv][c] = t; }
        for (int r = col + 1; r < 8; ++r) {
            const double f = A[r][col] / A[col][col];
            for (int c = col; c < 9; ++c) A[r][c] -= f * A[col][c];
        }
    }
    double h[8];
    for (int r = 7; r >= 0; --r) {
        double acc = A[r][8];
        for (int c = r + 1; c < 8; ++c) acc -= A[r][c] * h[c];
        h[r] = acc / A[r][r];
    }
    for (int i = 0; i < 8; ++i) H[i] = h[i];
    H[8] = 1.0;
    return true;
}

// ---------------------------------------------------------------------------
// Comparison form: scale by 1/max|h|, then to unit
// Frobenius norm, then flip the sign so that the largest-magnitude element
// (first one in row-major order on ties) is positive.
// ---------------------------------------------------------------------------
inline void normal_form(double H[9])
{
    double mx = 0.0;
    for (int i = 0; i < 9; ++i) if (std::fabs(H[i]) > mx) mx = std::fabs(H[i]);
    if (!(mx > 0.0) || !std::isfinite(mx)) return;
    double ss = 0.0;
    for (int i = 0; i < 9; ++i) { H[i] /= mx; ss += H[i] * H[i]; }
    const double nrm = std::sqrt(ss);
    int arg = 0;
    for (int i = 1; i < 9; ++i) if (std::fabs(H[i]) > std::fabs(H[arg])) arg = i;
    const double sgn = (H[arg] < 0.0) ? -1.0 : 1.0;
    for (int i = 0; i < 9; ++i) H[i] = sgn * H[i] / nrm;
}

// Forward transfer residual ||pi(H*[x;y;1]) - (u,v)||_2 (reading R9).  W == 0 -> +inf.
inline double transfer_residual(const double H[9], double x, double y, double u, double v)
{
    const double X = H[0] * x + H[1] * y + H[2];
    const double Y = H[3] * x + H[4] * y + H[5];
    const double W = H[6] * x + H[7] * y + H[8];
    if (W == 0.0) return INFINITY;
    const double ex = X / W - u, ey = Y / W - v;
    return std::sqrt(ex * ex + ey * ey);
}

// ---------------------------------------------------------------------------
// Sample check of the hypothesise-and-verify loop (reading R20).
// The paper names what a degenerate minimal sample is -- three of the four points collinear, or two of them
// the same ("both of which are degenerate configurations") -- but gives no test; R20 fixes one:
//   A_ijk = (p_j - p_i) x (p_k - p_i)   (twice the signed area of triangle i,j,k), for the four triangles
//   (0,1,2), (0,1,3), (0,2,3), (1,2,3) of the source quadruple and of the target quadruple;
//   reject  iff  some |A_ijk| <= 2 * min_area on either plane            (degenerate)
//            or  sign(A_ijk(source)) != sign(A_ijk(target)) for some triangle   (H would have to send part of
//                the quadruple through its line at infinity, or mirror the plane: not a view of that plane).
// Arithmetic: coordinates are fp32 values promoted to fp64; every difference, product and the final subtraction is
// one IEEE fp64 operation, in exactly this order (the comparison is a decision: both sides of a parity test take
// it in the same precision).  Returns true when the sample is REJECTED.
// ---------------------------------------------------------------------------
inline double signed_area2(const double* p, int i, int j, int k)
{
    const double ux = p[2 * j] - p[2 * i], uy = p[2 * j + 1] - p[2 * i + 1];
    const double vx = p[2 * k] - p[2 * i], vy = p[2 * k + 1] - p[2 * i + 1];
    const double a = ux * vy;
    const double b = uy * vx;
    return a - b;
}

inline bool sample_rejected(const double s[8], const double d[8], double min_area)
{
    static const int tri[4][3] = { {0, 1, 2}, {0, 1, 3}, {0, 2, 3}, {1, 2, 3} };
    const double lim = 2.0 * min_area;
    for (int t = 0; t < 4; ++t) {
        const double a1 = signed_area2(s, tri[t][0], tri[t][1], tri[t][2]);
        const double a2 = signed_area2(d, tri[t][0], tri[t][1], tri[t][2]);
        if (!(std::fabs(a1) > lim) || !(std::fabs(a2) > lim)) return true;     // also rejects NaN
        if ((a1 > 0.0) != (a2 > 0.0)) return true;
    }
    return false;
}

// ---------------------------------------------------------------------------
// Scalar type that counts arithmetic the way the paper does:
// add / sub / mul = 1 FLOP, division = 4 FLOPs.  Unary minus is free.
// ---------------------------------------------------------------------------
struct Counted {
    double v;
    static inline int64_t n_add = 0, n_mul = 0, n_div = 0;
    Counted() : v(0.0) {}
    Counted(double x) : v(x) {}
    static void reset() { n_add = n_mul = n_div = 0; }
    static int64_t flops() { return n_add + n_mul + 4 * n_div; }
};
inline Counted operator+(Counted a, Counted b) { ++Counted::n_add; return Counted(a.v + b.v); }
inline Counted operator-(Counted a, Counted b) { ++Counted::n_add; return Counted(a.v - b.v); }
inline Counted operator*(Counted a, Counted b) { ++Counted::n_mul; return Counted(a.v * b.v); }
inline Counted operator/(Counted a, Counted b) { ++Counted::n_div; return Counted(a.v / b.v); }
inline Counted operator-(Counted a) { return Counted(-a.v); }

// ---------------------------------------------------------------------------
// Forward-mode dual number with N partial derivatives: evaluating any of the
// templated solvers above on Dual<N> differentiates the paper's formulas step by
// step (sum, product and quotient rules only).  Used for the backward pass of the
// offsets -> H map ("ACA only uses basic arithmetic operations which are naturally
// differential").
// ---------------------------------------------------------------------------
template <int N>
struct Dual {
    double v;
    double g[N];
    Dual() : v(0.0) { for (int i = 0; i < N; ++i) g[i] = 0.0; }
    Dual(double x) : v(x) { for (int i = 0; i < N; ++i) g[i] = 0.0; }
    static Dual variable(double x, int k) { Dual r(x); r.g[k] = 1.0; return r; }
};
template <int N> inline Dual<N> operator+(const Dual<N>& a, const Dual<N>& b)
{ Dual<N> r(a.v + b.v); for (int i = 0; i < N; ++i) r.g[i] = a.g[i] + b.g[i]; return r; }
template <int N> inline Dual<N> operator-(const Dual<N>& a, const Dual<N>& b)
{ Dual<N> r(a.v - b.v); for (int i = 0; i < N; ++i) r.g[i] = a.g[i] - b.g[i]; return r; }
template <int N> inline Dual<N> operator*(const Dual<N>& a, const Dual<N>& b)
{ Dual<N> r(a.v * b.v); for (int i = 0; i < N; ++i) r.g[i] = a.g[i] * b.v + a.v * b.g[i]; return r; }
template <int N> inline Dual<N> operator/(const Dual<N>& a, const Dual<N>& b)
{ Dual<N> r(a.v / b.v); for (int i = 0; i < N; ++i) r.g[i] = (a.g[i] - r.v * b.g[i]) / b.v; return r; }
template <int N> inline Dual<N> operator-(const Dual<N>& a)
{ Dual<N> r(-a.v); for (int i = 0; i < N; ++i) r.g[i] = -a.g[i]; return r; }

// ---------------------------------------------------------------------------
// Counter-based generator for on-device hypothesis sampling ("RANSAC extras"): the
// published Philox4x32-10 (Salmon et al., SC'11), restated: 10 rounds of
//   (c0, c1, c2, c3) <- (hi(M1*c2) ^ c1 ^ k0, lo(M1*c2), hi(M0*c0) ^ c3 ^ k1, lo(M0*c0)),  k += (W0, W1).
// Pinned by the published known-answer vectors (tests/golden/philox4x32_10_kat.json).
// ---------------------------------------------------------------------------
inline void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    const uint64_t M0 = 0xD2511F53ull, M1 = 0xCD9E8D57ull;
    const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = M0 * c0, p1 = M1 * c2;
        const uint32_t n0 = static_cast<uint32_t>(p1 >> 32) ^ c1 ^ k0;
        const uint32_t n1 = static_cast<uint32_t>(p1);
        const uint32_t n2 = static_cast<uint32_t>(p0 >> 32) ^ c3 ^ k1;
        const uint32_t n3 = static_cast<uint32_t>(p0);
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += W0; k1 += W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// The 4 indices of hypothesis h (reading R19 of DESIGN.md): attempt a = 0, 1, ... draws
// Philox(counter = (lo32(h), hi32(h), a, 0), key = (lo32(seed), hi32(seed))) and maps each word r to
// floor(r * n_pts / 2^32); the first attempt whose 4 indices are pairwise distinct is taken; after 32
// failed attempts (only plausible for n_pts < 8) the sample is i, i+1, i+2, i+3 (mod n_pts), i = attempt 0's
// first index.
inline void sample4(uint64_t seed, uint64_t h, int32_t n_pts, int32_t idx[4])
{
    const uint32_t key[2] = { static_cast<uint32_t>(seed), static_cast<uint32_t>(seed >> 32) };
    int32_t first = 0;
    for (uint32_t a = 0; a < 32; ++a) {
        const uint32_t ctr[4] = { static_cast<uint32_t>(h), static_cast<uint32_t>(h >> 32), a, 0u };
        uint32_t r[4];
        philox4x32_10(ctr, key, r);
        for (int k = 0; k < 4; ++k)
            idx[k] = static_cast<int32_t>((static_cast<uint64_t>(r[k]) * static_cast<uint64_t>(n_pts)) >> 32);
        if (a == 0) first = idx[0];
        if (idx[0] != idx[1] && idx[0] != idx[2] && idx[0] != idx[3] && idx[1] != idx[2] && idx[1] != idx[3] && idx[2] != idx[3])
            return;
    }
    for (int k = 0; k < 4; ++k) idx[k] = (first + k) % n_pts;
}

}  // namespace hgo
