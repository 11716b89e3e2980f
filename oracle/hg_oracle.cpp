// ORACLE -- TEST INFRASTRUCTURE ONLY (see hg_oracle_core.hpp for the rules).
//
// C-ABI batch drivers around the scalar oracle functions, loaded by
// oracle/__init__.py through ctypes.  Inputs are the fp32 problem instance
// (promoted exactly to fp64); results are fp64.  AoS layouts throughout:
//   src, dst : float  [n][4][2]   (x,y of points M,N,P,Q)
//   H        : double [n][3][3]   row-major
// Batch loops are OpenMP-parallel over independent sets; that is the only
// parallelism, and nothing is tuned.
#include "hg_oracle_core.hpp"

#include <cstring>
#include <omp.h>

namespace {

inline void load_set(const float* p, double o[8])
{
    for (int i = 0; i < 8; ++i) o[i] = static_cast<double>(p[i]);
}

}  // namespace

extern "C" {

int hgo_num_threads(void) { return omp_get_max_threads(); }
void hgo_set_num_threads(int n) { omp_set_num_threads(n); }

// method: 0 = DLT-GE (h33 = 1), 1 = ACA (raw scale), 2 = SKS, 3 = closed form Eq. 33'
// ok (nullable): per-set flag, 0 where DLT-GE met a zero pivot (H then holds NaN).
void hgo_solve(int method, const float* src, const float* dst, double* H, int64_t n, uint8_t* ok)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        double s[8], d[8];
        load_set(src + 8 * i, s);
        load_set(dst + 8 * i, d);
        double* Hi = H + 9 * i;
        bool good = true;
        switch (method) {
            case 0: good = hgo::dlt_ge(s, d, Hi); break;
            case 1: hgo::aca<double>(s, d, Hi); break;
            case 2: hgo::sks<double>(s, d, Hi); break;
            default: hgo::closed_form<double>(s, d, Hi); break;
        }
        if (!good) for (int k = 0; k < 9; ++k) Hi[k] = NAN;
        if (ok) ok[i] = good ? 1 : 0;
    }
}

// Same with fp64 inputs (used by the exact-integer and homogeneity pins).
void hgo_solve_f64(int method, const double* src, const double* dst, double* H, int64_t n)
{
    for (int64_t i = 0; i < n; ++i) {
        const double* s = src + 8 * i;
        const double* d = dst + 8 * i;
        double* Hi = H + 9 * i;
        switch (method) {
            case 0: if (!hgo::dlt_ge(s, d, Hi)) for (int k = 0; k < 9; ++k) Hi[k] = NAN; break;
            case 1: hgo::aca<double>(s, d, Hi); break;
            case 2: hgo::sks<double>(s, d, Hi); break;
            default: hgo::closed_form<double>(s, d, Hi); break;
        }
    }
}

// ACA core parameters c11,c22,c33 (Eq. 32) and SKS kernel parameters aK,bK,uK,vK (Eq. 15).
void hgo_aca_core(const float* src, const float* dst, double* core3, int64_t n)
{
    for (int64_t i = 0; i < n; ++i) {
        double s[8], d[8], H[9];
        load_set(src + 8 * i, s);
        load_set(dst + 8 * i, d);
        hgo::aca<double>(s, d, H, core3 + 3 * i);
    }
}
void hgo_sks_kernel(const float* src, const float* dst, double* kern4, int64_t n)
{
    for (int64_t i = 0; i < n; ++i) {
        double s[8], d[8], H[9];
        load_set(src + 8 * i, s);
        load_set(dst + 8 * i, d);
        hgo::sks<double>(s, d, H, kern4 + 4 * i);
    }
}

// Normal form (unit Frobenius, sign-fixed) in place.
void hgo_normal_form(double* H, int64_t n)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) hgo::normal_form(H + 9 * i);
}

// Paper-style operation counts of one evaluation.  method: 1 = ACA, 2 = SKS, 3 = Algorithm 1, 4 = affine, 5 = SK.
// out = { add/sub, mul, div, FLOPs = add + mul + 4*div }.
void hgo_op_counts(int method, int64_t out[4])
{
    using hgo::Counted;
    // any non-degenerate quadrilateral pair
    const double sv[8] = { 10, 20, 310, 35, 290, 260, 25, 240 };
    const double dv[8] = { 40, 30, 350, 60, 300, 300, 15, 270 };
    Counted s[8], d[8], H[9];
    for (int i = 0; i < 8; ++i) { s[i] = Counted(sv[i]); d[i] = Counted(dv[i]); }
    Counted::reset();
    if (method == 1)      hgo::aca<Counted>(s, d, H);
    else if (method == 2) hgo::sks<Counted>(s, d, H);
    else if (method == 3) // Algorithm 1 (TensorACA-rect) on a 300 x 240 rectangle, r_rec = 1.25
        hgo::aca_rect<Counted>(Counted(10.0), Counted(20.0), Counted(300.0), Counted(1.25), d, d + 2, d + 6, d + 4, H);
    else if (method == 4) // affine from the first three correspondences (Eq. 41)
        hgo::affine<Counted>(s, d, H);
    else {                // 5 = simplified SK (Eq. 17); the pattern constants are not counted (Table 3: 0)
        Counted pat[5];
        hgo::sk_pattern<Counted>(Counted(0.3), Counted(1.7), Counted(-0.6), Counted(-1.2), pat);
        Counted::reset();
        hgo::sk<Counted>(pat, d, H);
    }
    out[0] = Counted::n_add;
    out[1] = Counted::n_mul;
    out[2] = Counted::n_div;
    out[3] = Counted::flops();
}

// Algorithm 1 (TensorACA-rect).  offsets float [n][4][2] in corner order TL,TR,BR,BL of the
// source rectangle TL=(x0,y0), extents (w,h); target corner = source corner + offset.
// Roles per R6: M=TL, N=TR, Q=BR, P=BL.
void hgo_aca_rect(const float* offsets, float x0, float y0, float w, float h, double* H, int64_t n)
{
    const double X0 = x0, Y0 = y0, Wd = w, Hd = h;
    const double cx[4] = { X0, X0 + Wd, X0 + Wd, X0 };
    const double cy[4] = { Y0, Y0, Y0 + Hd, Y0 + Hd };
    for (int64_t i = 0; i < n; ++i) {
        double t[4][2];
        for (int k = 0; k < 4; ++k) {
            t[k][0] = cx[k] + static_cast<double>(offsets[8 * i + 2 * k]);
            t[k][1] = cy[k] + static_cast<double>(offsets[8 * i + 2 * k + 1]);
        }
        hgo::aca_rect<double>(X0, Y0, Wd, Wd / Hd, t[0], t[1], t[3], t[2], H + 9 * i);
    }
}

// Backward pass of the deep-homography module: G(offsets) = H / h33 with H from
// Algorithm 1 (what hg_aca_rect_batched returns under HG_NORM_H33).  Given grad_G = dL/dG
// (double [n][9], the (3,3) entry is ignored because G33 == 1), returns
// grad_off[k] = sum_ij grad_G[ij] * dG_ij / d offsets[k]   (double [n][8]),
// the Jacobian taken by forward-mode dual numbers through aca_rect<> and the division by h33.
// jac (nullable): double [n][9][8], dG_ij / d offsets[k].
void hgo_aca_rect_backward(const float* offsets, float x0, float y0, float w, float h,
                           const double* grad_G, double* grad_off, double* jac, int64_t n)
{
    using D = hgo::Dual<8>;
    const double X0 = x0, Y0 = y0, Wd = w, Hd = h;
    const double cx[4] = { X0, X0 + Wd, X0 + Wd, X0 };
    const double cy[4] = { Y0, Y0, Y0 + Hd, Y0 + Hd };
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        D t[4][2];
        for (int k = 0; k < 4; ++k) {
            t[k][0] = D(cx[k]) + D::variable(static_cast<double>(offsets[8 * i + 2 * k]), 2 * k);
            t[k][1] = D(cy[k]) + D::variable(static_cast<double>(offsets[8 * i + 2 * k + 1]), 2 * k + 1);
        }
        D H[9];
        hgo::aca_rect<D>(D(X0), D(Y0), D(Wd), D(Wd / Hd), t[0], t[1], t[3], t[2], H);
        double go[8] = { 0, 0, 0, 0, 0, 0, 0, 0 };
        for (int e = 0; e < 9; ++e) {
            const D G = H[e] / H[8];
            if (jac) for (int k = 0; k < 8; ++k) jac[(9 * i + e) * 8 + k] = G.g[k];
            if (e == 8) continue;
            for (int k = 0; k < 8; ++k) go[k] += grad_G[9 * i + e] * G.g[k];
        }
        if (grad_off) for (int k = 0; k < 8; ++k) grad_off[8 * i + k] = go[k];
    }
}

// Affine from three correspondences: src3, dst3 float [n][3][2] -> H double [n][3][3] (raw scale, h33 = f_A1).
void hgo_affine(const float* src3, const float* dst3, double* H, int64_t n)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        double s[6], d[6];
        for (int k = 0; k < 6; ++k) { s[k] = static_cast<double>(src3[6 * i + k]); d[k] = static_cast<double>(dst3[6 * i + k]); }
        hgo::affine<double>(s, d, H + 9 * i);
    }
}

// Simplified SK: pattern points P3, Q3 in the anchor frame (doubles), dst float [n][4][2] -> Hbar double [n][3][3].
void hgo_sk(double P3x, double P3y, double Q3x, double Q3y, const float* dst, double* H, int64_t n)
{
    double pat[5];
    hgo::sk_pattern<double>(P3x, P3y, Q3x, Q3y, pat);
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        double d[8];
        load_set(dst + 8 * i, d);
        hgo::sk<double>(pat, d, H + 9 * i);
    }
}

// Offsets -> H -> dense grid (reading R10).  General ACA on corners in API order
// (M,N,P,Q = TL,TR,BR,BL), then grid[b][j][i] = pi(H_b * (x_i, y_j, 1)) with
// x_i = x0 + i*w/(grid_w-1), y_j = y0 + j*h/(grid_h-1) (x_i = x0 when grid_w == 1).
// H_out (nullable) double [n][9] raw scale; grid (nullable) double [n][grid_h][grid_w][2].
void hgo_offsets_to_grid(const float* offsets, float x0, float y0, float w, float h,
                         int32_t grid_w, int32_t grid_h, double* H_out, double* grid, int64_t n)
{
    const double X0 = x0, Y0 = y0, Wd = w, Hd = h;
    const double s[8] = { X0, Y0, X0 + Wd, Y0, X0 + Wd, Y0 + Hd, X0, Y0 + Hd };
#pragma omp parallel for schedule(static)
    for (int64_t b = 0; b < n; ++b) {
        double d[8], H[9];
        for (int k = 0; k < 8; ++k) d[k] = s[k] + static_cast<double>(offsets[8 * b + k]);
        hgo::aca<double>(s, d, H);
        if (H_out) std::memcpy(H_out + 9 * b, H, sizeof(H));
        if (!grid) continue;
        double* g = grid + static_cast<int64_t>(2) * grid_w * grid_h * b;
        for (int32_t j = 0; j < grid_h; ++j) {
            const double y = (grid_h > 1) ? Y0 + j * Hd / (grid_h - 1) : Y0;
            for (int32_t i = 0; i < grid_w; ++i) {
                const double x = (grid_w > 1) ? X0 + i * Wd / (grid_w - 1) : X0;
                const double X = H[0] * x + H[1] * y + H[2];
                const double Y = H[3] * x + H[4] * y + H[5];
                const double W = H[6] * x + H[7] * y + H[8];
                g[2 * (static_cast<int64_t>(j) * grid_w + i) + 0] = X / W;
                g[2 * (static_cast<int64_t>(j) * grid_w + i) + 1] = Y / W;
            }
        }
    }
}

// Backward pass of hgo_offsets_to_grid ("offsets -> H (-> grid)"; "naturally differential"):
// given grad_grid = dL/d grid (double [n][grid_h][grid_w][2]) returns
//   grad_off[b][k] = sum over pixels (j,i) and coordinates c of grad_grid[b][j][i][c] * d grid[b][j][i][c] / d offsets[b][k]
// (double [n][8]).  The derivative is taken by the plain chain rule in forward mode: the eight offsets are dual-number
// variables, the forward pass is the one of hgo_offsets_to_grid line by line (general ACA on the corners, then the
// projection of every lattice point), and every pixel contributes its two dual parts.
void hgo_offsets_to_grid_backward(const float* offsets, float x0, float y0, float w, float h,
                                  int32_t grid_w, int32_t grid_h, const double* grad_grid, double* grad_off, int64_t n)
{
    using D = hgo::Dual<8>;
    const double X0 = x0, Y0 = y0, Wd = w, Hd = h;
    const double sc[8] = { X0, Y0, X0 + Wd, Y0, X0 + Wd, Y0 + Hd, X0, Y0 + Hd };
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t b = 0; b < n; ++b) {
        D s[8], d[8], H[9];
        for (int k = 0; k < 8; ++k) {
            s[k] = D(sc[k]);
            d[k] = D(sc[k]) + D::variable(static_cast<double>(offsets[8 * b + k]), k);
        }
        hgo::aca<D>(s, d, H);
        double go[8] = { 0, 0, 0, 0, 0, 0, 0, 0 };
        const double* g = grad_grid + static_cast<int64_t>(2) * grid_w * grid_h * b;
        for (int32_t j = 0; j < grid_h; ++j) {
            const double y = (grid_h > 1) ? Y0 + j * Hd / (grid_h - 1) : Y0;
            for (int32_t i = 0; i < grid_w; ++i) {
                const double x = (grid_w > 1) ? X0 + i * Wd / (grid_w - 1) : X0;
                const D X = H[0] * D(x) + H[1] * D(y) + H[2];
                const D Y = H[3] * D(x) + H[4] * D(y) + H[5];
                const D W = H[6] * D(x) + H[7] * D(y) + H[8];
                const D u = X / W, v = Y / W;
                const double gu = g[2 * (static_cast<int64_t>(j) * grid_w + i) + 0];
                const double gv = g[2 * (static_cast<int64_t>(j) * grid_w + i) + 1];
                for (int k = 0; k < 8; ++k) go[k] += gu * u.g[k] + gv * v.g[k];
            }
        }
        for (int k = 0; k < 8; ++k) grad_off[8 * b + k] = go[k];
    }
}

// Offsets -> H -> warped image ("warp image with H"; reading R17):
//   warped[b][c][j][i] = bilinear(image[b][c], pi(H_b * (x_i, y_j, 1)))
// with the lattice (x_i, y_j) of hgo_offsets_to_grid.  The image is sampled in pixel units (pixel (col u,
// row v) has centre (u, v)); u0 = floor(u), fu = u - u0, the four taps (u0,v0), (u0+1,v0), (u0,v0+1),
// (u0+1,v0+1) carry weights (1-fu)(1-fv), fu(1-fv), (1-fu)fv, fu fv, and a tap outside the image
// contributes zero (zero padding).  A non-finite sampling position gives 0.
//   image  float  [n][channels][img_h][img_w];   warped double [n][channels][out_h][out_w]
void hgo_offsets_to_warp(const float* offsets, float x0, float y0, float w, float h,
                         int32_t out_w, int32_t out_h, const float* image, int32_t channels,
                         int32_t img_w, int32_t img_h, double* warped, int64_t n)
{
    const double X0 = x0, Y0 = y0, Wd = w, Hd = h;
    const double s[8] = { X0, Y0, X0 + Wd, Y0, X0 + Wd, Y0 + Hd, X0, Y0 + Hd };
#pragma omp parallel for schedule(static)
    for (int64_t b = 0; b < n; ++b) {
        double d[8], H[9];
        for (int k = 0; k < 8; ++k) d[k] = s[k] + static_cast<double>(offsets[8 * b + k]);
        hgo::aca<double>(s, d, H);
        for (int32_t j = 0; j < out_h; ++j) {
            const double y = (out_h > 1) ? Y0 + j * Hd / (out_h - 1) : Y0;
            for (int32_t i = 0; i < out_w; ++i) {
                const double x = (out_w > 1) ? X0 + i * Wd / (out_w - 1) : X0;
                const double X = H[0] * x + H[1] * y + H[2];
                const double Y = H[3] * x + H[4] * y + H[5];
                const double W = H[6] * x + H[7] * y + H[8];
                const double u = X / W, v = Y / W;
                const bool finite = std::isfinite(u) && std::isfinite(v);
                const double u0 = std::floor(u), v0 = std::floor(v);
                const double fu = u - u0, fv = v - v0;
                for (int32_t c = 0; c < channels; ++c) {
                    const float* img = image + (static_cast<int64_t>(b) * channels + c) * img_h * img_w;
                    double acc = 0.0;
                    if (finite && u0 >= -1.0 && u0 <= img_w && v0 >= -1.0 && v0 <= img_h) {
                        const int64_t iu = static_cast<int64_t>(u0), iv = static_cast<int64_t>(v0);
                        for (int dv = 0; dv < 2; ++dv)
                            for (int du = 0; du < 2; ++du) {
                                const int64_t tu = iu + du, tv = iv + dv;
                                if (tu < 0 || tu >= img_w || tv < 0 || tv >= img_h) continue;
                                const double wt = (du ? fu : 1.0 - fu) * (dv ? fv : 1.0 - fv);
                                acc += wt * static_cast<double>(img[tv * img_w + tu]);
                            }
                    }
                    warped[((static_cast<int64_t>(b) * channels + c) * out_h + j) * out_w + i] = acc;
                }
            }
        }
    }
}

// RANSAC hypothesise-and-score (reading R9).
//   src_xy, dst_xy : float [n_pts][2];  hyp_idx : int32 [n_hyp][4]
//   solver: 1 = ACA-fp64 (the parity reference), 0 = DLT-GE (cross-check)
//   counts[h]      = #{ k : r_k <= t },  r_k = forward transfer residual in fp64, W == 0 -> outlier
//   band_counts[h] = #{ k : |r_k - t| <= band_rel * t }   (the allowance of north_star)
//   best: max count, ties -> lowest hypothesis index; best_H = that H in normal form.
// Reading R20: reject flags of the 4-point samples (1 = rejected).
void hgo_sample_check(const float* src_xy, const float* dst_xy, const int32_t* hyp_idx, int64_t n_hyp,
                      double min_area, uint8_t* rejected)
{
#pragma omp parallel for schedule(static)
    for (int64_t hI = 0; hI < n_hyp; ++hI) {
        double s[8], d[8];
        for (int k = 0; k < 4; ++k) {
            const int32_t j = hyp_idx[4 * hI + k];
            s[2 * k] = src_xy[2 * j];     s[2 * k + 1] = src_xy[2 * j + 1];
            d[2 * k] = dst_xy[2 * j];     d[2 * k + 1] = dst_xy[2 * j + 1];
        }
        rejected[hI] = hgo::sample_rejected(s, d, min_area) ? 1 : 0;
    }
}

// reject_min_area < 0: no sample check (reading R9); >= 0: samples rejected by reading R20 score 0.
void hgo_ransac_opt(const float* src_xy, const float* dst_xy, int32_t n_pts,
                    const int32_t* hyp_idx, int64_t n_hyp, double t, double band_rel, int solver,
                    double reject_min_area, int32_t* counts, int32_t* band_counts,
                    double* best_H, int64_t* best_index, int32_t* best_count);

void hgo_ransac(const float* src_xy, const float* dst_xy, int32_t n_pts,
                const int32_t* hyp_idx, int64_t n_hyp, double t, double band_rel, int solver,
                int32_t* counts, int32_t* band_counts,
                double* best_H, int64_t* best_index, int32_t* best_count)
{
    hgo_ransac_opt(src_xy, dst_xy, n_pts, hyp_idx, n_hyp, t, band_rel, solver, -1.0, counts, band_counts, best_H, best_index,
                   best_count);
}

void hgo_ransac_opt(const float* src_xy, const float* dst_xy, int32_t n_pts,
                    const int32_t* hyp_idx, int64_t n_hyp, double t, double band_rel, int solver,
                    double reject_min_area, int32_t* counts, int32_t* band_counts,
                    double* best_H, int64_t* best_index, int32_t* best_count)
{
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t hI = 0; hI < n_hyp; ++hI) {
        double s[8], d[8], H[9];
        for (int k = 0; k < 4; ++k) {
            const int32_t j = hyp_idx[4 * hI + k];
            s[2 * k] = src_xy[2 * j];     s[2 * k + 1] = src_xy[2 * j + 1];
            d[2 * k] = dst_xy[2 * j];     d[2 * k + 1] = dst_xy[2 * j + 1];
        }
        bool good = true;
        if (reject_min_area >= 0.0 && hgo::sample_rejected(s, d, reject_min_area)) good = false;
        else if (solver == 0) good = hgo::dlt_ge(s, d, H);
        else                  hgo::aca<double>(s, d, H);
        int32_t c = 0, bc = 0;
        if (good) {
            for (int32_t k = 0; k < n_pts; ++k) {
                const double r = hgo::transfer_residual(H, src_xy[2 * k], src_xy[2 * k + 1],
                                                        dst_xy[2 * k], dst_xy[2 * k + 1]);
                if (r <= t) ++c;
                if (std::fabs(r - t) <= band_rel * t) ++bc;
            }
        }
        counts[hI] = c;
        if (band_counts) band_counts[hI] = bc;
    }
    int64_t bi = -1;
    int32_t bcnt = -1;
    for (int64_t hI = 0; hI < n_hyp; ++hI)
        if (counts[hI] > bcnt) { bcnt = counts[hI]; bi = hI; }
    if (best_index) *best_index = bi;
    if (best_count) *best_count = bcnt;
    if (best_H && bi >= 0) {
        double s[8], d[8];
        for (int k = 0; k < 4; ++k) {
            const int32_t j = hyp_idx[4 * bi + k];
            s[2 * k] = src_xy[2 * j];     s[2 * k + 1] = src_xy[2 * j + 1];
            d[2 * k] = dst_xy[2 * j];     d[2 * k + 1] = dst_xy[2 * j + 1];
        }
        hgo::aca<double>(s, d, best_H);
        hgo::normal_form(best_H);
    }
}

// Known-answer access to the generator, and the sampled indices of hypotheses [h0, h0 + n).
void hgo_philox4x32_10(const uint32_t* ctr, const uint32_t* key, uint32_t* out) { hgo::philox4x32_10(ctr, key, out); }

void hgo_ransac_sample(uint64_t seed, int64_t h0, int64_t n, int32_t n_pts, int32_t* idx)
{
    for (int64_t i = 0; i < n; ++i) hgo::sample4(seed, static_cast<uint64_t>(h0 + i), n_pts, idx + 4 * i);
}

// RANSAC with on-device-style sampling and adaptive termination ("99 %"; reading R19).
// Hypotheses are scored in rounds of round_hyp; after a round with `done` hypotheses scored and best count c,
//   w = c / n_pts,  s = done * log1p(-w^4) - log1p(-confidence);  stop iff s <= 0
// (i.e. done >= log(1 - confidence) / log(1 - w^4), the standard number of samples for an all-inlier draw);
// confidence <= 0 never stops early.  counts / idx_out / band_counts hold max_hyp entries (those past
// n_evaluated are left untouched); margins[r] = s after round r (NaN when not computed).
void hgo_ransac_adaptive(const float* src_xy, const float* dst_xy, int32_t n_pts, uint64_t seed,
                         int64_t max_hyp, int64_t round_hyp, double t, double confidence, double band_rel,
                         double reject_min_area, int32_t* idx_out, int32_t* counts, int32_t* band_counts, double* best_H,
                         int64_t* best_index, int32_t* best_count, int64_t* n_evaluated, double* margins)
{
    int64_t bi = -1, done = 0, round = 0;
    int32_t bc = -1;
    while (done < max_hyp) {
        const int64_t m = (max_hyp - done < round_hyp) ? (max_hyp - done) : round_hyp;
        hgo_ransac_sample(seed, done, m, n_pts, idx_out + 4 * done);
        int64_t rbi = -1;
        int32_t rbc = -1;
        hgo_ransac_opt(src_xy, dst_xy, n_pts, idx_out + 4 * done, m, t, band_rel, 1, reject_min_area, counts + done,
                       band_counts ? band_counts + done : nullptr, nullptr, &rbi, &rbc);
        if (rbc > bc) { bc = rbc; bi = done + rbi; }          // ties keep the lowest index
        done += m;
        double s = NAN;
        if (confidence > 0.0) {
            const double w = static_cast<double>(bc) / static_cast<double>(n_pts);
            const double q = w * w * w * w;
            s = static_cast<double>(done) * std::log1p(-q) - std::log1p(-confidence);
        }
        if (margins) margins[round] = s;
        ++round;
        if (confidence > 0.0 && s <= 0.0) break;
    }
    *n_evaluated = done;
    *best_index = bi;
    *best_count = bc;
    if (best_H && bi >= 0) {
        double sv[8], dv[8];
        for (int k = 0; k < 4; ++k) {
            const int32_t j = idx_out[4 * bi + k];
            sv[2 * k] = src_xy[2 * j];     sv[2 * k + 1] = src_xy[2 * j + 1];
            dv[2 * k] = dst_xy[2 * j];     dv[2 * k + 1] = dst_xy[2 * j + 1];
        }
        hgo::aca<double>(sv, dv, best_H);
        hgo::normal_form(best_H);
    }
}

// Residuals of one H against all correspondences (used by tests to look at single pairs).
void hgo_residuals(const double* H, const float* src_xy, const float* dst_xy, int32_t n_pts, double* r)
{
    for (int32_t k = 0; k < n_pts; ++k)
        r[k] = hgo::transfer_residual(H, src_xy[2 * k], src_xy[2 * k + 1], dst_xy[2 * k], dst_xy[2 * k + 1]);
}

}  // extern "C"
