/*
 * hg.h -- C ABI of libhg: batched minimal 4-point homography on one B200 (sm_100a).
 *
 * Implements the data-parallel hot path of arXiv 2402.18008 ("Fast and Interpretable 2D
 * Homography Decomposition: SKS and ACA transformations"); "P:<line>" cites
 * /root/reference/PAPER.md.  One 3x3 homography H (up to scale) is computed from each set of
 * four point correspondences {M,N,P,Q}_1 -> {M,N,P,Q}_2 (Eq. 1), for millions of
 * sets per call (Sec. 6.4: "each 4-point homography is assigned to one thread").
 *
 * Conventions shared by every entry point
 * ---------------------------------------
 *  - Every pointer is a DEVICE pointer owned by the caller unless the name ends in `_host`
 *    (those entry points take HOST pointers, pinned or pageable, and do the copies themselves).
 *  - The library allocates no device memory (the `_host` entry points allocate and free their
 *    own staging buffers and streams inside the call).  Its only state is internal to the RANSAC
 *    entry points, which stage tables of <= 4096 correspondences in the device's 64 KB constant
 *    bank: calls that do so are ordered against each other through an internal event, and a call made
 *    on a capturing stream stages its table in shared memory instead, so every entry point is
 *    thread-safe and may be issued on any streams, captured or not (the one exception is
 *    hg_ransac_hypothesize_score_noalloc, whose calls share a fixed scratch array -- see there).
 *  - Device entry points only ENQUEUE work on `cuda_stream` (a cudaStream_t passed as void*;
 *    NULL = the legacy default stream) and never synchronise; `_host` entry points return
 *    after their result is complete in host memory.
 *  - Return value: HG_OK (0) or a negative hg_status_t.  No exceptions, no errno.
 *    n == 0 (or n_hyp == 0) is HG_OK and a no-op.  Numerical conditions are never errors:
 *    a degenerate set (three collinear points on either plane) yields ACA's finite singular H
 *    and SKS's non-finite H (reading R8).
 *  - Point roles (reading R11): points 0,1,2,3 of a set are M,N,P,Q; ACA uses
 *    M,N,P as anchors, SKS uses M,N.
 *  - H is row-major h11,h12,h13,h21,...,h33 and defined up to scale; its sign is never fixed.
 */
#ifndef HG_H_
#define HG_H_

#include <stddef.h>
#include <stdint.h>

#if defined(__GNUC__)
#define HG_API __attribute__((visibility("default")))
#else
#define HG_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    HG_OK = 0,
    HG_ERR_INVALID_ARG = -1, /* NULL pointer with n > 0, negative size, unknown enum value        */
    HG_ERR_ALIGNMENT   = -2, /* a base pointer is not 16-byte aligned                             */
    HG_ERR_CUDA        = -3, /* a CUDA runtime call or kernel launch failed                       */
    HG_ERR_WORKSPACE   = -4, /* workspace_bytes < hg_ransac_workspace_bytes(...)                  */
    HG_ERR_TOO_LARGE   = -5  /* a size is beyond the fixed capacity of a no-allocation entry point  */
} hg_status_t;

/* Memory layout of the point sets and of H.
 *   HG_SOA: src/dst = float[8][n]  planes x0,y0,x1,y1,x2,y2,x3,y3 (plane stride n);
 *           H       = float[9][n]  planes h11,h12,h13,h21,...,h33.
 *           The streaming layout: every warp access is a full 128-byte line.
 *   HG_AOS: src/dst = float[n][4][2];  H = float[n][3][3] row-major.                              */
typedef enum { HG_SOA = 0, HG_AOS = 1 } hg_layout_t;

/* Scale of the returned H.
 *   HG_NORM_NONE:      the method's raw scale (ACA: Eq. 31-32; SKS: Eq. 11/16).  The
 *                      raw ACA H is a degree-7..9 polynomial of the inputs (Eq. 35),
 *                      about 1e23 for 640x480 coordinates: it overflows fp32 for |coords| >~ 1e4.
 *   HG_NORM_H33:       H / h33 (the 12-FLOP normalisation of P:301; h33 == 0 gives inf/NaN).
 *   HG_NORM_FROBENIUS: H / ||H||_F (overflow-safe).                                               */
typedef enum { HG_NORM_NONE = 0, HG_NORM_H33 = 1, HG_NORM_FROBENIUS = 2 } hg_norm_t;

/* Arithmetic used between the fp32 loads and the fp32 stores.
 *   HG_PREC_F64: inputs promoted exactly to fp64, the whole solve and the normalisation in fp64,
 *                H rounded to fp32 once.  Meets the parity tolerances; the default everywhere.
 *   HG_PREC_F32: plain fp32 (FMA-contracted).  Cancellation in c11-c33, c22-c33 makes h31,h32
 *                inaccurate for near-affine H; provided for measurement and for callers that
 *                accept ~1e-3 relative error.                                                     */
typedef enum { HG_PREC_F64 = 0, HG_PREC_F32 = 1 } hg_precision_t;

/* --------------------------------------------------------------------------------------------
 * hg_aca_batched -- Affine-Core-Affine solve, H = H_A2^-1 * H_C * H_A1 (Sec. 4.2-4.4,
 * Eq. 23-32, Table 4): 85 FLOPs and no division per homography before
 * normalisation.
 *   src, dst : n source / target 4-point sets in `layout`            (read,  64 B per set)
 *   H        : n homographies in `layout`, scaled per `norm`         (write, 36 B per set)
 *   n        : number of sets, >= 0.  HG_SOA planes have stride n; n need not be a multiple of 4
 *              (the 128-bit fast path needs n % 4 == 0, otherwise a scalar-load path is used).
 * Errors: HG_ERR_INVALID_ARG (NULL with n > 0, n < 0, bad enum), HG_ERR_ALIGNMENT (src, dst or H
 * not 16-byte aligned), HG_ERR_CUDA (launch failure).
 * -------------------------------------------------------------------------------------------- */
HG_API int hg_aca_batched(const float* src, const float* dst, float* H, int64_t n,
                   hg_layout_t layout, hg_norm_t norm, hg_precision_t prec, void* cuda_stream);

/* hg_sks_batched -- Similarity-Kernel-Similarity solve, H = H_S2^-1 * H_K * H_S1 with
 * H_K = H_E^-1 * H_S' * H_E (Sec. 3.1-3.4, Eq. 6-16, Table 3): five reciprocals per
 * homography.  Arguments, layouts and errors exactly as hg_aca_batched.                          */
HG_API int hg_sks_batched(const float* src, const float* dst, float* H, int64_t n,
                   hg_layout_t layout, hg_norm_t norm, hg_precision_t prec, void* cuda_stream);

/* Host-buffer forms of the two solves (the end-to-end path of bench.py): src/dst/H are HOST
 * pointers in `layout`.  If all three buffers are page-locked and device-mapped (cudaHostAlloc /
 * cudaHostRegister; torch pinned tensors are) and 16-byte aligned, ONE kernel reads and writes them
 * directly over PCIe (both directions of the bus at once, no staging memory; `chunk_sets` unused).
 * Otherwise the call splits the batch into chunks and pipelines host->device copies, the solve
 * kernel and device->host copies on internal streams.  Either way it returns after H is complete in
 * host memory.  `chunk_sets` = sets per chunk of the staged path (0 = library default).  Extra
 * error: HG_ERR_CUDA if staging memory cannot be allocated.                                        */
HG_API int hg_aca_batched_host(const float* src_host, const float* dst_host, float* H_host, int64_t n,
                        hg_layout_t layout, hg_norm_t norm, hg_precision_t prec,
                        int64_t chunk_sets);
HG_API int hg_sks_batched_host(const float* src_host, const float* dst_host, float* H_host, int64_t n,
                        hg_layout_t layout, hg_norm_t norm, hg_precision_t prec,
                        int64_t chunk_sets);

/* --------------------------------------------------------------------------------------------
 * hg_offsets_to_grid -- the deep-homography use (4-point parameterisation, P:25, P:131,
 * P:540-544): for each item, target corners = source-rectangle corners + predicted offsets,
 * H by ACA, then (fused, same kernel) the dense sampling grid of H over the patch
 * (reading R10: grid[b][j][i] = pi(H_b * (x_i, y_j, 1)), forward map, pixel units).
 *   offsets : float[n][4][2], corner order TL,TR,BR,BL                (read, 32 B per item)
 *   x0,y0,w,h : source rectangle: TL corner (x0,y0), extents w,h (C1/C5: 0,0,127,127).
 *               Requires w != 0 and h != 0.
 *   grid_w, grid_h : pixels per row / rows; x_i = x0 + i*w/(grid_w-1) (x0 if grid_w == 1),
 *               y_j likewise (C5: 128,128 -> integer pixels 0..127).  Ignored if grid == NULL.
 *   H       : nullable, float[n][3][3], scaled per `norm`              (write, 36 B per item)
 *   grid    : nullable, float[n][grid_h][grid_w][2], (x,y) order       (write, 8 B per pixel)
 * The solve is always fp64-internal.  Errors: HG_ERR_INVALID_ARG (offsets NULL with n > 0,
 * both outputs NULL is allowed and a no-op, grid != NULL with grid_w < 1 or grid_h < 1, w == 0
 * or h == 0, n < 0), HG_ERR_ALIGNMENT (offsets/grid not 16-byte aligned, H not 4-byte aligned),
 * HG_ERR_CUDA.
 * -------------------------------------------------------------------------------------------- */
HG_API int hg_offsets_to_grid(const float* offsets, float x0, float y0, float w, float h,
                       int32_t grid_w, int32_t grid_h, float* H, float* grid, int64_t n,
                       hg_norm_t norm, void* cuda_stream);

/* --------------------------------------------------------------------------------------------
 * hg_offsets_to_warp -- offsets -> H -> warped image in one kernel ("warp image with H"): as
 * hg_offsets_to_grid, but instead of writing the sampling grid the kernel samples `image` at it
 * (reading R17):  warped[b][c][j][i] = bilinear(image[b][c], pi(H_b * (x_i, y_j, 1))),
 * image coordinates in pixel units (pixel (col u, row v) has centre (u, v)), the four taps around
 * (floor(u), floor(v)), a tap outside the image contributes zero, a non-finite position gives 0.
 *   offsets, x0, y0, w, h : as hg_offsets_to_grid; out_w, out_h play the role of grid_w, grid_h
 *   image   : float[n][channels][img_h][img_w]                       (read,  4 B per tap, L1-cached)
 *   warped  : float[n][channels][out_h][out_w]                       (write, 4 B per pixel and channel)
 *   H       : nullable, float[n][3][3] per `norm`
 * Errors: HG_ERR_INVALID_ARG (NULL with n > 0, sizes < 1, w == 0 or h == 0, bad enum),
 * HG_ERR_ALIGNMENT (offsets not 16-byte aligned; image, warped, H not 4-byte aligned), HG_ERR_CUDA.
 * An image plane of up to about 160 x 160 pixels is staged in shared memory inside a frame of zeros, one CTA per
 * (item, channel) -- by bulk-async row copies when img_w % 4 == 0 and `image` is 16-byte aligned, by plain loads
 * otherwise; larger planes are gathered through L1.
 * -------------------------------------------------------------------------------------------- */
HG_API int hg_offsets_to_warp(const float* offsets, float x0, float y0, float w, float h,
                       int32_t out_w, int32_t out_h, const float* image, int32_t channels,
                       int32_t img_w, int32_t img_h, float* warped, float* H, int64_t n,
                       hg_norm_t norm, void* cuda_stream);

/* --------------------------------------------------------------------------------------------
 * hg_aca_rect_batched -- TensorACA for a rectangular source (Sec. 5.3, Eq. 42-45, Algorithm 1,
 * P:540-591): the source quadrangle is the fixed rectangle TL = (x0,y0), extents (w,h), shared by
 * the whole batch, so H_A1 is trivial, Q3 = (1,1,1) and H follows from the target corners alone
 * (47 FLOPs; 44 for a square).  Only the offsets are read: 32 B in + 36 B out per homography.
 *   offsets : corner offsets, target corner = source corner + offset, corner order TL,TR,BR,BL
 *             (roles M=TL, N=TR, Q=BR, P=BL, reading R6);
 *             HG_SOA: float[8][n] planes TL.x,TL.y,TR.x,...,BL.y;  HG_AOS: float[n][4][2]   (read)
 *   H       : HG_SOA float[9][n] / HG_AOS float[n][3][3], scaled per `norm`; HG_NORM_NONE returns
 *             Eq. 45's scale (a degree-2 polynomial of the target coordinates times w)       (write)
 * The same H (up to scale) as hg_aca_batched on the explicit corners.  Errors: HG_ERR_INVALID_ARG
 * (NULL with n > 0, n < 0, w == 0 or h == 0, bad enum), HG_ERR_ALIGNMENT (offsets or H not 16-byte
 * aligned), HG_ERR_CUDA.
 * -------------------------------------------------------------------------------------------- */
HG_API int hg_aca_rect_batched(const float* offsets, float x0, float y0, float w, float h, float* H,
                        int64_t n, hg_layout_t layout, hg_norm_t norm, hg_precision_t prec,
                        void* cuda_stream);

/* hg_aca_rect_backward -- backward pass of the deep-homography module (the training use of
 * TensorACA: "ACA only uses basic arithmetic operations which are naturally differential").
 * The forward map is G(offsets) = hg_aca_rect_batched(offsets, ..., HG_AOS, HG_NORM_H33), i.e. H/h33
 * of Algorithm 1.  Given grad_H = dL/dG, writes grad_offsets[b][k] = sum_ij grad_H[b][i][j] *
 * dG_ij/d offsets[b][k] (reverse mode through Algorithm 1 and the division by h33, fp64 internal).
 *   offsets      : float[n][4][2], corner order TL,TR,BR,BL               (read,  32 B per item)
 *   grad_H       : float[n][3][3]; entry (3,3) is ignored (G33 == 1)      (read,  36 B per item)
 *   grad_offsets : float[n][4][2]                                         (write, 32 B per item)
 * Errors: HG_ERR_INVALID_ARG (NULL with n > 0, n < 0, w == 0 or h == 0), HG_ERR_ALIGNMENT (any
 * pointer not 16-byte aligned), HG_ERR_CUDA.                                                      */
HG_API int hg_aca_rect_backward(const float* offsets, float x0, float y0, float w, float h,
                         const float* grad_H, float* grad_offsets, int64_t n, void* cuda_stream);

/* The same backward pass on structure-of-arrays planes (the streaming layout of every other entry point):
 *   offsets float[8][n] (planes TL.x,TL.y,TR.x,...,BL.y), grad_H float[9][n] (planes g11,g12,...,g33),
 *   grad_offsets float[8][n].  n % 4 == 0 takes the 128-bit path.  Errors as hg_aca_rect_backward.          */
HG_API int hg_aca_rect_backward_soa(const float* offsets, float x0, float y0, float w, float h,
                         const float* grad_H, float* grad_offsets, int64_t n, void* cuda_stream);

/* hg_offsets_to_grid_backward -- backward pass of hg_offsets_to_grid ("offsets -> H (-> grid)"; the
 * training use of the fused module): given grad_grid = dL/d grid, writes
 *   grad_offsets[b][k] = sum over pixels (j,i), c in {x,y} of grad_grid[b][j][i][c] * d grid[b][j][i][c] / d offsets[b][k],
 * grid[b][j][i] = pi(H_b (x_i, y_j, 1)) on the lattice of hg_offsets_to_grid (reading R10).  One kernel: H is re-derived from
 * the offsets (Algorithm 1, fp64), the item's gradient is streamed once (fp32 per-pixel partials of the projection, fp64
 * reduction), and the result goes through the reverse mode of hg_aca_rect_backward.
 *   offsets      : float[n][4][2], corner order TL,TR,BR,BL                         (read,  32 B per item)
 *   x0,y0,w,h, grid_w, grid_h : as hg_offsets_to_grid (w != 0, h != 0, grid_w >= 1, grid_h >= 1)
 *   grad_grid    : float[n][grid_h][grid_w][2]                                      (read,  8 B per pixel)
 *   grad_offsets : float[n][4][2]                                                   (write, 32 B per item)
 *   grad_G       : nullable, float[n][3][3]: dL/dG for G = H/h33 (what hg_aca_rect_backward takes; its (3,3) entry is
 *                  the formal partial and is not used)                              (write, 36 B per item)
 * An item whose H sends a lattice point to infinity (W = 0) gets non-finite gradients.
 * Errors: HG_ERR_INVALID_ARG (NULL with n > 0, n < 0, sizes < 1 or > 2^24 or grid_w * grid_h >= 2^30, w == 0 or h == 0),
 * HG_ERR_ALIGNMENT (offsets, grad_grid, grad_offsets not 16-byte aligned, grad_G not 4-byte aligned), HG_ERR_CUDA.        */
HG_API int hg_offsets_to_grid_backward(const float* offsets, float x0, float y0, float w, float h,
                         int32_t grid_w, int32_t grid_h, const float* grad_grid, float* grad_offsets,
                         float* grad_G, int64_t n, void* cuda_stream);

/* --------------------------------------------------------------------------------------------
 * hg_affine_batched -- 2D affine transformation from THREE correspondences by the ACA route
 * (Sec. 5.2, Eq. 41 first row): H_A = H_A2^-1 * H_A1, the core transformation being the
 * identity; 33 FLOPs, no division.  Returned as a 3x3 H "computed in the same way as projective
 * transformations": h31 = h32 = 0 and, under HG_NORM_NONE, h33 = f_A1 (Eq. 24).
 *   src3, dst3 : n sets of points M,N,P;  HG_SOA: float[6][n] planes x0,y0,x1,y1,x2,y2;
 *                HG_AOS: float[n][3][2]                                  (read,  48 B per set)
 *   H          : HG_SOA float[9][n] / HG_AOS float[n][3][3], per `norm`  (write, 36 B per set)
 * Collinear source points give the singular H (h33 = 0).  Errors as hg_aca_batched.
 * -------------------------------------------------------------------------------------------- */
HG_API int hg_affine_batched(const float* src3, const float* dst3, float* H, int64_t n,
                      hg_layout_t layout, hg_norm_t norm, hg_precision_t prec, void* cuda_stream);

/* --------------------------------------------------------------------------------------------
 * hg_sk_batched -- the simplified SK decomposition (Sec. 3.4 case ii, Eq. 17, Table 3 row "SK",
 * P:303-318): homography from a known planar pattern (object plane) to each of n images,
 * Hbar = H * H_S1^-1 = H_S2^-1 * H_K.  The pattern's coordinates are given in the frame of its two
 * anchors, M -> (-1,0), N -> (+1,0) (H_S1 = I), so only P3, Q3 describe it; everything that depends
 * on the pattern alone is computed once per call.  Hbar maps (-1,0), (1,0), P3, Q3 onto the image
 * points M2, N2, P2, Q2.  Two reciprocals per image.
 *   P3x..Q3y : the pattern's third and fourth point in the anchor frame (host doubles, by value)
 *   dst      : n image quadruples M2,N2,P2,Q2 in `layout` (as hg_aca_batched's dst) (read, 32 B)
 *   H        : Hbar in `layout`, per `norm`                                        (write, 36 B)
 * P3.y == 0 or Q3.y == 0 (pattern point on the anchor line) or a zero determinant of Eq. 14 give
 * non-finite output (reading R8).  Errors as hg_aca_batched, plus HG_ERR_INVALID_ARG for a NaN
 * pattern coordinate.
 * -------------------------------------------------------------------------------------------- */
HG_API int hg_sk_batched(double P3x, double P3y, double Q3x, double Q3y, const float* dst, float* H,
                  int64_t n, hg_layout_t layout, hg_norm_t norm, hg_precision_t prec,
                  void* cuda_stream);

/* hg_aca_batched_f64 / hg_sks_batched_f64 -- the two general solvers with fp64 STORAGE, the
 * precision of the paper's own GPU experiment (Sec. 6.4).  Layouts as hg_layout_t with
 * double in place of float (HG_SOA: double[8][n] -> double[9][n]); 128 B read + 72 B written per
 * homography.  Arguments and errors otherwise as hg_aca_batched.                                */
HG_API int hg_aca_batched_f64(const double* src, const double* dst, double* H, int64_t n,
                       hg_layout_t layout, hg_norm_t norm, void* cuda_stream);
HG_API int hg_sks_batched_f64(const double* src, const double* dst, double* H, int64_t n,
                       hg_layout_t layout, hg_norm_t norm, void* cuda_stream);

/* --------------------------------------------------------------------------------------------
 * hg_ransac_hypothesize_score -- RANSAC hypothesis generation fused with inlier scoring
 * (hypothesise-and-verify loop, Sec. 2.2; parallel hypotheses P:703).
 * For every hypothesis: gather its 4 correspondences, ACA solve (fp64 internal), then count
 * the correspondences whose forward transfer error ||pi(H*s) - d||_2 <= threshold_px
 * (reading R9: inclusive, W == 0 -> outlier, no degeneracy test, no local optimisation).
 * Scoring runs in fp32 with a per-hypothesis rigorous error band; every pair that falls inside
 * the band is decided in fp64 by the same kernel, so counts equal an fp64 evaluation.
 * Launches: a call of <= 9472 hypotheses (<= 20 480 on <= 2048 points) on <= 4096 points is one kernel behind a
 * one-CTA zeroing kernel (7 us for 1024 x 1000); larger calls are zero + prep + score
 * (+ best for calls of fewer than 148 x 512 hypotheses) + finalize.  Never synchronises.  Capturable in a CUDA graph: a
 * captured call reads its table from shared-memory stages rather than the constant bank (7-10 % slower on tables of <= 4096
 * points), which makes the graph self-contained -- its replays may overlap any other call of the library.
 *   src_xy, dst_xy : float[n_pts][2] correspondences                  (read)
 *   hyp_idx        : int32[n_hyp][4], the 4 indices of a row distinct and in [0,n_pts)
 *                    (out-of-range indices are undefined behaviour)   (read, 16 B per hyp.)
 *   threshold_px   : t > 0
 *   counts         : nullable, int32[n_hyp] inlier count per hypothesis (write, 4 B per hyp.)
 *   best_H         : nullable, float[9] row-major unit-Frobenius H of the best hypothesis
 *   best_index     : nullable, int64: argmax of counts, ties -> lowest hypothesis index
 *   best_count     : nullable, int32: its count
 *   workspace      : device scratch of >= hg_ransac_workspace_bytes(n_pts, n_hyp) bytes,
 *                    16-byte aligned; contents undefined before the call (the library zeroes what it
 *                    needs), statistics after it (below).  (Header, the packed table, and -- for calls
 *                    too small to fill the GPU with one hypothesis per thread -- 4 bytes per hypothesis
 *                    of partial counts, or the per-group result slots of the one-kernel path.)
 * Errors: HG_ERR_INVALID_ARG (NULL inputs, n_pts < 4, n_hyp < 0, threshold not > 0),
 * HG_ERR_ALIGNMENT, HG_ERR_WORKSPACE, HG_ERR_CUDA.
 * -------------------------------------------------------------------------------------------- */
HG_API size_t hg_ransac_workspace_bytes(int32_t n_pts, int64_t n_hyp);
HG_API int hg_ransac_hypothesize_score(const float* src_xy, const float* dst_xy, int32_t n_pts,
                                const int32_t* hyp_idx, int64_t n_hyp, float threshold_px,
                                int32_t* counts, float* best_H, int64_t* best_index,
                                int32_t* best_count, void* workspace, size_t workspace_bytes,
                                void* cuda_stream);

/* --------------------------------------------------------------------------------------------
 * hg_ransac_adaptive -- the same fused gather-solve-score with the two "RANSAC extras" of the
 * hypothesise-and-verify loop (Sec. 2.2; "99 %" sampling counts) done on the device
 * (reading R19):
 *  - sampling: hypothesis h takes its 4 indices from the counter-based generator Philox4x32-10,
 *    counter = (lo32(h), hi32(h), attempt, 0), key = (lo32(seed), hi32(seed)); word r -> index
 *    floor(r * n_pts / 2^32); the first attempt with 4 pairwise distinct indices is used (after 32
 *    failed attempts: i, i+1, i+2, i+3 mod n_pts, i = attempt 0's first index);
 *  - adaptive termination: hypotheses are scored in rounds of round_hyp; after a round with `done`
 *    hypotheses scored and best count c, w = c / n_pts and the run stops iff
 *    done * log1p(-w^4) <= log1p(-confidence) (fp64), i.e. done >= log(1-confidence)/log(1-w^4);
 *    confidence <= 0 scores all max_hyp hypotheses.  No host synchronisation: every round is
 *    enqueued, rounds after the stop return immediately.  A single round (round_hyp >= max_hyp) on a small table takes
 *    the one-kernel path of hg_ransac_hypothesize_score with the sampling done inside it.
 *   seed, max_hyp, round_hyp : max_hyp <= 2^31-1, round_hyp >= 1, at most 65536 rounds
 *   confidence     : < 1
 *   counts         : nullable, int32[max_hyp]; entries >= *n_evaluated are not written
 *   hyp_idx_out    : nullable, int32[max_hyp][4], 16-byte aligned: the sampled indices (same rule)
 *   best_H, best_index, best_count : as hg_ransac_hypothesize_score, over the hypotheses scored
 *   n_evaluated    : nullable, int64: hypotheses scored (a multiple of round_hyp, or max_hyp)
 *   workspace      : >= hg_ransac_workspace_bytes(n_pts, max_hyp) bytes, 16-byte aligned
 * Errors: as hg_ransac_hypothesize_score.
 * -------------------------------------------------------------------------------------------- */
HG_API int hg_ransac_adaptive(const float* src_xy, const float* dst_xy, int32_t n_pts, uint64_t seed,
                       int64_t max_hyp, int64_t round_hyp, float threshold_px, float confidence,
                       int32_t* counts, int32_t* hyp_idx_out, float* best_H, int64_t* best_index,
                       int32_t* best_count, int64_t* n_evaluated, void* workspace,
                       size_t workspace_bytes, void* cuda_stream);

/* Options of the `_ex` forms (a HOST struct, read during the call; NULL = all defaults = the plain entry points).
 *   HG_RANSAC_REJECT_DEGENERATE : test every 4-point sample before scoring it (reading R20; degenerate
 *                                 configurations P:786): rejected hypotheses score 0 and skip the sweep.
 *   HG_RANSAC_DECIDE_ALL_F64    : verification mode -- no fp32 sweep; every (hypothesis, point) pair is decided by
 *                                 the definition in fp64 from the kernel's own fp64 H.  Orders of magnitude slower;
 *                                 it exists so that the exactness of the fp32 sweep + error band can be checked
 *                                 bit for bit against it.                                                         */
#define HG_RANSAC_REJECT_DEGENERATE 1u
#define HG_RANSAC_DECIDE_ALL_F64    2u
typedef struct hg_ransac_options {
    uint32_t flags;          /* OR of HG_RANSAC_* bits; unknown bits -> HG_ERR_INVALID_ARG                       */
    float    min_area_px2;   /* HG_RANSAC_REJECT_DEGENERATE: epsilon of R20 in px^2 (>= 0; 0 rejects only exact
                                collinearity / coincidence and orientation flips)                                  */
} hg_ransac_options_t;

HG_API int hg_ransac_hypothesize_score_ex(const float* src_xy, const float* dst_xy, int32_t n_pts,
                                   const int32_t* hyp_idx, int64_t n_hyp, float threshold_px,
                                   const hg_ransac_options_t* options,
                                   int32_t* counts, float* best_H, int64_t* best_index,
                                   int32_t* best_count, void* workspace, size_t workspace_bytes,
                                   void* cuda_stream);
HG_API int hg_ransac_adaptive_ex(const float* src_xy, const float* dst_xy, int32_t n_pts, uint64_t seed,
                          int64_t max_hyp, int64_t round_hyp, float threshold_px, float confidence,
                          const hg_ransac_options_t* options,
                          int32_t* counts, int32_t* hyp_idx_out, float* best_H, int64_t* best_index,
                          int32_t* best_count, int64_t* n_evaluated, void* workspace,
                          size_t workspace_bytes, void* cuda_stream);

/* After a RANSAC call has completed on its stream, the first 6 int64 words of the workspace hold
 * statistics of that call (device memory; copy them out to read):
 *   [0] packed best key, [1] number of (hypothesis, table slice) combinations with at least one pair decided in fp64
 *   (= the number of such hypotheses when the launch does not split the table; the one-kernel path and the split launches
 *   count a hypothesis once per slice it was undecided in),
 *   [2] number of (hypothesis, point) pairs decided in fp64, [3] hypotheses scored (adaptive mode),
 *   [4] hypotheses rejected by HG_RANSAC_REJECT_DEGENERATE, [5] pairs that fell inside the table-wide
 *   fp32 band and were re-tested against the per-pair band.                  */
#define HG_RANSAC_STAT_WORDS 6

/* Host-buffer form: all pointers are HOST pointers; the call allocates device memory and the
 * workspace, copies in, runs, copies counts/best out and waits.                                  */
HG_API int hg_ransac_hypothesize_score_host(const float* src_xy_host, const float* dst_xy_host,
                                     int32_t n_pts, const int32_t* hyp_idx_host, int64_t n_hyp,
                                     float threshold_px, int32_t* counts_host, float* best_H_host,
                                     int64_t* best_index_host, int32_t* best_count_host);

/* --------------------------------------------------------------------------------------------
 * hg_ransac_hypothesize_score_noalloc -- hg_ransac_hypothesize_score for callers that have no device
 * memory to hand over as a workspace and no way of getting any.
 *
 * Who that is: code that runs where cudaMalloc / cudaFree are off limits or would break a promise --
 * a plugin or filter called from inside somebody else's frame loop (the host application owns the
 * memory pool and a cudaMalloc there stalls every stream of the device), a control loop with a
 * latency budget in which an allocator call is an unbounded wait, a process whose other threads are
 * capturing streams in the global capture mode (an allocation made meanwhile fails), and embedders
 * whose memory is accounted up front and who must not see the library grow the footprint later.
 * Such callers already own their inputs and outputs; the only thing the ordinary entry point asks of
 * them beyond that is the scratch workspace, and this entry point brings its own.
 *
 * Same operation, same results (bit for bit: it runs the one-kernel small-call path of
 * hg_ransac_hypothesize_score) and the same arguments minus
 * `workspace` / `workspace_bytes`.  The scratch -- the 128-byte header and one 96-byte result slot per
 * group of 32 hypotheses -- lives in a fixed array inside the library image:
 *   - capacity: n_pts <= HG_RANSAC_NOALLOC_MAX_PTS (4096) and n_hyp <= HG_RANSAC_NOALLOC_MAX_HYP
 *     (9472 = 296 groups); the array is HG_RANSAC_NOALLOC_SCRATCH_BYTES (28 672) of device memory
 *     that every GPU which loads libhg holds from module load until the process exits, used or not.
 *     Anything larger is refused with HG_ERR_TOO_LARGE before any work is enqueued -- take the
 *     ordinary entry point with a workspace of your own for that.
 *   - the call performs no cudaMalloc, no cudaFree and calls nothing that allocates (no event or stream
 *     creation either); it enqueues the zeroing kernel and the scoring kernel on `cuda_stream` and returns.
 *   - first call on each device: the library looks up the device address of the array (once per device,
 *     with that device current -- make the device of the buffers current before calling, as for every
 *     entry point) and remembers it.  Make that first call during start-up, outside any stream capture;
 *     later calls do no such set-up.
 *   - ONE array per device, shared by every call: each call zeroes the words it depends on (header and
 *     its slots) on the stream before using them and leaves its own statistics and slots behind, so the
 *     contents between calls are the last call's.  Two calls that can be on the GPU at the same time
 *     (different streams with no ordering between them, or two host threads) zero and write the same
 *     words: that is a race -- wrong best_* outputs, or a final step that waits for a slot the other call
 *     wiped and never finishes.  Keep all calls of a device on one stream, or order them with events.
 *     The statistics words (HG_RANSAC_STAT_WORDS) are not readable through this entry point.
 * Errors: as hg_ransac_hypothesize_score (HG_ERR_INVALID_ARG, HG_ERR_ALIGNMENT, HG_ERR_CUDA), never
 * HG_ERR_WORKSPACE; HG_ERR_TOO_LARGE as above.  n_hyp == 0 is HG_OK and does nothing.
 * -------------------------------------------------------------------------------------------- */
#define HG_RANSAC_NOALLOC_MAX_PTS       4096
#define HG_RANSAC_NOALLOC_MAX_HYP       9472
#define HG_RANSAC_NOALLOC_SCRATCH_BYTES 28672
HG_API int hg_ransac_hypothesize_score_noalloc(const float* src_xy, const float* dst_xy, int32_t n_pts,
                                        const int32_t* hyp_idx, int64_t n_hyp, float threshold_px,
                                        int32_t* counts, float* best_H, int64_t* best_index,
                                        int32_t* best_count, void* cuda_stream);

/* Human-readable name of a status code (static storage, never NULL). */
HG_API const char* hg_status_string(int status);

/* Library version (major*10000 + minor*100 + patch) and the SM architecture it was built for. */
HG_API int hg_version(void);
HG_API int hg_built_for_sm(void);

#ifdef __cplusplus
}
#endif
#endif /* HG_H_ */
