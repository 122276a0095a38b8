/* gsplat_b200.h -- C ABI of the single-GPU (sm_100a) differentiable 3D Gaussian splatting hot path.
 *
 * What this library computes is the data-parallel hot path inside the custom splatting
 * operators that arxiv/paper_2606_11390 distributes across GPUs (section 4:
 * "Gaussian spherical harmonics [10] and Gaussian projection operators ... each GPU processes
 * a segment of the input Gaussians and outputs colors and projected geometric quantities for
 * all cameras in the batch"; "the GPU sorts the Gaussians by depth, rasterizes them to obtain
 * the rendered image"; "atomics are needed to accumulate gradients in the backward
 * pass"; "per-pixel/tile intersection records").  The paper states no formula and
 * defers to its reference [10]; the mathematics is written out in SURVEY.md
 * section 8(c) (steps O-P1, O-B, O-R1, O-R2, O-P5) and restated in DESIGN.md.
 *
 * Conventions (all entry points)
 *   - Every pointer is a DEVICE pointer owned by the caller unless its comment says "host".
 *     The library never allocates or frees device memory and keeps no global state (one exception, stated at its
 *     declaration: gs_sort_pairs_static keeps its scratch in a static device array that every call on a device shares).
 *   - Arrays are dense, row-major, fp32 unless stated; counts are int64_t.
 *   - Calls are asynchronous on `stream` (a cudaStream_t passed as void*; NULL = default
 *     stream).  The only host synchronisation is in gs_bin_tiles when `M_out` is non-NULL.
 *   - Views of one call share width, height and the tile size; a "batch" is C >= 1 views.
 *     Per-(view, Gaussian) arrays are laid out [C, N, *]; entry e = c*N + i.
 *   - Return value: GS_OK (0) or a negative gs_status.  No exception crosses the ABI.
 *   - Culled (view, Gaussian) entries have radii == 0 and tiles_touched == 0; their other
 *     per-view fields are unspecified and are never read by later stages.
 */
#ifndef GSPLAT_B200_H_
#define GSPLAT_B200_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define GS_MAX_VIEWS 64 /* upper bound on C per call */

/* Visibility mask (optional fast path for scenes in which a small fraction of the C*N entries is visible).
 * uint32 words [C][GS_VIS_WORDS(N)], 16-byte aligned; bit (i & 31) of word c*GS_VIS_WORDS(N) + (i >> 5) is 1 iff entry
 * (view c, Gaussian i) is visible (radius > 0 and >= 1 tile); bits of i >= N are 0.  gs_project_fwd writes it; gs_bin_tiles,
 * gs_raster_bwd, gs_project_bwd and gs_adam_step_visible read it instead of scanning the dense radii[C,N]. */
#define GS_VIS_WORDS(N) ((((int64_t)(N) + 511) / 512) * 16)

typedef enum gs_status {
    GS_OK = 0,
    GS_ERR_INVALID_ARGUMENT = -1, /* null / misaligned pointer, N < 0, C out of range, bad config, views differ in size */
    GS_ERR_CAPACITY = -2,         /* gs_bin_tiles: capacity_M too small; needed M is in *M_out */
    GS_ERR_CUDA = -3,             /* a CUDA runtime call or launch failed (cudaGetLastError) */
    GS_ERR_UNSUPPORTED = -4       /* tile != 16, C*N >= 2^31, M >= 2^30 */
} gs_status;

/* Pinhole camera (host struct).  Pixel (row i, col j) samples the image plane at (j+0.5, i+0.5).
 * viewmat = world->camera [W | tau], row-major 3x4; camera axes +x right, +y down, +z forward
 * (SURVEY.md 8(c) reading A3). */
typedef struct gs_camera {
    int32_t width, height;
    float fx, fy, cx, cy;
    float viewmat[12];
    float near_plane, far_plane; /* cull t_z <= near or t_z >= far (reading A4) */
} gs_camera;

/* Constants of the method (host struct); gs_config_default fills the 3DGS values:
 * dilation 0.3, alpha_min 1/255, alpha_max 0.99, t_min 1e-4, extent 3, tile 16, sh_degree 3
 * (readings A6, A7, A11). */
typedef struct gs_config {
    float dilation, alpha_min, alpha_max, t_min, extent;
    int32_t tile;      /* only 16 is supported */
    int32_t sh_degree; /* 0..3; K = (sh_degree+1)^2 bases */
} gs_config;

int gs_config_default(gs_config* cfg /*host, out*/);
const char* gs_status_string(int status);

/* P1 -- per-Gaussian forward.
 * exp(log-scale), normalised quaternion (w,x,y,z) -> Sigma = R S S^T R^T; t = W p + tau; near/far
 * cull; EWA Jacobian with the 1.3x field-of-view clamp -> 2-D covariance + dilation -> conic and
 * det cull; radius = ceil(extent*sqrt(lambda_max)); mean2d, depth; fp32 tile rectangle and
 * tiles_touched; SH colour (+0.5, clamp >= 0) along the camera->Gaussian direction; sigmoid opacity.
 * in : means[N,3] log_scales[N,3] quats[N,4] opacity_logits[N] sh[N,K,3]; cams: host array of C.
 * out: means2d[C,N,2] depths[C,N] conics[C,N,3] (A,B,C) opacities[C,N] rgbs[C,N,3]
 *      radii[C,N] (int32, 0 = culled) tiles_touched[C,N] (uint32).
 * vis_mask (optional, out): when given, visibility is reported through the mask (see GS_VIS_WORDS) and radii /
 *   tiles_touched are written ONLY for visible entries -- the 8*C*N-byte dense zero-fill is skipped and the radii of culled
 *   entries keep whatever the caller's buffer held; every later stage must then be given the same mask.
 * log_scale_bound (optional, device scalar): an upper bound of every log-scale (gs_log_scale_bound computes it,
 *   gs_adam_step* can keep it up to date).  With it, a Gaussian whose largest possible 3-sigma radius cannot reach the
 *   image of a view is dropped while the means are streamed, before its own scales are read.  It never changes a result
 *   as long as it is a true upper bound (a NaN bound disables the test). */
int gs_project_fwd(const gs_config* cfg /*host*/, int64_t N, const float* means, const float* log_scales,
                   const float* quats, const float* opacity_logits, const float* sh, int32_t C,
                   const gs_camera* cams /*host*/, float* means2d, float* depths, float* conics,
                   float* opacities, float* rgbs, int32_t* radii, uint32_t* tiles_touched, uint32_t* vis_mask /*optional*/,
                   const float* log_scale_bound /*optional*/, void* stream);

/* bound[0] (device float) = max over the 3 N log-scales (N >= 1; NaNs are ignored).  Asynchronous on `stream`. */
int gs_log_scale_bound(int64_t N, const float* log_scales, float* bound, void* stream);

/* B1..B4 -- tile binning for a batch of views.
 * For every entry e = c*N + i with radii[e] > 0, in ascending e, one record per overlapped 16x16
 * tile (tile rectangle recomputed in fp32 from means2d and radii exactly as in P1 step 8):
 *   key = (uint64)(c*tiles + ty*Gx + tx) << 32 | bit pattern of depths[e],  value = e.
 * Records are put in stable key order (equal keys keep ascending e), and tile_ranges[t] =
 * [first, last+1) of the records whose key >> 32 == t ([0,0) when none), t in [0, C*tiles).
 * The order is produced by two stable radix sorts (depth bits on the visible entries, then the
 * tile id on the records), which is the same order as one stable sort on the 64-bit key.
 * workspace == NULL: only *workspace_bytes (host) is written (size query for N, C, capacity_M).
 * capacity_M: number of records isect_keys / isect_vals can hold.
 * M_dev (device, optional): receives the total record count M.
 * M_out (host, optional): if non-NULL the call synchronises `stream`, writes M, and returns
 *   GS_ERR_CAPACITY when M > capacity_M (outputs are then incomplete but nothing is written
 *   out of bounds).  With M_out == NULL the call never synchronises; overflow is reported only
 *   through M_dev.
 * isect_keys[capacity_M] (uint64, optional: NULL = the sorted keys are not materialised; the
 * rasteriser reads only values and ranges), isect_vals[capacity_M] (int32),
 * tile_ranges[C*tiles,2] (int64).  depths must be positive (they are: depth > near > 0).
 * vis_mask (optional): the mask gs_project_fwd wrote; the visible entries are then exactly its set bits (radii is read
 *   only for those) and no pass over the dense radii is made.
 * tile_sort: how the records are brought into tile order (same result bit for bit, GS_TILE_SORT_AUTO chooses by size):
 *   ONE_LEVEL = stable radix sort of the M (tile, entry) records on the tile id; GROUPS_4 / GROUPS_8 = the records that are
 *   generated and sorted are (group of 4x4 / 8x8 tiles, entry), 2..10 per visible entry instead of 19..80, and every group
 *   then expands its depth-ordered list into the lists of its tiles, one ballot per (tile, 32 entries), writing each record
 *   straight to its final place (GS_ERR_UNSUPPORTED beyond 8192 groups per batch). */
#define GS_TILE_SORT_AUTO 0
#define GS_TILE_SORT_ONE_LEVEL 1
#define GS_TILE_SORT_GROUPS_4 2
#define GS_TILE_SORT_GROUPS_8 3
int gs_bin_tiles(const gs_config* cfg /*host*/, int64_t N, int32_t C, const gs_camera* cams /*host*/,
                 const float* means2d, const float* depths, const int32_t* radii, const uint32_t* vis_mask /*optional*/, void* workspace,
                 size_t* workspace_bytes /*host*/, int64_t capacity_M, uint64_t* isect_keys,
                 int32_t* isect_vals, int64_t* tile_ranges, int64_t* M_dev, int64_t* M_out /*host*/,
                 int32_t tile_sort, void* stream);

/* Stand-alone stable LSD radix sort used by gs_bin_tiles (step B3), exported for testing and
 * measurement: sorts n (key, value) pairs on key bits [0, end_bit) -- bit 31 is skipped when
 * skip_bit31 != 0 (positive fp32 depth patterns).  keys/vals are overwritten with the result;
 * workspace as in gs_bin_tiles (NULL -> size query). */
int gs_sort_pairs(int64_t n, int32_t end_bit, int32_t skip_bit31, uint64_t* keys, int32_t* vals, void* workspace,
                  size_t* workspace_bytes /*host*/, void* stream);

/* gs_sort_pairs for callers that cannot allocate (stream capture into a CUDA graph, serving loops, harnesses that forbid
 * cudaMalloc): the same sort -- same kernels, same result bit for bit -- with NO workspace argument.  The scratch (pass
 * tickets, digit histograms, look-back status words, the ping-pong copy of keys and values) lives in one file-scope
 * `static __device__` array inside the library, sized for n <= GS_SORT_STATIC_MAX_N pairs (13.1 MB; every GPU that loads
 * the library holds it until the process exits).  The call allocates nothing: no cudaMalloc / cudaFree, no allocating
 * library routine; the caller passes only the inputs / outputs keys[n] (uint64, device) and vals[n] (int32, device), which
 * are overwritten with the result.  Asynchronous on `stream`.
 * The first call on a device (with that device current) resolves the array's device address once
 * (cudaGetSymbolAddress); make that call -- n == 0 is enough -- before stream capture starts.
 * Every call on a device shares the one array, which keeps the previous call's contents: the call itself clears what must
 * start at zero (tickets, histograms, status words), so calls in sequence on one stream need nothing from the caller, but
 * two calls that overlap on the GPU (different streams, or graphs launched concurrently) RACE on the scratch -- order them.
 * Errors: GS_ERR_UNSUPPORTED when n > GS_SORT_STATIC_MAX_N (nothing is launched; use gs_sort_pairs with a workspace) or the
 * bit range needs more than 8 passes; GS_ERR_INVALID_ARGUMENT (n < 0, end_bit outside [1, 64], null / misaligned pointers);
 * GS_ERR_CUDA. */
#define GS_SORT_STATIC_MAX_N (1 << 20)
int gs_sort_pairs_static(int64_t n, int32_t end_bit, int32_t skip_bit31, uint64_t* keys, int32_t* vals, void* stream);

/* R1 -- rasterisation forward.  Per pixel, front to back over
 * its tile's range: power = -1/2 d^T K d; skip power > 0; alpha = min(alpha_max, o*exp(power));
 * skip alpha < alpha_min; stop before T(1-alpha) < t_min; C += rgb*alpha*T.  image = C + T*bg.
 * out: image[C,H,W,3] final_T[C,H,W] n_contrib[C,H,W] (index+1 of the last composited record). */
int gs_raster_fwd(const gs_config* cfg /*host*/, int32_t C, const gs_camera* cams /*host*/,
                  const int32_t* isect_vals, const int64_t* tile_ranges, const float* means2d,
                  const float* conics, const float* opacities, const float* rgbs, const float* bg /*host[3]*/,
                  float* image, float* final_T, int32_t* n_contrib, void* stream);

/* R2 -- rasterisation backward.  Per pixel, back to front over
 * the first n_contrib records, recomputing alpha and recovering T by division; gradients are summed
 * per (view, Gaussian) entry with warp-shuffle + shared-memory reduction and device-scope atomics.
 * radii (optional): when given, only rows with radii > 0 are zero-filled before accumulation (rows of
 * culled entries are left untouched and are never read by gs_project_bwd); when NULL all C*N rows
 * are zero-filled.  N_total = C*N.  vis_mask (optional, takes precedence over radii): rows of its set bits are zero-filled.
 * out: dL_dmeans2d[C,N,2] dL_dconics[C,N,3] dL_dopacities[C,N] dL_drgbs[C,N,3]. */
int gs_raster_bwd(const gs_config* cfg /*host*/, int32_t C, const gs_camera* cams /*host*/, int64_t N_total,
                  const int32_t* isect_vals, const int64_t* tile_ranges, const float* means2d,
                  const float* conics, const float* opacities, const float* rgbs, const float* bg /*host[3]*/,
                  const float* final_T, const int32_t* n_contrib, const float* dL_dimage /*[C,H,W,3]*/,
                  const int32_t* radii /*optional*/, const uint32_t* vis_mask /*optional*/, float* dL_dmeans2d, float* dL_dconics,
                  float* dL_dopacities, float* dL_drgbs, void* stream);

/* Measurement aid (not a step of the hot path; bench.py calls it outside the timed region to count the work the method
 * itself does): replays the per-pixel decisions of O-R1 over the tile lists and writes
 *   stats[0] = (pixel, record) pairs composited,
 *   stats[1] = pairs the forward definition evaluates without compositing (rejected by a rule, or terminating the pixel),
 *   stats[2] = pairs the backward definition walks (list position <= n_contrib) without compositing,
 *   stats[3] = 256 x number of records (the dense bound).
 * stats: device uint64[4], overwritten.  Asynchronous on `stream`. */
int gs_raster_pair_stats(const gs_config* cfg /*host*/, int32_t C, const gs_camera* cams /*host*/,
                         const int32_t* isect_vals, const int64_t* tile_ranges, const float* means2d,
                         const float* conics, const float* opacities, uint64_t* stats, void* stream);

/* P5 -- per-Gaussian backward.  Chain rule through conic ->
 * 2-D covariance -> (J, Sigma) -> (mean, log-scale, quaternion), mean2d -> mean, rgb -> SH
 * coefficients and view direction -> mean, opacity -> logit; summed over the C views.  Gradients
 * are with respect to the RAW parameters (reading A1).
 * accumulate == 0: every row of every output is overwritten (zeros for Gaussians visible nowhere);
 * accumulate == 1: rows of Gaussians visible in >= 1 view are added to, other rows untouched;
 * accumulate == 2: rows of Gaussians visible in >= 1 view are OVERWRITTEN, other rows untouched (the visible-only
 *                  gradient that goes with gs_adam_step_visible; C <= 16, else GS_ERR_UNSUPPORTED).
 * Visibility comes from vis_mask when given (radii may then be NULL), else from radii > 0.
 * out: dL_dmeans[N,3] dL_dlog_scales[N,3] dL_dquats[N,4] dL_dopacity_logits[N] dL_dsh[N,K,3]. */
int gs_project_bwd(const gs_config* cfg /*host*/, int64_t N, const float* means, const float* log_scales,
                   const float* quats, const float* opacity_logits, const float* sh, int32_t C,
                   const gs_camera* cams /*host*/, const int32_t* radii, const uint32_t* vis_mask /*optional*/, const float* dL_dmeans2d,
                   const float* dL_dconics, const float* dL_dopacities, const float* dL_drgbs,
                   float* dL_dmeans, float* dL_dlog_scales, float* dL_dquats, float* dL_dopacity_logits,
                   float* dL_dsh, int32_t accumulate, void* stream);

/* The dense zero-fill of gs_project_bwd as a call of its own: zeroes all N rows of the five gradient arrays.
 * gs_grad_zero_fill followed by gs_project_bwd(accumulate = 1) gives exactly the result of gs_project_bwd(accumulate = 0).
 * It exists so that a caller can run the 236 N bytes of stores (SH degree 3) on a second stream while the rasterisation
 * kernels, which leave the HBM almost idle, run on the first (the paper's own remedy for memory stalls is to overlap,
 * PAPER.md:84).  Asynchronous on `stream`.  Errors: GS_ERR_INVALID_ARGUMENT, GS_ERR_CUDA. */
int gs_grad_zero_fill(int64_t N, int32_t sh_degree, float* dL_dmeans, float* dL_dlog_scales, float* dL_dquats,
                      float* dL_dopacity_logits, float* dL_dsh, void* stream);

/* Sparse clearing of the gradient arrays: zeroes the rows of every Gaussian that `vis_mask` (uint32 [C][GS_VIS_WORDS(N)],
 * the mask a gs_project_fwd call wrote) marks in at least one of its C views; all other rows are untouched.
 * Use: gradient arrays that persist from step to step hold non-zero rows only where the previous gs_project_bwd wrote
 * them.  gs_grad_zero_rows(mask of the PREVIOUS step) followed by gs_project_bwd(accumulate = 2, mask of this step) then
 * leaves exactly what gs_project_bwd(accumulate = 0) would: the dense gradient, zeros included, bit for bit -- for
 * 2 * 236 bytes per visible Gaussian instead of 236 bytes for every Gaussian (SH degree 3), provided the arrays were
 * zero-filled once (gs_grad_zero_fill) and nothing else writes to them in between.  Asynchronous on `stream`.
 * Errors: GS_ERR_INVALID_ARGUMENT (null / misaligned pointers, N < 0, sh_degree outside 0..3, C outside 1..GS_MAX_VIEWS),
 * GS_ERR_CUDA. */
int gs_grad_zero_rows(int64_t N, int32_t sh_degree, int32_t C, const uint32_t* vis_mask, float* dL_dmeans, float* dL_dlog_scales,
                      float* dL_dquats, float* dL_dopacity_logits, float* dL_dsh, void* stream);

/* Harness loss (SURVEY.md 8(c) reading A18): mean-reduced L1 against a target image.
 * dL_dimage[n] = sign(image - target) / n; *loss_sum (device, float, caller-zeroed) += sum |image - target| / n. */
int gs_l1_loss(int64_t n, const float* image, const float* target, float* dL_dimage, float* loss_sum, void* stream);

/* Fused L1 + SSIM image loss, forward and backward ("computes the loss", refs [31],
 * [20]):  L = (1 - lambda) mean|x - y| + lambda (1 - mean SSIM(x, y)), SSIM per channel with the 11 x 11 Gaussian window
 * (sigma 1.5, sum 1), zero padding (window not renormalised at the border), biased window variances, C1 = 0.01^2,
 * C2 = 0.03^2, means over all C * H * W * 3 values.
 * in : image, target [C, H, W, 3] fp32 (device), 0 <= lambda <= 1.
 * out: dL_dimage [C, H, W, 3] = dL/dimage (overwritten); *loss_sum (device, float, caller-zeroed) += L.
 * workspace (device, caller-owned): 3 * C * H * W * 3 floats; with workspace == NULL the call only writes the needed
 * size to *workspace_bytes.  Asynchronous on `stream`; no allocation, no host synchronisation.
 * Errors: GS_ERR_INVALID_ARGUMENT (null pointers, sizes < 1, lambda outside [0, 1], workspace too small), GS_ERR_CUDA. */
int gs_l1_ssim_loss(int32_t C, int32_t height, int32_t width, const float* image, const float* target, float lambda,
                    float* dL_dimage, float* loss_sum, void* workspace, size_t* workspace_bytes, void* stream);

/* 3-D Morton ordering of the Gaussian arrays ("sorted along a Morton curve").
 * Sequence: gs_bounds -> gs_morton_codes -> gs_sort_pairs(N, 63, 0, codes, index, ...) -> gs_gather_rows per array.
 * All pointers are device pointers; everything is asynchronous on `stream`; no allocation, no host synchronisation.
 *
 * gs_bounds: lo_hi[6] (device) = min x, y, z, max x, y, z of means[N,3] (N >= 1; NaNs order as their bit patterns).
 * gs_morton_codes: per Gaussian q_a = clamp(floor((p_a - lo_a) * (2^21 / (hi_a - lo_a))), 0, 2^21 - 1) in fp32 with one
 *   rounding per operation (scale 1 for a degenerate axis, q = 0 for a non-finite product); codes[i] = bits of
 *   (qx, qy, qz) interleaved, bit k of qx at 3k+2, qy at 3k+1, qz at 3k (63 bits); index[i] = i.  N < 2^31.
 * gs_gather_rows: dst[i, :] = src[perm[i], :] for rows of row_floats floats (src != dst; 16-byte accesses when
 *   row_floats % 4 == 0 and both pointers are 16-byte aligned).
 * Errors: GS_ERR_INVALID_ARGUMENT (null pointers, sizes out of range, src == dst), GS_ERR_CUDA. */
int gs_bounds(int64_t N, const float* means, float* lo_hi, void* stream);
int gs_morton_codes(int64_t N, const float* means, const float* lo_hi, uint64_t* codes, int32_t* index, void* stream);
int gs_gather_rows(int64_t N, int32_t row_floats, const float* src, const int32_t* perm, float* dst, void* stream);

/* Fused Adam step over one parameter array, in place:
 *   m <- beta1 m + (1 - beta1) g;  v <- beta2 v + (1 - beta2) g^2;
 *   p <- p - lr (m / (1 - beta1^step)) / (sqrt(v / (1 - beta2^step)) + eps)         (no weight decay, no amsgrad)
 * param, grad, m, v: [N, row_floats] fp32 (device); step >= 1.
 * radii == NULL: every element is updated (16-byte accesses when all four pointers are 16-byte aligned).
 * radii != NULL ([C, N] int32 as saved by gs_project_fwd): only the rows of Gaussians with radius > 0 in at least one
 * of the C views are updated; parameter and moments of every other row are left untouched.
 * running_max (optional, device float): *running_max = max(*running_max, every updated parameter value) -- pass the
 * log-scale bound of gs_project_fwd with the log_scales array so that it stays an upper bound while training.
 * Asynchronous on `stream`.  Errors: GS_ERR_INVALID_ARGUMENT, GS_ERR_CUDA. */
int gs_adam_step(int64_t N, int32_t row_floats, float* param, const float* grad, float* m, float* v, float lr, float beta1,
                 float beta2, float eps, int32_t step, const int32_t* radii, int32_t C, float* running_max /*optional*/, void* stream);

/* The visible-only Adam step over n_arrays (<= 8) parameter arrays in ONE launch: the radii [C, N] are scanned once.
 * row_floats, params, grads, ms, vs: HOST arrays of n_arrays entries (row sizes; device pointers to [N, row] arrays).
 * Same update and same row selection as gs_adam_step with radii != NULL.  vis_mask (optional, takes precedence over radii):
 * the rows are those of Gaussians with a set bit in any view.  running_max (optional): as in gs_adam_step, over the updated
 * values of array number max_array. */
int gs_adam_step_visible(int64_t N, int32_t n_arrays, const int32_t* row_floats, float* const* params, const float* const* grads,
                         float* const* ms, float* const* vs, float lr, float beta1, float beta2, float eps, int32_t step,
                         const int32_t* radii, const uint32_t* vis_mask /*optional*/, int32_t C, float* running_max /*optional*/,
                         int32_t max_array, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* GSPLAT_B200_H_ */
