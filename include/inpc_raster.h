/* inpc_raster.h -- C ABI of the B200-native differentiable bilinear point rasterizer.
 *
 * What it computes (INPC, arXiv 2403.16862; citations are lines of the paper text PAPER.md):
 *   RASTERIZE(C, P, A, F) -> I of Algorithm 1 (App. A.6): every point is projected
 *   with a pinhole camera (Eq. 6), splatted to the 2x2 nearest pixel centres with
 *   opacity alpha = alpha_h (1-|u-u_i|)(1-|v-v_i|) (Eq. 7), each pixel's fragments are
 *   ordered by depth ("blend all points in depth order"; ties by point index) and
 *   composited front to back, C = sum_i T_i alpha_i c_i, T_i = prod_{j<i}(1-alpha_j) (Eq. 1,
 *   PAPER.md:34), stopping once T < 1e-4 (BASELINE.json north_star; the paper has no cut-off).
 *   The backward pass returns gradients w.r.t. features, opacities and the projected
 *   screen position (u, v) of every point.  DESIGN.md section 3 lists every reading of the paper.
 *
 * Conventions
 *   - Pixel (i, j) has its centre at (i+0.5, j+0.5); +z forward, +y down; p_c = R p_w + t.
 *   - A point is kept iff near_z < z_c < far_z and u, v are finite; each of its four fragments is kept
 *     iff its pixel is inside [0,W)x[0,H).  Zero-weight / zero-opacity fragments are kept and counted.
 *   - The discrete quantities (cull, pixel, depth key) come from a fixed sequence of individually
 *     rounded fp32 operations (no FMA): x_c = ((R0 x + R1 y) + R2 z) + t0, ..., u = (fx x_c)/z_c + cx.
 *   - All arithmetic is fp32.  Images are [H][W][D] (pixel-interleaved), alpha is [H][W].
 *
 * Memory, ownership, streams
 *   - Every pointer is DEVICE memory owned by the caller unless marked "host".  The library allocates
 *     no device memory and keeps no state between calls, on the host or on the device (apart from one
 *     side stream, a few events and an occupancy figure per device, created on first use): scratch and the
 *     state saved for the backward pass (per-fragment transmittances, per-pixel blended counts and the
 *     blend order itself, 2 bytes per fragment) live in the caller's `workspace`, which starts with a small
 *     header (magic, shape, D, N, flags) the forward pass writes.  Later calls on a workspace
 *     (backward, get_*) are validated against THAT header, so a workspace may be copied, moved or
 *     freed by the caller at will; a workspace that holds no matching forward is never interpreted.
 *   - Device pointers must be 16-byte aligned; `workspace` must be 256-byte aligned (cudaMalloc and
 *     the PyTorch allocator return at least that).
 *   - Outputs and gradient buffers are OVERWRITTEN (not accumulated into).
 *   - All work is enqueued on `cuda_stream` (a cudaStream_t; NULL = the default stream).  Calls return
 *     without synchronising, except the inpc_raster_get_* introspection calls (they read back).
 *
 * Errors: every entry point returns INPC_OK (0) or a negative inpc_status; nothing aborts, throws or
 * prints.  There is no CPU fallback: without a CUDA device every compute call returns INPC_ERR_CUDA.
 * What only the device can know without a synchronisation -- whether the workspace handed to
 * inpc_raster_backward really holds the forward its arguments describe -- is checked by the first
 * kernel of that call: on a mismatch the backward kernels do nothing (the gradient buffers are left
 * untouched) and the reason is kept in the workspace header; inpc_raster_get_status returns it.
 */
#ifndef INPC_RASTER_H
#define INPC_RASTER_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct inpc_camera {
    float   fx, fy, cx, cy;  /* intrinsics, in pixels                                            */
    float   R[9], t[3];      /* world -> camera, row-major: p_c = R p_w + t                      */
    float   near_z, far_z;   /* kept iff near_z < z_c < far_z (paper: 0.01 / 100)  */
    int32_t width, height;
} inpc_camera;

typedef enum inpc_status {
    INPC_OK                      =  0,
    INPC_ERR_INVALID_ARG         = -1,  /* NULL / misaligned pointer, N < 0, W/H <= 0, near >= far, near < 0, N >= 2^30 */
    INPC_ERR_WORKSPACE_TOO_SMALL = -2,
    INPC_ERR_CUDA                = -3,  /* launch failure or sticky error; see inpc_raster_last_cuda_error   */
    INPC_ERR_NO_SAVED_STATE      = -4,  /* backward / get_* on a workspace no matching forward has filled (get_* return
                                           it at once; for backward it is reported by inpc_raster_get_status)  */
    INPC_ERR_UNSUPPORTED         = -5,  /* D not in {4, 8}, W or H > 4095                                     */
    INPC_ERR_STATIC_LIMIT        = -6   /* inpc_sample_view_static: n_leaves > inpc_sample_static_max_leaves()  */
} inpc_status;

/* flags of inpc_raster_forward / inpc_raster_workspace_bytes */
#define INPC_SAVE_FOR_BACKWARD 1u  /* keep what inpc_raster_backward needs in the workspace                 */
#define INPC_SAVE_SORTED       2u  /* also materialise every pixel's sorted fragment list (for get_sorted)  */
/* flags of the _ex / _levels / _multisample entry points only (NEXT row f3 of the scope table) */
#define INPC_OUT_PLANAR        4u  /* feature image (and its gradient) as [D][H][W] instead of [H][W][D]     */
#define INPC_ACCUMULATE        8u  /* forward: out += out_scale * result (out holds an earlier call's image) */
#define INPC_FUSED_SH         16u  /* workspace sizing for inpc_raster_forward_sh / _backward_sh (NEXT row f2)  */

typedef struct inpc_stats {          /* host struct filled by inpc_raster_get_stats                          */
    uint64_t n_points;               /* N of the last forward                                                 */
    uint64_t n_kept;                 /* points that survived the cull (= records binned)                      */
    uint64_t n_fragments;            /* emitted fragments = sum over pixels of count[p]                       */
    uint64_t n_tile_items;           /* screen-tile work items built for the blend kernel                     */
    uint64_t n_big_pixels;           /* pixels whose neighbourhood exceeds a tile, handled by the long-run path */
    uint64_t n_big_fragments;        /* fragments in those pixels                                             */
    uint64_t n_big_cells;            /* cells too large for the counting sort (bitonic-sorted, one CTA each)  */
} inpc_stats;

/* Upper bound (for 4N fragments) of the workspace needed for N points; 0 on invalid arguments. */
size_t inpc_raster_workspace_bytes(int64_t n_points, int32_t D, int32_t W, int32_t H, uint32_t flags);

/* Forward pass, Algorithm 1.
 *   pos[N][3], opacity[N] (in [0,1], not clamped), feat[N][D]; cam: host pointer, copied at call time.
 *   out_feat[H][W][D] = premultiplied composited features, out_alpha[H][W] = sum of blended T*alpha.
 *   N = 0 is valid (zero image).  `workspace_bytes` >= inpc_raster_workspace_bytes(N, D, W, H, flags). */
int inpc_raster_forward(const float* pos, const float* opacity, const float* feat, int64_t N, int32_t D,
                        const inpc_camera* cam, float* out_feat, float* out_alpha,
                        void* workspace, size_t workspace_bytes, uint32_t flags, void* cuda_stream);

/* Backward pass of L = <grad_out_feat, out_feat> + <grad_out_alpha, out_alpha>.
 *   Same pos / opacity / feat / N / D / cam and the workspace as left by a forward that had
 *   INPC_SAVE_FOR_BACKWARD set.  grad_out_alpha may be NULL (= 0).
 *   grad_feat[N][D], grad_opacity[N], grad_uv[N][2] = dL/d(u, v) in pixels.  Any of the three may be NULL: that
 *   gradient is then not written (its stores are skipped; the others are bit-identical to a call that asks for all).
 *   The same holds for every backward entry point below (grad_sh_coeff included).
 *   Culled points and fragments behind the cut-off get exactly 0. */
int inpc_raster_backward(const float* pos, const float* opacity, const float* feat, int64_t N, int32_t D,
                         const inpc_camera* cam,
                         const float* grad_out_feat, const float* grad_out_alpha,
                         float* grad_feat, float* grad_opacity, float* grad_uv,
                         void* workspace, size_t workspace_bytes, void* cuda_stream);

/* ---- NEXT row f3: the paper's real call pattern -- several resolution levels per call, several point clouds
 * averaged per pixel, [D][H][W] output (PAPER.md:100 "multisampling"; :126, :372 "multiple resolutions of feature
 * maps ... multiple instances of our rasterization module for each resolution level"; :130 CNN input). ----------
 *
 * inpc_raster_forward_ex = inpc_raster_forward plus
 *   flags INPC_OUT_PLANAR : out_feat is [D][H][W];
 *   flags INPC_ACCUMULATE : out_feat / out_alpha already hold an image and the new one is ADDED to it;
 *   out_scale             : factor on the image and on alpha (1/S for the average of S clouds).
 *   With flags <= 3 and out_scale = 1 it is bit-identical to inpc_raster_forward.
 * inpc_raster_backward_ex: grad_out_feat read as [D][H][W] with INPC_OUT_PLANAR, both output gradients multiplied
 *   by grad_scale; blend_weight may be NULL. */
int inpc_raster_forward_ex(const float* pos, const float* opacity, const float* feat, int64_t N, int32_t D,
                           const inpc_camera* cam, float* out_feat, float* out_alpha,
                           void* workspace, size_t workspace_bytes, uint32_t flags, float out_scale, void* cuda_stream);
int inpc_raster_backward_ex(const float* pos, const float* opacity, const float* feat, int64_t N, int32_t D,
                            const inpc_camera* cam,
                            const float* grad_out_feat, const float* grad_out_alpha,
                            float* grad_feat, float* grad_opacity, float* grad_uv, float* blend_weight,
                            void* workspace, size_t workspace_bytes, uint32_t flags, float grad_scale, void* cuda_stream);

/* ---- NEXT row f2: spherical harmonics fused into the rasterizer. ------------------------
 * sh_coeff[N][36] replaces feat: the 4-D feature of a point is  f[d] = sum_{b<9} Y_b(dir) sh_coeff[4 b + d]  with
 * Y_0..Y_8 the real SH basis of degree <= 2 (Condon-Shortley phase; reading R18) of the unit direction
 * from the camera centre (-R^T t) to the point.  D is 4.  The workspace must be sized with
 * inpc_raster_workspace_bytes(N, 4, W, H, flags | INPC_FUSED_SH).  Other arguments as inpc_raster_forward_ex /
 * inpc_raster_backward_ex; grad_sh_coeff[N][36] = Y_b dL/df[d] (exact zeros for culled points).  No gradient is
 * propagated into the position through the direction. */
int inpc_raster_forward_sh(const float* pos, const float* opacity, const float* sh_coeff, int64_t N,
                           const inpc_camera* cam, float* out_feat, float* out_alpha,
                           void* workspace, size_t workspace_bytes, uint32_t flags, float out_scale, void* cuda_stream);
int inpc_raster_backward_sh(const float* pos, const float* opacity, const float* sh_coeff, int64_t N,
                            const inpc_camera* cam,
                            const float* grad_out_feat, const float* grad_out_alpha,
                            float* grad_sh_coeff, float* grad_opacity, float* grad_uv, float* blend_weight,
                            void* workspace, size_t workspace_bytes, uint32_t flags, float grad_scale, void* cuda_stream);

/* Camera of resolution level l (host only, no device work): the image is halved l times,
 *   width_l = ceil(width / 2^l), height_l = ceil(height / 2^l), fx, fy, cx, cy multiplied by 2^-l (exact in fp32),
 * so a point that projects to (u, v) at level 0 projects to (u, v) / 2^l: pixel centres stay at (i+0.5, j+0.5). */
int inpc_raster_level_camera(const inpc_camera* cam, int32_t level, inpc_camera* out);

/* One point cloud rasterised at n_levels (<= 8) resolution levels: level l uses inpc_raster_level_camera(cam, l),
 * out_feat[l] / out_alpha[l] / workspaces[l] / workspace_bytes[l] are HOST arrays of n_levels device pointers /
 * sizes (workspace l sized for the level-l image; each keeps its own state for a later backward with that level's
 * camera).  flags / out_scale as for inpc_raster_forward_ex. */
int inpc_raster_forward_levels(const float* pos, const float* opacity, const float* feat, int64_t N, int32_t D,
                               const inpc_camera* cam, int32_t n_levels, float* const* out_feat, float* const* out_alpha,
                               void* const* workspaces, const size_t* workspace_bytes, uint32_t flags, float out_scale,
                               void* cuda_stream);

/* Inference multisampling: n_clouds (<= 64) independently sampled point clouds (HOST arrays of device pointers and
 * of point counts) are each rasterised at n_levels levels and averaged per pixel, out[l] = (1/S) sum_s image_s[l],
 * in cloud order (so the result is bit-reproducible).  Forward only: ONE workspace, sized for the largest cloud at
 * level 0, is reused; flags may only hold INPC_OUT_PLANAR. */
int inpc_raster_forward_multisample(int32_t n_clouds, const float* const* pos, const float* const* opacity,
                                    const float* const* feat, const int64_t* N, int32_t D, const inpc_camera* cam,
                                    int32_t n_levels, float* const* out_feat, float* const* out_alpha, void* workspace,
                                    size_t workspace_bytes, uint32_t flags, void* cuda_stream);

/* The same backward pass with the per-point BLENDING WEIGHT fused in (NEXT row f1 of the scope table):
 *   blend_weight[N] = max over the point's blended fragments of alpha_c T_c, alpha_c = opacity w_c (Eq. 7) and
 *   T_c the transmittance in front of that fragment (Eq. 1) -- "the transmitted blending weight b_j = alpha_j T_j"
 *   that the probability update p_i' = max(lambda_u p_i, max{b_0..b_n}) of the octree consumes (Eq. 3,
 *   PAPER.md:75-78; "the blending weight computation required for updating P [is] fused into this pipeline",
 *   PAPER.md:370).  Culled points and points none of whose fragments was blended get exactly 0.  The max over
 *   the points of a leaf (Eq. 3's outer max) is the sampler's business, not the rasterizer's.
 *   It costs one extra coalesced 4-byte store per point: the four T_c a_c are already formed for grad_feat. */
int inpc_raster_backward_weights(const float* pos, const float* opacity, const float* feat, int64_t N, int32_t D,
                                 const inpc_camera* cam,
                                 const float* grad_out_feat, const float* grad_out_alpha,
                                 float* grad_feat, float* grad_opacity, float* grad_uv, float* blend_weight,
                                 void* workspace, size_t workspace_bytes, void* cuda_stream);

/* Sticky status of the device-side checks since the last forward on this workspace (synchronises):
 * INPC_OK, or why the last inpc_raster_backward refused to run (INPC_ERR_NO_SAVED_STATE: no forward
 * with INPC_SAVE_FOR_BACKWARD has filled this workspace; INPC_ERR_INVALID_ARG: N, D, W or H differ from
 * that forward's). */
int inpc_raster_get_status(const void* workspace, void* cuda_stream);

/* Parity introspection.  All of these read the workspace of the last forward on it, take its shape from
 * the workspace header (W, H must match it) and synchronise the stream.
 * counts[H*W] = per-pixel fragment counts (step a2 of the path). */
int inpc_raster_get_counts(const void* workspace, int32_t W, int32_t H, uint32_t* counts, void* cuda_stream);

/* blended[H*W] = how many of a pixel's fragments the forward pass composited before the cut-off
 * (step a4; needs a forward with INPC_SAVE_FOR_BACKWARD). */
int inpc_raster_get_blended_counts(const void* workspace, int32_t W, int32_t H, uint32_t* blended, void* cuda_stream);

/* Needs a forward with INPC_SAVE_SORTED.  *total (host) = number of fragments.
 * With offsets == NULL only *total is returned.  Otherwise offsets[H*W+1] = exclusive sum of counts,
 * point_idx[total] / depth_bits[total] = every pixel's fragments in blend order (pixel-major), and, when
 * `transmittance` is not NULL, transmittance[total] = the fp32 transmittance T_k the kernel had in front of
 * each blended fragment (the value its cut-off test saw), -1 for fragments behind the cut-off. */
int inpc_raster_get_sorted(const void* workspace, int32_t W, int32_t H, uint32_t* offsets,
                           uint32_t* point_idx, uint32_t* depth_bits, float* transmittance, uint64_t* total,
                           void* cuda_stream);

/* Fills *stats (host) from the workspace of the last forward; synchronises the stream. */
int inpc_raster_get_stats(const void* workspace, inpc_stats* stats, void* cuda_stream);

/* ---- NEXT row f4: view-specific sampling of the implicit point cloud, the rasterizer's upstream neighbour
 * (Sec. 3.2, Eq. 4; depth Eq. 9; frustum re-sampling PAPER.md:322). -------------
 * Leaves of the probability octree: leaf_centre[L][3] (world), leaf_level[L] (side = root_side / 2^level),
 * leaf_prob[L] in [0,1]; L <= 2^24 (the paper's 256^3 cap).  Each leaf gets the weight
 *   p^ = visible * p / (d * 2^(level * 0.5)),   d = max(|z_view - near| / (far - near), 1e-8)
 * (visible: the leaf's cube can intersect the view frustum -- its centre or a corner is inside, or no frustum plane
 * has all eight corners outside; reading R19; a leaf_level outside [0, 30] gets p^ = 0), N leaves are drawn with replacement
 * from p^ / sum p^ (inverse CDF), each draw is offset uniformly inside its leaf, and a position outside the
 * frustum is drawn again (up to 8 times; then pos = NaN, leaf = -1: the rasterizer culls it).
 * pos[N][3] and leaf[N] are outputs; the result is a pure function of the inputs and `seed` (counter-based
 * SplitMix64, integer CDF; csrc/sampler.cuh states the exact arithmetic), bit-reproducible on any device.
 * workspace: inpc_sample_workspace_bytes(L) bytes, 256-byte aligned.  inpc_sample_get_stats synchronises and
 * returns how many samples are valid, the integer CDF total and max p^ of the last call on that workspace. */
size_t inpc_sample_workspace_bytes(int64_t n_leaves);
int inpc_sample_view(const float* leaf_centre, const int32_t* leaf_level, const float* leaf_prob, int64_t n_leaves,
                     float root_side, const inpc_camera* cam, uint64_t seed, int64_t N, float* pos, int32_t* leaf,
                     void* workspace, size_t workspace_bytes, void* cuda_stream);
int inpc_sample_get_stats(const void* workspace, uint64_t* n_valid, uint64_t* cdf_total, double* max_weight,
                          void* cuda_stream);
/* inpc_sample_view with flags.  INPC_SAMPLE_NO_RESAMPLE: the inference mode of PAPER.md:322 ("During inference, we use
 * multisampled point clouds and can therefore omit resampling, which also boosts performance"): every sample is drawn
 * ONCE; a position outside the frustum is returned as NaN / leaf -1 and culled by the rasterizer.  The random counters
 * are those of the first attempt of inpc_sample_view, so a sample whose first draw is inside the frustum is the same
 * bits in both modes.  flags = 0 is inpc_sample_view. */
#define INPC_SAMPLE_NO_RESAMPLE 1u
int inpc_sample_view_ex(const float* leaf_centre, const int32_t* leaf_level, const float* leaf_prob, int64_t n_leaves,
                        float root_side, const inpc_camera* cam, uint64_t seed, int64_t N, float* pos, int32_t* leaf,
                        void* workspace, size_t workspace_bytes, uint32_t flags, void* cuda_stream);

/* ---- The sampler for callers that cannot allocate device memory. ---------------------------------------------
 * inpc_sample_view needs a workspace, and somebody has to cudaMalloc it.  Not every caller can: a plugin inside a
 * host application whose allocator owns the whole GPU, a frame loop that must never hit cudaMalloc's device-wide
 * synchronisation, a process that is already at its memory budget.  inpc_sample_view_static is the same sampler
 * (same kernels, same checks, bit-identical pos / leaf) with its scratch in a fixed array that is part of the
 * library image, so the call itself and everything under it allocates and frees nothing.
 *   Limit:  n_leaves <= inpc_sample_static_max_leaves() = 262,144 (2^18).  More returns INPC_ERR_STATIC_LIMIT
 *           and enqueues nothing; use inpc_sample_view with a workspace of your own then.
 *   Cost:   the array is 4,458,240 bytes (16 per leaf + 258 KB) of every GPU that loads this library, from module
 *           load to process exit, used or not.
 *   Set-up: the first call on each device looks up that device's address of the array (cudaGetSymbolAddress, with
 *           that device current; no allocation, but it may make the runtime load the module).  Make that first
 *           call outside any stream capture.  Later calls on the device do no set-up.
 *   Sharing: there is ONE array per device and every call on that device uses it.  The call clears the words
 *           that must start at zero and overwrites the rest before reading it, so leftovers of the previous call are
 *           harmless -- but two calls that are in flight on the GPU at the same time (different streams, or
 *           different host threads on different streams) write over each other and both results are garbage.
 *           Calls on one stream are ordered and safe.  The statistics of inpc_sample_get_stats are not available.
 * pos[N][3], leaf[N] and the leaf arrays are the caller's device buffers exactly as for inpc_sample_view. */
int64_t inpc_sample_static_max_leaves(void);
int inpc_sample_view_static(const float* leaf_centre, const int32_t* leaf_level, const float* leaf_prob, int64_t n_leaves,
                            float root_side, const inpc_camera* cam, uint64_t seed, int64_t N, float* pos, int32_t* leaf,
                            void* cuda_stream);

const char* inpc_raster_strerror(int status);
/* CUDA error string of the last INPC_ERR_CUDA on this thread ("" if none). */
const char* inpc_raster_last_cuda_error(void);
/* Number of kernels this library has launched so far in this process (all entry points). */
uint64_t inpc_raster_launch_count(void);
/* Diagnostics: the distinct kernel template instantiations this process has launched since the last reset,
 * as a ';'-separated, sorted list ("k_back<4>;k_blend<4,0>;..."; k_blend<D,DUMP>, k_big<D,MODE> with MODE 0 =
 * forward, 1 = forward + INPC_SAVE_SORTED dump, 2 = backward) written to the HOST buffer `buf` (truncated to
 * buf_bytes, always NUL-terminated; buf may be NULL).  Returns the bytes needed for the whole list. */
size_t inpc_raster_launched_kernels(char* buf, size_t buf_bytes, int reset);

/* Profiling aid (bench.py's roofline).  With timing enabled every stage the library enqueues is
 * bracketed by two cudaEvents on the caller's stream (a few microseconds per stage; off by default).
 * inpc_raster_get_kernel_times waits for the recorded events and returns, per stage i in
 * [0, inpc_raster_kernel_count()), the summed device time ms[i] (milliseconds) and the number of
 * timed launches since the last reset; ms / launches are HOST arrays of that length. */
int         inpc_raster_set_kernel_timing(int enable);
int         inpc_raster_kernel_count(void);
const char* inpc_raster_kernel_name(int i);
int         inpc_raster_get_kernel_times(double* ms, uint64_t* launches, int reset);

#ifdef __cplusplus
}
#endif
#endif /* INPC_RASTER_H */
