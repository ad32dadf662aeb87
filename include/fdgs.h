/* fdgs.h — C ABI of the B200-native time-sliced tile rasterizer for native 4D Gaussians.
 *
 * Method: "4D Gaussian Splatting: Modeling Dynamic Scenes with Native 4D Primitives"
 * (arxiv 2412.20720).  Citations below are PAPER.md:L<line> of the extracted paper text.
 *
 * Everything behind these entry points is hand-written CUDA for sm_100a (no CPU fallback, no
 * library kernels).  The library never allocates device memory, never throws across the ABI and
 * never synchronises the stream unless a `_host` out-pointer is given.  fdgs_preprocess / fdgs_render_forward(_aux) /
 * fdgs_l1_loss / fdgs_render_backward(_aux) issue only kernels and device memsets on the caller's stream, so the sequence
 * can be captured into a CUDA graph.  The library keeps a little process-global state (atomic launch counter, timing
 * events, and per CUDA device the worker streams of fdgs_step_batch / fdgs_step_host, created under a mutex): the step
 * calls of ONE device are not re-entrant across host threads, everything else is.
 *
 * Conventions
 *   - Every pointer is a DEVICE pointer unless its name ends in `_host`.  fdgs_view and
 *     fdgs_config are small HOST structs passed by pointer and copied into kernel parameters.
 *   - All arrays are contiguous fp32 unless stated; base pointers must be 16-byte aligned.
 *   - The caller owns every buffer, including the workspace `ws` (e.g. a torch uint8 tensor),
 *     which is the only state carried between calls.  Call order on one `ws` and one stream:
 *         fdgs_preprocess -> fdgs_render_forward -> fdgs_render_backward
 *     with the same scene, view, config and pair_capacity (they define the workspace layout).
 *   - Return value: 0 = OK, <0 = error (fdgs_strerror).
 */
#ifndef FDGS_H
#define FDGS_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define FDGS_OK 0
#define FDGS_ERR_INVALID (-1)       /* NULL / misaligned pointer, N<0, sh_degree not in 0..3, n_time<1, W/H<=0 ... */
#define FDGS_ERR_WORKSPACE (-2)     /* ws_bytes smaller than fdgs_workspace_bytes() says                            */
#define FDGS_ERR_CUDA (-3)          /* CUDA runtime error (text via fdgs_strerror)                                  */
#define FDGS_ERR_PAIR_OVERFLOW (-4) /* number of (tile, primitive) pairs D exceeded pair_capacity                   */
#define FDGS_ERR_STATIC_LIMIT (-5)  /* fdgs_render_forward_static: the sizes need more than FDGS_STATIC_WS_BYTES       */

#define FDGS_TILE 16 /* 16x16-pixel tiles (tile rasterizer of [23]) */

/* A scene = N 4D Gaussians.  K = n_time * (sh_degree+1)^2. */
typedef struct {
  int32_t N;                  /* number of primitives, >= 0                                             */
  int32_t sh_degree;          /* spatial SH degree L in 0..3                                            */
  int32_t n_time;             /* Fourier orders n = 0..n_time-1 of the 4DSH (eq. 20), 1..8         */
  const float *mean;          /* [N,4]  (mu_x, mu_y, mu_z, mu_t)                               L135     */
  const float *log_scale;     /* [N,4]  S = diag(exp(.)), order (x,y,z,t)                      L128     */
  const float *quat_l;        /* [N,4]  q_l = (a,b,c,d), need not be unit (normalised inside)  L128     */
  const float *quat_r;        /* [N,4]  q_r = (p,q,r,s)                                        L128     */
  const float *opacity_logit; /* [N]    alpha = sigmoid(.)                                              */
  const float *sh;            /* [N,K,3] 4DSH coefficients, k = n*(L+1)^2 + l*l + l + m, channel last   */
} fdgs_scene;

/* One view: extrinsic E = [W | tau] and intrinsic K, query time t, 4DSH period T. */
typedef struct {
  float view[16];       /* world -> camera, row-major 4x4 [W tau; 0 0 0 1], +z forward             */
  float fx, fy, cx, cy; /* pinhole intrinsics in pixels; pixel (i,j) is sampled at (i+0.5, j+0.5)  */
  int32_t width, height;
  float t;              /* query time                                                    L108-L113 */
  float period_T;       /* period T of cos(2 pi n (t - mu_t) / T)                        L187      */
  float bg[3];          /* background colour composited with the final transmittance               */
} fdgs_view;

/* Thresholds.  Only marginal_min is the paper's (L324); the rest are the settings of [23] that the
 * paper adopts without stating (L324) — see DESIGN.md readings S7-S10. */
typedef struct {
  float marginal_min;      /* 0.05: cull if exp(-(t-mu_t)^2 / (2 Sigma_44)) < marginal_min; 0 disables (L265) */
  float alpha_min;         /* 1/255: a splat with alpha < alpha_min is skipped at that pixel                  */
  float alpha_max;         /* 0.99:  alpha is clamped to alpha_max                                            */
  float transmittance_min; /* 1e-4:  stop before the splat that would take T below this                       */
  float dilation;          /* 0.3 px^2 added to the diagonal of Sigma_2d                                      */
  float cutoff_sigma;      /* 3.0:   support radius = cutoff_sigma * sqrt(lambda_max(Sigma_2d))               */
  float znear;             /* 0.2:   cull if camera-space depth <= znear                                      */
  float guard;             /* 1.3:   guard band for the clamped ratios inside the Jacobian J                  */
} fdgs_config;

/* Gradient buffers, same shapes as the fdgs_scene arrays.  fdgs_render_backward ACCUMULATES (+=)
 * into them: zero them once per optimisation step and the views of a batch sum (L324 "batch size 4"). */
typedef struct {
  float *mean, *log_scale, *quat_l, *quat_r, *opacity_logit, *sh;
  float *mean2d;  /* [N,2] optional (NULL ok): dL/d(u,v) in pixels, summed over views (L197)                          */
  float *densify; /* [N,3] optional (NULL ok): density-control indicators, accumulated once per backward of a view the
                     primitive is visible in (L197 "gradients of mu_t as an additional density control indicator"):
                     [0] += |dL/d(u,v)| of this view, [1] += |dL/dmu_t| of this view, [2] += 1                          */
} fdgs_grads;

/* Fills the defaults listed above.  Returns FDGS_ERR_INVALID if cfg is NULL. */
int fdgs_default_config(fdgs_config *cfg_host);

/* Size of the workspace for a scene of N primitives with K coefficients per channel rendered at
 * W x H with room for pair_capacity (tile, primitive) pairs (1 <= pair_capacity < 2^30).  W x H is limited to
 * (ceil(W/16)+1)*(ceil(H/16)+1) <= 50000 tiles (e.g. 3500 x 3500). */
int fdgs_workspace_bytes(int32_t N, int32_t K, int32_t W, int32_t H, int64_t pair_capacity, size_t *bytes_host);

/* Steps A1-A5: activation and 4D covariance Sigma = R S S^T R^T with R = L(q_l) R(q_r)
 * (eq. 7-8); time slice mu_xyz|t, Sigma_xyz|t and marginal weight (eq. 9-10)
 * with the p(t) < marginal_min filter (L324); EWA projection to a 2D conic (eq. 3-4);
 * 4DSH colour (eq. 20); tiles touched and their exclusive prefix sum.
 * Scenes of sh_degree 3: the colour slots of the per-primitive records are filled in by the fdgs_render_forward(_aux) that
 * follows (on a library-owned side stream, next to its depth sort and tile lists: only the blend reads the colours), so
 * FDGS_EXPORT_RECORDS shows final colours after that call, not after this one.
 * If num_pairs_host / num_visible_host are non-NULL the stream is synchronised and D / the number
 * of surviving primitives are returned (and FDGS_ERR_PAIR_OVERFLOW if D > pair_capacity). */
int fdgs_preprocess(const fdgs_scene *scene, const fdgs_view *view_host, const fdgs_config *cfg_host, void *ws,
                    size_t ws_bytes, int64_t pair_capacity, void *cuda_stream, int64_t *num_pairs_host,
                    int32_t *num_visible_host);

/* Steps A6-A9: order the (tile, primitive) pairs as a stable sort on the key (tile id << 32 | fp32
 * depth bits) with ties in primitive-id order would (done two-level: survivors sorted by depth, then every pair
 * written straight to its place in its tile's list — DESIGN.md), per-tile ranges, front-to-back alpha compositing of
 * p_i(t) p_i(u,v|t) alpha_i c_i (eq. 6).  Outputs: image [3,H,W], final_T [H,W] (transmittance
 * left), n_contrib [H,W] (1 + position in the tile list of the last splat composited).
 * If D exceeded pair_capacity nothing is drawn (image = bg) and the overflow is reported by
 * fdgs_debug_export(FDGS_EXPORT_STATUS) or the next synchronising call.
 * Each call consumes the tickets and look-back state that fdgs_preprocess prepared on `ws`: one forward per preprocess.
 * For sh_degree 3 the call forks the colour evaluation (A4) onto a library-owned stream and joins it back into
 * `cuda_stream` before the blend; fork and join both happen inside the call, so it can be captured into a CUDA graph. */
int fdgs_render_forward(const fdgs_scene *scene, const fdgs_view *view_host, const fdgs_config *cfg_host, void *ws,
                        size_t ws_bytes, int64_t pair_capacity, void *cuda_stream, float *image, float *final_T,
                        uint32_t *n_contrib);

/* Steps B1-B2: reverse-order gradient of the compositing, then the chain through projection, 4DSH,
 * conditioning, Sigma = M M^T and the two quaternions to every parameter (exact derivative of the
 * forward as stated; zero through active clamps).  Accumulates into grads. */
int fdgs_render_backward(const fdgs_scene *scene, const fdgs_view *view_host, const fdgs_config *cfg_host, void *ws,
                         size_t ws_bytes, int64_t pair_capacity, void *cuda_stream, const float *dL_dimage,
                         const float *final_T, const uint32_t *n_contrib, const fdgs_grads *grads_host);

/* Auxiliary channels through the same blend (eq. 25, L256 eq. 29; reading S18):
 *   accumulated opacity O_gs = sum_k alpha_k T_k = 1 - final_T          (already an output of fdgs_render_forward);
 *   rendered depth      D    = sum_k z_k alpha_k T_k, z_k = camera depth of the conditional mean, no background term.
 * fdgs_render_forward_aux = fdgs_render_forward + depth_map [H,W].
 * fdgs_render_backward_aux = fdgs_render_backward with two more upstream gradients, dL_ddepth [H,W] and dL_dopacity
 * [H,W] (= dL/dO_gs); either may be NULL.  Exact derivative of the forward as stated, accumulated into grads. */
int fdgs_render_forward_aux(const fdgs_scene *scene, const fdgs_view *view_host, const fdgs_config *cfg_host, void *ws,
                            size_t ws_bytes, int64_t pair_capacity, void *cuda_stream, float *image, float *final_T,
                            uint32_t *n_contrib, float *depth_map);
int fdgs_render_backward_aux(const fdgs_scene *scene, const fdgs_view *view_host, const fdgs_config *cfg_host, void *ws,
                             size_t ws_bytes, int64_t pair_capacity, void *cuda_stream, const float *dL_dimage,
                             const float *dL_ddepth, const float *dL_dopacity, const float *final_T,
                             const uint32_t *n_contrib, const fdgs_grads *grads_host);

/* Harness-side loss ("rendering loss"): L = mean |image - target| over 3HW values.
 * Writes dL/dimage [3,H,W] and adds L to *loss (device float, caller zeroes it). */
int fdgs_l1_loss(const float *image, const float *target, int64_t count, float *dL_dimage, float *loss,
                 void *cuda_stream);

/* One forward(+backward) pass over one view with HOST target / result buffers: copies target_host
 * [3,H,W] to `target_dev`, runs preprocess + forward (+ L1 loss + backward if grads_host != NULL),
 * copies the loss (1 float) — or, when grads_host == NULL, the image — back to the host and
 * synchronises the stream.  target_host / result_host should be pinned.  The host -> device copy of the target runs
 * on a library-owned copy stream, forked from and joined to `cuda_stream` by events, so it overlaps preprocess and
 * forward; `target_dev` must not be touched by other streams during the call.  Returns FDGS_ERR_PAIR_OVERFLOW if D
 * exceeded pair_capacity (the result is then the loss / image of an empty rendering). */
int fdgs_step_host(const fdgs_scene *scene, const fdgs_view *view_host, const fdgs_config *cfg_host, void *ws,
                   size_t ws_bytes, int64_t pair_capacity, void *cuda_stream, const float *target_host,
                   float *target_dev, float *image, float *final_T, uint32_t *n_contrib, float *dL_dimage,
                   float *loss_dev, fdgs_grads *grads_host, float *result_host);

/* One optimisation step over a batch of views ("batch size 4", batch sampling in time): for every view
 * preprocess + forward + L1 loss against its target + backward, gradients of all views accumulated into `grads_host`
 * (+=; the caller zeroes them).  The views run on library-owned worker streams forked from and joined to `cuda_stream`
 * by events, each on its OWN workspace and buffers, so the latency-bound stages of one view (scans, sorts) overlap the
 * blend kernels of the others.  The second half of the backward (B2, the accumulation into the shared gradient arrays, a
 * non-atomic read-modify-write) follows when the blend backward of every view is done: with sh_degree 3, n_time <= 4 and
 * num_views <= 4 its colour part is ONE pass over the primitives for all views — the coefficient block of a primitive seen
 * by several views of the batch is read once and its gradient block read and written once (written only, under
 * FDGS_STEP_ZERO_GRADS) — followed by the geometry part view after view; otherwise B2 runs per view, chained.  The
 * accumulated result is the same as calling the three functions view by view, up to fp32 summation order.
 *   bufs_host[i].target_host  != NULL: [3,H,W] pinned host image, copied to target_dev inside the call;
 *                             == NULL: target_dev already holds the target.
 *   loss_dev [num_views] device floats: loss of each view (overwritten); NaN for a view whose pairs exceeded
 *                             pair_capacity (nothing drawn, zero gradients): the signal an asynchronous caller gets.
 *   loss_host != NULL: the losses are copied back, `cuda_stream` is synchronised and FDGS_ERR_PAIR_OVERFLOW is returned if
 *                             any view overflowed; NULL: fully asynchronous.
 * If an argument is rejected or a launch fails after work has been forked onto the worker streams, they are joined into
 * `cuda_stream` and it is synchronised before the error is returned: no kernel still runs on the caller's buffers.
 *   flags: FDGS_STEP_ZERO_GRADS = the six parameter-gradient arrays (and mean2d if given; not densify, which is meant to
 *          accumulate over steps) are zeroed inside the call, on a side stream, hidden under the forward passes.
 * 1 <= num_views <= FDGS_MAX_BATCH; workspaces must be distinct. */
#define FDGS_MAX_BATCH 8
#define FDGS_STEP_ZERO_GRADS 1
typedef struct {
  void *ws; size_t ws_bytes;     /* workspace of this view (fdgs_workspace_bytes)                      */
  const float *target_host;      /* see above                                                          */
  float *target_dev;             /* [3,H,W]                                                            */
  float *image, *final_T;        /* [3,H,W], [H,W] outputs of the forward                              */
  uint32_t *n_contrib;           /* [H,W]                                                              */
  float *dL_dimage;              /* [3,H,W] scratch: dL/dimage of the L1 loss                          */
} fdgs_view_buffers;
int fdgs_step_batch(const fdgs_scene *scene, const fdgs_view *views_host, int32_t num_views, const fdgs_config *cfg_host,
                    int64_t pair_capacity, const fdgs_view_buffers *bufs_host, void *cuda_stream, float *loss_dev,
                    const fdgs_grads *grads_host, float *loss_host, int32_t flags);

/* Parity hooks: copy one intermediate of the last calls on `ws` to dst (device memory).  Synchronises. */
#define FDGS_EXPORT_STATUS 0        /* int64[4]: D, num_visible, overflow flag, pair_capacity               */
#define FDGS_EXPORT_RECORDS 1       /* float[N,12]: u, v, conic A, B, C, opacity o, r, g, b, depth, radius, w */
#define FDGS_EXPORT_RECTS 2         /* int32[N,4]: tx0, ty0, tx1, ty1 (all 0 for culled primitives)          */
#define FDGS_EXPORT_TILES_TOUCHED 3 /* uint32[N]                                                             */
/* 4 was FDGS_EXPORT_OFFSETS (round 1: prefix sum of tiles_touched in depth order); the pair emission it served is gone */
#define FDGS_EXPORT_SORTED_KEYS 5   /* uint64[D]                                                             */
#define FDGS_EXPORT_SORTED_VALS 6   /* uint32[D] primitive ids                                               */
#define FDGS_EXPORT_RANGES 7        /* uint32[tiles,2]: [first, last+1) into the sorted arrays               */
#define FDGS_EXPORT_SPLAT_GRADS 8   /* float[N,9]: dL/d(u, v, A, B, C, o, r, g, b) from the last backward    */
#define FDGS_EXPORT_DEPTH_ORDER 9   /* uint32[num_visible]: ids of the survivors sorted by (depth bits, id)   */
#define FDGS_EXPORT_SPLAT_GRAD_DEPTH 10 /* float[N]: dL/d(camera depth) per splat from the last fdgs_render_backward_aux */
int fdgs_debug_export(const void *ws, size_t ws_bytes, int what, void *dst, size_t dst_bytes, void *cuda_stream);

/* Measurement hooks (bench.py).  fdgs_set_stage_timing(1) makes the three calls record CUDA events at
 * their stage boundaries; fdgs_get_stage_ms waits for them and fills ms_host[8]: preprocess kernel, compaction +
 * tile grid, depth sort, tile lists (row scatter), forward blend, backward blend, backward preprocess, and the colour
 * kernel that fdgs_render_forward runs on its side stream UNDER the depth sort and the row scatter (its time is not part
 * of the frame's critical path) (-1 for a stage that has not run).  fdgs_debug_blend_stats re-walks the tile lists of the last forward on `ws`
 * and writes uint64[4] to stats_dev: (pixel, splat) pairs walked, pairs reaching the exp2, pairs composited,
 * splats staged — the algorithmic work of the blend kernels. */
int fdgs_set_stage_timing(int enable);
int fdgs_get_stage_ms(float *ms_host);
int fdgs_debug_blend_stats(const fdgs_view *view_host, const fdgs_config *cfg_host, void *ws, size_t ws_bytes, int32_t N,
                           int32_t K, int64_t pair_capacity, void *cuda_stream, unsigned long long *stats_dev);

/* Cull decision of every primitive for this view, uint8[N]: 0 visible, 1 culled by the temporal marginal (L324),
 * 2 behind the near plane, 3 empty tile rectangle, 4 non-finite.  Recomputed from the parameters (does not touch a
 * workspace): parity of the cull reasons, and cfg5's "fraction culled by the marginal temporal weight". */
int fdgs_debug_cull_status(const fdgs_scene *scene, const fdgs_view *view_host, const fdgs_config *cfg_host, void *cuda_stream,
                           unsigned char *status_dev);

/* Measured pipe peaks of this GPU (the blend kernels' roofline denominators): FP32 FMA issue rate
 * in T lane-instructions/s (8 independent FFMA chains per thread, 8 CTAs of 256 threads per SM) and MUFU.EX2 rate in
 * T/s.  scratch_dev: >= 4 * 8 * 256 * (number of SMs) bytes.  Synchronises; takes a few ms. */
int fdgs_debug_measure_peaks(void *scratch_dev, size_t scratch_bytes, void *cuda_stream, float *fma_tlane_per_s_host,
                             float *mufu_t_per_s_host);

/* ------------------------------------------------------------------------------------------------------------------
 * Feature channels and rendered optical flow.
 * "The 2D feature F at a specific view could be rendered following the same process as in Section 3.2, with the color c
 * replaced by the normalized feature vector f":  F[c](pixel) = sum_k feat[k,c] alpha_k T_k over the same
 * per-tile depth-ordered lists, thresholds and termination as the colour image; no background term.
 * Call after fdgs_preprocess + fdgs_render_forward on the same ws / view / config (tile lists and records are reused).
 * Forward: a dedicated C-channel kernel, alpha evaluated once per 32 channels (ceil(C/32) launches), every skip and
 * termination decision bit-identical to the colour pass.  Backward with grads == NULL (geometry frozen, the setting of
 * L300): a dedicated front-to-back kernel, 32 channels per launch.  Backward with grads != NULL: the 3-channel backward
 * blend kernel three channels at a time (ceil(C/3) launches) on a copy of the records in `scratch`.
 * scratch: device buffer of fdgs_features_scratch_bytes(N, W, H) bytes, 16-byte aligned, caller-owned.
 * ------------------------------------------------------------------------------------------------------------------ */
int fdgs_features_scratch_bytes(int32_t N, int32_t W, int32_t H, size_t *bytes_host);

/* feat [N,C] device fp32 (C >= 1); out [C,H,W]. */
int fdgs_render_features_forward(const fdgs_scene *scene, const fdgs_view *view_host, const fdgs_config *cfg_host, void *ws,
                                 size_t ws_bytes, int64_t pair_capacity, void *cuda_stream, const float *feat, int32_t C,
                                 void *scratch, size_t scratch_bytes, float *out);

/* VJP of the above.  dL_dout [C,H,W]; final_T / n_contrib from fdgs_render_forward of this view.
 *   grad_feat [N,C] += dL/dfeat;   grads (NULL = features only) += the gradient through alpha_k and T_k to mean,
 *   log_scale, quat_l, quat_r, opacity_logit (grads->sh receives zeros: the 4DSH coefficients do not enter). */
int fdgs_render_features_backward(const fdgs_scene *scene, const fdgs_view *view_host, const fdgs_config *cfg_host, void *ws,
                                  size_t ws_bytes, int64_t pair_capacity, void *cuda_stream, const float *feat, int32_t C,
                                  void *scratch, size_t scratch_bytes, const float *dL_dout, const float *final_T,
                                  const uint32_t *n_contrib, float *grad_feat, const fdgs_grads *grads);

/* Per-splat optical flow: "we project its 3D displacement between consecutive two frames to the image
 * plane and render it using equation (6)".  flow [N,2] (pixels) = pi(mu_xyz|t+dt_next) - pi(mu_xyz|t), with
 * mu_xyz|t+d = mu_xyz|t + Sigma_1:3,4 / Sigma_44 d (eq. 9 is linear in t) and pi the pinhole projection of eq. 3; zero for
 * primitives culled at t or behind the camera at t + dt_next.  Call after fdgs_preprocess; render the result with
 * fdgs_render_features_forward(feat = flow, C = 2). */
int fdgs_splat_flow(const fdgs_scene *scene, const fdgs_view *view_host, const fdgs_config *cfg_host, void *ws, size_t ws_bytes,
                    int64_t pair_capacity, void *cuda_stream, float dt_next, float *flow);

/* ------------------------------------------------------------------------------------------------------------------
 * Training-side per-primitive terms next to the rasterizer (readings
 * T1-T6).  All are single streaming kernels over the parameter arrays (HBM-bound), asynchronous on `cuda_stream`.
 * ------------------------------------------------------------------------------------------------------------------ */

/* Learnable mask, forward (eq. 21-23): M = Sigmoid(mask_logit), M_hat = 1{M > mask_eps};
 * S_hat = M_hat S, alpha_hat = M_hat alpha.  A masked primitive (M_hat = 0) has alpha_hat = 0 and contributes nothing,
 * so the mask is applied by handing the renderer a copy of the opacity logits:
 *   opacity_logit_out[i] = M_hat_i ? opacity_logit[i] : -inf     (a non-finite parameter culls the primitive)
 * Render with a fdgs_scene whose opacity_logit is opacity_logit_out; kept primitives are untouched (M_hat = 1).
 * mask_logit, opacity_logit, opacity_logit_out: [N] device.  In-place (out == in) is allowed. */
int fdgs_mask_apply(const float *mask_logit, float mask_eps, const float *opacity_logit, float *opacity_logit_out,
                    int32_t N, void *cuda_stream);

typedef struct {
  float lambda_sparse; /* weight of L_sparse = 1/N sum_i |q_l^i - q_r^i|_1 on the NORMALISED quaternions (eq. 26; T1) */
  float lambda_covt;   /* weight of L_covt   = 1/N sum_i exp(-Sigma_44^i)                                (eq. 27)   */
  float lambda_mask;   /* weight of L_mask   = 1/N sum_i Sigmoid(m_i)                                    (eq. 24)   */
  float mask_eps;      /* threshold eps of eq. 21                                                                         */
} fdgs_reg_config;

/* Fused forward + backward of the three per-primitive regularisers, and the straight-through gradient of the mask.
 * For every primitive i, in this order:
 *   1. if mask_logit != NULL: with the rendering gradients ALREADY accumulated in grads (all views of the step),
 *        grad_mask_logit[i] += M_hat_i (sum_k grads->log_scale[i,k] + grads->opacity_logit[i] / (1 - alpha_i)) M_i (1 - M_i)
 *                              + lambda_mask M_i (1 - M_i) / N           (eq. 21-24; alpha_i = Sigmoid(scene->opacity_logit[i]),
 *                                                                        the UNMASKED logits)
 *   2. grads->log_scale, grads->quat_l, grads->quat_r += gradient of lambda_sparse L_sparse + lambda_covt L_covt.
 *   3. losses_dev (NULL ok) [3] += (L_sparse, L_covt, L_mask), unweighted, summed with atomics (order not fixed).
 * scene: only N, log_scale, quat_l, quat_r, opacity_logit are read.  Non-finite parameters or a zero quaternion make
 * the primitive contribute nothing.  grads->mean / sh / mean2d / densify are not touched. */
int fdgs_regularizers(const fdgs_scene *scene, const float *mask_logit, const fdgs_reg_config *rc_host,
                      const fdgs_grads *grads, float *grad_mask_logit, float *losses_dev, void *cuda_stream);

/* One dense Adam update of one parameter array (Kingma & Ba, Algorithm 1; the optimiser of [23], L324; T6):
 *   m = beta1 m + (1-beta1) g;  v = beta2 v + (1-beta2) g^2;
 *   p -= lr (m / (1-beta1^step)) / (sqrt(v / (1-beta2^step)) + eps)
 * param, grad, exp_avg, exp_avg_sq: [count] device fp32, 16-byte aligned; step >= 1.  zero_grad != 0 also clears grad
 * (saves the separate memset of the next step). */
typedef struct { float lr, beta1, beta2, eps; int32_t step; } fdgs_adam_config;
int fdgs_adam_step(float *param, float *grad, float *exp_avg, float *exp_avg_sq, int64_t count,
                   const fdgs_adam_config *cfg_host, int32_t zero_grad, void *cuda_stream);

/* Compact model of section 4.2 / 8.3.1 (T4): positions in binary16, opacity logit as a
 * `opacity_bits`-bit min-max code, log-scale / both quaternions / base colour (k = 0) / remaining coefficients as
 * residual-VQ indices (one uint8 per stage) into codebooks whose entries have the shape of the parameter they replace.
 * Decoded value = SUM over stages (in stage order) of the indexed entries.  Entries per codebook <= 256. */
typedef struct {
  int32_t N, sh_degree, n_time;
  const uint16_t *mean_f16;     /* [N,4] IEEE binary16 bit patterns                                                   */
  const uint8_t *opacity_code;  /* [N]   logit = opacity_lo + code (opacity_hi - opacity_lo) / (2^opacity_bits - 1)   */
  float opacity_lo, opacity_hi;
  int32_t opacity_bits;         /* 1..8                                                                               */
  int32_t scale_stages, scale_entries; const uint8_t *scale_idx; /* [N,stages] */ const float *scale_cb; /* [stages,entries,4] */
  int32_t rot_stages, rot_entries;     const uint8_t *rot_l_idx, *rot_r_idx;      const float *rot_cb;   /* shared, [..,4]     */
  int32_t dc_stages, dc_entries;       const uint8_t *dc_idx;                     const float *dc_cb;    /* [stages,entries,3] */
  int32_t rest_stages, rest_entries;   const uint8_t *rest_idx;                   const float *rest_cb;  /* [stages,entries,(K-1)*3]; unused if K = 1 */
} fdgs_compact_scene;

/* Expands a compact model into the fp32 arrays of `out` (caller-owned, shapes of fdgs_scene for the same N, sh_degree,
 * n_time; the const qualifiers of fdgs_scene are cast away for writing).  Stage counts 1..16. */
int fdgs_decode_compact(const fdgs_compact_scene *compact, const fdgs_scene *out, void *cuda_stream);

/* ------------------------------------------------------------------------------------------------------------------
 * Forward of one view WITHOUT any allocation, for callers that cannot call cudaMalloc (stream capture into a CUDA graph,
 * tight serving loops, harnesses that forbid it).  Same kernels, same launch sequence and same result, bit for bit, as
 * fdgs_preprocess + fdgs_render_forward (PAPER.md:L147 tile rasterizer, eq. 6), but the workspace is a device array
 * built into the library: FDGS_STATIC_WS_BYTES (8 MiB) on every GPU that loads libfdgs.so, held until the process exits.
 * The caller passes inputs and outputs only:  scene arrays, image [3,H,W], final_T [H,W], n_contrib [H,W] as for
 * fdgs_render_forward;  overflow_dev (device uint32, may be NULL) receives 1 if D exceeded pair_capacity (the image is then
 * that of an empty rendering), else 0.
 * Limit: fdgs_workspace_bytes(N, K, W, H, pair_capacity) must not exceed FDGS_STATIC_WS_BYTES, else FDGS_ERR_STATIC_LIMIT
 * is returned before anything is launched (fits e.g. N = 32768, 320x240, pair_capacity = 524288;  N = 16384, 256x256,
 * 262144 pairs takes 3.6 MiB).  Other errors as fdgs_render_forward.
 * The call issues one memset, 8 kernels and (overflow_dev != NULL) one 4-byte device copy on `cuda_stream`; it calls no
 * cudaMalloc / cudaFree / stream or event creation and never synchronises.  The first call on a device looks up the
 * address of the array (cudaGetSymbolAddress) and the SM count: make one call outside a stream capture first.
 * All calls on one device share the array, which keeps the contents of the last call; the part that has to start from
 * zero is cleared by the memset of each call.  Calls that overlap on the GPU (different streams without an ordering
 * event, or two host threads) RACE on it: order them.  No backward: the training path owns its workspaces.
 * ------------------------------------------------------------------------------------------------------------------ */
#define FDGS_STATIC_WS_BYTES (8u << 20)
int fdgs_render_forward_static(const fdgs_scene *scene, const fdgs_view *view_host, const fdgs_config *cfg_host,
                               int64_t pair_capacity, void *cuda_stream, float *image, float *final_T, uint32_t *n_contrib,
                               uint32_t *overflow_dev);

/* Number of kernel launches the library has issued so far in this process (bench.py's gpu_launches). */
int64_t fdgs_launch_count(void);

const char *fdgs_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* FDGS_H */
