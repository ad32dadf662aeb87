// api.cu — the C ABI of include/fdgs.h: argument validation, workspace carve-up, launch sequence.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <atomic>
#include <mutex>

#include "common.cuh"

namespace fdgs {

static char g_cuda_err[256] = "no CUDA error recorded";

int cuda_fail(cudaError_t e, const char* where) {
  snprintf(g_cuda_err, sizeof(g_cuda_err), "CUDA error in %s: %s", where, cudaGetErrorString(e));
  return FDGS_ERR_CUDA;
}
#define FDGS_CUDA(call, where) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return cuda_fail(e_, where); } while (0)

// Optional per-stage timing (fdgs_set_stage_timing): CUDA events recorded on the caller's stream at the stage
// boundaries; off by default so that the product path carries no event records.
enum { EV_PRE0, EV_PRE1, EV_PRE2, EV_FWD0, EV_FWD1, EV_FWD2, EV_FWD3, EV_BWD0, EV_BWD1, EV_BWD2, EV_COL0, EV_COL1, EV_COUNT };
static int g_timing = 0;
static cudaEvent_t g_ev[EV_COUNT];
static inline void mark(int which, cudaStream_t st) { if (g_timing) cudaEventRecord(g_ev[which], st); }

static bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

// Library-owned streams and events, one set per CUDA device (created on first use on that device): the worker streams
// of fdgs_step_batch, the zeroing stream, the copy stream of fdgs_step_host, and the SM count.
constexpr int SIDE_STREAMS = 8;
struct DeviceCtx {
  bool ready = false;
  int sms = 0;
  // side streams of fdgs_render_forward (colour of the survivors next to the depth sort and the row scatter): a call takes
  // the next slot, so concurrent frames on different caller streams do not queue behind each other
  cudaStream_t side[SIDE_STREAMS] = {};
  cudaEvent_t side_fork[SIDE_STREAMS] = {}, side_join[SIDE_STREAMS] = {};
  std::atomic<unsigned int> side_next{0};
  cudaStream_t worker[FDGS_MAX_BATCH] = {}, zero_stream = nullptr, copy_stream = nullptr;
  cudaEvent_t batch_fork = nullptr, b2_done[FDGS_MAX_BATCH] = {}, copy_done[FDGS_MAX_BATCH] = {}, zero_done = nullptr, copy_fork = nullptr, copy_join = nullptr, colour_done = nullptr;
};
constexpr int MAX_DEVICES = 64;
static DeviceCtx g_ctx[MAX_DEVICES];
static std::mutex g_ctx_mutex;

static int device_ctx(DeviceCtx** out) {
  int dev = 0;
  FDGS_CUDA(cudaGetDevice(&dev), "cudaGetDevice");
  if (dev < 0 || dev >= MAX_DEVICES) return FDGS_ERR_INVALID;
  std::lock_guard<std::mutex> lock(g_ctx_mutex);
  DeviceCtx& c = g_ctx[dev];
  if (!c.ready) {
    FDGS_CUDA(cudaDeviceGetAttribute(&c.sms, cudaDevAttrMultiProcessorCount, dev), "SM count");
    if (c.sms <= 0) c.sms = 148;
    for (int i = 0; i < FDGS_MAX_BATCH; ++i) {
      FDGS_CUDA(cudaStreamCreateWithFlags(&c.worker[i], cudaStreamNonBlocking), "worker stream");
      FDGS_CUDA(cudaEventCreateWithFlags(&c.b2_done[i], cudaEventDisableTiming), "worker event");
      FDGS_CUDA(cudaEventCreateWithFlags(&c.copy_done[i], cudaEventDisableTiming), "copy event");
    }
    for (int i = 0; i < SIDE_STREAMS; ++i) {
      FDGS_CUDA(cudaStreamCreateWithFlags(&c.side[i], cudaStreamNonBlocking), "side stream");
      FDGS_CUDA(cudaEventCreateWithFlags(&c.side_fork[i], cudaEventDisableTiming), "side event");
      FDGS_CUDA(cudaEventCreateWithFlags(&c.side_join[i], cudaEventDisableTiming), "side event");
    }
    FDGS_CUDA(cudaStreamCreateWithFlags(&c.zero_stream, cudaStreamNonBlocking), "zero stream");
    FDGS_CUDA(cudaStreamCreateWithFlags(&c.copy_stream, cudaStreamNonBlocking), "copy stream");
    FDGS_CUDA(cudaEventCreateWithFlags(&c.zero_done, cudaEventDisableTiming), "zero event");
    FDGS_CUDA(cudaEventCreateWithFlags(&c.batch_fork, cudaEventDisableTiming), "fork event");
    FDGS_CUDA(cudaEventCreateWithFlags(&c.copy_fork, cudaEventDisableTiming), "copy event");
    FDGS_CUDA(cudaEventCreateWithFlags(&c.copy_join, cudaEventDisableTiming), "copy event");
    FDGS_CUDA(cudaEventCreateWithFlags(&c.colour_done, cudaEventDisableTiming), "colour event");
    c.ready = true;
  }
  *out = &c;
  return FDGS_OK;
}

static int num_sms() {
  DeviceCtx* c = nullptr;
  return device_ctx(&c) == FDGS_OK ? c->sms : 148;
}

// The thresholds must describe a renderer: the backward divides by (1 - alpha), the radius takes a square root, ...
static int check_cfg(const fdgs_config* c) {
  if (!c) return FDGS_ERR_INVALID;
  if (!(c->alpha_min >= 0.f) || !(c->alpha_min <= c->alpha_max) || !(c->alpha_max <= 1.f)) return FDGS_ERR_INVALID;
  // alpha_max = 1 is the "pure eq. 6" setting: 1 - alpha can then only vanish where the forward has terminated already,
  // unless transmittance_min = 0 too; rcp(0) of such a pixel is excluded by requiring one of the two guards
  if (!(c->transmittance_min >= 0.f) || !(c->transmittance_min < 1.f)) return FDGS_ERR_INVALID;
  if (!(c->dilation >= 0.f) || !(c->cutoff_sigma > 0.f) || !(c->guard > 0.f) || !(c->znear > 0.f) || !(c->marginal_min >= 0.f)) return FDGS_ERR_INVALID;
  if (!std::isfinite(c->dilation) || !std::isfinite(c->cutoff_sigma) || !std::isfinite(c->guard) || !std::isfinite(c->znear) || !(c->marginal_min <= 1.f))
    return FDGS_ERR_INVALID;
  return FDGS_OK;
}

static int check_common(const fdgs_scene* sc, const fdgs_view* v, const fdgs_config* c, const void* ws) {
  if (!sc || !v || !c || !ws) return FDGS_ERR_INVALID;
  if (check_cfg(c)) return FDGS_ERR_INVALID;
  if (sc->N < 0 || sc->sh_degree < 0 || sc->sh_degree > 3 || sc->n_time < 1 || sc->n_time > 8) return FDGS_ERR_INVALID;
  if (v->width <= 0 || v->height <= 0 || !(v->fx > 0) || !(v->fy > 0) || !(v->period_T > 0)) return FDGS_ERR_INVALID;
  if (sc->N > 0) {
    if (!sc->mean || !sc->log_scale || !sc->quat_l || !sc->quat_r || !sc->opacity_logit || !sc->sh) return FDGS_ERR_INVALID;
    if (!aligned16(sc->mean) || !aligned16(sc->log_scale) || !aligned16(sc->quat_l) || !aligned16(sc->quat_r) || !aligned16(sc->sh))
      return FDGS_ERR_INVALID;
  }
  if (!aligned16(ws)) return FDGS_ERR_INVALID;
  const long long tx = (v->width + TILE - 1) / TILE, ty = (v->height + TILE - 1) / TILE;
  if ((tx + 1) * (ty + 1) > MAX_GRID_CELLS || tx > 65535 || ty > 65535) return FDGS_ERR_INVALID;
  return FDGS_OK;
}

static int check_grads(const fdgs_scene* sc, const fdgs_grads* g) {
  if (!g) return FDGS_ERR_INVALID;
  if (sc->N <= 0) return FDGS_OK;
  if (!g->mean || !g->log_scale || !g->quat_l || !g->quat_r || !g->opacity_logit || !g->sh) return FDGS_ERR_INVALID;
  // every array that the backward reads or writes with 128-bit accesses
  if (!aligned16(g->mean) || !aligned16(g->log_scale) || !aligned16(g->quat_l) || !aligned16(g->quat_r) || !aligned16(g->sh)) return FDGS_ERR_INVALID;
  if (g->mean2d && (reinterpret_cast<uintptr_t>(g->mean2d) & 7u)) return FDGS_ERR_INVALID;
  return FDGS_OK;
}

static void make_params(const fdgs_view* v, const fdgs_config* c, ViewParams& vp, CfgParams& cp) {
  for (int r = 0; r < 3; ++r) { for (int q = 0; q < 3; ++q) vp.W[r][q] = v->view[4 * r + q]; vp.tau[r] = v->view[4 * r + 3]; }
  for (int r = 0; r < 3; ++r) vp.cam[r] = -(vp.W[0][r] * vp.tau[0] + vp.W[1][r] * vp.tau[1] + vp.W[2][r] * vp.tau[2]);
  vp.fx = v->fx; vp.fy = v->fy; vp.cx = v->cx; vp.cy = v->cy;
  vp.width = v->width; vp.height = v->height;
  vp.tiles_x = (v->width + TILE - 1) / TILE; vp.tiles_y = (v->height + TILE - 1) / TILE;
  vp.t = v->t; vp.inv_T = 1.0f / v->period_T;
  for (int k = 0; k < 3; ++k) vp.bg[k] = v->bg[k];
  vp.limx = c->guard * v->width / (2.0f * v->fx); vp.limy = c->guard * v->height / (2.0f * v->fy);
  cp.marginal_min = c->marginal_min; cp.alpha_min = c->alpha_min; cp.alpha_max = c->alpha_max;
  cp.transmittance_min = c->transmittance_min; cp.dilation = c->dilation; cp.cutoff_sigma = c->cutoff_sigma;
  cp.znear = c->znear; cp.guard = c->guard;
  cp.log2_alpha_min = c->alpha_min > 0.f ? log2f(c->alpha_min) * (1.0f + 1e-6f) - 1e-6f : -INFINITY;
  cp.default_thresholds = c->alpha_min == FDGS_DEF_ALPHA_MIN && c->alpha_max == FDGS_DEF_ALPHA_MAX && c->transmittance_min == FDGS_DEF_T_MIN;
  if (cp.default_thresholds) cp.log2_alpha_min = FDGS_DEF_L2MIN;   // every kernel, specialised or not, compares against the same value
}

// ---- parity exports -----------------------------------------------------------------------------
__global__ void export_records_kernel(const SplatRec* __restrict__ rec, const unsigned int* __restrict__ tiles_touched, const int N,
                                      float* __restrict__ dst) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  float* o = dst + (size_t)12 * i;
  if (tiles_touched[i] == 0) { for (int k = 0; k < 12; ++k) o[k] = __int_as_float(0x7fc00000); return; }
  const SplatRec r = rec[i];
  const float ik = 1.0f / 0.72134752044448170f;     // conic from its exp2-scaled Cholesky factor
  o[0] = r.u; o[1] = r.v;
  o[2] = r.ca * r.ca * ik; o[3] = r.ca * r.cb * ik; o[4] = (r.cb * r.cb + r.cc * r.cc) * ik;
  o[5] = exp2f(r.lo); o[6] = r.r; o[7] = r.g; o[8] = r.b; o[9] = r.depth; o[10] = r.radius; o[11] = r.w;
}
__global__ void export_rects_kernel(const ushort4* __restrict__ rect, const int N, int4* __restrict__ dst) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < N) { const ushort4 r = rect[i]; dst[i] = make_int4(r.x, r.y, r.z, r.w); }
}
// the literal 64-bit key of every pair of the per-tile lists: tile id << 32 | fp32 depth bits; the tile of list position i
// is the one whose range holds i (binary search over the tile ranges: no key array exists on the product path)
__global__ void export_keys_kernel(const uint2* __restrict__ ranges, const int tiles, const unsigned int* __restrict__ ids,
                                   const SplatRec* __restrict__ rec, const unsigned int D, unsigned long long* __restrict__ dst) {
  const unsigned int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= D) return;
  int lo = 0, hi = tiles;                                  // LARGEST tile with ranges[tile].x <= i: an empty tile shares its x with
  while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (ranges[mid].x <= i) lo = mid; else hi = mid; }   // its successor, so this is the owner
  dst[i] = ((unsigned long long)(unsigned int)lo << 32) | __float_as_uint(rec[ids[i]].depth);
}

// ---- measured pipe peaks: the denominators of the blend kernels' roofline ------------------------
// 8 independent FFMA chains per thread: 1 lane-instruction per lane and issue slot, nothing else in the loop
__global__ void __launch_bounds__(256) peak_fma_kernel(float* out, const int iters, const float s) {
  float a[8];
#pragma unroll
  for (int k = 0; k < 8; ++k) a[k] = threadIdx.x * 1e-3f + k;
  for (int i = 0; i < iters; ++i)
#pragma unroll
    for (int u = 0; u < 8; ++u)
#pragma unroll
      for (int k = 0; k < 8; ++k) a[k] = fmaf(a[k], s, 1e-3f);
  float r = 0.f;
#pragma unroll
  for (int k = 0; k < 8; ++k) r += a[k];
  out[blockIdx.x * blockDim.x + threadIdx.x] = r;
}
__global__ void __launch_bounds__(256) peak_mufu_kernel(float* out, const int iters) {
  float a[8];
#pragma unroll
  for (int k = 0; k < 8; ++k) a[k] = -(threadIdx.x * 1e-3f + k);
  for (int i = 0; i < iters; ++i)
#pragma unroll
    for (int u = 0; u < 8; ++u)
#pragma unroll
      for (int k = 0; k < 8; ++k) asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(a[k]));
  float r = 0.f;
#pragma unroll
  for (int k = 0; k < 8; ++k) r += a[k];
  out[blockIdx.x * blockDim.x + threadIdx.x] = r;
}

}  // namespace fdgs

using namespace fdgs;

extern "C" {

int fdgs_default_config(fdgs_config* c) {
  if (!c) return FDGS_ERR_INVALID;
  c->marginal_min = 0.05f; c->alpha_min = 1.0f / 255.0f; c->alpha_max = 0.99f; c->transmittance_min = 1e-4f;
  c->dilation = 0.3f; c->cutoff_sigma = 3.0f; c->znear = 0.2f; c->guard = 1.3f;
  return FDGS_OK;
}

int fdgs_workspace_bytes(int32_t N, int32_t K, int32_t W, int32_t H, int64_t pair_capacity, size_t* bytes_host) {
  if (!bytes_host || N < 0 || K < 1 || W <= 0 || H <= 0 || pair_capacity < 1 || pair_capacity >= (1LL << 30)) return FDGS_ERR_INVALID;
  *bytes_host = carve(nullptr, N, K, W, H, pair_capacity).bytes;
  return FDGS_OK;
}

// split_colour: the preprocess kernel of a degree-3 scene stops after the geometry and the forward that follows evaluates
// the colours on a side stream under the binning (the public pair fdgs_preprocess / fdgs_render_forward: shortest frame);
// false: colour inside the preprocess kernel (fdgs_step_batch, whose views already overlap each other: least total work)
static int preprocess_impl(const fdgs_scene* sc, const fdgs_view* v, const fdgs_config* c, void* ws_ptr, size_t ws_bytes,
                           int64_t cap, void* stream, int64_t* num_pairs_host, int32_t* num_visible_host, bool split_colour) {
  int rc = check_common(sc, v, c, ws_ptr);
  if (rc) return rc;
  if (cap < 1 || cap >= (1LL << 30)) return FDGS_ERR_INVALID;
  const int K = sc->n_time * (sc->sh_degree + 1) * (sc->sh_degree + 1);
  const Workspace ws = carve(ws_ptr, sc->N, K, v->width, v->height, cap);
  if (ws.bytes > ws_bytes) return FDGS_ERR_WORKSPACE;
  cudaStream_t st = (cudaStream_t)stream;
  ViewParams vp; CfgParams cp;
  make_params(v, c, vp, cp);
  // header (tickets, counters), coverage difference grid, scan states, depth-digit counts and the look-back regions of
  // the depth sort start from zero: ONE memset per frame.  (The layout mirror for fdgs_debug_export is written by the
  // compaction launch from its by-value arguments: no host-memory copy on the stream, so the whole call sequence can be
  // captured into a CUDA graph.)
  FDGS_CUDA(cudaMemsetAsync(ws_ptr, 0, ws.zero_bytes, st), "memset(header)");
  mark(EV_PRE0, st);
  launch_preprocess_fwd(*sc, vp, cp, ws, st, split_colour);         // A1-A4 (+ coverage grid)
  mark(EV_PRE1, st);
  launch_compact_and_tile_grid(ws, sc->N, K, vp, cp, cap, st);          // survivors -> (depth bits, id); A5/A8: list lengths -> ranges, D
  mark(EV_PRE2, st);
  FDGS_CUDA(cudaGetLastError(), "preprocess launches");
  if (num_pairs_host || num_visible_host) {
    FDGS_CUDA(cudaStreamSynchronize(st), "preprocess sync");
    WsHeader hh;
    FDGS_CUDA(cudaMemcpy(&hh, ws.hdr, sizeof(hh), cudaMemcpyDeviceToHost), "read header");
    if (num_pairs_host) *num_pairs_host = hh.total_pairs;
    if (num_visible_host) *num_visible_host = (int32_t)hh.num_visible;
    if (hh.overflow) return FDGS_ERR_PAIR_OVERFLOW;
  }
  return FDGS_OK;
}

int fdgs_preprocess(const fdgs_scene* sc, const fdgs_view* v, const fdgs_config* c, void* ws_ptr, size_t ws_bytes,
                    int64_t cap, void* stream, int64_t* num_pairs_host, int32_t* num_visible_host) {
  return preprocess_impl(sc, v, c, ws_ptr, ws_bytes, cap, stream, num_pairs_host, num_visible_host, true);
}

}  // extern "C"

// A6-A9.  The depth order of the survivors (level 1) is kept in the workspace for the backward.
static int forward_impl(const fdgs_scene* sc, const ViewParams& vp, const CfgParams& cp, const Workspace& ws, int64_t cap,
                        cudaStream_t st, float* image, float* final_T, uint32_t* n_contrib, float* depth_map, bool split_colour) {
  (void)cap;
  DeviceCtx* ctx = nullptr;
  int rc = device_ctx(&ctx);
  if (rc) return rc;
  const int sms = ctx->sms;
  mark(EV_FWD0, st);
  // A4 of a degree-3 scene runs on a side stream while the survivors are sorted and scattered: only the blend needs the
  // colours, and the binning launches are latency-bound chains of a few hundred CTAs (fork here, join before the blend;
  // both inside this call, so the sequence stays capturable into a CUDA graph)
  cudaEvent_t join = nullptr;
  if (split_colour && sc->N > 0 && sc->sh_degree == 3) {
    const unsigned int slot = ctx->side_next.fetch_add(1u, std::memory_order_relaxed) % SIDE_STREAMS;
    FDGS_CUDA(cudaEventRecord(ctx->side_fork[slot], st), "fork(colour)");
    FDGS_CUDA(cudaStreamWaitEvent(ctx->side[slot], ctx->side_fork[slot], 0), "fork(colour) wait");
    mark(EV_COL0, ctx->side[slot]);
    launch_colour_fwd(*sc, ws, sms, ctx->side[slot]);
    mark(EV_COL1, ctx->side[slot]);
    FDGS_CUDA(cudaEventRecord(ctx->side_join[slot], ctx->side[slot]), "join(colour)");
    join = ctx->side_join[slot];
  }
  launch_sort_depth(ws, sc->N, sms, st);                            // level 1: survivors by fp32 depth bits
  mark(EV_FWD1, st);
  launch_row_ballots(ws, sc->N, vp, sms, st);                       // level 2: which survivors cover which tile row ...
  launch_row_scatter(ws, sc->N, vp, sms, st);                       // ... and the per-tile lists written in place, depth order
  mark(EV_FWD2, st);
  if (join) FDGS_CUDA(cudaStreamWaitEvent(st, join, 0), "join(colour) wait");
  launch_blend_fwd(ws, vp, cp, image, final_T, n_contrib, depth_map, st);
  mark(EV_FWD3, st);
  FDGS_CUDA(cudaGetLastError(), "forward launches");
  return FDGS_OK;
}

static int depth_buf() { return 0; }      // kept for the signature of launch_preprocess_bwd (unused there)

// after a synchronisation: has the last preprocess on this workspace exceeded the pair capacity?
static int read_overflow(const Workspace& ws) {
  unsigned int ov = 0;
  FDGS_CUDA(cudaMemcpy(&ov, &ws.hdr->overflow, sizeof(ov), cudaMemcpyDeviceToHost), "read overflow flag");
  return ov ? FDGS_ERR_PAIR_OVERFLOW : FDGS_OK;
}

extern "C" {

static int forward_entry(const fdgs_scene* sc, const fdgs_view* v, const fdgs_config* c, void* ws_ptr, size_t ws_bytes,
                         int64_t cap, void* stream, float* image, float* final_T, uint32_t* n_contrib, float* depth_map,
                         bool split_colour = true) {
  int rc = check_common(sc, v, c, ws_ptr);
  if (rc) return rc;
  if (!image || !final_T || !n_contrib || cap < 1 || cap >= (1LL << 30)) return FDGS_ERR_INVALID;
  const int K = sc->n_time * (sc->sh_degree + 1) * (sc->sh_degree + 1);
  const Workspace ws = carve(ws_ptr, sc->N, K, v->width, v->height, cap);
  if (ws.bytes > ws_bytes) return FDGS_ERR_WORKSPACE;
  ViewParams vp; CfgParams cp;
  make_params(v, c, vp, cp);
  return forward_impl(sc, vp, cp, ws, cap, (cudaStream_t)stream, image, final_T, n_contrib, depth_map, split_colour);
}

int fdgs_render_forward(const fdgs_scene* sc, const fdgs_view* v, const fdgs_config* c, void* ws_ptr, size_t ws_bytes,
                        int64_t cap, void* stream, float* image, float* final_T, uint32_t* n_contrib) {
  return forward_entry(sc, v, c, ws_ptr, ws_bytes, cap, stream, image, final_T, n_contrib, nullptr);
}

int fdgs_render_forward_aux(const fdgs_scene* sc, const fdgs_view* v, const fdgs_config* c, void* ws_ptr, size_t ws_bytes,
                            int64_t cap, void* stream, float* image, float* final_T, uint32_t* n_contrib, float* depth_map) {
  if (!depth_map) return FDGS_ERR_INVALID;
  return forward_entry(sc, v, c, ws_ptr, ws_bytes, cap, stream, image, final_T, n_contrib, depth_map);
}

}  // extern "C"

// B1 + B2.  `before_b2` (optional): an event the stream waits for between the two — fdgs_step_batch uses it to order the
// non-atomic gradient read-modify-writes of concurrent views while their blend kernels overlap.
static int backward_impl(const fdgs_scene* sc, const fdgs_view* v, const fdgs_config* c, void* ws_ptr, size_t ws_bytes, int64_t cap,
                         cudaStream_t st, const float* dL_dimage, const float* final_T, const uint32_t* n_contrib,
                         const fdgs_grads* g, cudaEvent_t before_b2, const float* dL_ddepth = nullptr, const float* dL_dopacity = nullptr,
                         bool b1_only = false) {
  int rc = check_common(sc, v, c, ws_ptr);
  if (rc) return rc;
  if (!dL_dimage || !final_T || !n_contrib || cap < 1 || cap >= (1LL << 30)) return FDGS_ERR_INVALID;
  if ((rc = check_grads(sc, g))) return rc;
  const int K = sc->n_time * (sc->sh_degree + 1) * (sc->sh_degree + 1);
  const Workspace ws = carve(ws_ptr, sc->N, K, v->width, v->height, cap);
  if (ws.bytes > ws_bytes) return FDGS_ERR_WORKSPACE;
  ViewParams vp; CfgParams cp;
  make_params(v, c, vp, cp);
  const int l1 = depth_buf();
  if (sc->N > 0) FDGS_CUDA(cudaMemsetAsync(ws.g9, 0, sizeof(float) * 9 * (size_t)sc->N, st), "memset(g9)");
  const bool aux = dL_ddepth || dL_dopacity;
  if (aux && sc->N > 0) FDGS_CUDA(cudaMemsetAsync(ws.gz, 0, sizeof(float) * (size_t)sc->N, st), "memset(gz)");
  mark(EV_BWD0, st);
  launch_blend_bwd(ws, vp, cp, dL_dimage, final_T, n_contrib, dL_ddepth, dL_dopacity, st);   // B1
  mark(EV_BWD1, st);
  if (b1_only) { FDGS_CUDA(cudaGetLastError(), "backward launches"); return FDGS_OK; }     // fdgs_step_batch: B2 of all views follows in one pass
  if (before_b2) FDGS_CUDA(cudaStreamWaitEvent(st, before_b2, 0), "wait before B2");
  launch_preprocess_bwd(*sc, vp, cp, ws, l1, *g, aux, st);                      // B2
  mark(EV_BWD2, st);
  FDGS_CUDA(cudaGetLastError(), "backward launches");
  return FDGS_OK;
}

extern "C" {

int fdgs_render_backward(const fdgs_scene* sc, const fdgs_view* v, const fdgs_config* c, void* ws_ptr, size_t ws_bytes,
                         int64_t cap, void* stream, const float* dL_dimage, const float* final_T, const uint32_t* n_contrib,
                         const fdgs_grads* g) {
  return backward_impl(sc, v, c, ws_ptr, ws_bytes, cap, (cudaStream_t)stream, dL_dimage, final_T, n_contrib, g, nullptr);
}

int fdgs_render_backward_aux(const fdgs_scene* sc, const fdgs_view* v, const fdgs_config* c, void* ws_ptr, size_t ws_bytes,
                             int64_t cap, void* stream, const float* dL_dimage, const float* dL_ddepth, const float* dL_dopacity,
                             const float* final_T, const uint32_t* n_contrib, const fdgs_grads* g) {
  return backward_impl(sc, v, c, ws_ptr, ws_bytes, cap, (cudaStream_t)stream, dL_dimage, final_T, n_contrib, g, nullptr, dL_ddepth, dL_dopacity);
}

int fdgs_l1_loss(const float* image, const float* target, int64_t count, float* dL_dimage, float* loss, void* stream) {
  if (!image || !target || !dL_dimage || !loss || count <= 0) return FDGS_ERR_INVALID;
  launch_l1_loss(image, target, count, dL_dimage, loss, nullptr, (cudaStream_t)stream);
  FDGS_CUDA(cudaGetLastError(), "l1 loss launch");
  return FDGS_OK;
}

// loss of a view inside the step calls: as fdgs_l1_loss, but a view whose pairs exceeded the capacity (nothing drawn, all
// gradients zero) reports NaN instead of the loss of a background image, so that even a fully asynchronous caller sees it
static int step_loss(const Workspace& ws, const float* image, const float* target, int64_t count, float* dL_dimage, float* loss, cudaStream_t st) {
  launch_l1_loss(image, target, count, dL_dimage, loss, &ws.hdr->overflow, st);
  FDGS_CUDA(cudaGetLastError(), "l1 loss launch");
  return FDGS_OK;
}

int fdgs_step_host(const fdgs_scene* sc, const fdgs_view* v, const fdgs_config* c, void* ws, size_t ws_bytes, int64_t cap,
                   void* stream, const float* target_host, float* target_dev, float* image, float* final_T,
                   uint32_t* n_contrib, float* dL_dimage, float* loss_dev, fdgs_grads* g, float* result_host) {
  if (!v || !result_host) return FDGS_ERR_INVALID;
  int rc = check_common(sc, v, c, ws);
  if (rc) return rc;
  if (g && (rc = check_grads(sc, g))) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  const size_t count = (size_t)3 * v->width * v->height;
  DeviceCtx* ctx = nullptr;
  if ((rc = device_ctx(&ctx))) return rc;
  bool forked = false;
  // after the fork nothing may return before the copy stream has been joined into `st` again (the caller may reuse
  // target_dev as soon as `st` is idle): errors fall through to the join
  if (g) {
    if (!target_host || !target_dev || !dL_dimage || !loss_dev) return FDGS_ERR_INVALID;
    // fork: the copy may start once everything queued on `st` so far (the previous user of target_dev) is done
    FDGS_CUDA(cudaEventRecord(ctx->copy_fork, st), "fork");
    FDGS_CUDA(cudaStreamWaitEvent(ctx->copy_stream, ctx->copy_fork, 0), "fork wait");
    forked = true;
    cudaMemcpyAsync(target_dev, target_host, count * sizeof(float), cudaMemcpyHostToDevice, ctx->copy_stream);
    cudaEventRecord(ctx->copy_join, ctx->copy_stream);
    cudaMemsetAsync(loss_dev, 0, sizeof(float), st);
  }
  rc = fdgs_preprocess(sc, v, c, ws, ws_bytes, cap, stream, nullptr, nullptr);
  if (!rc) rc = fdgs_render_forward(sc, v, c, ws, ws_bytes, cap, stream, image, final_T, n_contrib);
  if (forked) cudaStreamWaitEvent(st, ctx->copy_join, 0);
  if (rc) { cudaStreamSynchronize(st); return rc; }
  const int K = sc->n_time * (sc->sh_degree + 1) * (sc->sh_degree + 1);
  const Workspace wsv = carve(ws, sc->N, K, v->width, v->height, cap);
  if (g) {
    rc = step_loss(wsv, image, target_dev, (int64_t)count, dL_dimage, loss_dev, st);
    if (!rc) rc = fdgs_render_backward(sc, v, c, ws, ws_bytes, cap, stream, dL_dimage, final_T, n_contrib, g);
    if (!rc) FDGS_CUDA(cudaMemcpyAsync(result_host, loss_dev, sizeof(float), cudaMemcpyDeviceToHost, st), "D2H loss");
  } else {
    FDGS_CUDA(cudaMemcpyAsync(result_host, image, count * sizeof(float), cudaMemcpyDeviceToHost, st), "D2H image");
  }
  FDGS_CUDA(cudaStreamSynchronize(st), "step sync");
  if (rc) return rc;
  return read_overflow(wsv);         // D > pair_capacity: nothing was drawn and every gradient is zero — say so
}

int fdgs_step_batch(const fdgs_scene* sc, const fdgs_view* views, int32_t num_views, const fdgs_config* c, int64_t cap,
                    const fdgs_view_buffers* bufs, void* stream, float* loss_dev, const fdgs_grads* g, float* loss_host, int32_t flags) {
  if (!sc || !views || !c || !bufs || !loss_dev || !g || num_views < 1 || num_views > FDGS_MAX_BATCH) return FDGS_ERR_INVALID;
  if (cap < 1 || cap >= (1LL << 30)) return FDGS_ERR_INVALID;
  int rc = check_grads(sc, g);
  if (rc) return rc;
  const int K = sc->n_time * (sc->sh_degree + 1) * (sc->sh_degree + 1);
  for (int i = 0; i < num_views; ++i) {          // everything that can be rejected is rejected before the first fork
    const fdgs_view_buffers& b = bufs[i];
    if (!b.ws || !b.target_dev || !b.image || !b.final_T || !b.n_contrib || !b.dL_dimage) return FDGS_ERR_INVALID;
    for (int k = 0; k < i; ++k) if (bufs[k].ws == b.ws) return FDGS_ERR_INVALID;      // one workspace per view
    if ((rc = check_common(sc, &views[i], c, b.ws))) return rc;
    if (carve(nullptr, sc->N, K, views[i].width, views[i].height, cap).bytes > b.ws_bytes) return FDGS_ERR_WORKSPACE;
  }
  cudaStream_t st = (cudaStream_t)stream;
  DeviceCtx* ctx = nullptr;
  if ((rc = device_ctx(&ctx))) return rc;
  FDGS_CUDA(cudaEventRecord(ctx->batch_fork, st), "fork");
  const bool zero = (flags & FDGS_STEP_ZERO_GRADS) && sc->N > 0;
  if (zero) {   // the gradient arrays are first touched by the first view's backward preprocess: zeroing them hides under the forward passes
    const size_t N = (size_t)sc->N;
    cudaStreamWaitEvent(ctx->zero_stream, ctx->batch_fork, 0);
    cudaMemsetAsync(g->mean, 0, 16 * N, ctx->zero_stream);
    cudaMemsetAsync(g->log_scale, 0, 16 * N, ctx->zero_stream);
    cudaMemsetAsync(g->quat_l, 0, 16 * N, ctx->zero_stream);
    cudaMemsetAsync(g->quat_r, 0, 16 * N, ctx->zero_stream);
    cudaMemsetAsync(g->opacity_logit, 0, 4 * N, ctx->zero_stream);
    cudaMemsetAsync(g->sh, 0, 12 * (size_t)K * N, ctx->zero_stream);
    if (g->mean2d) cudaMemsetAsync(g->mean2d, 0, 8 * N, ctx->zero_stream);
    cudaEventRecord(ctx->zero_done, ctx->zero_stream);
  }
  // From here on work is forked onto library streams: an error stops issuing, but every stream that was given work is
  // still joined into `st` before the call returns, so the caller can never free or reuse buffers under running kernels.
  // host targets travel on the copy stream, view after view, while the views' preprocess and forward passes run: a view
  // only waits for its own target right before its loss kernel
  bool copies = false;
  for (int i = 0; i < num_views; ++i) {
    if (!bufs[i].target_host) continue;
    if (!copies) { cudaStreamWaitEvent(ctx->copy_stream, ctx->batch_fork, 0); copies = true; }
    cudaMemcpyAsync(bufs[i].target_dev, bufs[i].target_host, (size_t)3 * views[i].width * views[i].height * sizeof(float), cudaMemcpyHostToDevice, ctx->copy_stream);
    cudaEventRecord(ctx->copy_done[i], ctx->copy_stream);
  }
  // sh_degree 3 with up to 4 Fourier orders and up to 4 views (every benchmark configuration): one colour pass for the whole batch
  const bool batched_b2 = sc->sh_degree == 3 && sc->n_time <= 4 && num_views > 1 && num_views <= 4;
  int launched = 0;
  for (int i = 0; i < num_views && !rc; ++i) {
    const fdgs_view_buffers& b = bufs[i];
    cudaStream_t w = ctx->worker[i];
    const size_t count = (size_t)3 * views[i].width * views[i].height;
    cudaStreamWaitEvent(w, ctx->batch_fork, 0);
    launched = i + 1;
    cudaMemsetAsync(loss_dev + i, 0, sizeof(float), w);
    // colour inside the preprocess kernel: the views' front ends already run side by side, a side stream per view only adds work
    rc = preprocess_impl(sc, &views[i], c, b.ws, b.ws_bytes, cap, w, nullptr, nullptr, false);
    if (!rc) rc = forward_entry(sc, &views[i], c, b.ws, b.ws_bytes, cap, w, b.image, b.final_T, b.n_contrib, nullptr, false);
    if (b.target_host) cudaStreamWaitEvent(w, ctx->copy_done[i], 0);     // also on the error path: the copy is joined through this stream
    if (!rc) rc = step_loss(carve(b.ws, sc->N, K, views[i].width, views[i].height, cap), b.image, b.target_dev, (int64_t)count, b.dL_dimage, loss_dev + i, w);
    // blend backward of this view overlaps everything of the others.  B2: with the batched colour pass every view stops
    // after B1 and the backward preprocess of all views follows below; otherwise B2 runs here, chained view after view
    if (!rc) rc = backward_impl(sc, &views[i], c, b.ws, b.ws_bytes, cap, w, b.dL_dimage, b.final_T, b.n_contrib, g,
                                batched_b2 ? nullptr : (i > 0 ? ctx->b2_done[i - 1] : (zero ? ctx->zero_done : nullptr)), nullptr, nullptr, batched_b2);
    cudaEventRecord(ctx->b2_done[i], w);
  }
  if (batched_b2 && !rc && launched == num_views) {
    // One pass over the primitives does the colour part (A4) for every view that sees them: coefficient and gradient
    // blocks of a primitive shared by several views move once.  Then the geometry part view by view (each reads its own
    // dcol and read-modify-writes the caller's arrays, so they stay in order on one stream).
    cudaStream_t w0 = ctx->worker[0];
    for (int i = 1; i < num_views; ++i) cudaStreamWaitEvent(w0, ctx->b2_done[i], 0);
    if (zero) cudaStreamWaitEvent(w0, ctx->zero_done, 0);
    Workspace wss[FDGS_MAX_BATCH]; float inv_T[FDGS_MAX_BATCH];
    for (int i = 0; i < num_views; ++i) { wss[i] = carve(bufs[i].ws, sc->N, K, views[i].width, views[i].height, cap); inv_T[i] = 1.0f / views[i].period_T; }
    launch_colour_bwd_batch(*sc, num_views, wss, inv_T, *g, zero, w0);
    cudaEventRecord(ctx->colour_done, w0);
    for (int i = 0; i < num_views; ++i) {      // geometry part: the views side by side on their own streams, sums by reductions
      ViewParams vp; CfgParams cp;
      make_params(&views[i], c, vp, cp);
      if (i > 0) cudaStreamWaitEvent(ctx->worker[i], ctx->colour_done, 0);
      launch_geom_bwd(*sc, vp, cp, wss[i], *g, ctx->worker[i]);
      cudaEventRecord(ctx->b2_done[i], ctx->worker[i]);
    }
  }
  for (int i = 0; i < launched; ++i) cudaStreamWaitEvent(st, ctx->b2_done[i], 0);
  if (zero) cudaStreamWaitEvent(st, ctx->zero_done, 0);
  if (copies) { cudaEventRecord(ctx->copy_join, ctx->copy_stream); cudaStreamWaitEvent(st, ctx->copy_join, 0); }
  if (rc) { cudaStreamSynchronize(st); return rc; }
  FDGS_CUDA(cudaGetLastError(), "batch launches");
  if (loss_host) {
    FDGS_CUDA(cudaMemcpyAsync(loss_host, loss_dev, sizeof(float) * num_views, cudaMemcpyDeviceToHost, st), "D2H loss");
    FDGS_CUDA(cudaStreamSynchronize(st), "batch sync");
    for (int i = 0; i < num_views; ++i)
      if ((rc = read_overflow(carve(bufs[i].ws, sc->N, K, views[i].width, views[i].height, cap)))) return rc;
  }
  return FDGS_OK;
}

}  // extern "C"

// ---- feature channels and optical flow (features.cu) ---------------------------------------------------------------
struct FeatScratch { SplatRec* rec; float* img3; float* final_T; unsigned int* n_contrib; size_t bytes; };
static FeatScratch carve_feat(void* base, long long N, long long W, long long H) {
  FeatScratch f; size_t off = 0;
  auto take = [&](size_t b) { void* p = base ? (char*)base + off : nullptr; off += align_up(b); return p; };
  f.rec = (SplatRec*)take(sizeof(SplatRec) * (size_t)(N > 0 ? N : 1));
  f.img3 = (float*)take(sizeof(float) * 3 * W * H);
  f.final_T = (float*)take(sizeof(float) * W * H);
  f.n_contrib = (unsigned int*)take(sizeof(unsigned int) * W * H);
  f.bytes = off;
  return f;
}

int fdgs_features_scratch_bytes(int32_t N, int32_t W, int32_t H, size_t* bytes_host) {
  if (!bytes_host || N < 0 || W <= 0 || H <= 0) return FDGS_ERR_INVALID;
  *bytes_host = carve_feat(nullptr, N, W, H).bytes;
  return FDGS_OK;
}

static int features_common(const fdgs_scene* sc, const fdgs_view* v, const fdgs_config* c, void* ws_ptr, size_t ws_bytes, int64_t cap,
                           const float* feat, int32_t C, void* scratch, size_t scratch_bytes, Workspace& ws, FeatScratch& fs,
                           ViewParams& vp, CfgParams& cp, int* l1, int* l2) {
  int rc = check_common(sc, v, c, ws_ptr);
  if (rc) return rc;
  if (C < 1 || cap < 1 || cap >= (1LL << 30) || !scratch || !aligned16(scratch) || (sc->N > 0 && !feat)) return FDGS_ERR_INVALID;
  if (!aligned16(feat)) return FDGS_ERR_INVALID;          // rows of feat[N,C] are read with 128-bit loads when C % 4 == 0
  const int K = sc->n_time * (sc->sh_degree + 1) * (sc->sh_degree + 1);
  ws = carve(ws_ptr, sc->N, K, v->width, v->height, cap);
  if (ws.bytes > ws_bytes) return FDGS_ERR_WORKSPACE;
  fs = carve_feat(scratch, sc->N, v->width, v->height);
  if (fs.bytes > scratch_bytes) return FDGS_ERR_WORKSPACE;
  make_params(v, c, vp, cp);
  vp.bg[0] = vp.bg[1] = vp.bg[2] = 0.f;                 // features have no background term
  *l1 = depth_buf(); *l2 = 0;
  return FDGS_OK;
}

extern "C" {

int fdgs_render_features_forward(const fdgs_scene* sc, const fdgs_view* v, const fdgs_config* c, void* ws_ptr, size_t ws_bytes,
                                 int64_t cap, void* stream, const float* feat, int32_t C, void* scratch, size_t scratch_bytes,
                                 float* out) {
  Workspace ws; FeatScratch fs; ViewParams vp; CfgParams cp; int l1, l2;
  int rc = features_common(sc, v, c, ws_ptr, ws_bytes, cap, feat, C, scratch, scratch_bytes, ws, fs, vp, cp, &l1, &l2);
  if (rc) return rc;
  if (!out) return FDGS_ERR_INVALID;
  cudaStream_t st = (cudaStream_t)stream;
  const size_t HW = (size_t)v->width * v->height;
  (void)HW;
  // dedicated C-channel kernel: alpha evaluated once per 16 channels, features gathered by id next to the records
  launch_blend_feat_fwd(ws, vp, cp, feat, C, out, st);
  FDGS_CUDA(cudaGetLastError(), "feature forward launches");
  return FDGS_OK;
}

int fdgs_render_features_backward(const fdgs_scene* sc, const fdgs_view* v, const fdgs_config* c, void* ws_ptr, size_t ws_bytes,
                                  int64_t cap, void* stream, const float* feat, int32_t C, void* scratch, size_t scratch_bytes,
                                  const float* dL_dout, const float* final_T, const uint32_t* n_contrib, float* grad_feat,
                                  const fdgs_grads* g) {
  Workspace ws; FeatScratch fs; ViewParams vp; CfgParams cp; int l1, l2;
  int rc = features_common(sc, v, c, ws_ptr, ws_bytes, cap, feat, C, scratch, scratch_bytes, ws, fs, vp, cp, &l1, &l2);
  if (rc) return rc;
  if (!dL_dout || !final_T || !n_contrib || (sc->N > 0 && !grad_feat)) return FDGS_ERR_INVALID;
  if (g && (rc = check_grads(sc, g))) return rc;
  if (sc->N == 0) return FDGS_OK;
  cudaStream_t st = (cudaStream_t)stream;
  if (!g) {   // geometry frozen: dL/dfeat only needs the weights alpha_k T_k — dedicated front-to-back kernel
    launch_blend_feat_bwd(ws, vp, cp, dL_dout, C, grad_feat, st);
    FDGS_CUDA(cudaGetLastError(), "feature backward launches");
    return FDGS_OK;
  }
  FDGS_CUDA(cudaMemsetAsync(ws.g9, 0, sizeof(float) * 9 * (size_t)sc->N, st), "memset(g9)");
  // one C-channel pass per 32 channels: dL/dfeat to grad_feat, the gradient through alpha_k and T_k to the geometry slots of g9
  launch_blend_feat_bwd_geom(ws, vp, cp, feat, dL_dout, C, final_T, n_contrib, grad_feat, st);
  // chain (u, v, conic, opacity) to the parameters once; the colour slots are zero, so the 4DSH coefficients get nothing
  if (g) launch_preprocess_bwd(*sc, vp, cp, ws, l1, *g, false, st);
  FDGS_CUDA(cudaGetLastError(), "feature backward launches");
  return FDGS_OK;
}

int fdgs_splat_flow(const fdgs_scene* sc, const fdgs_view* v, const fdgs_config* c, void* ws_ptr, size_t ws_bytes, int64_t cap,
                    void* stream, float dt_next, float* flow) {
  int rc = check_common(sc, v, c, ws_ptr);
  if (rc) return rc;
  if (cap < 1 || cap >= (1LL << 30) || (sc->N > 0 && (!flow || (reinterpret_cast<uintptr_t>(flow) & 7u)))) return FDGS_ERR_INVALID;
  const int K = sc->n_time * (sc->sh_degree + 1) * (sc->sh_degree + 1);
  const Workspace ws = carve(ws_ptr, sc->N, K, v->width, v->height, cap);
  if (ws.bytes > ws_bytes) return FDGS_ERR_WORKSPACE;
  if (sc->N == 0) return FDGS_OK;
  ViewParams vp; CfgParams cp;
  make_params(v, c, vp, cp);
  launch_splat_flow(*sc, vp, cp, ws, dt_next, flow, (cudaStream_t)stream);
  FDGS_CUDA(cudaGetLastError(), "flow launch");
  return FDGS_OK;
}

}  // extern "C"

extern "C" {

int64_t fdgs_launch_count(void) { return launch_count_value(); }

int fdgs_set_stage_timing(int enable) {
  if (enable && !g_timing) for (int i = 0; i < EV_COUNT; ++i) FDGS_CUDA(cudaEventCreate(&g_ev[i]), "event create");
  if (!enable && g_timing) for (int i = 0; i < EV_COUNT; ++i) cudaEventDestroy(g_ev[i]);
  g_timing = enable ? 1 : 0;
  return FDGS_OK;
}

int fdgs_get_stage_ms(float* ms_host) {
  if (!ms_host || !g_timing) return FDGS_ERR_INVALID;
  const int pairs[8][2] = {{EV_PRE0, EV_PRE1}, {EV_PRE1, EV_PRE2}, {EV_FWD0, EV_FWD1}, {EV_FWD1, EV_FWD2},
                           {EV_FWD2, EV_FWD3}, {EV_BWD0, EV_BWD1}, {EV_BWD1, EV_BWD2}, {EV_COL0, EV_COL1}};
  for (int k = 0; k < 8; ++k) {
    ms_host[k] = -1.f;
    if (cudaEventSynchronize(g_ev[pairs[k][1]]) == cudaSuccess) cudaEventElapsedTime(&ms_host[k], g_ev[pairs[k][0]], g_ev[pairs[k][1]]);
  }
  cudaGetLastError();   // stages that never ran leave an error state behind: clear it
  return FDGS_OK;
}

int fdgs_debug_blend_stats(const fdgs_view* v, const fdgs_config* c, void* ws_ptr, size_t ws_bytes, int32_t N, int32_t K,
                           int64_t cap, void* stream, unsigned long long* stats_dev) {
  if (!v || !c || !ws_ptr || !stats_dev) return FDGS_ERR_INVALID;
  const Workspace ws = carve(ws_ptr, N, K, v->width, v->height, cap);
  if (ws.bytes > ws_bytes) return FDGS_ERR_WORKSPACE;
  ViewParams vp; CfgParams cp;
  make_params(v, c, vp, cp);
  FDGS_CUDA(cudaMemsetAsync(stats_dev, 0, 4 * sizeof(unsigned long long), (cudaStream_t)stream), "memset(stats)");
  launch_blend_stats(ws, vp, cp, stats_dev, (cudaStream_t)stream);
  FDGS_CUDA(cudaGetLastError(), "stats launch");
  return FDGS_OK;
}

int fdgs_debug_cull_status(const fdgs_scene* sc, const fdgs_view* v, const fdgs_config* c, void* stream, unsigned char* status_dev) {
  if (!sc || !v || !c || !status_dev || sc->N < 0 || v->width <= 0 || v->height <= 0 || !(v->period_T > 0) || check_cfg(c)) return FDGS_ERR_INVALID;
  ViewParams vp; CfgParams cp;
  make_params(v, c, vp, cp);
  launch_cull_status(*sc, vp, cp, status_dev, (cudaStream_t)stream);
  FDGS_CUDA(cudaGetLastError(), "cull status launch");
  return FDGS_OK;
}

int fdgs_debug_measure_peaks(void* scratch_dev, size_t scratch_bytes, void* stream, float* fma_tlane_per_s_host, float* mufu_t_per_s_host) {
  if (!scratch_dev || !fma_tlane_per_s_host || !mufu_t_per_s_host) return FDGS_ERR_INVALID;
  const int blocks = 8 * num_sms(), threads = 256;
  if (scratch_bytes < sizeof(float) * (size_t)blocks * threads) return FDGS_ERR_WORKSPACE;
  cudaStream_t st = (cudaStream_t)stream;
  cudaEvent_t e0, e1;
  FDGS_CUDA(cudaEventCreate(&e0), "event create");
  FDGS_CUDA(cudaEventCreate(&e1), "event create");
  float best_fma = 0.f, best_mufu = 0.f;
  for (int rep = 0; rep < 4; ++rep) {          // first repetition warms up; best of the rest
    const int it_f = 4000, it_m = 1000;
    float ms = 0.f;
    cudaEventRecord(e0, st);
    peak_fma_kernel<<<blocks, threads, 0, st>>>((float*)scratch_dev, it_f, 0.999f);
    cudaEventRecord(e1, st);
    FDGS_CUDA(cudaEventSynchronize(e1), "peak sync");
    cudaEventElapsedTime(&ms, e0, e1);
    if (rep) best_fma = fmaxf(best_fma, (float)((double)blocks * threads * it_f * 64.0 / (ms * 1e-3) / 1e12));
    cudaEventRecord(e0, st);
    peak_mufu_kernel<<<blocks, threads, 0, st>>>((float*)scratch_dev, it_m);
    cudaEventRecord(e1, st);
    FDGS_CUDA(cudaEventSynchronize(e1), "peak sync");
    cudaEventElapsedTime(&ms, e0, e1);
    if (rep) best_mufu = fmaxf(best_mufu, (float)((double)blocks * threads * it_m * 64.0 / (ms * 1e-3) / 1e12));
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  FDGS_CUDA(cudaGetLastError(), "peak kernels");
  *fma_tlane_per_s_host = best_fma; *mufu_t_per_s_host = best_mufu;
  return FDGS_OK;
}

const char* fdgs_strerror(int code) {
  switch (code) {
    case FDGS_OK: return "ok";
    case FDGS_ERR_INVALID: return "invalid argument";
    case FDGS_ERR_WORKSPACE: return "workspace too small (see fdgs_workspace_bytes)";
    case FDGS_ERR_CUDA: return g_cuda_err;
    case FDGS_ERR_PAIR_OVERFLOW: return "number of (tile, primitive) pairs exceeds pair_capacity";
    case FDGS_ERR_STATIC_LIMIT: return "sizes exceed the built-in workspace of fdgs_render_forward_static (FDGS_STATIC_WS_BYTES)";
    default: return "unknown error";
  }
}

}  // extern "C"

extern "C" int fdgs_debug_export(const void* ws_ptr, size_t ws_bytes, int what, void* dst, size_t dst_bytes, void* stream) {
  if (!ws_ptr || !dst) return FDGS_ERR_INVALID;
  cudaStream_t st = (cudaStream_t)stream;
  FDGS_CUDA(cudaStreamSynchronize(st), "export sync");
  WsHeader h;
  FDGS_CUDA(cudaMemcpy(&h, ws_ptr, sizeof(h), cudaMemcpyDeviceToHost), "export header");
  const Workspace ws = carve(const_cast<void*>(ws_ptr), h.N, h.K, h.W, h.H, h.pair_capacity);
  if (ws.bytes > ws_bytes) return FDGS_ERR_WORKSPACE;
  const long long N = h.N, D = h.num_pairs;
  const int l1 = depth_buf();
  size_t need = 0;
  const void* src = nullptr;
  switch (what) {
    case FDGS_EXPORT_STATUS: {
      const long long status[4] = {(long long)h.total_pairs, (long long)h.num_visible, (long long)h.overflow, h.pair_capacity};
      if (dst_bytes < sizeof(status)) return FDGS_ERR_INVALID;
      FDGS_CUDA(cudaMemcpy(dst, status, sizeof(status), cudaMemcpyHostToDevice), "export status");
      return h.overflow ? FDGS_ERR_PAIR_OVERFLOW : FDGS_OK;
    }
    case FDGS_EXPORT_RECORDS:
      if (dst_bytes < sizeof(float) * 12 * (size_t)N) return FDGS_ERR_INVALID;
      if (N > 0) export_records_kernel<<<(unsigned)((N + 255) / 256), 256, 0, st>>>(ws.rec, ws.tiles_touched, (int)N, (float*)dst);
      break;
    case FDGS_EXPORT_RECTS:
      if (dst_bytes < sizeof(int) * 4 * (size_t)N) return FDGS_ERR_INVALID;
      if (N > 0) export_rects_kernel<<<(unsigned)((N + 255) / 256), 256, 0, st>>>(ws.rect, (int)N, (int4*)dst);
      break;
    case FDGS_EXPORT_TILES_TOUCHED: src = ws.tiles_touched; need = 4 * (size_t)N; break;
    case FDGS_EXPORT_DEPTH_ORDER: src = ws.sorted_ids; need = 4 * (size_t)h.num_visible; break;
    case FDGS_EXPORT_SORTED_KEYS:
      if (dst_bytes < 8 * (size_t)D) return FDGS_ERR_INVALID;
      if (D > 0) export_keys_kernel<<<(unsigned)((D + 255) / 256), 256, 0, st>>>(ws.ranges, (int)h.tiles, ws.pair_ids, ws.rec, (unsigned)D, (unsigned long long*)dst);
      break;
    case FDGS_EXPORT_SORTED_VALS: src = ws.pair_ids; need = 4 * (size_t)D; break;
    case FDGS_EXPORT_RANGES: src = ws.ranges; need = 8 * (size_t)h.tiles; break;
    case FDGS_EXPORT_SPLAT_GRADS: src = ws.g9; need = 36 * (size_t)N; break;
    case FDGS_EXPORT_SPLAT_GRAD_DEPTH: src = ws.gz; need = 4 * (size_t)N; break;
    default: return FDGS_ERR_INVALID;
  }
  if (src) {
    if (dst_bytes < need) return FDGS_ERR_INVALID;
    if (need) FDGS_CUDA(cudaMemcpyAsync(dst, src, need, cudaMemcpyDeviceToDevice, st), "export copy");
  }
  FDGS_CUDA(cudaGetLastError(), "export launch");
  FDGS_CUDA(cudaStreamSynchronize(st), "export sync");
  return FDGS_OK;
}

// ---- fdgs_render_forward_static: the forward of one view on a workspace that nobody allocates ----------------------
// The workspace of this entry point is a file-scope device array: it exists on every GPU that loads the library, from
// the load to the exit of the process.  In host code `g_static_ws` is only the host-side stand-in of the symbol, not a
// device address — a kernel given that name would fault, or write somewhere in host memory where the GPU can reach it —
// so the address is asked for once per device, with that device current, and it is the answer that reaches the kernels.
namespace fdgs {

static __device__ __align__(256) unsigned char g_static_ws[FDGS_STATIC_WS_BYTES];

struct StaticCtx {
  bool ready = false;
  void* ws = nullptr;   // device address of g_static_ws on this device
  int sms = 0;
};
static StaticCtx g_static[MAX_DEVICES];
static std::mutex g_static_mutex;

static int static_ctx(StaticCtx** out) {
  int dev = 0;
  FDGS_CUDA(cudaGetDevice(&dev), "cudaGetDevice");
  if (dev < 0 || dev >= MAX_DEVICES) return FDGS_ERR_INVALID;
  std::lock_guard<std::mutex> lock(g_static_mutex);
  StaticCtx& c = g_static[dev];
  if (!c.ready) {
    void* p = nullptr;
    FDGS_CUDA(cudaGetSymbolAddress(&p, g_static_ws), "cudaGetSymbolAddress(static workspace)");
    if (!p || (reinterpret_cast<uintptr_t>(p) & 255u)) return cuda_fail(cudaErrorInvalidSymbol, "static workspace address");
    FDGS_CUDA(cudaDeviceGetAttribute(&c.sms, cudaDevAttrMultiProcessorCount, dev), "SM count");
    if (c.sms <= 0) c.sms = 148;
    c.ws = p;
    c.ready = true;
  }
  *out = &c;
  return FDGS_OK;
}

}  // namespace fdgs

extern "C" int fdgs_render_forward_static(const fdgs_scene* sc, const fdgs_view* v, const fdgs_config* c, int64_t cap, void* stream,
                                          float* image, float* final_T, uint32_t* n_contrib, uint32_t* overflow_dev) {
  if (!sc || !v || !c || !image || !final_T || !n_contrib || cap < 1 || cap >= (1LL << 30)) return FDGS_ERR_INVALID;
  // the size check comes before anything touches the device: the layout is a function of the sizes alone
  if (sc->N < 0 || v->width <= 0 || v->height <= 0 || sc->n_time < 1 || sc->sh_degree < 0) return FDGS_ERR_INVALID;
  const int K = sc->n_time * (sc->sh_degree + 1) * (sc->sh_degree + 1);
  if (carve(nullptr, sc->N, K, v->width, v->height, cap).bytes > (size_t)FDGS_STATIC_WS_BYTES) return FDGS_ERR_STATIC_LIMIT;
  StaticCtx* ctx = nullptr;
  int rc = static_ctx(&ctx);
  if (rc) return rc;
  if ((rc = check_common(sc, v, c, ctx->ws))) return rc;
  const Workspace ws = carve(ctx->ws, sc->N, K, v->width, v->height, cap);
  cudaStream_t st = (cudaStream_t)stream;
  ViewParams vp; CfgParams cp;
  make_params(v, c, vp, cp);
  // same sequence as fdgs_preprocess + fdgs_render_forward.  The array keeps what the last call left in it: everything
  // that has to start from zero (header, coverage grid, scan states, digit counts, look-back regions) is the prefix
  // cleared here; the rest is written before it is read.
  FDGS_CUDA(cudaMemsetAsync(ctx->ws, 0, ws.zero_bytes, st), "memset(static header)");
  launch_preprocess_fwd(*sc, vp, cp, ws, st, false);       // colour inside the kernel: this entry point creates nothing, not even a side stream
  launch_compact_and_tile_grid(ws, sc->N, K, vp, cp, cap, st);
  launch_sort_depth(ws, sc->N, ctx->sms, st);
  launch_row_ballots(ws, sc->N, vp, ctx->sms, st);
  launch_row_scatter(ws, sc->N, vp, ctx->sms, st);
  launch_blend_fwd(ws, vp, cp, image, final_T, n_contrib, nullptr, st);
  if (overflow_dev) FDGS_CUDA(cudaMemcpyAsync(overflow_dev, &ws.hdr->overflow, sizeof(uint32_t), cudaMemcpyDeviceToDevice, st), "copy overflow flag");
  FDGS_CUDA(cudaGetLastError(), "static forward launches");
  return FDGS_OK;
}
