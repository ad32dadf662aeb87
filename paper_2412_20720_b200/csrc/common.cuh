// common.cuh — shared declarations of the fdgs CUDA path (sm_100a).  Product code: shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string.h>

#include "../../include/fdgs.h"

namespace fdgs {

constexpr int TILE = FDGS_TILE;
constexpr int TILE_PIX = TILE * TILE;

// Per-primitive record written by preprocess (48 B, 16-B aligned; gathered by id in the blend).
//   q0 = (u, v, ca, cb)   q1 = (cc, lo, r, g)   q2 = (b, depth, radius, w)
// (ca, cb, cc) is the Cholesky-like factor of the conic scaled for exp2:
//   log2(alpha) = lo - e1^2 - e2^2,  e1 = ca*dx + cb*dy,  e2 = cc*dy,  dx = u - px, dy = v - py
//   with ca = sqrt(k A), cb = k B / ca, cc = sqrt(k (C - B^2/A)), k = log2(e)/2, lo = log2(o).
// The exponent is <= lo by construction, so no "power > 0" clamp is needed (S10).
struct __align__(16) SplatRec {
  float u, v, ca, cb;
  float cc, lo, r, g;
  float b, depth, radius, w;
};
static_assert(sizeof(SplatRec) == 48, "SplatRec must be 48 bytes");

struct ViewParams {   // by-value kernel parameter
  float W[3][3], tau[3];
  float cam[3];       // camera centre -W^T tau
  float fx, fy, cx, cy;
  int width, height, tiles_x, tiles_y;
  float t, inv_T;     // query time, 1 / period_T
  float bg[3];
  float limx, limy;   // guard band: guard * W / (2 fx), guard * H / (2 fy)
};

struct CfgParams {
  float marginal_min, alpha_min, alpha_max, transmittance_min, dilation, cutoff_sigma, znear, guard;
  float log2_alpha_min;   // log2(alpha_min) (-inf if alpha_min == 0)
  int default_thresholds; // 1: alpha_min, alpha_max, transmittance_min are the values of [23] (S8) — the blend
                          // kernels then run an instantiation with the four thresholds as immediates
};

// Thresholds of [23] ("adopted the settings of [23]"; S8).  A kernel argument used in the
// blend loops costs a constant-bank load per use on sm_100a (LDCU / LDC in SASS: ptxas does not keep it in a register),
// so the hot kernels have an instantiation with these as immediates.
#define FDGS_DEF_ALPHA_MIN (1.0f / 255.0f)
#define FDGS_DEF_ALPHA_MAX 0.99f
#define FDGS_DEF_T_MIN 1e-4f
#define FDGS_DEF_L2MIN (-0x1.ffa3ap+2f)   // log2f(1/255) * (1 + 1e-6) - 1e-6 in fp32 (= -7.994362)

// Device-side header at the start of the workspace (zeroed by fdgs_preprocess; the layout mirror is then written by the
// preprocess kernel's first thread).
struct WsHeader {
  unsigned int num_pairs;         // D (written by the tile-grid role of the compaction kernel); 0 if D > pair_capacity
  unsigned int num_visible;       // survivors of all culls (written by the compaction scan)
  unsigned int overflow;          // 1 if D > pair_capacity
  unsigned int scan_ticket[2];    // dynamic tile ids of the two chained scans
  unsigned int sort_ticket[4];    // one per radix pass of the depth sort
  unsigned int total_pairs;       // D even when it overflows
  unsigned int pad[6];
  long long N, K, W, H, pair_capacity, tiles;   // layout mirror for fdgs_debug_export
};

// Depth sort: LSD radix sort of key' = fp32 bits of the camera depth - fp32 bits of znear (every survivor has
// z > znear, so key' > 0 and the order is that of the depth bits).  9-bit digits: three passes cover key' < 2^27, i.e. depths
// up to 2^16 znear (13 km at znear = 0.2); a fourth pass over the remaining five bits is launched as well but returns at
// once unless a survivor has such a depth (the digit counts of all four passes come from the compaction kernel).
constexpr int RADIX_BITS = 9;
constexpr int RADIX = 1 << RADIX_BITS;
constexpr int SORT_THREADS = 256;
#ifndef FDGS_SORT_ITEMS
#define FDGS_SORT_ITEMS 8
#endif
constexpr int SORT_ITEMS_L1 = FDGS_SORT_ITEMS;   // 2048-key tiles: 0.206 ms per 4 views at cfg3 (4: 0.212, 16: 0.259)    // depth sort of <= N survivors: small tiles, more CTAs
constexpr int DEPTH_PASSES = 4;                  // 3 x 9 bits + the optional pass over bits 27..31
constexpr int SCAN_THREADS = 256;
#ifndef FDGS_SCAN_ITEMS
#define FDGS_SCAN_ITEMS 8
#endif
constexpr int SCAN_ITEMS = FDGS_SCAN_ITEMS;
static_assert(RADIX == 2 * SCAN_THREADS && RADIX == 2 * SORT_THREADS, "a thread of the compaction / sort kernels owns two digits");
constexpr int SCAN_TILE = SCAN_THREADS * SCAN_ITEMS;
constexpr int RS_MIN_CHUNK = 2048, RS_MAX_CHUNK = 32768;   // survivors per chunk of the row scatter (scan_dup.cu)
constexpr int RS_MAX_ITERS = RS_MAX_CHUNK / 32;
constexpr int MAX_GRID_CELLS = 50000;   // (tiles_x+1)*(tiles_y+1) must fit the shared memory of the tile-grid / scatter kernels

// Host-side view of the carved-up workspace.
//
// Binning is two-level: survivors are first sorted by their fp32 depth bits (level 1, <= N items,
// hand-written onesweep radix sort); the (tile, id) pairs are then written in that order straight to their final
// position in the per-tile lists by a stable, rectangle-aware scatter (level 2, "row scatter": one CTA per chunk of
// survivors and tile row; no key array exists).  The resulting per-tile lists are exactly those of one stable sort on the
// 64-bit key tile<<32 | depth-bits with ties in id order.
struct Workspace {
  WsHeader* hdr;
  int* tile_diff;                    // [(tiles_y+1)*(tiles_x+1)] 2D difference array of tile coverage
  unsigned long long* scan_state[2]; // look-back words of the two scans
  unsigned int* sort_hist;           // [4][RADIX] digit counts of the 4 depth passes (raw, accumulated by the compaction kernel)
  unsigned int* sort_lookback;       // [4][depth-sort tiles][RADIX]: one region per pass, cleared with the header
  size_t lookback_stride;            // words per pass
  SplatRec* rec;                     // [N] indexed by primitive id
  ushort4* rect;                     // [N] tx0, ty0, tx1, ty1
  unsigned int* tiles_touched;       // [N]
  unsigned int* l1_keys[2];          // [N] depth keys of the survivors (fp32 depth bits - fp32 bits of znear; double buffer)
  unsigned int* l1_vals[2];          // [N] primitive ids of the survivors (double buffer of the sort)
  unsigned int* vis_ids;             // [N] primitive ids of survivors in ascending id order (kept for the backward)
  unsigned int* sorted_ys;           // [N] tile rows   y0 | y1 << 16 of the survivors in depth order (written by the last depth-sort pass)
  unsigned int* sorted_xs;           // [N] tile columns x0 | x1 << 16, same order
  unsigned int* sorted_ids;          // [N] primitive ids of the survivors in depth order (same pass: the pass count is decided on the device)
  unsigned int* row_ballots;         // [tiles_y][rb_stride] bit i of word (y, it): survivor 32 it + i (depth order) covers tile row y
  size_t rb_stride;                  // words per tile row (>= ceil(N / 32))
  unsigned int rs_chunk, rs_chunks;  // survivors per chunk of the row scatter; chunks N is divided into
  unsigned int* rs_state;            // [rs_chunks][tiles] look-back words of the row scatter (count of chunk c in tile T), cleared with the header
  unsigned int* pair_ids;            // [cap] primitive ids of the per-tile lists, tile after tile (ranges), depth order inside
  uint2* ranges;                     // [tiles] [first, last+1)
  float* g9;                         // [N,9] per-splat gradients of the blend backward
  float4* aux;                       // [N] survivors: view direction (x, y, z) and (t - mu_t) / T, written by preprocess
  float4* dcol;                      // [N] survivors: colour backward -> geometry backward: dL/d dir (x, y, z), dL/d Delta
  float* gz;                         // [N] auxiliary depth channel: dL/d(camera depth) per splat
  size_t zero_bytes;                 // prefix of the workspace cleared by fdgs_preprocess
  size_t bytes;
};

inline size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

// what the compaction kernel subtracts from the fp32 depth bits of a survivor (see RADIX_BITS above)
inline unsigned int depth_key_base(const CfgParams& cp) { unsigned int u; memcpy(&u, &cp.znear, sizeof(u)); return u; }

inline Workspace carve(void* base, long long N, long long K, long long W, long long H, long long cap) {
  Workspace w;
  char* p = (char*)base;
  size_t off = 0;
  auto take = [&](size_t bytes) { char* q = p ? p + off : nullptr; off += align_up(bytes); return q; };
  const long long tx = (W + TILE - 1) / TILE, ty = (H + TILE - 1) / TILE, tiles = tx * ty;
  const long long Np = N > 0 ? N : 1;
  w.hdr = (WsHeader*)take(sizeof(WsHeader));
  w.tile_diff = (int*)take(4 * (size_t)(tx + 1) * (ty + 1));
  for (int i = 0; i < 2; ++i) w.scan_state[i] = (unsigned long long*)take(8 * (Np / 256 + 2));   // chained-scan tiles of >= 256 items
  w.sort_hist = (unsigned int*)take(4 * DEPTH_PASSES * RADIX);     // accumulated by the compaction kernel
  const long long t1 = (Np + SORT_THREADS * SORT_ITEMS_L1 - 1) / (SORT_THREADS * SORT_ITEMS_L1);
  w.lookback_stride = (size_t)RADIX * (size_t)(t1 + 1);
  w.sort_lookback = (unsigned int*)take(4 * w.lookback_stride * DEPTH_PASSES);
  long long ch = ((Np + 127) / 128 + 255) / 256 * 256;    // <= 128 chunks unless that makes them larger than RS_MAX_CHUNK
  if (ch < RS_MIN_CHUNK) ch = RS_MIN_CHUNK;
  if (ch > RS_MAX_CHUNK) ch = RS_MAX_CHUNK;
  w.rs_chunk = (unsigned int)ch;
  w.rs_chunks = (unsigned int)((Np + ch - 1) / ch);
  w.rs_state = (unsigned int*)take(4 * (size_t)w.rs_chunks * (size_t)tiles);
  w.zero_bytes = off;
  w.rec = (SplatRec*)take(sizeof(SplatRec) * Np);
  w.rect = (ushort4*)take(sizeof(ushort4) * Np);
  w.tiles_touched = (unsigned int*)take(4 * Np);
  for (int i = 0; i < 2; ++i) w.l1_keys[i] = (unsigned int*)take(4 * Np);
  for (int i = 0; i < 2; ++i) w.l1_vals[i] = (unsigned int*)take(4 * Np);
  w.vis_ids = (unsigned int*)take(4 * Np);
  w.sorted_ys = (unsigned int*)take(4 * Np);
  w.sorted_xs = (unsigned int*)take(4 * Np);
  w.sorted_ids = (unsigned int*)take(4 * Np);
  w.rb_stride = (size_t)((Np + 31) / 32 + 31) / 32 * 32;
  w.row_ballots = (unsigned int*)take(4 * w.rb_stride * (size_t)ty);
  w.pair_ids = (unsigned int*)take(4 * (size_t)cap);
  w.ranges = (uint2*)take(sizeof(uint2) * tiles);
  w.g9 = (float*)take(4 * 9 * Np);
  w.aux = (float4*)take(16 * Np);
  w.dcol = (float4*)take(16 * Np);
  w.gz = (float*)take(4 * Np);
  (void)K;
  w.bytes = off;
  return w;
}

#ifdef __CUDACC__
// Ask L2 for every 128-byte line of [p, p + bytes): the request costs no register and no scoreboard slot, so a thread
// can have its whole record on the way while it is still doing arithmetic.
__device__ __forceinline__ void prefetch_l2(const void* p, const int bytes) {
  const char* c = reinterpret_cast<const char*>(reinterpret_cast<uintptr_t>(p) & ~(uintptr_t)127);
  const char* end = reinterpret_cast<const char*>(p) + bytes;
  for (; c < end; c += 128) asm volatile("prefetch.global.L2 [%0];" ::"l"(c));
}
#endif

// Launch counter (fdgs_launch_count) — bumped by every launcher (atomic: launchers may run on several host threads).
void count_launch(int n = 1);
long long launch_count_value();
// Records the CUDA error text for fdgs_strerror and returns FDGS_ERR_CUDA (api.cu).
int cuda_fail(cudaError_t e, const char* where);

// Launchers (each file implements its own; all asynchronous on `st`).
// split_colour (degree-3 scenes only): stop after the geometry (A1-A3) and leave the colour slots of the records to
// launch_colour_fwd, which fdgs_render_forward runs on a side stream under the binning launches
void launch_preprocess_fwd(const fdgs_scene& sc, const ViewParams& vp, const CfgParams& cp, const Workspace& ws, cudaStream_t st, bool split_colour);
// A4 of a degree-3 scene: colour of the visible survivors into the records (after the compaction; only the blend reads it).
// false: nothing to do (the preprocess kernel of the other degrees evaluates the colour itself).
bool launch_colour_fwd(const fdgs_scene& sc, const Workspace& ws, int num_sms, cudaStream_t st);
// compaction scan: survivors (tiles_touched > 0) in id order -> l1_keys[0] (depth bits), l1_vals[0] (ids), hdr->num_visible;
// the same launch carries, as the role of its first CTA, the 2D prefix of the coverage difference array -> ranges, D, overflow
void launch_compact_and_tile_grid(const Workspace& ws, int N, int K, const ViewParams& vp, const CfgParams& cp, long long cap, cudaStream_t st);
// Stable LSD radix sort of the survivors' (depth key, id) pairs on all key bits (three 9-bit passes, a fourth if a key
// needs it); the count is read on the device and ws.sort_hist[pass] holds the digit counts of the pass.  The last pass
// that runs also writes the ids and the tile rectangles of the survivors in the final order (sorted_ids / sorted_ys /
// sorted_xs).
void launch_sort_depth(const Workspace& ws, long long max_count, int num_sms, cudaStream_t st);
// level 2, first half: which survivors (depth order) cover which tile row, one ballot word per (row, 32 survivors)
void launch_row_ballots(const Workspace& ws, int N, const ViewParams& vp, int num_sms, cudaStream_t st);
// level 2: per-tile lists in depth order written straight to their final place (scan_dup.cu "row scatter")
void launch_row_scatter(const Workspace& ws, int N, const ViewParams& vp, int num_sms, cudaStream_t st);
void launch_blend_fwd(const Workspace& ws, const ViewParams& vp, const CfgParams& cp, float* image, float* final_T,
                      unsigned int* n_contrib, float* depth_map /*NULL = no auxiliary channel*/, cudaStream_t st);
void launch_blend_stats(const Workspace& ws, const ViewParams& vp, const CfgParams& cp, unsigned long long* stats, cudaStream_t st);
void launch_blend_bwd(const Workspace& ws, const ViewParams& vp, const CfgParams& cp, const float* dL_dimage,
                      const float* final_T, const unsigned int* n_contrib, const float* dL_ddepth, const float* dL_dopacity,
                      cudaStream_t st);
void launch_preprocess_bwd(const fdgs_scene& sc, const ViewParams& vp, const CfgParams& cp, const Workspace& ws, int l1_buf,
                           const fdgs_grads& g, bool with_gz, cudaStream_t st);
// batched step: colour part of the backward preprocess of all V views in one pass (false: not available for this scene),
// and the geometry part of one view
// grads_are_zero: g.sh was cleared for this step, so the pass writes its sums instead of adding to what it would have to read
bool launch_colour_bwd_batch(const fdgs_scene& sc, int V, const Workspace* ws, const float* inv_T, const fdgs_grads& g, bool grads_are_zero,
                             cudaStream_t st);
void launch_geom_bwd(const fdgs_scene& sc, const ViewParams& vp, const CfgParams& cp, const Workspace& ws, const fdgs_grads& g, cudaStream_t st);
void launch_cull_status(const fdgs_scene& sc, const ViewParams& vp, const CfgParams& cp, unsigned char* dst, cudaStream_t st);
void launch_blend_feat_fwd(const Workspace& ws, const ViewParams& vp, const CfgParams& cp, const float* feat, int C,
                           float* out, cudaStream_t st);
void launch_blend_feat_bwd(const Workspace& ws, const ViewParams& vp, const CfgParams& cp, const float* dL_dout, int C,
                           float* grad_feat, cudaStream_t st);
// feature backward with geometry gradients: dL/dfeat -> grad_feat, dL/d(u, v, A, B, C, o) -> ws.g9 (+=), 32 channels per launch
void launch_blend_feat_bwd_geom(const Workspace& ws, const ViewParams& vp, const CfgParams& cp, const float* feat, const float* dL_dout, int C,
                                const float* final_T, const unsigned int* n_contrib, float* grad_feat, cudaStream_t st);
void launch_splat_flow(const fdgs_scene& sc, const ViewParams& vp, const CfgParams& cp, const Workspace& ws, float dt_next, float* flow,
                       cudaStream_t st);
// overflow_flag (NULL ok): device word; if non-zero the loss written is NaN (fdgs_step_batch / fdgs_step_host)
void launch_l1_loss(const float* image, const float* target, long long count, float* dL, float* loss, const unsigned int* overflow_flag,
                    cudaStream_t st);

}  // namespace fdgs
