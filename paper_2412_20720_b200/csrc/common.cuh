// common.cuh — shared declarations of the fdgs CUDA path (sm_100a).  Product code: shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

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

// Device-side header at the start of the workspace (zeroed by fdgs_preprocess).
struct WsHeader {
  unsigned int num_pairs;         // D (written by the tile-grid kernel)
  unsigned int num_visible;       // survivors of all culls (written by the compaction scan)
  unsigned int overflow;          // 1 if D > pair_capacity
  unsigned int scan_ticket[2];    // dynamic tile ids of the two chained scans
  unsigned int sort_ticket[8];    // one per radix pass (4 depth passes + up to 4 tile-id passes)
  unsigned int pad[3];
  long long N, K, W, H, pair_capacity, tiles;   // layout mirror for fdgs_debug_export
};

constexpr int RADIX_BITS = 8;
constexpr int RADIX = 1 << RADIX_BITS;
constexpr int SORT_THREADS = 256;
constexpr int SORT_ITEMS_L1 = 4;    // depth sort of <= N survivors: small tiles, more CTAs
constexpr int SORT_ITEMS_L2 = 16;   // tile-id sort of D pairs
constexpr int SCAN_THREADS = 256;
constexpr int SCAN_ITEMS = 8;
constexpr int SCAN_TILE = SCAN_THREADS * SCAN_ITEMS;
constexpr int DUP_CHUNK = 2048;         // output pairs per CTA of the pair emission
constexpr int MAX_GRID_CELLS = 50000;   // (tiles_x+1)*(tiles_y+1) must fit the tile-grid kernel's shared memory

// Host-side view of the carved-up workspace.
//
// Sorting is two-level: survivors are first sorted by their fp32 depth bits
// (level 1, <= N items); pairs (tile, id) are then emitted in that order and stably sorted by tile id
// (level 2, D items, ceil(log2 tiles) bits).  The resulting per-tile lists are exactly those of one
// stable sort on the 64-bit key tile<<32 | depth-bits with ties in id order.
struct Workspace {
  WsHeader* hdr;
  int* tile_diff;                    // [(tiles_y+1)*(tiles_x+1)] 2D difference array of tile coverage
  unsigned long long* scan_state[2]; // look-back words of the two scans
  SplatRec* rec;                     // [N] indexed by primitive id
  ushort4* rect;                     // [N] tx0, ty0, tx1, ty1
  unsigned int* tiles_touched;       // [N]
  unsigned int* l1_keys[2];          // [N] fp32 depth bits of survivors (double buffer)
  unsigned int* l1_vals[2];          // [N] primitive ids of survivors; after the sort: depth order
  unsigned int* vis_ids;             // [N] primitive ids of survivors in ascending id order (kept for the backward)
  unsigned int* offsets;             // [N] exclusive prefix sum of tiles_touched in depth order
  unsigned int* chunk_first;         // [cap / DUP_CHUNK + 2] survivor (depth order) that owns output position k * DUP_CHUNK
  unsigned int* l2_keys[2];          // [cap] tile ids
  unsigned int* l2_vals[2];          // [cap] primitive ids
  unsigned int* sort_hist;           // [8][RADIX] digit counts of the 4 depth passes (raw) and exclusive bases of the tile-id passes
  unsigned int* sort_lookback;       // [max sort tiles][RADIX]
  uint2* ranges;                     // [tiles] [first, last+1)
  float* g9;                         // [N,9] per-splat gradients of the blend backward
  float4* aux;                       // [N] survivors: view direction (x, y, z) and (t - mu_t) / T, written by preprocess
  float4* dcol;                      // [N] survivors: colour backward -> geometry backward: dL/d dir (x, y, z), dL/d Delta
  float* gz;                         // [N] auxiliary depth channel: dL/d(camera depth) per splat
  size_t lookback_bytes, zero_bytes; // zero_bytes: prefix of the workspace cleared by fdgs_preprocess
  size_t bytes;
};

inline size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

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
  w.sort_hist = (unsigned int*)take(4 * 8 * RADIX);     // level-1 digit counts are accumulated by the compaction kernel
  w.zero_bytes = off;
  w.rec = (SplatRec*)take(sizeof(SplatRec) * Np);
  w.rect = (ushort4*)take(sizeof(ushort4) * Np);
  w.tiles_touched = (unsigned int*)take(4 * Np);
  for (int i = 0; i < 2; ++i) w.l1_keys[i] = (unsigned int*)take(4 * Np);
  for (int i = 0; i < 2; ++i) w.l1_vals[i] = (unsigned int*)take(4 * Np);
  w.vis_ids = (unsigned int*)take(4 * Np);
  w.offsets = (unsigned int*)take(4 * Np);
  w.chunk_first = (unsigned int*)take(4 * ((size_t)cap / DUP_CHUNK + 2));
  for (int i = 0; i < 2; ++i) w.l2_keys[i] = (unsigned int*)take(4 * (size_t)cap);
  for (int i = 0; i < 2; ++i) w.l2_vals[i] = (unsigned int*)take(4 * (size_t)cap);
  const long long t1 = (Np + SORT_THREADS * SORT_ITEMS_L1 - 1) / (SORT_THREADS * SORT_ITEMS_L1);
  const long long t2 = (cap + SORT_THREADS * SORT_ITEMS_L2 - 1) / (SORT_THREADS * SORT_ITEMS_L2);
  w.lookback_bytes = 4 * (size_t)RADIX * ((t1 > t2 ? t1 : t2) + 1);
  w.sort_lookback = (unsigned int*)take(w.lookback_bytes);
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

// Launch counter (fdgs_launch_count) — bumped by every launcher.
extern long long g_launches;
// Records the CUDA error text for fdgs_strerror and returns FDGS_ERR_CUDA (api.cu).
int cuda_fail(cudaError_t e, const char* where);

// Launchers (each file implements its own; all asynchronous on `st`).
void launch_preprocess_fwd(const fdgs_scene& sc, const ViewParams& vp, const CfgParams& cp, const Workspace& ws, cudaStream_t st);
// compaction scan: survivors (tiles_touched > 0) in id order -> l1_keys[0] (depth bits), l1_vals[0] (ids), hdr->num_visible
void launch_compact(const Workspace& ws, int N, cudaStream_t st);
// Stable LSD radix sort of (key, val) u32 pairs on key bits [0, bits); the count is read on the device.
// ws.sort_hist[ticket_base + pass] holds the digit counts of the pass (bases_exclusive = false: every CTA scans them
// itself) or their exclusive prefix (true).  Returns the result buffer (0/1).
int launch_sort_pairs(const Workspace& ws, unsigned int* const keys[2], unsigned int* const vals[2],
                      const unsigned int* count_dev, long long max_count, int bits, int items_per_thread, int ticket_base,
                      bool bases_exclusive, int num_sms, cudaStream_t st);
// 2D prefix of the coverage difference array -> ranges, D, overflow flag, level-2 digit bases
void launch_tile_grid(const Workspace& ws, const ViewParams& vp, long long cap, int l2_passes, cudaStream_t st);
// exclusive prefix sum of tiles_touched in depth order -> offsets
void launch_offsets(const Workspace& ws, int l1_buf, int N, cudaStream_t st);
void launch_duplicate(const Workspace& ws, int l1_buf, int N, long long cap, const ViewParams& vp, cudaStream_t st);
void launch_blend_fwd(const Workspace& ws, int l2_buf, const ViewParams& vp, const CfgParams& cp, float* image, float* final_T,
                      unsigned int* n_contrib, float* depth_map /*NULL = no auxiliary channel*/, cudaStream_t st);
void launch_blend_stats(const Workspace& ws, int l2_buf, const ViewParams& vp, const CfgParams& cp, unsigned long long* stats, cudaStream_t st);
void launch_blend_bwd(const Workspace& ws, int l2_buf, const ViewParams& vp, const CfgParams& cp, const float* dL_dimage,
                      const float* final_T, const unsigned int* n_contrib, const float* dL_ddepth, const float* dL_dopacity,
                      cudaStream_t st);
void launch_preprocess_bwd(const fdgs_scene& sc, const ViewParams& vp, const CfgParams& cp, const Workspace& ws, int l1_buf,
                           const fdgs_grads& g, bool with_gz, cudaStream_t st);
void launch_cull_status(const fdgs_scene& sc, const ViewParams& vp, const CfgParams& cp, unsigned char* dst, cudaStream_t st);
void launch_blend_feat_fwd(const Workspace& ws, int l2_buf, const ViewParams& vp, const CfgParams& cp, const float* feat, int C,
                           float* out, cudaStream_t st);
void launch_blend_feat_bwd(const Workspace& ws, int l2_buf, const ViewParams& vp, const CfgParams& cp, const float* dL_dout, int C,
                           float* grad_feat, cudaStream_t st);
void launch_feature_records(const Workspace& ws, const float* feat, int C, int c0, int N, SplatRec* dst, cudaStream_t st);
void launch_extract_feature_grads(const Workspace& ws, float* grad_feat, int C, int c0, int N, cudaStream_t st);
void launch_splat_flow(const fdgs_scene& sc, const ViewParams& vp, const CfgParams& cp, const Workspace& ws, float dt_next, float* flow,
                       cudaStream_t st);
void launch_l1_loss(const float* image, const float* target, long long count, float* dL, float* loss, cudaStream_t st);

}  // namespace fdgs
