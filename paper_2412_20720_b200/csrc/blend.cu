// blend.cu — A9 (forward compositing) and B1 (its reverse-order gradient) for sm_100a.
// One CTA per 16x16 tile, one pixel per thread; each warp covers an 8x4 pixel patch so that early
// termination and alpha-skips stay coherent inside a warp.  Splat records are gathered by id into shared
// memory in batches of 256 and converted once per (tile, splat) to tile-local form:
//     e1 = k1 - ca*x - cb*y,  e2 = k2 - cc*y,  log2(alpha) = lo - e1^2 - e2^2      (x, y tile-local pixel centres)
// i.e. 5 FFMA + 1 MUFU.EX2 per (pixel, splat) evaluation; tile-local coordinates keep |e| small so fp32
// cancellation stays ~1e-7.
#include "common.cuh"

namespace fdgs {

constexpr int BATCH = 256;

struct TileSplat {   // 48 B in shared memory, read as three broadcast LDS.128
  float nca, ncb, ncc, k1;   // -ca, -cb, -cc, ca*(u-ox) + cb*(v-oy)
  float k2, lo, r, g;        // cc*(v-oy), log2(o)
  float b, u, v, pad;        // (u, v) tile-local, for the backward
};

__device__ __forceinline__ float ex2_approx(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

__device__ __forceinline__ void stage_splat(const SplatRec* __restrict__ rec, const unsigned int id, const float ox, const float oy,
                                            float4* s0, float4* s1, float4* s2) {
  const float4* src = reinterpret_cast<const float4*>(rec + id);
  const float4 q0 = __ldg(src), q1 = __ldg(src + 1), q2 = __ldg(src + 2);
  const float ul = q0.x - ox, vl = q0.y - oy;
  *s0 = make_float4(-q0.z, -q0.w, -q1.x, fmaf(q0.z, ul, q0.w * vl));
  *s1 = make_float4(q1.x * vl, q1.y, q1.z, q1.w);
  *s2 = make_float4(q2.x, ul, vl, 0.f);
}

// Conservative test "can this splat reach alpha >= alpha_min anywhere on the warp's 8x4 pixel patch?": in the whitened
// coordinates (e1, e2) the patch is a parallelogram; its bounding box gives the lower bound
//   min(e1^2 + e2^2) >= max(0,|e1(c)| - ca*hw - |cb|*hh)^2 + max(0,|e2(c)| - cc*hh)^2     (c = patch centre)
// A splat is dropped only if even that bound (shrunk by a rounding slack) puts log2(alpha) below the skip threshold,
// i.e. only pairs every pixel of the patch would skip anyway are removed: the result is bit-identical.
__device__ __forceinline__ bool patch_hit(const float4 a, const float4 b, const float xm, const float ym, const float l2min) {
  const float e1c = fmaf(a.x, xm, fmaf(a.y, ym, a.w)), e2c = fmaf(a.z, ym, b.x);
  const float r1 = fmaf(-a.x, 3.5f, 1.5f * fabsf(a.y)), r2 = -a.z * 1.5f;      // half extents: 3.5 px in x, 1.5 px in y
  const float m1 = fmaxf(0.f, fabsf(e1c) - r1), m2 = fmaxf(0.f, fabsf(e2c) - r2);
  const float qmin = fmaf(m1, m1, m2 * m2);
  return !(fmaf(qmin, 0.999f, -1e-3f) > b.y - l2min);
}

// STATS = true: same walk, but counts the work instead of writing the image (fdgs_debug_blend_stats):
//   stats[0] pairs walked (pixel x splat, until the pixel terminates), [1] pairs that reach the exp2,
//   [2] pairs composited, [3] splats staged into shared memory (summed over tiles)
template <bool STATS>
__global__ void __launch_bounds__(256) blend_fwd_kernel(const uint2* __restrict__ ranges, const unsigned int* __restrict__ vals,
                                                        const SplatRec* __restrict__ rec, const ViewParams vp, const CfgParams cp,
                                                        float* __restrict__ image, float* __restrict__ final_T,
                                                        unsigned int* __restrict__ n_contrib, unsigned long long* stats) {
  __shared__ float4 s0[BATCH], s1[BATCH], s2[BATCH];
  const int tile = blockIdx.x, tx = tile % vp.tiles_x, ty = tile / vp.tiles_x;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int lx = ((warp & 1) << 3) + (lane & 7), ly = ((warp >> 1) << 2) + (lane >> 3);
  const int px = tx * TILE + lx, py = ty * TILE + ly;
  const bool inside = px < vp.width && py < vp.height;
  const float x = lx + 0.5f, y = ly + 0.5f, ox = (float)(tx * TILE), oy = (float)(ty * TILE);
  const float xm = (float)((warp & 1) << 3) + 4.0f, ym = (float)((warp >> 1) << 2) + 2.0f;   // patch centre (tile-local)
  const uint2 range = ranges[tile];
  const int n = (int)(range.y - range.x);
  float T = 1.f, Cr = 0.f, Cg = 0.f, Cb = 0.f;
  unsigned int last = 0;
  unsigned int st_walk = 0, st_exp = 0, st_comp = 0, st_stage = 0;
  bool done = !inside;
  for (int base = 0; base < n; base += BATCH) {
    if (__syncthreads_and(done)) break;
    const int m = min(BATCH, n - base);
    if (STATS && threadIdx.x == 0) st_stage += m;
    if ((int)threadIdx.x < m) stage_splat(rec, vals[range.x + base + threadIdx.x], ox, oy, &s0[threadIdx.x], &s1[threadIdx.x], &s2[threadIdx.x]);
    __syncthreads();
    if (__all_sync(0xffffffffu, done)) continue;     // whole 8x4 patch saturated: skip the batch (warp-uniform)
    for (int jb = 0; jb < m; jb += 32) {
      // lane l tests splat jb+l against the warp's patch; the ballot is the list of splats worth evaluating per pixel
      unsigned int hits;
      if (STATS) hits = jb + 32 <= m ? 0xffffffffu : ((1u << (m - jb)) - 1u);
      else hits = __ballot_sync(0xffffffffu, jb + lane < m && patch_hit(s0[jb + lane], s1[jb + lane], xm, ym, cp.log2_alpha_min));
      while (hits) {
        const int j = jb + __ffs(hits) - 1;
        hits &= hits - 1;
        const float4 a = s0[j], b = s1[j];
        const float e1 = fmaf(a.x, x, fmaf(a.y, y, a.w));
        const float e2 = fmaf(a.z, y, b.x);
        const float l2a = fmaf(-e2, e2, fmaf(-e1, e1, b.y));
        if (STATS && !done) ++st_walk;
        if (done || l2a < cp.log2_alpha_min) continue;                 // alpha < alpha_min: skipped
        const float alpha = fminf(cp.alpha_max, ex2_approx(l2a));
        if (STATS) ++st_exp;
        if (alpha < cp.alpha_min) continue;
        const float Tn = fmaf(-T, alpha, T);
        if (Tn < cp.transmittance_min) { done = true; continue; }      // the terminating splat is not composited
        const float wgt = alpha * T;
        Cr = fmaf(b.z, wgt, Cr); Cg = fmaf(b.w, wgt, Cg); Cb = fmaf(s2[j].x, wgt, Cb);
        T = Tn;
        last = base + j + 1;
        if (STATS) ++st_comp;
      }
      if (__all_sync(0xffffffffu, done)) break;
    }
  }
  if (STATS) {
    unsigned int v[4] = {st_walk, st_exp, st_comp, st_stage};
#pragma unroll
    for (int k = 0; k < 4; ++k) {
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) v[k] += __shfl_xor_sync(0xffffffffu, v[k], o);
      if (lane == 0 && v[k]) atomicAdd(stats + k, (unsigned long long)v[k]);
    }
    return;
  }
  if (inside) {
    const size_t hw = (size_t)vp.width * vp.height, pix = (size_t)py * vp.width + px;
    image[pix] = fmaf(T, vp.bg[0], Cr); image[hw + pix] = fmaf(T, vp.bg[1], Cg); image[2 * hw + pix] = fmaf(T, vp.bg[2], Cb);
    final_T[pix] = T; n_contrib[pix] = last;
  }
}

// ---------------------------------------------------------------------------------------------
// Sum of 8 values over the 32 lanes with 9 shuffles (halving exchange), result k lands on lane 4k.
__device__ __forceinline__ float warp_reduce8(float v[8], const int lane) {
  const bool b4 = lane & 16, b3 = lane & 8, b2 = lane & 4;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const float keep = b4 ? v[i + 4] : v[i], send = b4 ? v[i] : v[i + 4];
    v[i] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
  }
#pragma unroll
  for (int i = 0; i < 2; ++i) {
    const float keep = b3 ? v[i + 2] : v[i], send = b3 ? v[i] : v[i + 2];
    v[i] = keep + __shfl_xor_sync(0xffffffffu, send, 8);
  }
  {
    const float keep = b2 ? v[1] : v[0], send = b2 ? v[0] : v[1];
    v[0] = keep + __shfl_xor_sync(0xffffffffu, send, 4);
  }
  v[0] += __shfl_xor_sync(0xffffffffu, v[0], 2);
  v[0] += __shfl_xor_sync(0xffffffffu, v[0], 1);
  return v[0];
}

// B1.  Walks each tile list back to front from the last contributor of the tile.  Per (pixel, splat) the lane
// produces two scalars, wgt = alpha T (for dL/dc) and dpow = alpha dL/dalpha (for everything that flows through the
// exponent), and nine products of them with per-pixel quantities:
//     dpow * {dx, dy, dx^2, dx dy, dy^2, 1}   and   wgt * dL/dpixel{r,g,b}        (dx = u - px, dy = v - py)
// which are reduced over the warp by shuffles, then over the eight warps in shared memory; one thread per splat
// turns the nine sums into dL/d(u, v, A, B, C, o, r, g, b) and flushes nine global atomics per (tile, splat):
//     dL/du = -(A Sx + B Sy), dL/dv = -(B Sx + C Sy), dL/dA = -Sxx/2, dL/dB = -Sxy, dL/dC = -Syy/2, dL/do = S1 / o.
// The colour behind the current splat enters only through its dot product with dL/dpixel, so one scalar s is carried:
//     dL/dalpha_k = T_k (g.c_k) - s_k / (1 - alpha_k),   s_{k-1} = s_k + (g.c_k) alpha_k T_k,   s_last = T_final (g.bg).
constexpr int ACC_STRIDE = BATCH + 1;   // odd stride: the eight lanes that hold the warp sums hit eight different banks

struct BwdShared {
  float4 s0[BATCH], s1[BATCH], s2[BATCH];
  float acc[9 * ACC_STRIDE];
  unsigned int id[BATCH];
  int max_contrib;
};

__device__ __forceinline__ float rcp_approx(float x) { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

__global__ void __launch_bounds__(256) blend_bwd_kernel(const uint2* __restrict__ ranges, const unsigned int* __restrict__ vals,
                                                        const SplatRec* __restrict__ rec, const ViewParams vp, const CfgParams cp,
                                                        const float* __restrict__ dL_dimage, const float* __restrict__ final_T,
                                                        const unsigned int* __restrict__ n_contrib, float* __restrict__ g9) {
  __shared__ BwdShared sm;
  const int tile = blockIdx.x, tx = tile % vp.tiles_x, ty = tile / vp.tiles_x;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int lx = ((warp & 1) << 3) + (lane & 7), ly = ((warp >> 1) << 2) + (lane >> 3);
  const int px = tx * TILE + lx, py = ty * TILE + ly;
  const bool inside = px < vp.width && py < vp.height;
  const float x = lx + 0.5f, y = ly + 0.5f, ox = (float)(tx * TILE), oy = (float)(ty * TILE);
  const float xm = (float)((warp & 1) << 3) + 4.0f, ym = (float)((warp >> 1) << 2) + 2.0f;
  const uint2 range = ranges[tile];
  const size_t hw = (size_t)vp.width * vp.height, pix = (size_t)py * vp.width + px;
  float T = 1.f, gr = 0.f, gg = 0.f, gb = 0.f;
  int mine = 0;
  if (inside) { T = final_T[pix]; mine = (int)n_contrib[pix]; gr = dL_dimage[pix]; gg = dL_dimage[hw + pix]; gb = dL_dimage[2 * hw + pix]; }
  if (threadIdx.x == 0) sm.max_contrib = 0;
  __syncthreads();
  int warp_max = mine;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) warp_max = max(warp_max, __shfl_xor_sync(0xffffffffu, warp_max, o));
  if (lane == 0) atomicMax(&sm.max_contrib, warp_max);
  __syncthreads();
  const int total = sm.max_contrib;
  float s = T * (gr * vp.bg[0] + gg * vp.bg[1] + gb * vp.bg[2]);
  // warp_reduce8 leaves sum k on lane 4k; the ninth sum (butterfly, on every lane) is flushed by lane 1: one atomic
  // instruction for all nine rows, nine different banks
  const bool flusher = (lane & 3) == 0 || lane == 1;
  float* const acc_lane = sm.acc + (lane == 1 ? 8 : lane >> 2) * ACC_STRIDE;
  for (int hi = total; hi > 0; hi -= BATCH) {           // batch covers list positions [lo_pos, hi)
    const int lo_pos = max(0, hi - BATCH), m = hi - lo_pos;
    __syncthreads();                                    // previous batch fully flushed
    if ((int)threadIdx.x < m) {
      const unsigned int id = vals[range.x + lo_pos + threadIdx.x];
      sm.id[threadIdx.x] = id;
      stage_splat(rec, id, ox, oy, &sm.s0[threadIdx.x], &sm.s1[threadIdx.x], &sm.s2[threadIdx.x]);
    }
#pragma unroll
    for (int k = 0; k < 9; ++k) sm.acc[k * ACC_STRIDE + threadIdx.x] = 0.f;
    __syncthreads();
    if (lo_pos < warp_max) {
     for (int jb = ((m - 1) >> 5) << 5; jb >= 0; jb -= 32) {
      unsigned int hits = __ballot_sync(0xffffffffu, jb + lane < m && lo_pos + jb + lane < warp_max &&
                                                     patch_hit(sm.s0[jb + lane], sm.s1[jb + lane], xm, ym, cp.log2_alpha_min));
      while (hits) {
        const int bit = 31 - __clz(hits);
        hits &= ~(1u << bit);
        const int j = jb + bit;
        const float4 a = sm.s0[j], b = sm.s1[j];
        const float e1 = fmaf(a.x, x, fmaf(a.y, y, a.w));
        const float e2 = fmaf(a.z, y, b.x);
        const float l2a = fmaf(-e2, e2, fmaf(-e1, e1, b.y));
        bool active = (lo_pos + j < mine) && !(l2a < cp.log2_alpha_min);
        float alpha = 0.f, araw = 0.f;
        if (active) { araw = ex2_approx(l2a); alpha = fminf(cp.alpha_max, araw); active = !(alpha < cp.alpha_min); }
        if (!__any_sync(0xffffffffu, active)) continue;
        float v[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f}, v1 = 0.f;
        if (active) {
          const float4 c = sm.s2[j];
          const float iom = rcp_approx(1.f - alpha);
          T *= iom;                                                    // T_k
          const float wgt = alpha * T;
          v[5] = wgt * gr; v[6] = wgt * gg; v[7] = wgt * gb;           // dL/dc
          const float gc = fmaf(gr, b.z, fmaf(gg, b.w, gb * c.x));     // dL/dpixel . c_k
          const float dalpha = fmaf(T, gc, -s * iom);
          s = fmaf(gc, wgt, s);
          if (!(araw > cp.alpha_max)) {                                // alpha clamp inactive: d alpha / d power = alpha
            const float dpow = alpha * dalpha, dx = c.y - x, dy = c.z - y;
            v1 = dpow;
            v[0] = dpow * dx; v[1] = dpow * dy;
            v[2] = v[0] * dx; v[3] = v[0] * dy; v[4] = v[1] * dy;
          }
        }
        const float red = warp_reduce8(v, lane);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v1 += __shfl_xor_sync(0xffffffffu, v1, o);
        if (flusher) atomicAdd(acc_lane + j, lane == 1 ? v1 : red);
      }
     }
    }
    __syncthreads();
    if ((int)threadIdx.x < m) {
      const int j = threadIdx.x;
      const float Sx = sm.acc[j], Sy = sm.acc[ACC_STRIDE + j], Sxx = sm.acc[2 * ACC_STRIDE + j], Sxy = sm.acc[3 * ACC_STRIDE + j];
      const float Syy = sm.acc[4 * ACC_STRIDE + j], S1 = sm.acc[8 * ACC_STRIDE + j];
      const float4 a = sm.s0[j];
      const float ik = 1.0f / 0.72134752044448170f;                    // conic (A, B, C) from its exp2-scaled factor
      const float A = a.x * a.x * ik, B = a.x * a.y * ik, C = fmaf(a.y, a.y, a.z * a.z) * ik;
      float out[9];
      out[0] = -fmaf(A, Sx, B * Sy); out[1] = -fmaf(B, Sx, C * Sy);
      out[2] = -0.5f * Sxx; out[3] = -Sxy; out[4] = -0.5f * Syy;
      out[5] = S1 * exp2f(-sm.s1[j].y);
      out[6] = sm.acc[5 * ACC_STRIDE + j]; out[7] = sm.acc[6 * ACC_STRIDE + j]; out[8] = sm.acc[7 * ACC_STRIDE + j];
      float* dst = g9 + (size_t)9 * sm.id[j];
#pragma unroll
      for (int k = 0; k < 9; ++k) if (out[k] != 0.f) atomicAdd(dst + k, out[k]);
    }
  }
}

void launch_blend_fwd(const Workspace& ws, int l2_buf, const ViewParams& vp, const CfgParams& cp, float* image, float* final_T,
                      unsigned int* n_contrib, cudaStream_t st) {
  blend_fwd_kernel<false><<<vp.tiles_x * vp.tiles_y, 256, 0, st>>>(ws.ranges, ws.l2_vals[l2_buf], ws.rec, vp, cp, image, final_T, n_contrib, nullptr);
  ++g_launches;
}

void launch_blend_stats(const Workspace& ws, int l2_buf, const ViewParams& vp, const CfgParams& cp, unsigned long long* stats, cudaStream_t st) {
  blend_fwd_kernel<true><<<vp.tiles_x * vp.tiles_y, 256, 0, st>>>(ws.ranges, ws.l2_vals[l2_buf], ws.rec, vp, cp, nullptr, nullptr, nullptr, stats);
  ++g_launches;
}

void launch_blend_bwd(const Workspace& ws, int l2_buf, const ViewParams& vp, const CfgParams& cp, const float* dL_dimage,
                      const float* final_T, const unsigned int* n_contrib, cudaStream_t st) {
  blend_bwd_kernel<<<vp.tiles_x * vp.tiles_y, 256, 0, st>>>(ws.ranges, ws.l2_vals[l2_buf], ws.rec, vp, cp, dL_dimage, final_T, n_contrib, ws.g9);
  ++g_launches;
}

}  // namespace fdgs
