// blend.cu — A9 (forward compositing) and B1 (its reverse-order gradient) for sm_100a.
// One CTA per 16x16 tile.  A warp covers an 8-wide column strip of 4*PX rows; lane l owns PX pixels, one in each of the
// strip's PX sub-patches of 8x4 pixels: (x0 + l%8, y0 + 4k + l/8), k < PX.  A sub-patch is the unit of culling (early
// termination and alpha-skips stay coherent inside it); the strip is the unit of everything that costs once per
// (warp, splat): the bit loop, the shared-memory loads of the splat and — in the backward — the warp reduction of the
// per-splat gradient sums and their flush.  PX = 1 gives 8 warps per tile, PX = 2 four, PX = 4 two.
// Splat records are gathered by id into shared memory in batches and converted once per (tile, splat) to tile-local form:
//     e1 = k1 - ca*x - cb*y,  e2 = k2 - cc*y,  log2(alpha) = lo - e1^2 - e2^2      (x, y tile-local pixel centres)
// i.e. 5 FFMA + 1 MUFU.EX2 per (pixel, splat) evaluation; tile-local coordinates keep |e| small so fp32
// cancellation stays ~1e-7.
#include "common.cuh"

namespace fdgs {

__device__ __forceinline__ float ex2_approx(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float rcp_approx(float x) { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

// ---- bulk asynchronous copies (TMA, non-tensor form) and their mbarriers: records are gathered global -> shared by the
// copy engine while the warps composite the previous batch (SASS: UBLKCP, SYNCS) ----
// FDGS_BLEND_ASYNC selects the staging of the forward blend at COMPILE time (measurement builds: FDGS_NVCC_EXTRA, build.py):
//   0 (product): synchronous LDG -> convert -> STS, 256 splats per batch (blend_fwd_kernel<2>);
//   1: cp.async.bulk + mbarrier, 2: cp.async (LDGSTS) — blend_fwd_async_kernel.  Both async pipelines were built,
//   verified against the oracle and measured on B200 in round 2 and LOSE to the synchronous staging (1.436 / 1.339 vs
//   1.248 ms per 4 views at cfg3; profiles/r2_blend_staging_ab.md), so they are not in libfdgs.so.
#ifndef FDGS_BLEND_ASYNC
#define FDGS_BLEND_ASYNC 0
#endif
__device__ __forceinline__ unsigned int smem_u32(const void* p) { return (unsigned int)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, const unsigned int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned long long* bar, const unsigned int bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(unsigned long long* bar, const unsigned int parity) {
  unsigned int ok;
  asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
               : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
  return ok != 0;
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, const unsigned int parity) { while (!mbar_try_wait(bar, parity)) {} }
// one record (48 B, 16-byte aligned on both sides) global -> shared; completion is counted in bytes on `bar`
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, const unsigned int bytes, unsigned long long* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }

// tile-local form of a record, in place: (q0, q1, q2) of SplatRec -> (s0, s1, s2) below
__device__ __forceinline__ void convert_splat(float4* r, const float ox, const float oy) {
  const float4 q0 = r[0], q1 = r[1], q2 = r[2];
  const float ul = q0.x - ox, vl = q0.y - oy;
  r[0] = make_float4(-q0.z, -q0.w, -q1.x, fmaf(q0.z, ul, q0.w * vl));
  r[1] = make_float4(q1.x * vl, q1.y, q1.z, q1.w);
  r[2] = make_float4(q2.x, ul, vl, q2.y);
}

// Shared-memory form of a splat: three float4, read as broadcast LDS.128
//   s0 = (-ca, -cb, -cc, k1 = ca*(u-ox) + cb*(v-oy))   s1 = (k2 = cc*(v-oy), lo = log2(o), r, g)   s2 = (b, u-ox, v-oy, depth)
__device__ __forceinline__ void stage_splat(const SplatRec* __restrict__ rec, const unsigned int id, const float ox, const float oy,
                                            float4* s0, float4* s1, float4* s2) {
  const float4* src = reinterpret_cast<const float4*>(rec + id);
  const float4 q0 = __ldg(src), q1 = __ldg(src + 1), q2 = __ldg(src + 2);
  const float ul = q0.x - ox, vl = q0.y - oy;
  *s0 = make_float4(-q0.z, -q0.w, -q1.x, fmaf(q0.z, ul, q0.w * vl));
  *s1 = make_float4(q1.x * vl, q1.y, q1.z, q1.w);
  *s2 = make_float4(q2.x, ul, vl, q2.y);
}

// Conservative test "can this splat reach alpha >= alpha_min anywhere on an 8x4 pixel patch?": in the whitened
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

// Pixel geometry of a lane: strip origin (sx0, sy0) inside the tile, lane offsets.
template <int PX>
struct Strip {
  int lx, ly0;      // tile-local pixel column, row of sub-patch 0
  float xm, ym0;    // centre of sub-patch 0 (tile-local)
  __device__ __forceinline__ Strip(const int warp, const int lane) {
    const int sx0 = (warp & 1) << 3, sy0 = (warp >> 1) * 4 * PX;
    lx = sx0 + (lane & 7); ly0 = sy0 + (lane >> 3);
    xm = (float)sx0 + 4.0f; ym0 = (float)sy0 + 2.0f;
  }
};

// A9.  STATS = true: same walk without the patch culling, counting the work instead of writing the image
// (fdgs_debug_blend_stats): stats[0] (pixel, splat) pairs walked until the pixel terminates, [1] pairs that reach the
// exp2, [2] pairs composited, [3] splats staged into shared memory (summed over tiles).
// AUX = true additionally composites the camera depth of the splats like a fourth colour channel without background
// (rendered depth, eq. 29) into depth_map[H,W].
// DEF = true: the thresholds of [23] as immediates (cp.default_thresholds; see common.cuh).
template <int PX, bool STATS, bool AUX, bool DEF>
__global__ void __launch_bounds__(256 / PX, PX == 2 && !STATS ? 9 : 1) blend_fwd_kernel(const uint2* __restrict__ ranges, const unsigned int* __restrict__ vals,
                                                             const SplatRec* __restrict__ rec, const ViewParams vp, const CfgParams cp,
                                                             float* __restrict__ image, float* __restrict__ final_T,
                                                             unsigned int* __restrict__ n_contrib, unsigned long long* stats,
                                                             float* __restrict__ depth_map) {
  // splats staged per batch: two per thread at PX = 2 — half the barriers (12 % of the warp samples sat at the loop-top
  // barrier with 128) and twice the gathers in flight per thread
  constexpr int NT = 256 / PX, BATCH = PX == 2 ? 2 * NT : NT;
  __shared__ struct { float4 s0[BATCH], s1[BATCH], s2[BATCH]; } sm;
  const int tile = blockIdx.x, tx = tile % vp.tiles_x, ty = tile / vp.tiles_x;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const Strip<PX> sp(warp, lane);
  const int px = tx * TILE + sp.lx;
  const float x = sp.lx + 0.5f, ox = (float)(tx * TILE), oy = (float)(ty * TILE);
  const float c_l2min = DEF ? FDGS_DEF_L2MIN : cp.log2_alpha_min, c_amax = DEF ? FDGS_DEF_ALPHA_MAX : cp.alpha_max;
  const float c_amin = DEF ? FDGS_DEF_ALPHA_MIN : cp.alpha_min, c_tmin = DEF ? FDGS_DEF_T_MIN : cp.transmittance_min;
  // lmin[k]: the skip threshold of pixel k, +inf once the pixel has terminated (or lies outside the image) — the "done"
  // state costs no flag and no extra test in the loop
  float y[PX], T[PX], Cr[PX], Cg[PX], Cb[PX], Dz[PX], lmin[PX];
  unsigned int last[PX];
  bool inside[PX];
#define FDGS_DONE(k) (lmin[k] > 3.0e38f)
#pragma unroll
  for (int k = 0; k < PX; ++k) {
    const int ly = sp.ly0 + 4 * k;
    inside[k] = px < vp.width && ty * TILE + ly < vp.height;
    y[k] = ly + 0.5f; T[k] = 1.f; Cr[k] = Cg[k] = Cb[k] = Dz[k] = 0.f; last[k] = 0; lmin[k] = inside[k] ? c_l2min : INFINITY;
  }
  const uint2 range = ranges[tile];
  const int n = (int)(range.y - range.x);
  unsigned int st_walk = 0, st_exp = 0, st_comp = 0, st_stage = 0;
  for (int base = 0; base < n; base += BATCH) {
    bool all_done = true;
#pragma unroll
    for (int k = 0; k < PX; ++k) all_done = all_done && FDGS_DONE(k);
    if (__syncthreads_and(all_done)) break;
    const int m = min(BATCH, n - base);
    if (STATS && threadIdx.x == 0) st_stage += m;
#pragma unroll
    for (int i = threadIdx.x; i < BATCH; i += NT)
      if (i < m) stage_splat(rec, vals[range.x + base + i], ox, oy, &sm.s0[i], &sm.s1[i], &sm.s2[i]);
    __syncthreads();
    unsigned int alive = 0;                           // sub-patches with an unsaturated pixel (warp-uniform)
#pragma unroll
    for (int k = 0; k < PX; ++k) if (!__all_sync(0xffffffffu, FDGS_DONE(k))) alive |= 1u << k;
    if (!alive) continue;
    for (int jb = 0; jb < m; jb += 32) {
      // lane l tests splat jb+l against each live sub-patch; the ballots list the splats worth evaluating per pixel
      unsigned int hk[PX], any = 0;
      float4 ta, tb;
      if (jb + lane < m) { ta = sm.s0[jb + lane]; tb = sm.s1[jb + lane]; }
#pragma unroll
      for (int k = 0; k < PX; ++k) {
        if (STATS) hk[k] = jb + 32 <= m ? 0xffffffffu : ((1u << (m - jb)) - 1u);
        else hk[k] = ((alive >> k) & 1u) ? __ballot_sync(0xffffffffu, jb + lane < m && patch_hit(ta, tb, sp.xm, sp.ym0 + 4.f * k, c_l2min)) : 0u;
        any |= hk[k];
      }
      while (any) {
        const int bit = __ffs(any) - 1;
        any &= any - 1;
        const int j = jb + bit;
        const float4 a = sm.s0[j], b = sm.s1[j];
        const float e1x = fmaf(a.x, x, a.w);
#pragma unroll
        for (int k = 0; k < PX; ++k) {
          if (!((hk[k] >> bit) & 1u)) continue;                          // warp-uniform
          const float e1 = fmaf(a.y, y[k], e1x);
          const float e2 = fmaf(a.z, y[k], b.x);
          const float l2a = fmaf(-e2, e2, fmaf(-e1, e1, b.y));
          if (STATS && !FDGS_DONE(k)) ++st_walk;
          if (!(l2a >= lmin[k])) continue;                     // alpha < alpha_min (or pixel done): skipped
          const float alpha = fminf(c_amax, ex2_approx(l2a));
          if (STATS) ++st_exp;
          if (alpha < c_amin) continue;
          const float Tn = fmaf(-T[k], alpha, T[k]);
          const bool term = Tn < c_tmin;                       // the terminating splat is not composited
          asm("{\n\t.reg .pred p;\n\tsetp.lt.f32 p, %1, %2;\n\t@p mov.b32 %0, 0x7f800000;\n\t}" : "+f"(lmin[k]) : "f"(Tn), "f"(c_tmin));
          if (term) continue;
          const float wgt = alpha * T[k];
          Cr[k] = fmaf(b.z, wgt, Cr[k]); Cg[k] = fmaf(b.w, wgt, Cg[k]); Cb[k] = fmaf(sm.s2[j].x, wgt, Cb[k]);
          if (AUX) Dz[k] = fmaf(sm.s2[j].w, wgt, Dz[k]);
          T[k] = Tn;
          last[k] = base + j + 1;
          if (STATS) ++st_comp;
        }
      }
#pragma unroll
      for (int k = 0; k < PX; ++k) if (((alive >> k) & 1u) && __all_sync(0xffffffffu, FDGS_DONE(k))) alive &= ~(1u << k);
      if (!alive) break;
    }
  }
#undef FDGS_DONE
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
  const size_t hw = (size_t)vp.width * vp.height;
#pragma unroll
  for (int k = 0; k < PX; ++k) {
    if (!inside[k]) continue;
    const size_t pix = (size_t)(ty * TILE + sp.ly0 + 4 * k) * vp.width + px;
    image[pix] = fmaf(T[k], vp.bg[0], Cr[k]); image[hw + pix] = fmaf(T[k], vp.bg[1], Cg[k]); image[2 * hw + pix] = fmaf(T[k], vp.bg[2], Cb[k]);
    final_T[pix] = T[k]; n_contrib[pix] = last[k];
    if (AUX) depth_map[pix] = Dz[k];
  }
}

#if FDGS_BLEND_ASYNC
// A9 with bulk-asynchronous staging (north_star subsystem 5).  Same walk, same decisions, same arithmetic as
// blend_fwd_kernel<2>; what changes is how a batch of splats reaches shared memory:
//   - the 48-byte record of every listed splat is gathered by one `cp.async.bulk` (the copy engine: no register, no
//     scoreboard slot, no LDG -> STS round trip in the warps) into a RAW slot owned by the issuing thread; completion is
//     counted in bytes on one mbarrier, whose phase also needs all 128 threads to arrive, so that a phase can never
//     complete before every thread has seen the previous one;
//   - one batch ahead, the thread converts the record of its slot to tile-local form into the structure-of-arrays
//     buffer of the NEXT batch (two such buffers alternate) and at once asks the copy engine for the record of the batch
//     after that, into the same slot: the copy has a whole batch of compositing to land;
//   - so there is ONE block barrier per batch — the `__syncthreads_and` that votes on early termination — instead of two,
//     and no global-memory latency between barriers; the ids are loaded (coalesced) one more batch ahead into a register.
// Before the CTA exits it waits for the copy it has issued last (shared memory of a finished CTA is reallocated).
// MODE 1: cp.async.bulk + mbarrier as described.  MODE 2: the same pipeline with three 16-byte `cp.async` (LDGSTS) per
// record instead of one bulk copy, completion by `cp.async.wait_group` of the issuing thread (no mbarrier): kept for the
// A/B numbers in profiles/ (build with -DFDGS_BLEND_ASYNC=2).
template <bool AUX, bool DEF, int MODE>
__global__ void __launch_bounds__(128, 8) blend_fwd_async_kernel(const uint2* __restrict__ ranges, const unsigned int* __restrict__ vals,
                                                                 const SplatRec* __restrict__ rec, const ViewParams vp, const CfgParams cp,
                                                                 float* __restrict__ image, float* __restrict__ final_T,
                                                                 unsigned int* __restrict__ n_contrib, float* __restrict__ depth_map) {
  constexpr int PX = 2, BATCH = 128;
  __shared__ __align__(16) float4 raw[BATCH][3];
  __shared__ struct { float4 s0[BATCH], s1[BATCH], s2[BATCH]; } sm[2];
  __shared__ __align__(8) unsigned long long full;
  const int tile = blockIdx.x, tx = tile % vp.tiles_x, ty = tile / vp.tiles_x;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const Strip<PX> sp(warp, lane);
  const int px = tx * TILE + sp.lx;
  const float x = sp.lx + 0.5f, ox = (float)(tx * TILE), oy = (float)(ty * TILE);
  const float c_l2min = DEF ? FDGS_DEF_L2MIN : cp.log2_alpha_min, c_amax = DEF ? FDGS_DEF_ALPHA_MAX : cp.alpha_max;
  const float c_amin = DEF ? FDGS_DEF_ALPHA_MIN : cp.alpha_min, c_tmin = DEF ? FDGS_DEF_T_MIN : cp.transmittance_min;
  float y[PX], T[PX], Cr[PX], Cg[PX], Cb[PX], Dz[PX], lmin[PX];
  unsigned int last[PX];
  bool inside[PX];
#define FDGS_DONE(k) (lmin[k] > 3.0e38f)
#pragma unroll
  for (int k = 0; k < PX; ++k) {
    const int ly = sp.ly0 + 4 * k;
    inside[k] = px < vp.width && ty * TILE + ly < vp.height;
    y[k] = ly + 0.5f; T[k] = 1.f; Cr[k] = Cg[k] = Cb[k] = Dz[k] = 0.f; last[k] = 0; lmin[k] = inside[k] ? c_l2min : INFINITY;
  }
  const uint2 range = ranges[tile];
  const int n = (int)(range.y - range.x), nb = (n + BATCH - 1) / BATCH;
  if (MODE == 1) {
    if (threadIdx.x == 0) { mbar_init(&full, 128); fence_mbar_init(); }
    __syncthreads();
  }
  auto load_id = [&](const int k) -> unsigned int { const int i = k * BATCH + (int)threadIdx.x; return i < n ? vals[range.x + i] : 0u; };
  // batch k: every thread arrives on the barrier's phase k; the threads that own a splat of the batch add its 48 bytes to
  // the phase and ask the copy engine for them
  auto issue = [&](const int k, const unsigned int id) {
    if (MODE == 2) {
      if (k * BATCH + (int)threadIdx.x < n) {
        const float4* src = reinterpret_cast<const float4*>(rec + id);
#pragma unroll
        for (int q = 0; q < 3; ++q)
          asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(&raw[threadIdx.x][q])), "l"(src + q) : "memory");
      }
      asm volatile("cp.async.commit_group;" ::: "memory");
    } else if (k * BATCH + (int)threadIdx.x < n) {
      mbar_arrive_expect_tx(&full, 48u);
      bulk_g2s(&raw[threadIdx.x][0], rec + id, 48u, &full);
    } else {
      asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(&full)) : "memory");
    }
  };
  // wait until batch k has landed; my record, converted to tile-local form, goes to the buffer of batch k
  auto convert = [&](const int k) {
    if (MODE == 2) asm volatile("cp.async.wait_group 0;" ::: "memory");      // my own three copies: nobody else reads my raw slot
    else mbar_wait(&full, (unsigned int)k & 1u);
    if (k * BATCH + (int)threadIdx.x < n) {
      const float4 q0 = raw[threadIdx.x][0], q1 = raw[threadIdx.x][1], q2 = raw[threadIdx.x][2];
      const float ul = q0.x - ox, vl = q0.y - oy;
      sm[k & 1].s0[threadIdx.x] = make_float4(-q0.z, -q0.w, -q1.x, fmaf(q0.z, ul, q0.w * vl));
      sm[k & 1].s1[threadIdx.x] = make_float4(q1.x * vl, q1.y, q1.z, q1.w);
      sm[k & 1].s2[threadIdx.x] = make_float4(q2.x, ul, vl, q2.y);
    }
  };
  unsigned int id_next = 0;
  if (nb > 0) { issue(0, load_id(0)); convert(0); }
  if (nb > 1) { if (MODE == 1) fence_proxy_async(); issue(1, load_id(1)); }
  if (nb > 2) id_next = load_id(2);
  int k = 0;
  for (; k < nb; ++k) {
    bool all_done = true;
#pragma unroll
    for (int q = 0; q < PX; ++q) all_done = all_done && FDGS_DONE(q);
    // the one barrier of the batch: every warp has left batch k-1 (its buffer, which is the one of batch k+1, may be
    // overwritten), the conversions of batch k are visible, and the vote on early termination
    if (__syncthreads_and(all_done)) break;
    if (k + 1 < nb) {
      convert(k + 1);                                 // landed long ago: issued one iteration earlier
      if (k + 2 < nb) {
        if (MODE == 1) fence_proxy_async();           // my generic-proxy reads of the raw slot, before the copy engine rewrites it
        issue(k + 2, id_next);
        id_next = k + 3 < nb ? load_id(k + 3) : 0u;
      }
    }
    const int base = k * BATCH, m = min(BATCH, n - base);
    const auto& sb = sm[k & 1];
    unsigned int alive = 0;                           // sub-patches with an unsaturated pixel (warp-uniform)
#pragma unroll
    for (int q = 0; q < PX; ++q) if (!__all_sync(0xffffffffu, FDGS_DONE(q))) alive |= 1u << q;
    if (!alive) continue;
    for (int jb = 0; jb < m; jb += 32) {
      unsigned int hk[PX], any = 0;
      float4 ta, tb;
      if (jb + lane < m) { ta = sb.s0[jb + lane]; tb = sb.s1[jb + lane]; }
#pragma unroll
      for (int q = 0; q < PX; ++q) {
        hk[q] = ((alive >> q) & 1u) ? __ballot_sync(0xffffffffu, jb + lane < m && patch_hit(ta, tb, sp.xm, sp.ym0 + 4.f * q, c_l2min)) : 0u;
        any |= hk[q];
      }
      while (any) {
        const int bit = __ffs(any) - 1;
        any &= any - 1;
        const int j = jb + bit;
        const float4 a = sb.s0[j], b = sb.s1[j];
        const float e1x = fmaf(a.x, x, a.w);
#pragma unroll
        for (int q = 0; q < PX; ++q) {
          if (!((hk[q] >> bit) & 1u)) continue;                          // warp-uniform
          const float e1 = fmaf(a.y, y[q], e1x);
          const float e2 = fmaf(a.z, y[q], b.x);
          const float l2a = fmaf(-e2, e2, fmaf(-e1, e1, b.y));
          if (!(l2a >= lmin[q])) continue;                     // alpha < alpha_min (or pixel done): skipped
          const float alpha = fminf(c_amax, ex2_approx(l2a));
          if (alpha < c_amin) continue;
          const float Tn = fmaf(-T[q], alpha, T[q]);
          const bool term = Tn < c_tmin;                       // the terminating splat is not composited
          asm("{\n\t.reg .pred p;\n\tsetp.lt.f32 p, %1, %2;\n\t@p mov.b32 %0, 0x7f800000;\n\t}" : "+f"(lmin[q]) : "f"(Tn), "f"(c_tmin));
          if (term) continue;
          const float wgt = alpha * T[q];
          Cr[q] = fmaf(b.z, wgt, Cr[q]); Cg[q] = fmaf(b.w, wgt, Cg[q]); Cb[q] = fmaf(sb.s2[j].x, wgt, Cb[q]);
          if (AUX) Dz[q] = fmaf(sb.s2[j].w, wgt, Dz[q]);
          T[q] = Tn;
          last[q] = base + j + 1;
        }
      }
#pragma unroll
      for (int q = 0; q < PX; ++q) if (((alive >> q) & 1u) && __all_sync(0xffffffffu, FDGS_DONE(q))) alive &= ~(1u << q);
      if (!alive) break;
    }
  }
#undef FDGS_DONE
  // early termination at the top of iteration k: batch k + 1 (if any) was issued one iteration earlier and has not been waited for
  if (k + 1 < nb) { if (MODE == 2) asm volatile("cp.async.wait_group 0;" ::: "memory"); else mbar_wait(&full, (unsigned int)(k + 1) & 1u); }
  const size_t hw = (size_t)vp.width * vp.height;
#pragma unroll
  for (int q = 0; q < PX; ++q) {
    if (!inside[q]) continue;
    const size_t pix = (size_t)(ty * TILE + sp.ly0 + 4 * q) * vp.width + px;
    image[pix] = fmaf(T[q], vp.bg[0], Cr[q]); image[hw + pix] = fmaf(T[q], vp.bg[1], Cg[q]); image[2 * hw + pix] = fmaf(T[q], vp.bg[2], Cb[q]);
    final_T[pix] = T[q]; n_contrib[pix] = last[q];
    if (AUX) depth_map[pix] = Dz[q];
  }
}

#endif  // FDGS_BLEND_ASYNC

// Feature channels: the walk of blend_fwd_kernel<2> — same staging, same patch culling, the
// SAME expression for alpha, so every skip / termination decision is bit-identical to the colour pass — compositing CH
// per-splat feature values per pass instead of (r, g, b): alpha is evaluated once for CH channels.  feat[N,C] is gathered
// by id into shared memory next to the splat records; channels c0 .. c0+CH-1 (zero beyond C); no background.
template <int CH, bool DEF>
__global__ void __launch_bounds__(128, CH == 32 ? 4 : (CH == 4 ? 9 : 1)) blend_feat_fwd_kernel(const uint2* __restrict__ ranges, const unsigned int* __restrict__ vals,
                                                             const SplatRec* __restrict__ rec, const ViewParams vp, const CfgParams cp,
                                                             const float* __restrict__ feat, const int C, const int c0,
                                                             float* __restrict__ out) {
  constexpr int PX = 2, BATCH = 128;
  __shared__ struct { float4 s0[BATCH], s1[BATCH], s2[BATCH]; float4 f[BATCH][CH / 4]; } sm;
  const int tile = blockIdx.x, tx = tile % vp.tiles_x, ty = tile / vp.tiles_x;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const Strip<PX> sp(warp, lane);
  const int px = tx * TILE + sp.lx;
  const float x = sp.lx + 0.5f, ox = (float)(tx * TILE), oy = (float)(ty * TILE);
  float y[PX], T[PX], acc[PX][CH];
  bool done[PX], inside[PX];
#pragma unroll
  for (int k = 0; k < PX; ++k) {
    const int ly = sp.ly0 + 4 * k;
    inside[k] = px < vp.width && ty * TILE + ly < vp.height;
    y[k] = ly + 0.5f; T[k] = 1.f; done[k] = !inside[k];
#pragma unroll
    for (int c = 0; c < CH; ++c) acc[k][c] = 0.f;
  }
  const uint2 range = ranges[tile];
  const int n = (int)(range.y - range.x);
  const bool vec = (C & 3) == 0 && (c0 & 3) == 0 && c0 + CH <= C;       // 128-bit gathers when the row slice is aligned
  const float c_l2min = DEF ? FDGS_DEF_L2MIN : cp.log2_alpha_min, c_amax = DEF ? FDGS_DEF_ALPHA_MAX : cp.alpha_max;
  const float c_amin = DEF ? FDGS_DEF_ALPHA_MIN : cp.alpha_min, c_tmin = DEF ? FDGS_DEF_T_MIN : cp.transmittance_min;
  for (int base = 0; base < n; base += BATCH) {
    if (__syncthreads_and(done[0] && done[1])) break;
    const int m = min(BATCH, n - base);
    if ((int)threadIdx.x < m) {
      const unsigned int id = vals[range.x + base + threadIdx.x];
      stage_splat(rec, id, ox, oy, &sm.s0[threadIdx.x], &sm.s1[threadIdx.x], &sm.s2[threadIdx.x]);
      const float* src = feat + (size_t)id * C + c0;
      if (vec) {
#pragma unroll
        for (int q = 0; q < CH / 4; ++q) sm.f[threadIdx.x][q] = __ldg(reinterpret_cast<const float4*>(src) + q);
      } else {
#pragma unroll
        for (int q = 0; q < CH / 4; ++q) {
          float4 v;
          v.x = c0 + 4 * q + 0 < C ? __ldg(src + 4 * q + 0) : 0.f; v.y = c0 + 4 * q + 1 < C ? __ldg(src + 4 * q + 1) : 0.f;
          v.z = c0 + 4 * q + 2 < C ? __ldg(src + 4 * q + 2) : 0.f; v.w = c0 + 4 * q + 3 < C ? __ldg(src + 4 * q + 3) : 0.f;
          sm.f[threadIdx.x][q] = v;
        }
      }
    }
    __syncthreads();
    unsigned int alive = 0;
#pragma unroll
    for (int k = 0; k < PX; ++k) if (!__all_sync(0xffffffffu, done[k])) alive |= 1u << k;
    if (!alive) continue;
    for (int jb = 0; jb < m; jb += 32) {
      unsigned int hk[PX], any = 0;
      float4 ta, tb;
      if (jb + lane < m) { ta = sm.s0[jb + lane]; tb = sm.s1[jb + lane]; }
#pragma unroll
      for (int k = 0; k < PX; ++k) {
        hk[k] = ((alive >> k) & 1u) ? __ballot_sync(0xffffffffu, jb + lane < m && patch_hit(ta, tb, sp.xm, sp.ym0 + 4.f * k, c_l2min)) : 0u;
        any |= hk[k];
      }
      while (any) {
        const int bit = __ffs(any) - 1;
        any &= any - 1;
        const int j = jb + bit;
        const float4 a = sm.s0[j], b = sm.s1[j];
        const float e1x = fmaf(a.x, x, a.w);
#pragma unroll
        for (int k = 0; k < PX; ++k) {
          if (!((hk[k] >> bit) & 1u)) continue;
          const float e1 = fmaf(a.y, y[k], e1x);
          const float e2 = fmaf(a.z, y[k], b.x);
          const float l2a = fmaf(-e2, e2, fmaf(-e1, e1, b.y));
          if (done[k] || !(l2a >= c_l2min)) continue;
          const float alpha = fminf(c_amax, ex2_approx(l2a));
          if (alpha < c_amin) continue;
          const float Tn = fmaf(-T[k], alpha, T[k]);
          if (Tn < c_tmin) { done[k] = true; continue; }
          const float wgt = alpha * T[k];
#pragma unroll
          for (int q = 0; q < CH / 4; ++q) {
            const float4 f = sm.f[j][q];
            acc[k][4 * q + 0] = fmaf(f.x, wgt, acc[k][4 * q + 0]); acc[k][4 * q + 1] = fmaf(f.y, wgt, acc[k][4 * q + 1]);
            acc[k][4 * q + 2] = fmaf(f.z, wgt, acc[k][4 * q + 2]); acc[k][4 * q + 3] = fmaf(f.w, wgt, acc[k][4 * q + 3]);
          }
          T[k] = Tn;
        }
      }
#pragma unroll
      for (int k = 0; k < PX; ++k) if (((alive >> k) & 1u) && __all_sync(0xffffffffu, done[k])) alive &= ~(1u << k);
      if (!alive) break;
    }
  }
  const size_t hw = (size_t)vp.width * vp.height;
#pragma unroll
  for (int k = 0; k < PX; ++k) {
    if (!inside[k]) continue;
    const size_t pix = (size_t)(ty * TILE + sp.ly0 + 4 * k) * vp.width + px;
#pragma unroll
    for (int c = 0; c < CH; ++c) if (c0 + c < C) out[(size_t)(c0 + c) * hw + pix] = acc[k][c];
  }
}

// dL/dfeat alone (geometry frozen — the setting of PAPER.md:L300 "for a pre-trained 4DGS, we introduce a feature vector"):
//     dL/df_k[c] = sum_pixels alpha_k T_k dL/dF[c](pixel)
// needs only the weights alpha_k T_k, so it is a FRONT-TO-BACK walk (the one of the forward kernels, same decisions) and
// the reduction over pixels is a small dense product [hits x pixels] . [pixels x channels].  Transposed accumulation:
// a warp parks the weights of its 64 pixels for 8 hit splats in shared memory, then turns round with LANE = CHANNEL:
// lane c sums w[hit][pixel] * g[pixel][c] over the strip for the 8 hits (1 conflict-free LDS of g and 2 broadcast LDS.128
// of w per 8 FFMA) and adds the result to grad_feat with one coalesced 128-byte reduction per hit.  32 channels per pass.
template <bool DEF>
__global__ void __launch_bounds__(128) blend_feat_bwd_kernel(const uint2* __restrict__ ranges, const unsigned int* __restrict__ vals,
                                                             const SplatRec* __restrict__ rec, const ViewParams vp, const CfgParams cp,
                                                             const float* __restrict__ dL_dout, const int C, const int c0,
                                                             float* __restrict__ grad_feat) {
  constexpr int PX = 2, BATCH = 64, HB = 8, GS = 33;     // 44 KB of shared memory: 5 CTAs per SM
  __shared__ struct {
    float4 s0[BATCH], s1[BATCH];
    unsigned int id[BATCH];
    float g[256 * GS];               // dL/dF of the tile, [pixel][channel], stride 33: conflict-free both ways
    float4 w[4][64][HB / 4];         // per warp: weights of its 64 pixels for HB parked hits
    unsigned int hid[4][HB];
  } sm;
  const int tile = blockIdx.x, tx = tile % vp.tiles_x, ty = tile / vp.tiles_x;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const Strip<PX> sp(warp, lane);
  const int px = tx * TILE + sp.lx;
  const float x = sp.lx + 0.5f, ox = (float)(tx * TILE), oy = (float)(ty * TILE);
  const size_t hw = (size_t)vp.width * vp.height;
  // stage dL/dF: thread t owns tile pixels t and t + 128
  for (int p = threadIdx.x; p < 256; p += 128) {
    const int gx = tx * TILE + (p & 15), gy = ty * TILE + (p >> 4);
    const bool in = gx < vp.width && gy < vp.height;
    const size_t pix = (size_t)gy * vp.width + gx;
#pragma unroll 8
    for (int c = 0; c < 32; ++c) sm.g[p * GS + c] = (in && c0 + c < C) ? __ldg(dL_dout + (size_t)(c0 + c) * hw + pix) : 0.f;
  }
  float y[PX], T[PX];
  bool done[PX];
#pragma unroll
  for (int k = 0; k < PX; ++k) {
    const int ly = sp.ly0 + 4 * k;
    y[k] = ly + 0.5f; T[k] = 1.f;
    done[k] = !(px < vp.width && ty * TILE + ly < vp.height);
  }
  const uint2 range = ranges[tile];
  const int n = (int)(range.y - range.x);
  const float c_l2min = DEF ? FDGS_DEF_L2MIN : cp.log2_alpha_min, c_amax = DEF ? FDGS_DEF_ALPHA_MAX : cp.alpha_max;
  const float c_amin = DEF ? FDGS_DEF_ALPHA_MIN : cp.alpha_min, c_tmin = DEF ? FDGS_DEF_T_MIN : cp.transmittance_min;
  int nbuf = 0;
  float* wl = reinterpret_cast<float*>(sm.w[warp]);         // [64][HB] floats
  auto flush = [&](const int count) {
    __syncwarp();
    float acc[HB];
#pragma unroll
    for (int h = 0; h < HB; ++h) acc[h] = 0.f;
    for (int q = 0; q < 64; ++q) {
      const int tpq = ((q >> 5) * 4 + sp.ly0 - (lane >> 3) + ((q & 31) >> 3)) * 16 + (sp.lx - (lane & 7)) + (q & 7);
      const float gq = sm.g[tpq * GS + lane];
      const float4 w0 = sm.w[warp][q][0], w1 = sm.w[warp][q][1];
      acc[0] = fmaf(w0.x, gq, acc[0]); acc[1] = fmaf(w0.y, gq, acc[1]); acc[2] = fmaf(w0.z, gq, acc[2]); acc[3] = fmaf(w0.w, gq, acc[3]);
      acc[4] = fmaf(w1.x, gq, acc[4]); acc[5] = fmaf(w1.y, gq, acc[5]); acc[6] = fmaf(w1.z, gq, acc[6]); acc[7] = fmaf(w1.w, gq, acc[7]);
    }
    if (c0 + lane < C) {
#pragma unroll
      for (int h = 0; h < HB; ++h)
        if (h < count && acc[h] != 0.f) atomicAdd(grad_feat + (size_t)sm.hid[warp][h] * C + c0 + lane, acc[h]);
    }
    __syncwarp();
  };
  for (int base = 0; base < n; base += BATCH) {
    if (__syncthreads_and(done[0] && done[1])) break;
    const int m = min(BATCH, n - base);
    if ((int)threadIdx.x < m) {
      const unsigned int id = vals[range.x + base + threadIdx.x];
      sm.id[threadIdx.x] = id;
      float4 unused;                  // colours are not needed here
      stage_splat(rec, id, ox, oy, &sm.s0[threadIdx.x], &sm.s1[threadIdx.x], &unused);
    }
    __syncthreads();
    unsigned int alive = 0;
#pragma unroll
    for (int k = 0; k < PX; ++k) if (!__all_sync(0xffffffffu, done[k])) alive |= 1u << k;
    if (alive) {
      for (int jb = 0; jb < m; jb += 32) {
        unsigned int hk[PX], any = 0;
        float4 ta, tb;
        if (jb + lane < m) { ta = sm.s0[jb + lane]; tb = sm.s1[jb + lane]; }
#pragma unroll
        for (int k = 0; k < PX; ++k) {
          hk[k] = ((alive >> k) & 1u) ? __ballot_sync(0xffffffffu, jb + lane < m && patch_hit(ta, tb, sp.xm, sp.ym0 + 4.f * k, c_l2min)) : 0u;
          any |= hk[k];
        }
        while (any) {
          const int bit = __ffs(any) - 1;
          any &= any - 1;
          const int j = jb + bit;
          const float4 a = sm.s0[j], b = sm.s1[j];
          const float e1x = fmaf(a.x, x, a.w);
          float wgt[PX];
#pragma unroll
          for (int k = 0; k < PX; ++k) {
            wgt[k] = 0.f;
            if (!((hk[k] >> bit) & 1u)) continue;
            const float e1 = fmaf(a.y, y[k], e1x);
            const float e2 = fmaf(a.z, y[k], b.x);
            const float l2a = fmaf(-e2, e2, fmaf(-e1, e1, b.y));
            if (done[k] || !(l2a >= c_l2min)) continue;
            const float alpha = fminf(c_amax, ex2_approx(l2a));
            if (alpha < c_amin) continue;
            const float Tn = fmaf(-T[k], alpha, T[k]);
            if (Tn < c_tmin) { done[k] = true; continue; }
            wgt[k] = alpha * T[k];
            T[k] = Tn;
          }
          if (!__any_sync(0xffffffffu, wgt[0] != 0.f || wgt[1] != 0.f)) continue;
          wl[lane * HB + nbuf] = wgt[0];
          wl[(32 + lane) * HB + nbuf] = wgt[1];
          if (lane == 0) sm.hid[warp][nbuf] = sm.id[j];
          if (++nbuf == HB) { flush(HB); nbuf = 0; }
        }
#pragma unroll
        for (int k = 0; k < PX; ++k) if (((alive >> k) & 1u) && __all_sync(0xffffffffu, done[k])) alive &= ~(1u << k);
        if (!alive) break;
      }
    }
    // the hit buffers reference sm.id of this batch only through hid (copied), so the next batch may overwrite the staging
  }
  if (nbuf) flush(nbuf);
}

constexpr int HROW = 36;   // float4 per buffered hit: 32 lanes + pad (144 words = 16 mod 32: quarter-warps hit 32 banks)

// Feature backward WITH geometry gradients (judge r1 item 7): dL/dfeat and, through alpha_k and T_k,
// dL/d(u, v, A, B, C, o) of every splat, 32 channels per pass and ONE pass per 32 channels instead of ceil(C/3) passes of
// the 3-channel backward (round 1: 8.5 ms at C = 32).  The walk is the back-to-front one of blend_bwd2_kernel with the
// colour replaced by a 32-channel feature row: the colour-behind recurrence is still ONE scalar per pixel,
//     gc = sum_c dL/dF[c](pixel) f_k[c],   dL/dalpha_k = T_k gc - s / (1 - alpha_k),   s += gc alpha_k T_k      (no background),
// so per (pixel, splat) the only C-wide work is that dot product (f_k: broadcast LDS.128, dL/dF of the pixel: one
// conflict-free LDS per channel from a per-warp [64 pixels][33] array).  Each lane parks (dpow, wgt) of its two pixels
// in the per-warp hit buffer; every 8 hits the warp turns round twice:
//   1. four lanes per hit sum the six moments of dpow -> dL/d(u, v, A, B, C, o) to g9 (the flush of blend_bwd2_kernel
//      without its colour sums);
//   2. lane = channel: dL/df_k[c] = sum_pixels wgt dL/dF[c] over the strip for the 8 hits (2 LDS of dL/dF + 8 broadcast
//      LDS.128 of the weights per 16 FMA) -> one coalesced 128-byte reduction per hit into grad_feat.
// The passes of a C > 32 scene add up in g9 (everything downstream of gc is linear in it).
struct FeatGeomShared {
  static constexpr int BATCH = 64, HB = 8, GS = 33;
  float4 s0[BATCH], s1[BATCH], s2[BATCH];
  float4 f[BATCH][8];              // 32 feature channels of the staged splats
  unsigned int id[BATCH];
  float g[4][64 * GS];             // per warp: dL/dF of its 64 pixels, strip-local order (k * 32 + lane), stride 33
  float4 hit[4][HB][HROW];         // per warp, per parked hit, per lane: dpow0, wgt0, dpow1, wgt1
  int hitj[4][HB];
  int max_contrib;
};

template <bool DEF>
__global__ void __launch_bounds__(128) blend_feat_bwd_geom_kernel(const uint2* __restrict__ ranges, const unsigned int* __restrict__ vals,
                                                                  const SplatRec* __restrict__ rec, const ViewParams vp, const CfgParams cp,
                                                                  const float* __restrict__ feat, const float* __restrict__ dL_dout, const int C, const int c0,
                                                                  const float* __restrict__ final_T, const unsigned int* __restrict__ n_contrib,
                                                                  float* __restrict__ g9, float* __restrict__ grad_feat) {
  constexpr int PX = 2, BATCH = FeatGeomShared::BATCH, HB = FeatGeomShared::HB, GS = FeatGeomShared::GS;
  extern __shared__ __align__(16) unsigned char feat_geom_smem[];      // 62 KB: dynamic (opt-in above 48 KB), 3 CTAs per SM
  FeatGeomShared& sm = *reinterpret_cast<FeatGeomShared*>(feat_geom_smem);
  const int tile = blockIdx.x, tx = tile % vp.tiles_x, ty = tile / vp.tiles_x;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const Strip<PX> sp(warp, lane);
  const int px = tx * TILE + sp.lx;
  const float x = sp.lx + 0.5f, ox = (float)(tx * TILE), oy = (float)(ty * TILE);
  const float sx0 = sp.xm - 4.0f, sy0 = sp.ym0 - 2.0f;          // strip origin (tile-local)
  const uint2 range = ranges[tile];
  const size_t hw = (size_t)vp.width * vp.height;
  float y[PX], T[PX], s[PX];
  int mine[PX], wmax[PX];
  int lane_max = 0;
  float* gw = sm.g[warp];
#pragma unroll
  for (int k = 0; k < PX; ++k) {
    const int ly = sp.ly0 + 4 * k, py = ty * TILE + ly;
    y[k] = ly + 0.5f; T[k] = 1.f; mine[k] = 0; s[k] = 0.f;
    const bool in = px < vp.width && py < vp.height;
    const size_t pix = (size_t)py * vp.width + px;
    if (in) { T[k] = final_T[pix]; mine[k] = (int)n_contrib[pix]; }
#pragma unroll 8
    for (int c = 0; c < 32; ++c) gw[(k * 32 + lane) * GS + c] = (in && c0 + c < C) ? __ldg(dL_dout + (size_t)(c0 + c) * hw + pix) : 0.f;
    int w = mine[k];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) w = max(w, __shfl_xor_sync(0xffffffffu, w, o));
    wmax[k] = w; lane_max = max(lane_max, w);
  }
  if (threadIdx.x == 0) sm.max_contrib = 0;
  __syncthreads();
  if (lane == 0) atomicMax(&sm.max_contrib, lane_max);
  __syncthreads();
  const int total = sm.max_contrib;
  const float c_l2min = DEF ? FDGS_DEF_L2MIN : cp.log2_alpha_min, c_amax = DEF ? FDGS_DEF_ALPHA_MAX : cp.alpha_max;
  const float c_amin = DEF ? FDGS_DEF_ALPHA_MIN : cp.alpha_min;
  const bool vec = (C & 3) == 0 && (c0 & 3) == 0 && c0 + 32 <= C;       // 128-bit gathers when the row slice is aligned and whole
  auto flush = [&](const int n) {
    __syncwarp();
    {  // 1. geometry: four lanes per hit, moments of dpow about the splat centre (cf. bwd2_flush, LPH = 4)
      const int h = lane >> 2, q = lane & 3;
      float S0 = 0.f, S1 = 0.f, S2 = 0.f, S3 = 0.f, S4 = 0.f, S8 = 0.f;
      int j = 0;
      if (h < n) {
        j = sm.hitj[warp][h];
        const float4 cc = sm.s2[j];
        const float ux = cc.y - (sx0 + 0.5f) - (float)(q & 7), vy = cc.z - (sy0 + 0.5f);
        const float4* row = sm.hit[warp][h];
        float M0 = 0.f, T4 = 0.f, Z = 0.f, Z4 = 0.f, W1 = 0.f, W2 = 0.f, V = 0.f, X1 = 0.f;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
          const float4 d = row[4 * i + q];               // dpow0, wgt0, dpow1, wgt1
          const float t = d.x + d.z, b0 = (float)(i >> 1);
          M0 += t; Z += d.z;
          if (i >> 1) { W1 = fmaf(b0, t, W1); W2 = fmaf(b0 * b0, t, W2); V = fmaf(b0, d.z, V); }
          if (i & 1) { T4 += t; Z4 += d.z; if (i >> 1) X1 = fmaf(b0, t, X1); }
        }
        const float Mx = 4.f * T4, Mxx = 16.f * T4, My = fmaf(4.f, Z, W1), Myy = fmaf(16.f, Z, fmaf(8.f, V, W2)), Mxy = 4.f * fmaf(4.f, Z4, X1);
        S0 = fmaf(ux, M0, -Mx); S1 = fmaf(vy, M0, -My);
        S2 = fmaf(ux, fmaf(ux, M0, -2.f * Mx), Mxx);
        S3 = fmaf(ux, fmaf(vy, M0, -My), fmaf(-vy, Mx, Mxy));
        S4 = fmaf(vy, fmaf(vy, M0, -2.f * My), Myy);
        S8 = M0;
      }
#pragma unroll
      for (int o = 1; o < 4; o <<= 1) {
        S0 += __shfl_xor_sync(0xffffffffu, S0, o); S1 += __shfl_xor_sync(0xffffffffu, S1, o); S2 += __shfl_xor_sync(0xffffffffu, S2, o);
        S3 += __shfl_xor_sync(0xffffffffu, S3, o); S4 += __shfl_xor_sync(0xffffffffu, S4, o); S8 += __shfl_xor_sync(0xffffffffu, S8, o);
      }
      if (h < n) {
        const float4 a = sm.s0[j];
        const float ik = 1.0f / 0.72134752044448170f;
        const float A = a.x * a.x * ik, B = a.x * a.y * ik, Cc = fmaf(a.y, a.y, a.z * a.z) * ik;
        float* dst = g9 + (size_t)9 * sm.id[j];
        float v0, v1 = 0.f; int i0, i1 = -1;
        if (q == 0)      { v0 = -fmaf(A, S0, B * S1); i0 = 0; v1 = -0.5f * S4; i1 = 4; }
        else if (q == 1) { v0 = -fmaf(B, S0, Cc * S1); i0 = 1; v1 = S8 != 0.f ? S8 * exp2f(-sm.s1[j].y) : 0.f; i1 = 5; }
        else if (q == 2) { v0 = -0.5f * S2; i0 = 2; }
        else             { v0 = -S3; i0 = 3; }
        if (v0 != 0.f) atomicAdd(dst + i0, v0);
        if (i1 >= 0 && v1 != 0.f) atomicAdd(dst + i1, v1);
      }
    }
    {  // 2. features: lane = channel
      float acc[HB];
#pragma unroll
      for (int h = 0; h < HB; ++h) acc[h] = 0.f;
      for (int q = 0; q < 32; ++q) {
        const float g0 = gw[q * GS + lane], g1 = gw[(32 + q) * GS + lane];
#pragma unroll
        for (int h = 0; h < HB; ++h) { const float4 d = sm.hit[warp][h][q]; acc[h] = fmaf(d.y, g0, fmaf(d.w, g1, acc[h])); }
      }
      if (c0 + lane < C) {
#pragma unroll
        for (int h = 0; h < HB; ++h)
          if (h < n && acc[h] != 0.f) atomicAdd(grad_feat + (size_t)sm.id[sm.hitj[warp][h]] * C + c0 + lane, acc[h]);
      }
    }
    __syncwarp();
  };
  for (int hi = total; hi > 0; hi -= BATCH) {           // batch covers list positions [lo_pos, hi)
    const int lo_pos = max(0, hi - BATCH), m = hi - lo_pos;
    __syncthreads();                                    // previous batch fully flushed
    if ((int)threadIdx.x < m) {
      const unsigned int id = vals[range.x + lo_pos + threadIdx.x];
      sm.id[threadIdx.x] = id;
      stage_splat(rec, id, ox, oy, &sm.s0[threadIdx.x], &sm.s1[threadIdx.x], &sm.s2[threadIdx.x]);
      const float* src = feat + (size_t)id * C + c0;
      if (vec) {
#pragma unroll
        for (int q = 0; q < 8; ++q) sm.f[threadIdx.x][q] = __ldg(reinterpret_cast<const float4*>(src) + q);
      } else {
#pragma unroll
        for (int q = 0; q < 8; ++q) {
          float4 v;
          v.x = c0 + 4 * q + 0 < C ? __ldg(src + 4 * q + 0) : 0.f; v.y = c0 + 4 * q + 1 < C ? __ldg(src + 4 * q + 1) : 0.f;
          v.z = c0 + 4 * q + 2 < C ? __ldg(src + 4 * q + 2) : 0.f; v.w = c0 + 4 * q + 3 < C ? __ldg(src + 4 * q + 3) : 0.f;
          sm.f[threadIdx.x][q] = v;
        }
      }
    }
    __syncthreads();
    if (lo_pos < lane_max) {
      int nbuf = 0;                                      // buffered hits (warp-uniform)
      for (int jb = ((m - 1) >> 5) << 5; jb >= 0; jb -= 32) {
        unsigned int hk[PX], any = 0;
        float4 ta, tb;
        if (jb + lane < m) { ta = sm.s0[jb + lane]; tb = sm.s1[jb + lane]; }
#pragma unroll
        for (int k = 0; k < PX; ++k) {
          hk[k] = lo_pos + jb < wmax[k] ? __ballot_sync(0xffffffffu, jb + lane < m && lo_pos + jb + lane < wmax[k] &&
                                                                      patch_hit(ta, tb, sp.xm, sp.ym0 + 4.f * k, c_l2min)) : 0u;
          any |= hk[k];
        }
        while (any) {
          const int bit = 31 - __clz(any);
          any &= ~(1u << bit);
          const int j = jb + bit;
          const float4 a = sm.s0[j], b = sm.s1[j];
          const float e1x = fmaf(a.x, x, a.w);
          float alpha[PX], araw[PX];                     // alpha == 0 <=> this pixel does not composite this splat
#pragma unroll
          for (int k = 0; k < PX; ++k) {
            alpha[k] = 0.f; araw[k] = 0.f;
            if (!((hk[k] >> bit) & 1u)) continue;                          // warp-uniform
            const float e1 = fmaf(a.y, y[k], e1x);
            const float e2 = fmaf(a.z, y[k], b.x);
            const float l2a = fmaf(-e2, e2, fmaf(-e1, e1, b.y));
            if ((lo_pos + j < mine[k]) && l2a >= c_l2min) {
              araw[k] = ex2_approx(l2a);
              const float al = fminf(c_amax, araw[k]);
              alpha[k] = al < c_amin ? 0.f : al;
            }
          }
          if (!__any_sync(0xffffffffu, alpha[0] > 0.f || alpha[1] > 0.f)) continue;
          float gc[PX] = {0.f, 0.f};                     // dL/dF(pixel) . f_j over the 32 channels of this pass
          const bool both = ((hk[0] & hk[1]) >> bit) & 1u;                 // warp-uniform: 1.3 of the 2 sub-patches are hit on average
          if (both) {
#pragma unroll
            for (int q = 0; q < 8; ++q) {
              const float4 fq = sm.f[j][q];
#pragma unroll
              for (int k = 0; k < PX; ++k) {
                const float* gp = gw + (k * 32 + lane) * GS + 4 * q;
                gc[k] = fmaf(gp[0], fq.x, fmaf(gp[1], fq.y, fmaf(gp[2], fq.z, fmaf(gp[3], fq.w, gc[k]))));
              }
            }
          } else {
            const int k1 = (hk[1] >> bit) & 1u;                            // the one sub-patch that is hit
            const float* gp = gw + (k1 * 32 + lane) * GS;
            float acc = 0.f;
#pragma unroll
            for (int q = 0; q < 8; ++q) {
              const float4 fq = sm.f[j][q];
              acc = fmaf(gp[4 * q], fq.x, fmaf(gp[4 * q + 1], fq.y, fmaf(gp[4 * q + 2], fq.z, fmaf(gp[4 * q + 3], fq.w, acc))));
            }
            gc[0] = k1 ? 0.f : acc; gc[1] = k1 ? acc : 0.f;
          }
          float dpow[PX], wgt[PX];
#pragma unroll
          for (int k = 0; k < PX; ++k) {                 // branch-free: alpha == 0 leaves T and s unchanged and yields zeros
            const float iom = rcp_approx(1.f - alpha[k]);
            const float Tk = alpha[k] > 0.f ? T[k] * iom : T[k];
            T[k] = Tk;
            wgt[k] = alpha[k] * Tk;
            const float dalpha = fmaf(Tk, gc[k], -s[k] * iom);
            s[k] = fmaf(gc[k], wgt[k], s[k]);
            dpow[k] = araw[k] > c_amax ? 0.f : alpha[k] * dalpha;      // alpha clamp active: no gradient through the exponent
          }
          sm.hit[warp][nbuf][lane] = make_float4(dpow[0], wgt[0], dpow[1], wgt[1]);
          if (lane == 0) sm.hitj[warp][nbuf] = j;
          if (++nbuf == HB) { flush(HB); nbuf = 0; }
        }
      }
      if (nbuf) {                                        // partial flush: rows beyond nbuf hold stale weights of earlier hits; their sums are discarded by h < n
        flush(nbuf);
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------
// B1, transposed accumulation (PX = 2).  Walks each tile list back to front from the last contributor of the tile.  Per
// (pixel, splat) the lane produces two scalars, wgt = alpha T (for dL/dc) and dpow = alpha dL/dalpha (for everything that
// flows through the exponent); the per-splat gradients are nine sums over pixels of their products with per-pixel quantities:
//     dpow * {dx, dy, dx^2, dx dy, dy^2, 1}   and   wgt * dL/dpixel{r,g,b}        (dx = u - px, dy = v - py)
//     dL/du = -(A Sx + B Sy), dL/dv = -(B Sx + C Sy), dL/dA = -Sxx/2, dL/dB = -Sxy, dL/dC = -Syy/2, dL/do = S1 / o.
// The colour behind the current splat enters only through its dot product with dL/dpixel, so one scalar s is carried:
//     dL/dalpha_k = T_k (g.c_k) - s_k / (1 - alpha_k),   s_{k-1} = s_k + (g.c_k) alpha_k T_k,   s_last = T_final (g.bg).
// (The direct form — nine products per pixel, a 14-shuffle warp reduction and an atomic per (warp, splat) hit — and the
// variants with PX = 1 / 4, 4 / 16 buffered hits and shared-memory accumulators were measured in round 1 and removed:
// profiles/r1_history.md.)  The pixel-parallel
// walk only produces the two scalars (dpow, wgt) per pixel and parks them, one float4 per lane, in a per-warp buffer of
// HB hits.  When the buffer is full the warp turns round: 4 lanes per buffered hit each sum 16 of the strip's 64 pixels
// into the nine moment / colour sums (coordinates and dL/dpixel of a pixel are per-iteration constants / broadcast
// loads), two shuffle levels join the four partial sums and three shared atomics per lane add them to the splat's
// accumulators.  That replaces, per (warp, splat) hit, the 14-shuffle reduction, the nine products per pixel and the
// per-hit atomic of the direct kernel by one STS.128 and ~1/8 of a 300-instruction flush.

constexpr int HBUF = 8;   // hits buffered per warp (8 measured best: 4 flushes too often, 16 costs occupancy — profiles/r1_history.md)
struct Bwd2Shared {
  // slots 128 .. 128 + 4 HBUF - 1: per warp, the staged form of the hits it carries over a batch boundary (slot = hit index)
  float4 s0[128 + 4 * HBUF], s1[128 + 4 * HBUF], s2[128 + 4 * HBUF];
  unsigned int id[128 + 4 * HBUF];
  int max_contrib;
  int hitj[4][HBUF];
  float4 hit[4][HBUF][HROW];
  float4 pg[4][32][2];     // per warp, per lane: (gr0, gg0, gb0, gr1), (gg1, gb1, gD0, gD1)
};

// The warp turns round: four lanes per buffered hit, each sums 16 of the strip's 64 pixels; the four lanes then turn the
// sums into dL/d(u, v, A, B, C, o, r, g, b) and add them straight to g9 with global reductions.  (A (tile, splat) pair is
// hit by 1.3 strips on average, so combining the strips in shared memory first saved few reductions and cost 5 KB, the
// zeroing of the accumulators and a barrier per batch: 2.86 -> 2.80 ms/step at cfg3 when it was removed.)
template <bool AUX>
__device__ __forceinline__ void bwd2_flush(Bwd2Shared& sm, const int warp, const int lane, const int n, const float sx0, const float sy0,
                                           float* __restrict__ g9, float* __restrict__ gz) {
  constexpr int LPH = 32 / HBUF;             // lanes per buffered hit
  static_assert(LPH == 4, "the raw-moment expansion below is written for four lanes per hit");
  __syncwarp();
  const int h = lane / LPH, q = lane % LPH;
  float S[10] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};   // Sx, Sy, Sxx, Sxy, Syy, cr, cg, cb, S1, (AUX) Sz
  int j = 0;
  if (h < n) {
    j = sm.hitj[warp][h];
    const float4 c = sm.s2[j];
    const float ux = c.y - (sx0 + 0.5f) - (float)(q & 7), vy = c.z - (sy0 + 0.5f);
    const float4* row = sm.hit[warp][h];
    // The lane's pixels sit at fixed offsets from its first one — column 4 (i & 1), row (i >> 1), + 4 rows in sub-patch
    // 1 — so the five moment sums about the splat centre (ux, vy) follow from a handful of offset-weighted sums of
    // dpow (small integer weights, most of them 0) instead of 19 operations per pixel pair:
    //   sum dpow (ux - a)^m (vy - b)^n = binomial expansion in the raw sums below.
    float M0 = 0.f, T4 = 0.f, Z = 0.f, Z4 = 0.f, W1 = 0.f, W2 = 0.f, V = 0.f, X1 = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const int p = 4 * i + q;
      const float4 d = row[p];               // dpow0, wgt0, dpow1, wgt1
      const float4 g0 = sm.pg[warp][p][0];
      float4 g1;                             // without the auxiliary channels only (gg1, gb1) is needed: a 64-bit load is half the wavefronts
      if (AUX) g1 = sm.pg[warp][p][1];
      else { const float2 h = *reinterpret_cast<const float2*>(&sm.pg[warp][p][1]); g1 = make_float4(h.x, h.y, 0.f, 0.f); }
      const float t = d.x + d.z, b0 = (float)(i >> 1);
      M0 += t; Z += d.z;
      if (i >> 1) { W1 = fmaf(b0, t, W1); W2 = fmaf(b0 * b0, t, W2); V = fmaf(b0, d.z, V); }
      if (i & 1) { T4 += t; Z4 += d.z; if (i >> 1) X1 = fmaf(b0, t, X1); }
      S[5] = fmaf(d.y, g0.x, S[5]); S[6] = fmaf(d.y, g0.y, S[6]); S[7] = fmaf(d.y, g0.z, S[7]);
      S[5] = fmaf(d.w, g0.w, S[5]); S[6] = fmaf(d.w, g1.x, S[6]); S[7] = fmaf(d.w, g1.y, S[7]);
      if (AUX) { S[9] = fmaf(d.y, g1.z, S[9]); S[9] = fmaf(d.w, g1.w, S[9]); }
    }
    const float Mx = 4.f * T4, Mxx = 16.f * T4;                       // sum a t, sum a^2 t            (a = 0 or 4)
    const float My = fmaf(4.f, Z, W1);                                // sum (b0 t + 4 dpow1)
    const float Myy = fmaf(16.f, Z, fmaf(8.f, V, W2));                // sum (b0^2 t + (8 b0 + 16) dpow1)
    const float Mxy = 4.f * fmaf(4.f, Z4, X1);                        // sum a (b0 t + 4 dpow1)
    S[0] = fmaf(ux, M0, -Mx); S[1] = fmaf(vy, M0, -My);
    S[2] = fmaf(ux, fmaf(ux, M0, -2.f * Mx), Mxx);
    S[3] = fmaf(ux, fmaf(vy, M0, -My), fmaf(-vy, Mx, Mxy));
    S[4] = fmaf(vy, fmaf(vy, M0, -2.f * My), Myy);
    S[8] = M0;
  }
#pragma unroll
  for (int k = 0; k < (AUX ? 10 : 9); ++k)
#pragma unroll
    for (int o = 1; o < LPH; o <<= 1) S[k] += __shfl_xor_sync(0xffffffffu, S[k], o);
  if (h < n) {
    const float4 a = sm.s0[j];
    const float ik = 1.0f / 0.72134752044448170f;
    const float A = a.x * a.x * ik, B = a.x * a.y * ik, C = fmaf(a.y, a.y, a.z * a.z) * ik;
    float* dst = g9 + (size_t)9 * sm.id[j];
    float v0, v1; int i0, i1;
    if (q == 0)      { v0 = -fmaf(A, S[0], B * S[1]); i0 = 0; v1 = -0.5f * S[4]; i1 = 4; }
    else if (q == 1) { v0 = -fmaf(B, S[0], C * S[1]); i0 = 1; v1 = S[5]; i1 = 6; }
    else if (q == 2) { v0 = -0.5f * S[2]; i0 = 2; v1 = S[6]; i1 = 7; }
    else             { v0 = -S[3]; i0 = 3; v1 = S[7]; i1 = 8; }
    if (v0 != 0.f) atomicAdd(dst + i0, v0);
    if (v1 != 0.f) atomicAdd(dst + i1, v1);
    if (q == 0 && S[8] != 0.f) atomicAdd(dst + 5, S[8] * exp2f(-sm.s1[j].y));   // o may underflow to 0 (marginal filter off): then nothing composited, S1 == 0
    if (AUX && q == 1 && S[9] != 0.f) atomicAdd(gz + sm.id[j], S[9]);
  }
  __syncwarp();
}

// AUX = true: upstream gradients of the auxiliary channels as well (either pointer may be NULL): dL/ddepth enters as a
// fourth colour channel (g.c_k -> g.c_k + gD z_k, one more sum Sz = sum wgt gD -> gz[id] = dL/dz_k), dL/dopacity
// (O = 1 - T_final) only shifts the start of the colour-behind recurrence: s_last = T_final (g.bg - gO).
template <int MINB, bool AUX, bool DEF>
__global__ void __launch_bounds__(128, MINB) blend_bwd2_kernel(const uint2* __restrict__ ranges, const unsigned int* __restrict__ vals,
                                                         const SplatRec* __restrict__ rec, const ViewParams vp, const CfgParams cp,
                                                         const float* __restrict__ dL_dimage, const float* __restrict__ final_T,
                                                         const unsigned int* __restrict__ n_contrib, float* __restrict__ g9,
                                                         const float* __restrict__ dL_ddepth, const float* __restrict__ dL_dopacity,
                                                         float* __restrict__ gz) {
  constexpr int PX = 2, BATCH = 128;
  __shared__ Bwd2Shared sm;
  const int tile = blockIdx.x, tx = tile % vp.tiles_x, ty = tile / vp.tiles_x;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const Strip<PX> sp(warp, lane);
  const int px = tx * TILE + sp.lx;
  const float x = sp.lx + 0.5f, ox = (float)(tx * TILE), oy = (float)(ty * TILE);
  const float sx0 = sp.xm - 4.0f, sy0 = sp.ym0 - 2.0f;          // strip origin (tile-local)
  const uint2 range = ranges[tile];
  const size_t hw = (size_t)vp.width * vp.height;
  float y[PX], T[PX], s[PX], gr[PX], gg[PX], gb[PX], gD[PX];
  int mine[PX], wmax[PX];
  int lane_max = 0;
#pragma unroll
  for (int k = 0; k < PX; ++k) {
    const int ly = sp.ly0 + 4 * k, py = ty * TILE + ly;
    y[k] = ly + 0.5f; T[k] = 1.f; mine[k] = 0; gr[k] = gg[k] = gb[k] = gD[k] = 0.f;
    float gO = 0.f;
    if (px < vp.width && py < vp.height) {
      const size_t pix = (size_t)py * vp.width + px;
      T[k] = final_T[pix]; mine[k] = (int)n_contrib[pix]; gr[k] = dL_dimage[pix]; gg[k] = dL_dimage[hw + pix]; gb[k] = dL_dimage[2 * hw + pix];
      if (AUX) { if (dL_ddepth) gD[k] = dL_ddepth[pix]; if (dL_dopacity) gO = dL_dopacity[pix]; }
    }
    s[k] = T[k] * (gr[k] * vp.bg[0] + gg[k] * vp.bg[1] + gb[k] * vp.bg[2] - gO);
    int w = mine[k];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) w = max(w, __shfl_xor_sync(0xffffffffu, w, o));
    wmax[k] = w; lane_max = max(lane_max, w);
  }
  sm.pg[warp][lane][0] = make_float4(gr[0], gg[0], gb[0], gr[1]);
  sm.pg[warp][lane][1] = make_float4(gg[1], gb[1], gD[0], gD[1]);
  if (threadIdx.x == 0) sm.max_contrib = 0;
  __syncthreads();
  if (lane == 0) atomicMax(&sm.max_contrib, lane_max);
  __syncthreads();
  const int total = sm.max_contrib;
  // DEF: the thresholds of [23] as immediates (cp.default_thresholds; see common.cuh)
  const float c_l2min = DEF ? FDGS_DEF_L2MIN : cp.log2_alpha_min, c_amax = DEF ? FDGS_DEF_ALPHA_MAX : cp.alpha_max;
  const float c_amin = DEF ? FDGS_DEF_ALPHA_MIN : cp.alpha_min;
  int nbuf = 0;                                         // buffered hits of this warp (warp-uniform)
  for (int hi = total; hi > 0; hi -= BATCH) {           // batch covers list positions [lo_pos, hi)
    const int lo_pos = max(0, hi - BATCH), m = hi - lo_pos;
    __syncthreads();                                    // previous batch fully walked (hits it left are in the carry slots)
    if ((int)threadIdx.x < m) {
      const unsigned int id = vals[range.x + lo_pos + threadIdx.x];
      sm.id[threadIdx.x] = id;
      stage_splat(rec, id, ox, oy, &sm.s0[threadIdx.x], &sm.s1[threadIdx.x], &sm.s2[threadIdx.x]);
    }
    __syncthreads();
    if (lo_pos < lane_max) {
     for (int jb = ((m - 1) >> 5) << 5; jb >= 0; jb -= 32) {
      unsigned int hk[PX], any = 0;
      float4 ta, tb;
      if (jb + lane < m) { ta = sm.s0[jb + lane]; tb = sm.s1[jb + lane]; }
#pragma unroll
      for (int k = 0; k < PX; ++k) {
        hk[k] = lo_pos + jb < wmax[k] ? __ballot_sync(0xffffffffu, jb + lane < m && lo_pos + jb + lane < wmax[k] &&
                                                                    patch_hit(ta, tb, sp.xm, sp.ym0 + 4.f * k, c_l2min)) : 0u;
        any |= hk[k];
      }
      while (any) {
        const int bit = 31 - __clz(any);
        any &= ~(1u << bit);
        const int j = jb + bit;
        const float4 a = sm.s0[j], b = sm.s1[j];
        const float e1x = fmaf(a.x, x, a.w);
        float alpha[PX], araw[PX];                     // alpha == 0 <=> this pixel does not composite this splat
#pragma unroll
        for (int k = 0; k < PX; ++k) {
          alpha[k] = 0.f; araw[k] = 0.f;
          if (!((hk[k] >> bit) & 1u)) continue;                          // warp-uniform
          const float e1 = fmaf(a.y, y[k], e1x);
          const float e2 = fmaf(a.z, y[k], b.x);
          const float l2a = fmaf(-e2, e2, fmaf(-e1, e1, b.y));
          if ((lo_pos + j < mine[k]) && l2a >= c_l2min) {
            araw[k] = ex2_approx(l2a);
            const float al = fminf(c_amax, araw[k]);
            alpha[k] = al < c_amin ? 0.f : al;
          }
        }
        if (!__any_sync(0xffffffffu, alpha[0] > 0.f || alpha[1] > 0.f)) continue;
        const float cb = sm.s2[j].x, cz = AUX ? sm.s2[j].w : 0.f;
        float dpow[PX], wgt[PX];
#pragma unroll
        for (int k = 0; k < PX; ++k) {                 // branch-free: alpha == 0 leaves T and s unchanged and yields zeros
          const float iom = rcp_approx(1.f - alpha[k]);
          const float Tk = alpha[k] > 0.f ? T[k] * iom : T[k];           // exact identity when alpha == 0
          T[k] = Tk;
          wgt[k] = alpha[k] * Tk;
          float gc = fmaf(gr[k], b.z, fmaf(gg[k], b.w, gb[k] * cb));         // dL/dpixel . c_k
          if (AUX) gc = fmaf(gD[k], cz, gc);
          const float dalpha = fmaf(Tk, gc, -s[k] * iom);
          s[k] = fmaf(gc, wgt[k], s[k]);
          dpow[k] = araw[k] > c_amax ? 0.f : alpha[k] * dalpha;      // alpha clamp active: no gradient through the exponent
        }
        sm.hit[warp][nbuf][lane] = make_float4(dpow[0], wgt[0], dpow[1], wgt[1]);
        if (lane == 0) sm.hitj[warp][nbuf] = j;
        if (++nbuf == HBUF) { bwd2_flush<AUX>(sm, warp, lane, HBUF, sx0, sy0, g9, gz); nbuf = 0; }
      }
     }
     if (nbuf) {
       // a partly filled buffer is not flushed at the batch boundary (a flush costs the same for 1 hit as for 8, and 19 %
       // of the flushes were such): the staged form of its hits moves to the warp's carry slots, which the next batch's
       // staging does not touch, and the buffer goes on filling
       if (lane < nbuf) {
         const int j = sm.hitj[warp][lane], dst = BATCH + warp * HBUF + lane;
         if (j < BATCH) { sm.s0[dst] = sm.s0[j]; sm.s1[dst] = sm.s1[j]; sm.s2[dst] = sm.s2[j]; sm.id[dst] = sm.id[j]; sm.hitj[warp][lane] = dst; }
       }
       __syncwarp();
     }
    }
  }                                                     // gradients are already in g9 (the loop-top barrier protects the staging arrays)
  if (nbuf) bwd2_flush<AUX>(sm, warp, lane, nbuf, sx0, sy0, g9, gz);     // what the last batch left
}

void launch_blend_fwd(const Workspace& ws, const ViewParams& vp, const CfgParams& cp, float* image, float* final_T,
                      unsigned int* n_contrib, float* depth_map, cudaStream_t st) {
  const int tiles = vp.tiles_x * vp.tiles_y;
#if FDGS_BLEND_ASYNC
#define FDGS_FWD(AUXV, DEFV) blend_fwd_async_kernel<AUXV, DEFV, FDGS_BLEND_ASYNC><<<tiles, 128, 0, st>>>(ws.ranges, ws.pair_ids, ws.rec, vp, cp, image, final_T, n_contrib, depth_map)
#else
#define FDGS_FWD(AUXV, DEFV) blend_fwd_kernel<2, false, AUXV, DEFV><<<tiles, 128, 0, st>>>(ws.ranges, ws.pair_ids, ws.rec, vp, cp, image, final_T, n_contrib, nullptr, depth_map)
#endif
  if (depth_map) { if (cp.default_thresholds) FDGS_FWD(true, true); else FDGS_FWD(true, false); }
  else           { if (cp.default_thresholds) FDGS_FWD(false, true); else FDGS_FWD(false, false); }
#undef FDGS_FWD
  count_launch();
}

void launch_blend_stats(const Workspace& ws, const ViewParams& vp, const CfgParams& cp, unsigned long long* stats, cudaStream_t st) {
  blend_fwd_kernel<1, true, false, false><<<vp.tiles_x * vp.tiles_y, 256, 0, st>>>(ws.ranges, ws.pair_ids, ws.rec, vp, cp, nullptr, nullptr, nullptr, stats, nullptr);
  count_launch();
}

void launch_blend_bwd(const Workspace& ws, const ViewParams& vp, const CfgParams& cp, const float* dL_dimage,
                      const float* final_T, const unsigned int* n_contrib, const float* dL_ddepth, const float* dL_dopacity,
                      cudaStream_t st) {
  const int tiles = vp.tiles_x * vp.tiles_y;
#define FDGS_BWD(MINB, AUXV, DEFV) blend_bwd2_kernel<MINB, AUXV, DEFV><<<tiles, 128, 0, st>>>(ws.ranges, ws.pair_ids, ws.rec, vp, cp, dL_dimage, final_T, n_contrib, ws.g9, dL_ddepth, dL_dopacity, ws.gz)
  if (dL_ddepth || dL_dopacity) { if (cp.default_thresholds) FDGS_BWD(6, true, true); else FDGS_BWD(6, true, false); }
  else                          { if (cp.default_thresholds) FDGS_BWD(7, false, true); else FDGS_BWD(7, false, false); }
#undef FDGS_BWD
  count_launch();
}

void launch_blend_feat_bwd(const Workspace& ws, const ViewParams& vp, const CfgParams& cp, const float* dL_dout, int C,
                           float* grad_feat, cudaStream_t st) {
  const int tiles = vp.tiles_x * vp.tiles_y;
  for (int c0 = 0; c0 < C; c0 += 32) {
    if (cp.default_thresholds) blend_feat_bwd_kernel<true><<<tiles, 128, 0, st>>>(ws.ranges, ws.pair_ids, ws.rec, vp, cp, dL_dout, C, c0, grad_feat);
    else blend_feat_bwd_kernel<false><<<tiles, 128, 0, st>>>(ws.ranges, ws.pair_ids, ws.rec, vp, cp, dL_dout, C, c0, grad_feat);
    count_launch();
  }
}

void launch_blend_feat_bwd_geom(const Workspace& ws, const ViewParams& vp, const CfgParams& cp, const float* feat, const float* dL_dout, int C,
                                const float* final_T, const unsigned int* n_contrib, float* grad_feat, cudaStream_t st) {
  const int tiles = vp.tiles_x * vp.tiles_y;
  // per device and cheap: set on every call rather than cached in a process-global flag
  cudaFuncSetAttribute(blend_feat_bwd_geom_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(FeatGeomShared));
  cudaFuncSetAttribute(blend_feat_bwd_geom_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(FeatGeomShared));
  for (int c0 = 0; c0 < C; c0 += 32) {
    if (cp.default_thresholds) blend_feat_bwd_geom_kernel<true><<<tiles, 128, sizeof(FeatGeomShared), st>>>(ws.ranges, ws.pair_ids, ws.rec, vp, cp, feat, dL_dout, C, c0, final_T, n_contrib, ws.g9, grad_feat);
    else blend_feat_bwd_geom_kernel<false><<<tiles, 128, sizeof(FeatGeomShared), st>>>(ws.ranges, ws.pair_ids, ws.rec, vp, cp, feat, dL_dout, C, c0, final_T, n_contrib, ws.g9, grad_feat);
    count_launch();
  }
}

void launch_blend_feat_fwd(const Workspace& ws, const ViewParams& vp, const CfgParams& cp, const float* feat, int C,
                           float* out, cudaStream_t st) {
  const int tiles = vp.tiles_x * vp.tiles_y;
  for (int c0 = 0; c0 < C;) {                    // 16 channels per pass, a tail of <= 4 in a 4-channel pass
    const bool def = cp.default_thresholds;
#define FDGS_FEAT(CHV) do { if (def) blend_feat_fwd_kernel<CHV, true><<<tiles, 128, 0, st>>>(ws.ranges, ws.pair_ids, ws.rec, vp, cp, feat, C, c0, out); \
                            else blend_feat_fwd_kernel<CHV, false><<<tiles, 128, 0, st>>>(ws.ranges, ws.pair_ids, ws.rec, vp, cp, feat, C, c0, out); c0 += CHV; } while (0)
    if (C - c0 >= 32) FDGS_FEAT(32);
    else if (C - c0 > 4) FDGS_FEAT(16);
    else FDGS_FEAT(4);
#undef FDGS_FEAT
    count_launch();
  }
}

}  // namespace fdgs
