// train.cu — per-primitive training-side kernels next to the rasterizer:
//   mask (eq. 21-24), L_sparse / L_covt (eq. 26-27), dense Adam ([23]'s optimiser, L324),
//   decode of the compact model (section 4.2 / 8.3.1, L209, L501).
// All of them stream over the parameter arrays once: HBM-bound (the colour decode is bound by the L2 gather of its
// codebook rows), one thread (or one warp) per primitive, 128-bit accesses where the layout allows.
#include <cmath>
#include <cstdint>

#include <cuda_fp16.h>

#include "common.cuh"
#include "geom.cuh"

namespace fdgs {

#define TRAIN_CUDA(call, where) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return cuda_fail(e_, where); } while (0)

static bool al16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

__device__ __forceinline__ float sigmoidf_(const float x) { return 1.0f / (1.0f + expf(-x)); }

// ---- eq. 21-23: mask forward ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) mask_apply_kernel(const float* __restrict__ mask_logit, const float eps,
                                                         const float* __restrict__ logit, float* __restrict__ out, const int N) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  const bool keep = sigmoidf_(mask_logit[i]) > eps;                 // M_hat = 1{M > eps}
  out[i] = keep ? logit[i] : -INFINITY;                            // alpha_hat = M_hat alpha
}

// ---- eq. 24, 26, 27 fused forward + backward, eq. 21 straight-through gradient --------------------------------------
__global__ void __launch_bounds__(256) regularizers_kernel(const fdgs_scene sc, const float* __restrict__ mask_logit,
                                                           const fdgs_reg_config rc, const fdgs_grads g,
                                                           float* __restrict__ grad_mask, float* __restrict__ losses) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const float invN = 1.0f / (float)sc.N;
  float l_sparse = 0.f, l_covt = 0.f, l_mask = 0.f;
  if (i < sc.N) {
    const float4 ls4 = __ldg(reinterpret_cast<const float4*>(sc.log_scale) + i);
    const float4 ql4 = __ldg(reinterpret_cast<const float4*>(sc.quat_l) + i);
    const float4 qr4 = __ldg(reinterpret_cast<const float4*>(sc.quat_r) + i);
    float4* gls_p = reinterpret_cast<float4*>(g.log_scale) + i;
    float4* gql_p = reinterpret_cast<float4*>(g.quat_l) + i;
    float4* gqr_p = reinterpret_cast<float4*>(g.quat_r) + i;
    float4 gls = *gls_p, gql = *gql_p, gqr = *gqr_p;
    // 1. mask: needs the RENDERING gradient of log_scale, i.e. before the regularisers are added below
    if (mask_logit) {
      const float m = mask_logit[i];
      const float M = sigmoidf_(m), dM = M * sigmoidf_(-m);        // M (1 - M) without cancellation
      float gm = rc.lambda_mask * dM * invN;
      l_mask = M;
      if (M > rc.mask_eps) {
        const float logit = sc.opacity_logit[i];
        const float one_minus_alpha = sigmoidf_(-logit);
        const float go = g.opacity_logit[i];
        float dMhat = (gls.x + gls.y) + (gls.z + gls.w);
        if (go != 0.f) dMhat += go / one_minus_alpha;              // 0 / 0 when a saturated logit has no gradient
        if (isfinite(dMhat)) gm = fmaf(dMhat, dM, gm);
      }
      if (isfinite(gm)) grad_mask[i] += gm;
    }
    // 2. regularisers on the normalised quaternions and exp(log_scale)
    const float qlr[4] = {ql4.x, ql4.y, ql4.z, ql4.w}, qrr[4] = {qr4.x, qr4.y, qr4.z, qr4.w};
    const float lsv[4] = {ls4.x, ls4.y, ls4.z, ls4.w};
    float nl2 = 0.f, nr2 = 0.f;
#pragma unroll
    for (int k = 0; k < 4; ++k) { nl2 = fmaf(qlr[k], qlr[k], nl2); nr2 = fmaf(qrr[k], qrr[k], nr2); }
    const float chk = nl2 + nr2 + lsv[0] + lsv[1] + lsv[2] + lsv[3];
    if (isfinite(chk) && nl2 > 0.f && nr2 > 0.f) {
      const float inl = rsqrtf(nl2), inr = rsqrtf(nr2);
      float ql[4], qr[4], dql[4], dqr[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) { ql[k] = qlr[k] * inl; qr[k] = qrr[k] * inr; }
      // eq. 26: |q_l - q_r|_1, sign(0) = 0
      const float ws = rc.lambda_sparse * invN;
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const float d = ql[k] - qr[k];
        l_sparse += fabsf(d);
        const float sg = d > 0.f ? ws : (d < 0.f ? -ws : 0.f);
        dql[k] = sg; dqr[k] = -sg;
      }
      // eq. 27: Sigma_44 = sum_k (R_4k s_k)^2, R_4. = l^T R(q_r) with l = time row of L(q_l) = (d, -c, b, a)
      const float l[4] = {ql[3], -ql[2], ql[1], ql[0]};
      float Rm[4][4];
      quat_right(qr, Rm);
      float r4[4], s2[4], S44 = 0.f;
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        r4[k] = fmaf(l[0], Rm[0][k], fmaf(l[1], Rm[1][k], fmaf(l[2], Rm[2][k], l[3] * Rm[3][k])));
        const float s = expf(lsv[k]);
        s2[k] = s * s;
        S44 = fmaf(r4[k] * r4[k], s2[k], S44);
      }
      const float e = expf(-S44);
      if (e > 0.f && isfinite(S44)) {     // e == 0 (Sigma_44 large or overflowed): loss and gradient vanish, 0 * inf must not appear
        l_covt = e;
        const float gS = -rc.lambda_covt * e * invN;
        float gr[4], gl[4];
        gls.x = fmaf(gS, 2.f * r4[0] * r4[0] * s2[0], gls.x); gls.y = fmaf(gS, 2.f * r4[1] * r4[1] * s2[1], gls.y);
        gls.z = fmaf(gS, 2.f * r4[2] * r4[2] * s2[2], gls.z); gls.w = fmaf(gS, 2.f * r4[3] * r4[3] * s2[3], gls.w);
#pragma unroll
        for (int k = 0; k < 4; ++k) gr[k] = gS * 2.f * r4[k] * s2[k];
#pragma unroll
        for (int j = 0; j < 4; ++j) gl[j] = fmaf(gr[0], Rm[j][0], fmaf(gr[1], Rm[j][1], fmaf(gr[2], Rm[j][2], gr[3] * Rm[j][3])));
        dql[0] += gl[3]; dql[1] += gl[2]; dql[2] -= gl[1]; dql[3] += gl[0];
        // G[j][k] = l_j gr_k against the sign pattern of R(q_r)
#define G_(j, k) (l[j] * gr[k])
        dqr[0] += G_(0, 0) + G_(1, 1) + G_(2, 2) + G_(3, 3);
        dqr[1] += -G_(0, 1) + G_(1, 0) + G_(2, 3) - G_(3, 2);
        dqr[2] += -G_(0, 2) - G_(1, 3) + G_(2, 0) + G_(3, 1);
        dqr[3] += -G_(0, 3) + G_(1, 2) - G_(2, 1) + G_(3, 0);
#undef G_
      }
      // through the normalisation: dq = (dq_hat - q_hat (q_hat . dq_hat)) / |q|
      float dl = 0.f, dr = 0.f;
#pragma unroll
      for (int k = 0; k < 4; ++k) { dl = fmaf(ql[k], dql[k], dl); dr = fmaf(qr[k], dqr[k], dr); }
      gql.x += (dql[0] - ql[0] * dl) * inl; gql.y += (dql[1] - ql[1] * dl) * inl;
      gql.z += (dql[2] - ql[2] * dl) * inl; gql.w += (dql[3] - ql[3] * dl) * inl;
      gqr.x += (dqr[0] - qr[0] * dr) * inr; gqr.y += (dqr[1] - qr[1] * dr) * inr;
      gqr.z += (dqr[2] - qr[2] * dr) * inr; gqr.w += (dqr[3] - qr[3] * dr) * inr;
      *gls_p = gls; *gql_p = gql; *gqr_p = gqr;
    }
  }
  // 3. loss sums: warp shuffle, then one atomic per warp and loss
  if (losses) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      l_sparse += __shfl_xor_sync(0xffffffffu, l_sparse, o);
      l_covt += __shfl_xor_sync(0xffffffffu, l_covt, o);
      l_mask += __shfl_xor_sync(0xffffffffu, l_mask, o);
    }
    __shared__ float red[3][8];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0) { red[0][warp] = l_sparse; red[1][warp] = l_covt; red[2][warp] = l_mask; }
    __syncthreads();
    if (threadIdx.x < 3) {
      float s = 0.f;
#pragma unroll
      for (int w = 0; w < 8; ++w) s += red[threadIdx.x][w];
      if (s != 0.f) atomicAdd(losses + threadIdx.x, s * invN);
    }
  }
}

// ---- dense Adam ------------------------------------------------------------------------------------------------------
// 28 B (32 with zero_grad) of HBM traffic per element and ~10 flops: a pure streaming kernel.  Two float4 per thread and
// array keep 8 independent 128-bit loads in flight per thread; streaming cache hints (no reuse).
struct AdamK { float b1, b2, omb1, omb2, step_size, inv_sqrt_bc2, eps; };

__device__ __forceinline__ void adam_one(float& p, const float g, float& m, float& v, const AdamK& a) {
  m = fmaf(a.b1, m, a.omb1 * g);
  v = fmaf(a.b2, v, a.omb2 * g * g);
  const float denom = fmaf(sqrtf(v), a.inv_sqrt_bc2, a.eps);
  p = p - a.step_size * (m / denom);
}

__global__ void __launch_bounds__(256) adam_kernel(float* __restrict__ param, float* __restrict__ grad, float* __restrict__ ea,
                                                   float* __restrict__ eas, const long long count, const AdamK a, const int zero_grad) {
  const long long nvec = count >> 2;
  const long long base = ((long long)blockIdx.x * blockDim.x) * 2 + threadIdx.x;
  float4 p[2], g[2], m[2], v[2];
  bool on[2];
#pragma unroll
  for (int u = 0; u < 2; ++u) {
    const long long j = base + (long long)u * blockDim.x;
    on[u] = j < nvec;
    if (on[u]) {
      g[u] = __ldcs(reinterpret_cast<const float4*>(grad) + j);
      p[u] = __ldcs(reinterpret_cast<const float4*>(param) + j);
      m[u] = __ldcs(reinterpret_cast<const float4*>(ea) + j);
      v[u] = __ldcs(reinterpret_cast<const float4*>(eas) + j);
    }
  }
#pragma unroll
  for (int u = 0; u < 2; ++u) {
    if (!on[u]) continue;
    const long long j = base + (long long)u * blockDim.x;
    adam_one(p[u].x, g[u].x, m[u].x, v[u].x, a); adam_one(p[u].y, g[u].y, m[u].y, v[u].y, a);
    adam_one(p[u].z, g[u].z, m[u].z, v[u].z, a); adam_one(p[u].w, g[u].w, m[u].w, v[u].w, a);
    __stcs(reinterpret_cast<float4*>(param) + j, p[u]);
    __stcs(reinterpret_cast<float4*>(ea) + j, m[u]);
    __stcs(reinterpret_cast<float4*>(eas) + j, v[u]);
    if (zero_grad) __stcs(reinterpret_cast<float4*>(grad) + j, make_float4(0.f, 0.f, 0.f, 0.f));
  }
  // ragged tail (count % 4 elements): first threads of the first block
  if (blockIdx.x == 0 && threadIdx.x < (int)(count & 3)) {
    const long long j = (nvec << 2) + threadIdx.x;
    float pp = param[j], mm = ea[j], vv = eas[j];
    adam_one(pp, grad[j], mm, vv, a);
    param[j] = pp; ea[j] = mm; eas[j] = vv;
    if (zero_grad) grad[j] = 0.f;
  }
}

// ---- compact model decode ------------------------------------------------------------------------------------------
__device__ __forceinline__ float4 rvq4(const uint8_t* __restrict__ idx, const float* __restrict__ cb, const int stages,
                                       const int entries, const long long i) {
  float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
  for (int s = 0; s < stages; ++s) {
    const int e = idx[i * stages + s];
    const float4 c = __ldg(reinterpret_cast<const float4*>(cb) + (size_t)s * entries + e);
    acc.x += c.x; acc.y += c.y; acc.z += c.z; acc.w += c.w;
  }
  return acc;
}

// geometry + opacity: one thread per primitive, 27 B in, 68 B out; the three small codebooks stay in L1
__global__ void __launch_bounds__(256) decode_geom_kernel(const fdgs_compact_scene c, float4* __restrict__ mean, float4* __restrict__ ls,
                                                          float4* __restrict__ ql, float4* __restrict__ qr, float* __restrict__ logit) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= c.N) return;
  const uint2 h = __ldg(reinterpret_cast<const uint2*>(c.mean_f16) + i);
  const __half2 h01 = *reinterpret_cast<const __half2*>(&h.x), h23 = *reinterpret_cast<const __half2*>(&h.y);
  const float2 f01 = __half22float2(h01), f23 = __half22float2(h23);
  mean[i] = make_float4(f01.x, f01.y, f23.x, f23.y);
  ls[i] = rvq4(c.scale_idx, c.scale_cb, c.scale_stages, c.scale_entries, i);
  ql[i] = rvq4(c.rot_l_idx, c.rot_cb, c.rot_stages, c.rot_entries, i);
  qr[i] = rvq4(c.rot_r_idx, c.rot_cb, c.rot_stages, c.rot_entries, i);
  const float step = (c.opacity_hi - c.opacity_lo) / (float)((1 << c.opacity_bits) - 1);
  logit[i] = fmaf((float)c.opacity_code[i], step, c.opacity_lo);
}

// colour: one warp per primitive; lane e, e+32, ... owns element e of the 3K-float row: e < 3 from the base-colour
// codebooks, the others from the rest codebooks (rows of (K-1)*3 floats, read coalesced from L2)
__global__ void __launch_bounds__(256) decode_colour_kernel(const fdgs_compact_scene c, float* __restrict__ sh, const int K) {
  const long long i = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (i >= c.N) return;                                             // whole warps leave together
  const int lane = threadIdx.x & 31;
  const int row = 3 * K, rest_row = row - 3;
  float* dst = sh + (size_t)i * row;
  // lane s holds the row offset of stage s (stages <= 16): the index bytes are read once, the gathers of all stages of
  // an element are independent loads in flight together
  unsigned int off_dc = 0, off_rest = 0;
  if (lane < c.dc_stages) off_dc = ((unsigned)lane * c.dc_entries + c.dc_idx[i * c.dc_stages + lane]) * 3u;
  if (K > 1 && lane < c.rest_stages) off_rest = ((unsigned)lane * c.rest_entries + c.rest_idx[i * c.rest_stages + lane]) * (unsigned)rest_row;
  for (int e0 = 0; e0 < row; e0 += 32) {
    const int e = e0 + lane;
    const bool live = e < row;
    float acc = 0.f;
    if (e0 == 0) {                                                  // lanes 0..2: base colour, lanes 3..31: first rest elements
#pragma unroll 4
      for (int s = 0; s < c.dc_stages; ++s) {
        const unsigned int o = __shfl_sync(0xffffffffu, off_dc, s);
        if (e < 3) acc += __ldg(c.dc_cb + o + e);
      }
    }
#pragma unroll 8
    for (int s = 0; s < c.rest_stages; ++s) {
      const unsigned int o = __shfl_sync(0xffffffffu, off_rest, s);
      if (live && e >= 3) acc += __ldg(c.rest_cb + o + (e - 3));
    }
    if (live) dst[e] = acc;
  }
}

}  // namespace fdgs

using namespace fdgs;

extern "C" {

int fdgs_mask_apply(const float* mask_logit, float mask_eps, const float* opacity_logit, float* out, int32_t N, void* stream) {
  if (N < 0 || (N > 0 && (!mask_logit || !opacity_logit || !out))) return FDGS_ERR_INVALID;
  if (N == 0) return FDGS_OK;
  mask_apply_kernel<<<(N + 255) / 256, 256, 0, (cudaStream_t)stream>>>(mask_logit, mask_eps, opacity_logit, out, N);
  count_launch();
  TRAIN_CUDA(cudaGetLastError(), "mask apply launch");
  return FDGS_OK;
}

int fdgs_regularizers(const fdgs_scene* sc, const float* mask_logit, const fdgs_reg_config* rc, const fdgs_grads* g,
                      float* grad_mask_logit, float* losses_dev, void* stream) {
  if (!sc || !rc || !g || sc->N < 0) return FDGS_ERR_INVALID;
  if (sc->N == 0) return FDGS_OK;
  if (!sc->log_scale || !sc->quat_l || !sc->quat_r || !g->log_scale || !g->quat_l || !g->quat_r) return FDGS_ERR_INVALID;
  if (!al16(sc->log_scale) || !al16(sc->quat_l) || !al16(sc->quat_r) || !al16(g->log_scale) || !al16(g->quat_l) || !al16(g->quat_r))
    return FDGS_ERR_INVALID;
  if (mask_logit && (!grad_mask_logit || !sc->opacity_logit || !g->opacity_logit)) return FDGS_ERR_INVALID;
  regularizers_kernel<<<(sc->N + 255) / 256, 256, 0, (cudaStream_t)stream>>>(*sc, mask_logit, *rc, *g, grad_mask_logit, losses_dev);
  count_launch();
  TRAIN_CUDA(cudaGetLastError(), "regularizers launch");
  return FDGS_OK;
}

int fdgs_adam_step(float* param, float* grad, float* exp_avg, float* exp_avg_sq, int64_t count, const fdgs_adam_config* c,
                   int32_t zero_grad, void* stream) {
  if (!c || count < 0 || c->step < 1 || !(c->beta1 >= 0.f && c->beta1 < 1.f) || !(c->beta2 >= 0.f && c->beta2 < 1.f)) return FDGS_ERR_INVALID;
  if (count == 0) return FDGS_OK;
  if (!param || !grad || !exp_avg || !exp_avg_sq) return FDGS_ERR_INVALID;
  if (!al16(param) || !al16(grad) || !al16(exp_avg) || !al16(exp_avg_sq)) return FDGS_ERR_INVALID;
  const double bc1 = 1.0 - pow((double)c->beta1, (double)c->step), bc2 = 1.0 - pow((double)c->beta2, (double)c->step);
  AdamK a;
  a.b1 = c->beta1; a.b2 = c->beta2; a.omb1 = (float)(1.0 - (double)c->beta1); a.omb2 = (float)(1.0 - (double)c->beta2);
  a.step_size = (float)((double)c->lr / bc1); a.inv_sqrt_bc2 = (float)(1.0 / sqrt(bc2)); a.eps = c->eps;
  const long long nvec = count >> 2;
  const long long blocks = nvec > 0 ? (nvec + 511) / 512 : 1;
  adam_kernel<<<(unsigned)blocks, 256, 0, (cudaStream_t)stream>>>(param, grad, exp_avg, exp_avg_sq, count, a, zero_grad);
  count_launch();
  TRAIN_CUDA(cudaGetLastError(), "adam launch");
  return FDGS_OK;
}

int fdgs_decode_compact(const fdgs_compact_scene* c, const fdgs_scene* out, void* stream) {
  if (!c || !out || c->N < 0 || c->N != out->N || c->sh_degree != out->sh_degree || c->n_time != out->n_time) return FDGS_ERR_INVALID;
  if (c->sh_degree < 0 || c->sh_degree > 3 || c->n_time < 1 || c->n_time > 8) return FDGS_ERR_INVALID;
  if (c->N == 0) return FDGS_OK;
  const int K = c->n_time * (c->sh_degree + 1) * (c->sh_degree + 1);
  auto bad = [](int stages, int entries) { return stages < 1 || stages > 16 || entries < 1 || entries > 256; };
  if (bad(c->scale_stages, c->scale_entries) || bad(c->rot_stages, c->rot_entries) || bad(c->dc_stages, c->dc_entries)) return FDGS_ERR_INVALID;
  if (K > 1 && (bad(c->rest_stages, c->rest_entries) || !c->rest_idx || !c->rest_cb)) return FDGS_ERR_INVALID;
  if (c->opacity_bits < 1 || c->opacity_bits > 8) return FDGS_ERR_INVALID;
  if (!c->mean_f16 || !c->opacity_code || !c->scale_idx || !c->scale_cb || !c->rot_l_idx || !c->rot_r_idx || !c->rot_cb || !c->dc_idx || !c->dc_cb)
    return FDGS_ERR_INVALID;
  if (!out->mean || !out->log_scale || !out->quat_l || !out->quat_r || !out->opacity_logit || !out->sh) return FDGS_ERR_INVALID;
  if (!al16(out->mean) || !al16(out->log_scale) || !al16(out->quat_l) || !al16(out->quat_r) || !al16(c->scale_cb) || !al16(c->rot_cb) ||
      (reinterpret_cast<uintptr_t>(c->mean_f16) & 7u))
    return FDGS_ERR_INVALID;
  cudaStream_t st = (cudaStream_t)stream;
  decode_geom_kernel<<<(c->N + 255) / 256, 256, 0, st>>>(*c, (float4*)out->mean, (float4*)out->log_scale, (float4*)out->quat_l,
                                                        (float4*)out->quat_r, (float*)out->opacity_logit);
  count_launch();
  const long long threads = (long long)c->N * 32;
  decode_colour_kernel<<<(unsigned)((threads + 255) / 256), 256, 0, st>>>(*c, (float*)out->sh, K);
  count_launch();
  TRAIN_CUDA(cudaGetLastError(), "decode launch");
  return FDGS_OK;
}

}  // extern "C"
