// features.cu — feature channels through the blend kernels ("rendered following the
// same process as in Section 3.2, with the color c replaced by the ... feature vector") and the per-splat optical flow
// of L410 (projected displacement of mu_xyz|t between two frames, then rendered with eq. 6 as a 2-channel feature).
//
// Design of this first version: the C channels go through the existing 3-channel blend kernels three at a time, over
// the SAME sorted tile lists; per pass a copy of the splat records carries the three feature values in the colour
// slots.  alpha is re-evaluated per pass (cost ~ C/3 blend launches); a dedicated C-channel kernel that evaluates
// alpha once is the next step.
#include "common.cuh"
#include "geom.cuh"

namespace fdgs {

// records of the visible primitives with (r, g, b) <- feat[i, c0 .. c0+2] (zero beyond C)
__global__ void __launch_bounds__(256) feature_records_kernel(const SplatRec* __restrict__ src, const unsigned int* __restrict__ tiles_touched,
                                                              const float* __restrict__ feat, const int C, const int c0, const int N,
                                                              SplatRec* __restrict__ dst) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N || tiles_touched[i] == 0) return;
  SplatRec r = src[i];
  const float* f = feat + (size_t)i * C + c0;
  r.r = f[0];
  r.g = c0 + 1 < C ? f[1] : 0.f;
  r.b = c0 + 2 < C ? f[2] : 0.f;
  dst[i] = r;
}

// dL/df of one pass sits in the colour slots of g9: move it to grad_feat (+=) and clear the slots for the next pass
__global__ void __launch_bounds__(256) extract_feature_grads_kernel(float* __restrict__ g9, const unsigned int* __restrict__ tiles_touched,
                                                                    float* __restrict__ grad_feat, const int C, const int c0, const int N) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N || tiles_touched[i] == 0) return;
  float* g = g9 + (size_t)9 * i + 6;
  float* d = grad_feat + (size_t)i * C + c0;
#pragma unroll
  for (int j = 0; j < 3; ++j) {
    if (c0 + j < C) d[j] += g[j];
    g[j] = 0.f;
  }
}

// flow[i] = pi(mu_c(t + d)) - pi(mu_c(t)) with mu_c(t + d) = mu_c(t) + Sigma_1:3,4 / Sigma_44 d (eq. 9 is linear in t).
// Evaluated without the cancellation of two pixel coordinates: u' - u = fx (dx z - x dz) / (z z'), (dx, dy, dz) = W vel d.
__global__ void __launch_bounds__(128) splat_flow_kernel(const fdgs_scene sc, const ViewParams vp, const CfgParams cp, const float dt_next,
                                                         const unsigned int* __restrict__ tiles_touched, float2* __restrict__ flow) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= sc.N) return;
  float2 out = make_float2(0.f, 0.f);
  if (tiles_touched[i] != 0) {
    Geom g;
    const float4 mean = __ldg(reinterpret_cast<const float4*>(sc.mean) + i), ls = __ldg(reinterpret_cast<const float4*>(sc.log_scale) + i);
    const float4 ql = __ldg(reinterpret_cast<const float4*>(sc.quat_l) + i), qr = __ldg(reinterpret_cast<const float4*>(sc.quat_r) + i);
    if (geom_forward(mean, ls, ql, qr, sc.opacity_logit[i], vp, cp, g) == G_VISIBLE) {
      const float k = dt_next / g.b;
      const float vel[3] = {g.c[0] * k, g.c[1] * k, g.c[2] * k};                 // 3D displacement of the conditional mean
      float d[3];
#pragma unroll
      for (int r = 0; r < 3; ++r) d[r] = fmaf(vp.W[r][0], vel[0], fmaf(vp.W[r][1], vel[1], vp.W[r][2] * vel[2]));
      const float z = g.p[2], z2 = z + d[2];
      if (z2 > 0.f) {
        const float inv = 1.0f / (z * z2);
        out.x = vp.fx * (d[0] * z - g.p[0] * d[2]) * inv;
        out.y = vp.fy * (d[1] * z - g.p[1] * d[2]) * inv;
      }
    }
  }
  flow[i] = out;
}

void launch_feature_records(const Workspace& ws, const float* feat, int C, int c0, int N, SplatRec* dst, cudaStream_t st) {
  feature_records_kernel<<<(N + 255) / 256, 256, 0, st>>>(ws.rec, ws.tiles_touched, feat, C, c0, N, dst);
  count_launch();
}
void launch_extract_feature_grads(const Workspace& ws, float* grad_feat, int C, int c0, int N, cudaStream_t st) {
  extract_feature_grads_kernel<<<(N + 255) / 256, 256, 0, st>>>(ws.g9, ws.tiles_touched, grad_feat, C, c0, N);
  count_launch();
}
void launch_splat_flow(const fdgs_scene& sc, const ViewParams& vp, const CfgParams& cp, const Workspace& ws, float dt_next, float* flow,
                       cudaStream_t st) {
  splat_flow_kernel<<<(sc.N + 127) / 128, 128, 0, st>>>(sc, vp, cp, dt_next, ws.tiles_touched, reinterpret_cast<float2*>(flow));
  count_launch();
}

}  // namespace fdgs
