// features.cu — feature channels through the blend kernels ("rendered following the
// same process as in Section 3.2, with the color c replaced by the ... feature vector") and the per-splat optical flow
// of L410 (projected displacement of mu_xyz|t between two frames, then rendered with eq. 6 as a 2-channel feature).
//
// The C-channel blend kernels themselves live in blend.cu (blend_feat_fwd_kernel, blend_feat_bwd_kernel for frozen
// geometry, blend_feat_bwd_geom_kernel with geometry gradients: alpha is evaluated once per 32 channels in all three);
// this file holds the per-splat flow.
#include "common.cuh"
#include "geom.cuh"

namespace fdgs {

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

void launch_splat_flow(const fdgs_scene& sc, const ViewParams& vp, const CfgParams& cp, const Workspace& ws, float dt_next, float* flow,
                       cudaStream_t st) {
  splat_flow_kernel<<<(sc.N + 127) / 128, 128, 0, st>>>(sc, vp, cp, dt_next, ws.tiles_touched, reinterpret_cast<float2*>(flow));
  count_launch();
}

}  // namespace fdgs
