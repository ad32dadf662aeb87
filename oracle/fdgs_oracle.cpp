// fdgs_oracle.cpp — float64 CPU ORACLE for the time-sliced tile rasterizer of native 4D Gaussians.
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
// bench.py's cpu_baseline / --impl reference leg may build, load or call it.  It shares no code,
// header, table or constant generator with the CUDA path (paper_2412_20720_b200/csrc).
//
// Everything is written out step by step in the paper's order and notation, in double precision,
// with no blocking, fusion or reordering beyond what the definition states.  Citations are
// PAPER.md:L<line> (+ equation) of arxiv 2412.20720; "DESIGN §R" are the readings listed in
// DESIGN.md where the paper is silent or garbled.
//
// Pins (tests/test_oracle_pins.py, `-m "not gpu"`): eq. 8 against the Hamilton product, eq. 7 by
// its eigenvalues, eq. 9-10 by brute-force factorisation with a library inverse, eq. 15, the
// SH table against scipy's spherical harmonics and quadrature, EWA against a numerical
// Jacobian, tile lists against brute force, the blend loop against closed forms and a direct
// evaluation of eq. 6, the backward against central finite differences.
// Parity unpinned by the paper (conventions only, DESIGN §R S5/S8-S16): SH sign convention,
// 0.5 colour offset, alpha/transmittance thresholds, 3-sigma support, dilation, near plane.
//
// Build: g++ -O2 -fopenmp -shared -fPIC -std=c++17 fdgs_oracle.cpp -o libfdgs_oracle.so
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

constexpr int TILE = 16;  // 16x16-pixel tiles (BASELINE.json north_star; tile rasterizer of [23])
constexpr double PI = 3.14159265358979323846264338327950288;

struct Cfg {               // thresholds: data shared with the GPU side only as numbers (DESIGN §R S8)
  double marginal_min;     // 0.05, "Gaussian filter with marginal p(t) < 0.05"
  double alpha_min;        // 1/255   (paper silent; settings of [23], L324)
  double alpha_max;        // 0.99
  double transmittance_min;// 1e-4
  double dilation;         // 0.3 px^2 low-pass added to the 2D covariance
  double cutoff_sigma;     // 3.0
  double znear;            // 0.2
  double guard;            // 1.3  guard band for the clamped ratio inside J
  int full_support;        // 1 = "pure eq. 6" helper: every primitive is listed in every tile
};

struct View {
  double Wm[3][3], tau[3];   // E = [W | tau], world -> camera
  double fx, fy, cx, cy;     // K
  int width, height;
  double t, period_T;        // query time t, 4DSH period T (eq. 20)
  double bg[3];
};

// status codes of a primitive after preprocess
enum { VISIBLE = 0, CULL_TIME = 1, CULL_NEAR = 2, CULL_RECT = 3, CULL_NONFINITE = 4 };

struct Prim {  // everything the per-primitive chain produces (kept for parity checks and backward)
  int status = CULL_NONFINITE;
  double s[4], ql[4], qr[4], nl, nr;   // activations: s = exp(log s); unit quaternions and the norms
  double Lm[4][4], Rm[4][4], R4[4][4], M[4][4], Sig[4][4];
  double dt, b, w;                     // Delta = t - mu_t, b = Sigma_44, marginal weight w (eq. 10)
  double a[3], mu_c[3], Sig_c[3][3];   // eq. 9
  double p[3];                         // camera-space mean
  double u, v;                         // eq. 3
  int clampx, clampy; double xr, yr;   // guard-band clamp state and the (clamped) ratios x'/z, y'/z
  double J[2][3], T[2][3], S2[2][2];   // Jacobian, T = J W, Sigma_2d (eq. 4 + dilation)
  double A, B, C;                      // conic = Sigma_2d^{-1}
  double radius;
  int rect[4];                         // tx0, ty0, tx1, ty1 (half-open)
  double dir[3], rho;                  // view direction (camera centre -> mu_c), distance
  double raw[3], rgb[3];               // colour before / after the clamp at 0
  double sig, o;                       // sigmoid(logit), o = sigmoid * w
  float depth32;                       // sort key: fp32 rounding of p_z (DESIGN §R S12)
  double frag;                         // fragility: smallest relative margin to any discrete decision
};

struct Oracle {
  int N = 0, L = 0, n_time = 1, K = 1, Kd = 1;
  std::vector<double> mean, log_scale, quat_l, quat_r, logit, sh;
  View view; Cfg cfg;
  int tiles_x = 0, tiles_y = 0;
  std::vector<Prim> prims;
  std::vector<int64_t> tile_off;   // [tiles+1]
  std::vector<int32_t> tile_ids;   // [D] primitive ids, per tile sorted by (depth32 bits, id)
  // forward products
  std::vector<double> image, final_T, margin;
  std::vector<double> depth_map;   // auxiliary channel: rendered depth sum_k z_k alpha_k T_k (eq. 29, DESIGN S18)
  std::vector<int32_t> n_contrib;
  // per-splat gradients from the blend backward: g_u,g_v,g_A,g_B,g_C,g_o,g_r,g_g,g_b
  std::vector<double> g9;
  std::vector<double> gz;          // per-splat dL/d(camera depth z_k) from the auxiliary depth channel
  bool colour_override = false;    // feature channels: P.rgb holds free per-splat values, not eq. 20
};

// ---------------------------------------------------------------------------------------------
// eq. 8 (de-garbled sign pattern, DESIGN §R G1): the left- and
// right-isoclinic 4x4 matrices of q_l = (a,b,c,d) and q_r = (p,q,r,s).
void left_matrix(const double q[4], double Lm[4][4]) {
  const double a = q[0], b = q[1], c = q[2], d = q[3];
  const double m[4][4] = {{a, -b, -c, -d}, {b, a, -d, c}, {c, d, a, -b}, {d, -c, b, a}};
  std::memcpy(Lm, m, sizeof(m));
}
void right_matrix(const double q[4], double Rm[4][4]) {
  const double p = q[0], qq = q[1], r = q[2], s = q[3];
  const double m[4][4] = {{p, -qq, -r, -s}, {qq, p, s, -r}, {r, -s, p, qq}, {s, r, -qq, p}};
  std::memcpy(Rm, m, sizeof(m));
}
void matmul4(const double X[4][4], const double Y[4][4], double Z[4][4]) {
  for (int i = 0; i < 4; ++i)
    for (int j = 0; j < 4; ++j) {
      double acc = 0;
      for (int k = 0; k < 4; ++k) acc += X[i][k] * Y[k][j];
      Z[i][j] = acc;
    }
}

// Real orthonormal spherical harmonics up to degree 3 on a unit vector (x,y,z), index l*l+l+m.
// "Y_l^m is the 3D spherical harmonics"; sign convention = Condon-Shortley phase
// kept in the real combinations (DESIGN §R S5), constants from the closed forms.
// If grad != nullptr also returns the gradient of the polynomial extension wrt (x,y,z).
void sh_basis(int L, const double d[3], double* Y, double (*grad)[3]) {
  const double x = d[0], y = d[1], z = d[2];
  const double c0 = 0.5 * std::sqrt(1.0 / PI);
  Y[0] = c0;
  if (grad) { grad[0][0] = grad[0][1] = grad[0][2] = 0; }
  if (L < 1) return;
  const double c1 = std::sqrt(3.0 / (4.0 * PI));
  Y[1] = -c1 * y; Y[2] = c1 * z; Y[3] = -c1 * x;
  if (grad) {
    grad[1][0] = 0;   grad[1][1] = -c1; grad[1][2] = 0;
    grad[2][0] = 0;   grad[2][1] = 0;   grad[2][2] = c1;
    grad[3][0] = -c1; grad[3][1] = 0;   grad[3][2] = 0;
  }
  if (L < 2) return;
  const double c2 = 0.5 * std::sqrt(15.0 / PI), c20 = 0.25 * std::sqrt(5.0 / PI);
  Y[4] = c2 * x * y;
  Y[5] = -c2 * y * z;
  Y[6] = c20 * (2 * z * z - x * x - y * y);
  Y[7] = -c2 * x * z;
  Y[8] = 0.5 * c2 * (x * x - y * y);
  if (grad) {
    grad[4][0] = c2 * y;        grad[4][1] = c2 * x;         grad[4][2] = 0;
    grad[5][0] = 0;             grad[5][1] = -c2 * z;        grad[5][2] = -c2 * y;
    grad[6][0] = -2 * c20 * x;  grad[6][1] = -2 * c20 * y;   grad[6][2] = 4 * c20 * z;
    grad[7][0] = -c2 * z;       grad[7][1] = 0;              grad[7][2] = -c2 * x;
    grad[8][0] = c2 * x;        grad[8][1] = -c2 * y;        grad[8][2] = 0;
  }
  if (L < 3) return;
  const double c3 = 0.25 * std::sqrt(35.0 / (2.0 * PI)), c4 = 0.5 * std::sqrt(105.0 / PI);
  const double c5 = 0.25 * std::sqrt(21.0 / (2.0 * PI)), c6 = 0.25 * std::sqrt(7.0 / PI);
  const double xx = x * x, yy = y * y, zz = z * z;
  Y[9]  = -c3 * y * (3 * xx - yy);
  Y[10] = c4 * x * y * z;
  Y[11] = -c5 * y * (4 * zz - xx - yy);
  Y[12] = c6 * z * (2 * zz - 3 * xx - 3 * yy);
  Y[13] = -c5 * x * (4 * zz - xx - yy);
  Y[14] = 0.5 * c4 * z * (xx - yy);
  Y[15] = -c3 * x * (xx - 3 * yy);
  if (grad) {
    grad[9][0]  = -c3 * 6 * x * y;            grad[9][1]  = -c3 * (3 * xx - 3 * yy);       grad[9][2]  = 0;
    grad[10][0] = c4 * y * z;                 grad[10][1] = c4 * x * z;                    grad[10][2] = c4 * x * y;
    grad[11][0] = c5 * 2 * x * y;             grad[11][1] = -c5 * (4 * zz - xx - 3 * yy);  grad[11][2] = -c5 * 8 * y * z;
    grad[12][0] = -c6 * 6 * x * z;            grad[12][1] = -c6 * 6 * y * z;               grad[12][2] = c6 * (6 * zz - 3 * xx - 3 * yy);
    grad[13][0] = -c5 * (4 * zz - 3 * xx - yy); grad[13][1] = c5 * 2 * x * y;              grad[13][2] = -c5 * 8 * x * z;
    grad[14][0] = c4 * x * z;                 grad[14][1] = -c4 * y * z;                   grad[14][2] = 0.5 * c4 * (xx - yy);
    grad[15][0] = -c3 * (3 * xx - 3 * yy);    grad[15][1] = c3 * 6 * x * y;                grad[15][2] = 0;
  }
}

inline double rel_margin(double value, double threshold) {
  return std::fabs(value - threshold) / std::max(std::fabs(threshold), 1e-300);
}

// ---------------------------------------------------------------------------------------------
// Per-primitive chain, steps 1-9 of DESIGN.md "what the path computes".
void preprocess_one(const Oracle& O, int i, Prim& P) {
  const Cfg& c = O.cfg; const View& V = O.view;
  const double* mu = &O.mean[4 * i];
  P = Prim();
  P.frag = 1e300;
  // non-finite parameters or a zero quaternion: the primitive is culled (boundary contract)
  bool finite = std::isfinite(O.logit[i]);
  for (int k = 0; k < 4; ++k)
    finite = finite && std::isfinite(mu[k]) && std::isfinite(O.log_scale[4 * i + k]) &&
             std::isfinite(O.quat_l[4 * i + k]) && std::isfinite(O.quat_r[4 * i + k]);
  double nl = 0, nr = 0;
  for (int k = 0; k < 4; ++k) { nl += O.quat_l[4 * i + k] * O.quat_l[4 * i + k]; nr += O.quat_r[4 * i + k] * O.quat_r[4 * i + k]; }
  nl = std::sqrt(nl); nr = std::sqrt(nr);
  if (!finite || !(nl > 0) || !(nr > 0) || !std::isfinite(nl) || !std::isfinite(nr)) { P.status = CULL_NONFINITE; return; }
  // 1. activations (DESIGN §R S1): S = diag(s), s = exp(log s) (L128); unit quaternions
  P.nl = nl; P.nr = nr;
  for (int k = 0; k < 4; ++k) {
    P.s[k] = std::exp(O.log_scale[4 * i + k]);
    P.ql[k] = O.quat_l[4 * i + k] / nl;
    P.qr[k] = O.quat_r[4 * i + k] / nr;
  }
  // 2. R = L(q_l) R(q_r) (eq. 8), Sigma = R S S^T R^T (eq. 7); rows/cols ordered (x,y,z,t)
  left_matrix(P.ql, P.Lm); right_matrix(P.qr, P.Rm); matmul4(P.Lm, P.Rm, P.R4);
  for (int r = 0; r < 4; ++r) for (int k = 0; k < 4; ++k) P.M[r][k] = P.R4[r][k] * P.s[k];
  for (int r = 0; r < 4; ++r)
    for (int q = 0; q < 4; ++q) {
      double acc = 0;
      for (int k = 0; k < 4; ++k) acc += P.M[r][k] * P.M[q][k];
      P.Sig[r][q] = acc;
    }
  // 3. temporal marginal p(t) = N(t; mu_4, Sigma_44), unnormalised (eq. 10); filter p(t) < 0.05 (L324)
  P.dt = V.t - mu[3];
  P.b = P.Sig[3][3];
  P.w = std::exp(-0.5 * P.dt * P.dt / P.b);
  if (!std::isfinite(P.w) || !std::isfinite(P.b) || !(P.b > 0)) { P.status = CULL_NONFINITE; return; }
  if (c.marginal_min > 0) P.frag = std::min(P.frag, rel_margin(P.w, c.marginal_min));
  if (P.w < c.marginal_min) { P.status = CULL_TIME; return; }
  // 4. conditional 3D Gaussian (eq. 9), evaluated literally
  for (int r = 0; r < 3; ++r) {
    P.a[r] = P.Sig[r][3];
    P.mu_c[r] = mu[r] + P.a[r] * P.dt / P.b;
  }
  for (int r = 0; r < 3; ++r)
    for (int q = 0; q < 3; ++q) P.Sig_c[r][q] = P.Sig[r][q] - P.a[r] * P.a[q] / P.b;
  // 5. camera space and pinhole projection (eq. 3; DESIGN §R S11)
  for (int r = 0; r < 3; ++r)
    P.p[r] = V.Wm[r][0] * P.mu_c[0] + V.Wm[r][1] * P.mu_c[1] + V.Wm[r][2] * P.mu_c[2] + V.tau[r];
  const double x = P.p[0], y = P.p[1], z = P.p[2];
  P.depth32 = (float)z;
  if (!std::isfinite(z) || !std::isfinite(x) || !std::isfinite(y)) { P.status = CULL_NONFINITE; return; }
  P.frag = std::min(P.frag, rel_margin(z, c.znear));
  if (z <= c.znear) { P.status = CULL_NEAR; return; }
  P.u = V.fx * x / z + V.cx;
  P.v = V.fy * y / z + V.cy;
  // 6. J = Jacobian of the perspective projection at the (guard-band clamped) point (L104); eq. 4 + dilation
  const double limx = c.guard * V.width / (2.0 * V.fx), limy = c.guard * V.height / (2.0 * V.fy);
  P.xr = x / z; P.yr = y / z; P.clampx = 0; P.clampy = 0;
  if (P.xr > limx) { P.xr = limx; P.clampx = 1; } else if (P.xr < -limx) { P.xr = -limx; P.clampx = 1; }
  if (P.yr > limy) { P.yr = limy; P.clampy = 1; } else if (P.yr < -limy) { P.yr = -limy; P.clampy = 1; }
  const double xc = P.xr * z, yc = P.yr * z;
  P.J[0][0] = V.fx / z; P.J[0][1] = 0;        P.J[0][2] = -V.fx * xc / (z * z);
  P.J[1][0] = 0;        P.J[1][1] = V.fy / z; P.J[1][2] = -V.fy * yc / (z * z);
  for (int r = 0; r < 2; ++r)
    for (int q = 0; q < 3; ++q)
      P.T[r][q] = P.J[r][0] * V.Wm[0][q] + P.J[r][1] * V.Wm[1][q] + P.J[r][2] * V.Wm[2][q];
  for (int r = 0; r < 2; ++r)
    for (int q = 0; q < 2; ++q) {
      double acc = 0;
      for (int k = 0; k < 3; ++k)
        for (int l = 0; l < 3; ++l) acc += P.T[r][k] * P.Sig_c[k][l] * P.T[q][l];
      P.S2[r][q] = acc + (r == q ? c.dilation : 0.0);
    }
  const double a2 = P.S2[0][0], b2 = P.S2[0][1], c2 = P.S2[1][1];
  const double det = a2 * c2 - b2 * b2;
  if (!(det > 0) || !std::isfinite(det)) { P.status = CULL_NONFINITE; return; }
  P.A = c2 / det; P.B = -b2 / det; P.C = a2 / det;
  // 7. support: r = cutoff_sigma * sqrt(lambda_max), real valued; tile rectangle (DESIGN §R S9)
  const double lam = 0.5 * (a2 + c2) + std::sqrt(std::max(0.0, 0.25 * (a2 - c2) * (a2 - c2) + b2 * b2));
  P.radius = c.cutoff_sigma * std::sqrt(lam);
  if (c.full_support) {
    P.rect[0] = 0; P.rect[1] = 0; P.rect[2] = O.tiles_x; P.rect[3] = O.tiles_y;
  } else {
    const double ex[4] = {(P.u - P.radius) / TILE, (P.v - P.radius) / TILE, (P.u + P.radius) / TILE, (P.v + P.radius) / TILE};
    const double scale = std::max({std::fabs(P.u), std::fabs(P.v), P.radius, (double)TILE});
    for (int k = 0; k < 4; ++k) {   // distance (pixels) of the footprint edge to the nearest tile boundary
      const double dist = std::fabs(ex[k] - std::nearbyint(ex[k])) * TILE;
      P.frag = std::min(P.frag, dist / scale);
    }
    P.rect[0] = (int)std::min<double>(std::max<double>(std::floor(ex[0]), 0), O.tiles_x);
    P.rect[1] = (int)std::min<double>(std::max<double>(std::floor(ex[1]), 0), O.tiles_y);
    P.rect[2] = (int)std::min<double>(std::max<double>(std::ceil(ex[2]), 0), O.tiles_x);
    P.rect[3] = (int)std::min<double>(std::max<double>(std::ceil(ex[3]), 0), O.tiles_y);
  }
  if ((P.rect[2] - P.rect[0]) * (P.rect[3] - P.rect[1]) <= 0) { P.status = CULL_RECT; return; }
  // 8. colour: 4D spherindrical harmonics Z_nl^m = cos(2 pi n Delta / T) Y_l^m(dir) (eq. 20;
  //    argument Delta = t - mu_t per L183, DESIGN §R S2; direction to the conditional mean, S6)
  double ccam[3];
  for (int r = 0; r < 3; ++r) ccam[r] = -(V.Wm[0][r] * V.tau[0] + V.Wm[1][r] * V.tau[1] + V.Wm[2][r] * V.tau[2]);
  double dv[3] = {P.mu_c[0] - ccam[0], P.mu_c[1] - ccam[1], P.mu_c[2] - ccam[2]};
  P.rho = std::sqrt(dv[0] * dv[0] + dv[1] * dv[1] + dv[2] * dv[2]);
  for (int r = 0; r < 3; ++r) P.dir[r] = dv[r] / P.rho;
  double Y[16];
  sh_basis(O.L, P.dir, Y, nullptr);
  const double* coef = &O.sh[(size_t)i * O.K * 3];
  for (int ch = 0; ch < 3; ++ch) {
    double acc = 0.5;
    for (int n = 0; n < O.n_time; ++n) {
      const double cn = std::cos(2.0 * PI * n * P.dt / V.period_T);
      for (int k = 0; k < O.Kd; ++k) acc += coef[(n * O.Kd + k) * 3 + ch] * cn * Y[k];
    }
    P.raw[ch] = acc;
    P.rgb[ch] = std::max(0.0, acc);
  }
  // 9. opacity times marginal: alpha_i p_i(t) of eq. 6 (L118)
  P.sig = 1.0 / (1.0 + std::exp(-O.logit[i]));
  P.o = P.sig * P.w;
  P.status = VISIBLE;
}

void build_tile_lists(Oracle& O) {
  const int tiles = O.tiles_x * O.tiles_y;
  std::vector<std::vector<int32_t>> lists(tiles);
  for (int i = 0; i < O.N; ++i) {            // in id order, so each list starts sorted by id
    const Prim& P = O.prims[i];
    if (P.status != VISIBLE) continue;
    for (int ty = P.rect[1]; ty < P.rect[3]; ++ty)
      for (int tx = P.rect[0]; tx < P.rect[2]; ++tx) lists[ty * O.tiles_x + tx].push_back(i);
  }
  O.tile_off.assign(tiles + 1, 0);
#pragma omp parallel for schedule(dynamic, 8)
  for (int tl = 0; tl < tiles; ++tl) {
    // "sorted according to their depth" (L83): ascending fp32 depth bits, ties by primitive id (S12, S13)
    std::stable_sort(lists[tl].begin(), lists[tl].end(), [&](int32_t p, int32_t q) {
      uint32_t bp, bq;
      std::memcpy(&bp, &O.prims[p].depth32, 4); std::memcpy(&bq, &O.prims[q].depth32, 4);
      return bp < bq;
    });
  }
  for (int tl = 0; tl < tiles; ++tl) O.tile_off[tl + 1] = O.tile_off[tl] + (int64_t)lists[tl].size();
  O.tile_ids.resize(O.tile_off[tiles]);
  for (int tl = 0; tl < tiles; ++tl) std::copy(lists[tl].begin(), lists[tl].end(), O.tile_ids.begin() + O.tile_off[tl]);
}

// alpha of splat P at pixel centre (px,py): opacity x marginal x planar conditional Gaussian (eq. 6).
// Returns false if the splat is skipped (alpha < alpha_min).  power is clamped at 0 (S10).
inline bool eval_alpha(const Prim& P, const Cfg& c, double px, double py, double& alpha, double& G,
                       double& dx, double& dy, bool& pclamp, bool& aclamp) {
  dx = P.u - px; dy = P.v - py;
  double power = -0.5 * (P.A * dx * dx + P.C * dy * dy) - P.B * dx * dy;
  pclamp = power > 0;
  if (pclamp) power = 0;
  G = std::exp(power);
  alpha = P.o * G;
  aclamp = alpha > c.alpha_max;
  if (aclamp) alpha = c.alpha_max;
  return !(alpha < c.alpha_min);
}

void forward(Oracle& O) {
  const View& V = O.view; const Cfg& c = O.cfg;
  const int W = V.width, H = V.height;
  O.image.assign((size_t)3 * W * H, 0); O.final_T.assign((size_t)W * H, 1);
  O.margin.assign((size_t)W * H, 1e300); O.n_contrib.assign((size_t)W * H, 0);
  O.depth_map.assign((size_t)W * H, 0);
#pragma omp parallel for schedule(dynamic, 1)
  for (int tl = 0; tl < O.tiles_x * O.tiles_y; ++tl) {
    const int tx = tl % O.tiles_x, ty = tl / O.tiles_x;
    for (int py = ty * TILE; py < std::min(H, (ty + 1) * TILE); ++py)
      for (int px = tx * TILE; px < std::min(W, (tx + 1) * TILE); ++px) {
        double T = 1, C[3] = {0, 0, 0}, Dz = 0, marg = 1e300;
        int last = 0;
        for (int64_t k = O.tile_off[tl]; k < O.tile_off[tl + 1]; ++k) {   // front to back (eq. 6)
          const Prim& P = O.prims[O.tile_ids[k]];
          double alpha, G, dx, dy; bool pc, ac;
          const bool keep = eval_alpha(P, c, px + 0.5, py + 0.5, alpha, G, dx, dy, pc, ac);
          if (c.alpha_min > 0) marg = std::min(marg, rel_margin(P.o * G, c.alpha_min));
          if (!keep) continue;
          const double Tn = T * (1 - alpha);
          if (c.transmittance_min > 0) marg = std::min(marg, rel_margin(Tn, c.transmittance_min));
          if (Tn < c.transmittance_min) break;           // the terminating splat does not contribute (S14)
          for (int ch = 0; ch < 3; ++ch) C[ch] += P.rgb[ch] * alpha * T;
          Dz += P.p[2] * alpha * T;                        // depth is composited like a colour channel, no background
          T = Tn;
          last = (int)(k - O.tile_off[tl]) + 1;
        }
        const size_t pix = (size_t)py * W + px;
        for (int ch = 0; ch < 3; ++ch) O.image[(size_t)ch * W * H + pix] = C[ch] + T * V.bg[ch];
        O.final_T[pix] = T; O.n_contrib[pix] = last; O.margin[pix] = marg; O.depth_map[pix] = Dz;
      }
  }
}

inline void add(double& dst, double v) {
#pragma omp atomic
  dst += v;
}

// Reverse-order gradient of the blend (VJP of eq. 6 with the truncations of forward()).
// For contributors k = 1..m, T_k = prod_{j<k}(1-alpha_j), out = sum c_k alpha_k T_k + T_{m+1} bg:
//   dL/dc_k = alpha_k T_k g;   dL/dalpha_k = g . (T_k c_k - S_k / (1 - alpha_k)),  S_k = everything behind k.
// Auxiliary channels (eq. 25, L256 eq. 29): depth D = sum_k z_k alpha_k T_k and accumulated opacity
// O_gs = sum_k alpha_k T_k = 1 - T_{m+1}.  With upstream gD = dL/dD and gO = dL/dO_gs (either may be NULL):
//   dL/dz_k += gD alpha_k T_k;   dL/dalpha_k += gD (T_k z_k - Sz_k / (1 - alpha_k)) + gO T_{m+1} / (1 - alpha_k),
// Sz_k = depth accumulated behind k (no background term).
void backward_blend(Oracle& O, const double* dL_dimage, const double* dL_ddepth = nullptr, const double* dL_dopacity = nullptr) {
  const View& V = O.view; const Cfg& c = O.cfg;
  const int W = V.width, H = V.height;
  O.g9.assign((size_t)O.N * 9, 0);
  O.gz.assign((size_t)O.N, 0);
  const int tiles = O.tiles_x * O.tiles_y;
  std::vector<double>& acc = O.g9;
#pragma omp parallel
  {
#pragma omp for schedule(dynamic, 1)
    for (int tl = 0; tl < tiles; ++tl) {
      const int tx = tl % O.tiles_x, ty = tl / O.tiles_x;
      for (int py = ty * TILE; py < std::min(H, (ty + 1) * TILE); ++py)
        for (int px = tx * TILE; px < std::min(W, (tx + 1) * TILE); ++px) {
          const size_t pix = (size_t)py * W + px;
          const double g[3] = {dL_dimage[pix], dL_dimage[(size_t)W * H + pix], dL_dimage[(size_t)2 * W * H + pix]};
          double T = O.final_T[pix];
          const double T_final = T, gD = dL_ddepth ? dL_ddepth[pix] : 0.0, gO = dL_dopacity ? dL_dopacity[pix] : 0.0;
          double Sz = 0;
          double S[3] = {T * V.bg[0], T * V.bg[1], T * V.bg[2]};   // S_m = T_{m+1} bg
          for (int64_t k = O.tile_off[tl] + O.n_contrib[pix] - 1; k >= O.tile_off[tl]; --k) {
            const int id = O.tile_ids[k];
            const Prim& P = O.prims[id];
            double alpha, G, dx, dy; bool pc, ac;
            if (!eval_alpha(P, c, px + 0.5, py + 0.5, alpha, G, dx, dy, pc, ac)) continue;
            T = T / (1 - alpha);                                      // T_k
            double* a9 = &acc[(size_t)id * 9];
            double dalpha = 0;
            for (int ch = 0; ch < 3; ++ch) {
              add(a9[6 + ch], alpha * T * g[ch]);
              dalpha += g[ch] * (T * P.rgb[ch] - S[ch] / (1 - alpha));
              S[ch] += P.rgb[ch] * alpha * T;                         // S_{k-1}
            }
            add(O.gz[id], gD * alpha * T);
            dalpha += gD * (T * P.p[2] - Sz / (1 - alpha)) + gO * T_final / (1 - alpha);
            Sz += P.p[2] * alpha * T;
            if (ac) continue;                                         // alpha clamped at alpha_max: zero slope (S16)
            add(a9[5], G * dalpha);                                     // d alpha / d o = G
            if (pc) continue;                                         // power clamped at 0: zero slope (S10)
            const double dpow = P.o * G * dalpha;
            add(a9[0], dpow * -(P.A * dx + P.B * dy));                  // d power / d u  (dx = u - px)
            add(a9[1], dpow * -(P.C * dy + P.B * dx));
            add(a9[2], dpow * -0.5 * dx * dx);
            add(a9[3], dpow * -dx * dy);
            add(a9[4], dpow * -0.5 * dy * dy);
          }
        }
    }
  }
}

// VJP of preprocess_one for a visible primitive (chain of Appendix D of SURVEY.md re-derived in DESIGN.md;
// finite differences in tests/ are the authority).  Accumulates (+=) into the gradient arrays.
void backward_one(const Oracle& O, int i, const double g9[9], double* d_mean, double* d_ls, double* d_ql,
                  double* d_qr, double* d_logit, double* d_sh, double* d_mean2d, const double g_z = 0.0,
                  double* densify3 = nullptr) {
  const Prim& P = O.prims[i]; const View& V = O.view; const Cfg& c = O.cfg;
  if (P.status != VISIBLE) return;
  const double g_u = g9[0], g_v = g9[1], g_A = g9[2], g_B = g9[3], g_C = g9[4], g_o = g9[5];
  if (d_mean2d) { d_mean2d[2 * i] += g_u; d_mean2d[2 * i + 1] += g_v; }
  double d_muc[3] = {0, 0, 0}, d_dt = 0, d_b = 0;
  // (A4) colour — skipped when the composited channels are free per-splat features (their gradient is g9[6..8] itself)
  if (!O.colour_override) {
    double Y[16], dY[16][3];
    sh_basis(O.L, P.dir, Y, dY);
    const double* coef = &O.sh[(size_t)i * O.K * 3];
    double ddir[3] = {0, 0, 0};
    for (int ch = 0; ch < 3; ++ch) {
      if (!(P.raw[ch] > 0)) continue;            // clamp at 0 active: zero slope
      const double gc = g9[6 + ch];
      for (int n = 0; n < O.n_time; ++n) {
        const double om = 2.0 * PI * n / V.period_T;
        const double cn = std::cos(om * P.dt), sn = std::sin(om * P.dt);
        for (int k = 0; k < O.Kd; ++k) {
          const double cf = coef[(n * O.Kd + k) * 3 + ch];
          d_sh[((size_t)i * O.K + n * O.Kd + k) * 3 + ch] += gc * cn * Y[k];
          d_dt += gc * cf * (-om * sn) * Y[k];
          for (int r = 0; r < 3; ++r) ddir[r] += gc * cf * cn * dY[k][r];
        }
      }
    }
    const double dd = ddir[0] * P.dir[0] + ddir[1] * P.dir[1] + ddir[2] * P.dir[2];
    for (int r = 0; r < 3; ++r) d_muc[r] += (ddir[r] - P.dir[r] * dd) / P.rho;   // through the normalisation
  }
  // conic = Sigma_2d^{-1}:  G2 = -Q G_Q Q with G_Q = [[g_A, g_B/2],[g_B/2, g_C]]
  const double Q[2][2] = {{P.A, P.B}, {P.B, P.C}};
  const double GQ[2][2] = {{g_A, 0.5 * g_B}, {0.5 * g_B, g_C}};
  double QG[2][2], G2[2][2];
  for (int r = 0; r < 2; ++r) for (int q = 0; q < 2; ++q) QG[r][q] = Q[r][0] * GQ[0][q] + Q[r][1] * GQ[1][q];
  for (int r = 0; r < 2; ++r) for (int q = 0; q < 2; ++q) G2[r][q] = -(QG[r][0] * Q[0][q] + QG[r][1] * Q[1][q]);
  // Sigma_2d = T Sigma_c T^T + dilation I:  G_c = T^T G2 T,  dT = 2 G2 T Sigma_c
  double Gc[3][3], G2T[2][3], dT[2][3];
  for (int r = 0; r < 2; ++r) for (int q = 0; q < 3; ++q) G2T[r][q] = G2[r][0] * P.T[0][q] + G2[r][1] * P.T[1][q];
  for (int r = 0; r < 3; ++r) for (int q = 0; q < 3; ++q) Gc[r][q] = P.T[0][r] * G2T[0][q] + P.T[1][r] * G2T[1][q];
  for (int r = 0; r < 2; ++r)
    for (int q = 0; q < 3; ++q) {
      double acc = 0;
      for (int k = 0; k < 3; ++k) acc += G2T[r][k] * P.Sig_c[k][q];
      dT[r][q] = 2 * acc;
    }
  // T = J W:  dJ = dT W^T
  double dJ[2][3];
  for (int r = 0; r < 2; ++r)
    for (int q = 0; q < 3; ++q) dJ[r][q] = dT[r][0] * V.Wm[q][0] + dT[r][1] * V.Wm[q][1] + dT[r][2] * V.Wm[q][2];
  // J(p) and the pinhole map (u,v)(p)
  const double x = P.p[0], y = P.p[1], z = P.p[2];
  double dp[3];
  dp[0] = g_u * V.fx / z;
  dp[1] = g_v * V.fy / z;
  dp[2] = -g_u * V.fx * x / (z * z) - g_v * V.fy * y / (z * z);
  dp[2] += g_z;                                   // auxiliary depth channel: z_k = p_z directly
  dp[2] += dJ[0][0] * (-V.fx / (z * z)) + dJ[1][1] * (-V.fy / (z * z));
  if (!P.clampx) { dp[0] += dJ[0][2] * (-V.fx / (z * z)); dp[2] += dJ[0][2] * (2 * V.fx * x / (z * z * z)); }
  else           { dp[2] += dJ[0][2] * (V.fx * P.xr / (z * z)); }      // J02 = -fx * xr / z with xr constant
  if (!P.clampy) { dp[1] += dJ[1][2] * (-V.fy / (z * z)); dp[2] += dJ[1][2] * (2 * V.fy * y / (z * z * z)); }
  else           { dp[2] += dJ[1][2] * (V.fy * P.yr / (z * z)); }
  for (int r = 0; r < 3; ++r) d_muc[r] += V.Wm[0][r] * dp[0] + V.Wm[1][r] * dp[1] + V.Wm[2][r] * dp[2];
  // o = sigmoid(logit) w;  w = exp(-Delta^2 / (2 b))
  d_logit[i] += g_o * P.w * P.sig * (1 - P.sig);
  const double d_w = g_o * P.sig;
  d_dt += d_w * P.w * (-P.dt / P.b);
  d_b += d_w * P.w * (0.5 * P.dt * P.dt / (P.b * P.b));
  // eq. 9: mu_c = mu_1:3 + a Delta / b;  Sigma_c = Sigma_1:3,1:3 - a a^T / b
  double d_a[3];
  double muc_a = 0, aGa = 0;
  for (int r = 0; r < 3; ++r) muc_a += d_muc[r] * P.a[r];
  for (int r = 0; r < 3; ++r) for (int q = 0; q < 3; ++q) aGa += P.a[r] * Gc[r][q] * P.a[q];
  for (int r = 0; r < 3; ++r) {
    double Ga = 0;
    for (int q = 0; q < 3; ++q) Ga += Gc[r][q] * P.a[q];
    d_a[r] = d_muc[r] * P.dt / P.b - 2 * Ga / P.b;
  }
  d_dt += muc_a / P.b;
  d_b += -muc_a * P.dt / (P.b * P.b) + aGa / (P.b * P.b);
  for (int r = 0; r < 3; ++r) d_mean[4 * i + r] += d_muc[r];
  d_mean[4 * i + 3] += -d_dt;                                             // Delta = t - mu_t
  // density-control indicators of this view: magnitude of the screen-space position gradient, magnitude
  // of the mu_t gradient, and the number of views the primitive was visible in
  if (densify3) { densify3[3 * i] += std::sqrt(g_u * g_u + g_v * g_v); densify3[3 * i + 1] += std::fabs(d_dt); densify3[3 * i + 2] += 1.0; }
  // gradient wrt the full symmetric 4x4 Sigma, then Sigma = M M^T, M = R4 diag(s)
  double GS[4][4];
  for (int r = 0; r < 3; ++r) for (int q = 0; q < 3; ++q) GS[r][q] = Gc[r][q];
  for (int r = 0; r < 3; ++r) { GS[r][3] = 0.5 * d_a[r]; GS[3][r] = 0.5 * d_a[r]; }
  GS[3][3] = d_b;
  double dM[4][4], dR4[4][4];
  for (int r = 0; r < 4; ++r)
    for (int k = 0; k < 4; ++k) {
      double acc = 0;
      for (int q = 0; q < 4; ++q) acc += GS[r][q] * P.M[q][k];
      dM[r][k] = 2 * acc;
    }
  for (int k = 0; k < 4; ++k) {
    double ds = 0;
    for (int r = 0; r < 4; ++r) { ds += dM[r][k] * P.R4[r][k]; dR4[r][k] = dM[r][k] * P.s[k]; }
    d_ls[4 * i + k] += ds * P.s[k];                                        // s = exp(log s)
  }
  // R4 = L(q_l) R(q_r)
  double dL[4][4], dR[4][4];
  for (int r = 0; r < 4; ++r)
    for (int q = 0; q < 4; ++q) {
      double accL = 0, accR = 0;
      for (int k = 0; k < 4; ++k) { accL += dR4[r][k] * P.Rm[q][k]; accR += P.Lm[k][r] * dR4[k][q]; }
      dL[r][q] = accL; dR[r][q] = accR;
    }
  double dql[4], dqr[4];
  dql[0] = dL[0][0] + dL[1][1] + dL[2][2] + dL[3][3];
  dql[1] = -dL[0][1] + dL[1][0] - dL[2][3] + dL[3][2];
  dql[2] = -dL[0][2] + dL[1][3] + dL[2][0] - dL[3][1];
  dql[3] = -dL[0][3] - dL[1][2] + dL[2][1] + dL[3][0];
  dqr[0] = dR[0][0] + dR[1][1] + dR[2][2] + dR[3][3];
  dqr[1] = -dR[0][1] + dR[1][0] + dR[2][3] - dR[3][2];
  dqr[2] = -dR[0][2] - dR[1][3] + dR[2][0] + dR[3][1];
  dqr[3] = -dR[0][3] + dR[1][2] - dR[2][1] + dR[3][0];
  // normalisation q_hat = q / |q|
  double dl = 0, dr = 0;
  for (int k = 0; k < 4; ++k) { dl += P.ql[k] * dql[k]; dr += P.qr[k] * dqr[k]; }
  for (int k = 0; k < 4; ++k) {
    d_ql[4 * i + k] += (dql[k] - P.ql[k] * dl) / P.nl;
    d_qr[4 * i + k] += (dqr[k] - P.qr[k] * dr) / P.nr;
  }
  (void)c;
}

}  // namespace

// ---------------------------------------------------------------------------------------------
// C ABI of the oracle (its own; unrelated to include/fdgs.h).  All arrays are host float64 unless noted.
extern "C" {

void* fdgs_oracle_create(int N, int sh_degree, int n_time, const double* mean, const double* log_scale,
                         const double* quat_l, const double* quat_r, const double* opacity_logit,
                         const double* sh) {
  if (N < 0 || sh_degree < 0 || sh_degree > 3 || n_time < 1) return nullptr;
  Oracle* O = new Oracle();
  O->N = N; O->L = sh_degree; O->n_time = n_time; O->Kd = (sh_degree + 1) * (sh_degree + 1); O->K = n_time * O->Kd;
  O->mean.assign(mean, mean + (size_t)4 * N); O->log_scale.assign(log_scale, log_scale + (size_t)4 * N);
  O->quat_l.assign(quat_l, quat_l + (size_t)4 * N); O->quat_r.assign(quat_r, quat_r + (size_t)4 * N);
  O->logit.assign(opacity_logit, opacity_logit + (size_t)N);
  O->sh.assign(sh, sh + (size_t)N * O->K * 3);
  return O;
}
void fdgs_oracle_destroy(void* h) { delete (Oracle*)h; }

// view16: row-major 4x4 world->camera [W|tau; 0 0 0 1]; intr = fx,fy,cx,cy; cfg9 = marginal_min, alpha_min,
// alpha_max, transmittance_min, dilation, cutoff_sigma, znear, guard, full_support(0/1)
int fdgs_oracle_preprocess(void* h, const double* view16, const double* intr, int width, int height, double t,
                           double period_T, const double* bg, const double* cfg9) {
  Oracle& O = *(Oracle*)h;
  if (width <= 0 || height <= 0) return -1;
  O.colour_override = false;
  for (int r = 0; r < 3; ++r) { for (int q = 0; q < 3; ++q) O.view.Wm[r][q] = view16[4 * r + q]; O.view.tau[r] = view16[4 * r + 3]; }
  O.view.fx = intr[0]; O.view.fy = intr[1]; O.view.cx = intr[2]; O.view.cy = intr[3];
  O.view.width = width; O.view.height = height; O.view.t = t; O.view.period_T = period_T;
  for (int k = 0; k < 3; ++k) O.view.bg[k] = bg[k];
  O.cfg.marginal_min = cfg9[0]; O.cfg.alpha_min = cfg9[1]; O.cfg.alpha_max = cfg9[2]; O.cfg.transmittance_min = cfg9[3];
  O.cfg.dilation = cfg9[4]; O.cfg.cutoff_sigma = cfg9[5]; O.cfg.znear = cfg9[6]; O.cfg.guard = cfg9[7];
  O.cfg.full_support = cfg9[8] != 0;
  O.tiles_x = (width + TILE - 1) / TILE; O.tiles_y = (height + TILE - 1) / TILE;
  O.prims.resize(O.N);
#pragma omp parallel for schedule(static)
  for (int i = 0; i < O.N; ++i) preprocess_one(O, i, O.prims[i]);
  build_tile_lists(O);
  return 0;
}

int64_t fdgs_oracle_num_pairs(void* h) { return (int64_t)((Oracle*)h)->tile_ids.size(); }
int fdgs_oracle_num_tiles(void* h) { Oracle& O = *(Oracle*)h; return O.tiles_x * O.tiles_y; }

// tile_off[tiles+1] int64, tile_ids[D] int32
void fdgs_oracle_get_tile_lists(void* h, int64_t* tile_off, int32_t* tile_ids) {
  Oracle& O = *(Oracle*)h;
  std::copy(O.tile_off.begin(), O.tile_off.end(), tile_off);
  std::copy(O.tile_ids.begin(), O.tile_ids.end(), tile_ids);
}

// Per-primitive record, 40 doubles per primitive (NaN where not computed because of an earlier cull):
//  0 status  1 w  2 Sigma_44  3 Delta  4-6 mu_c  7-12 Sigma_c (xx,xy,xz,yy,yz,zz)  13-15 p_cam  16 u  17 v
//  18-20 conic A,B,C  21 radius  22-25 rect tx0,ty0,tx1,ty1  26-28 rgb  29 clamp bits (colour ch0..2 |
//  clampx<<3 | clampy<<4)  30 o  31 depth32  32 fragility  33-35 raw colour  36-39 Sigma_2d a,b,c, spare
void fdgs_oracle_get_prims(void* h, double* out) {
  Oracle& O = *(Oracle*)h;
  const double nan = std::nan("");
  for (int i = 0; i < O.N; ++i) {
    const Prim& P = O.prims[i];
    double* r = out + (size_t)40 * i;
    for (int k = 0; k < 40; ++k) r[k] = nan;
    r[0] = P.status; r[32] = P.frag;
    if (P.status == CULL_NONFINITE) continue;
    r[1] = P.w; r[2] = P.b; r[3] = P.dt;
    if (P.status == CULL_TIME) continue;
    for (int k = 0; k < 3; ++k) { r[4 + k] = P.mu_c[k]; r[13 + k] = P.p[k]; }
    r[7] = P.Sig_c[0][0]; r[8] = P.Sig_c[0][1]; r[9] = P.Sig_c[0][2]; r[10] = P.Sig_c[1][1]; r[11] = P.Sig_c[1][2]; r[12] = P.Sig_c[2][2];
    r[31] = P.depth32;
    if (P.status == CULL_NEAR) continue;
    r[16] = P.u; r[17] = P.v; r[18] = P.A; r[19] = P.B; r[20] = P.C; r[21] = P.radius;
    for (int k = 0; k < 4; ++k) r[22 + k] = P.rect[k];
    r[36] = P.S2[0][0]; r[37] = P.S2[0][1]; r[38] = P.S2[1][1];
    if (P.status == CULL_RECT) continue;
    int bits = 0;
    for (int k = 0; k < 3; ++k) { r[26 + k] = P.rgb[k]; r[33 + k] = P.raw[k]; if (!(P.raw[k] > 0)) bits |= 1 << k; }
    bits |= P.clampx << 3; bits |= P.clampy << 4;
    r[29] = bits; r[30] = P.o;
  }
}

// 4D rotation and covariance of primitive i (row-major 4x4 each) — for the eq. 7/8 pins
void fdgs_oracle_get_rot_cov(void* h, int i, double* R16, double* Sigma16) {
  Oracle& O = *(Oracle*)h;
  std::memcpy(R16, O.prims[i].R4, 16 * sizeof(double));
  std::memcpy(Sigma16, O.prims[i].Sig, 16 * sizeof(double));
}

// real SH basis values Y[(L+1)^2] at unit direction dir3 — for the quadrature / library pins
void fdgs_oracle_sh_basis(int sh_degree, const double* dir3, double* Y) { sh_basis(sh_degree, dir3, Y, nullptr); }
// the same with the hand-written gradient rows grad[(L+1)^2][3] of the polynomial extension — exported so that a
// `-m "not gpu"` test can pin them against central differences of the values (tests/test_oracle_pins.py)
void fdgs_oracle_sh_basis_grad(int sh_degree, const double* dir3, double* Y, double* grad) {
  sh_basis(sh_degree, dir3, Y, reinterpret_cast<double (*)[3]>(grad));
}

// image[3,H,W], final_T[H,W], n_contrib[H,W] int32 (1 + list position of the last contributor),
// margin[H,W] (min relative margin of any alpha / transmittance test at that pixel)
void fdgs_oracle_forward(void* h, double* image, double* final_T, int32_t* n_contrib, double* margin) {
  Oracle& O = *(Oracle*)h;
  forward(O);
  std::copy(O.image.begin(), O.image.end(), image);
  std::copy(O.final_T.begin(), O.final_T.end(), final_T);
  std::copy(O.n_contrib.begin(), O.n_contrib.end(), n_contrib);
  if (margin) std::copy(O.margin.begin(), O.margin.end(), margin);
}

// Requires fdgs_oracle_forward on the same state.  All gradient arrays are accumulated into (+=).
// g9[N,9] (may be NULL) receives (=) the per-splat blend gradients g_u,g_v,g_A,g_B,g_C,g_o,g_rgb.
void fdgs_oracle_backward(void* h, const double* dL_dimage, double* d_mean, double* d_log_scale, double* d_quat_l,
                          double* d_quat_r, double* d_logit, double* d_sh, double* d_mean2d, double* g9) {
  Oracle& O = *(Oracle*)h;
  backward_blend(O, dL_dimage);
  if (g9) std::copy(O.g9.begin(), O.g9.end(), g9);
#pragma omp parallel for schedule(static)
  for (int i = 0; i < O.N; ++i)
    backward_one(O, i, &O.g9[(size_t)9 * i], d_mean, d_log_scale, d_quat_l, d_quat_r, d_logit, d_sh, d_mean2d);
}

// Auxiliary channels.  depth_map[H,W] of the last fdgs_oracle_forward.
void fdgs_oracle_get_depth_map(void* h, double* depth_map) {
  Oracle& O = *(Oracle*)h;
  std::copy(O.depth_map.begin(), O.depth_map.end(), depth_map);
}

// fdgs_oracle_backward with upstream gradients of the auxiliary channels as well: dL_ddepth[H,W], dL_dopacity[H,W]
// (either may be NULL).  gz[N] (may be NULL) receives the per-splat dL/dz.  densify3[N,3] (may be NULL) is accumulated
// into (+=): |dL/d(u,v)|, |dL/dmu_t|, visibility count of this view (density-control indicators).
void fdgs_oracle_backward_aux(void* h, const double* dL_dimage, const double* dL_ddepth, const double* dL_dopacity,
                              double* d_mean, double* d_log_scale, double* d_quat_l, double* d_quat_r, double* d_logit,
                              double* d_sh, double* d_mean2d, double* g9, double* gz, double* densify3) {
  Oracle& O = *(Oracle*)h;
  backward_blend(O, dL_dimage, dL_ddepth, dL_dopacity);
  if (g9) std::copy(O.g9.begin(), O.g9.end(), g9);
  if (gz) std::copy(O.gz.begin(), O.gz.end(), gz);
#pragma omp parallel for schedule(static)
  for (int i = 0; i < O.N; ++i)
    backward_one(O, i, &O.g9[(size_t)9 * i], d_mean, d_log_scale, d_quat_l, d_quat_r, d_logit, d_sh, d_mean2d, O.gz[i], densify3);
}

// Feature channels ("rendered following the same process as in Section 3.2, with the color c replaced by
// the ... feature vector"; L410: the projected displacement rendered "using equation (6)" as optical flow): replaces the
// colour of every visible primitive by rgb[N,3] (three channels at a time; more channels = more passes).  The override
// stays until the next fdgs_oracle_preprocess; while it is active the backward returns dL/d(feature) in g9[:,6:9] and
// chains only the geometry (u, v, conic, opacity) to the parameters.
void fdgs_oracle_set_colour_override(void* h, const double* rgb) {
  Oracle& O = *(Oracle*)h;
  O.colour_override = true;
  for (int i = 0; i < O.N; ++i)
    if (O.prims[i].status == VISIBLE)
      for (int ch = 0; ch < 3; ++ch) O.prims[i].rgb[ch] = rgb[(size_t)3 * i + ch];
}

// threads used by the OpenMP loops from now on (timing only: bench.py reports single-thread and all-core times; no arithmetic)
void fdgs_oracle_set_num_threads(int n) {
#ifdef _OPENMP
  if (n > 0) omp_set_num_threads(n);
#else
  (void)n;
#endif
}

int fdgs_oracle_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

}  // extern "C"
