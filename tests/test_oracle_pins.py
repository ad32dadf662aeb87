"""Pins for the float64 oracle: what the paper and the mathematics fix, by routes that do not
retype the oracle's own formulas (Hamilton product, eigenvalues, library inverse, scipy SH,
quadrature, numerical Jacobian, brute force).  Part 1: the per-primitive chain (eq. 3-4, 7-10, 20)."""
import os

import numpy as np
import pytest

import oracle
from helpers import hand_scene, make_oracle, oracle_for, run_pre
from paper_2412_20720_b200 import scenes

GOLD = os.path.join(os.path.dirname(__file__), "golden", "eq8_worked_example.txt")


def _hamilton(p, q):
    a1, b1, c1, d1 = p
    a2, b2, c2, d2 = q
    return np.array([a1 * a2 - b1 * b2 - c1 * c2 - d1 * d2,
                     a1 * b2 + b1 * a2 + c1 * d2 - d1 * c2,
                     a1 * c2 - b1 * d2 + c1 * a2 + d1 * b2,
                     a1 * d2 + b1 * c2 - c1 * b2 + d1 * a2])


def _rot_from_hamilton(ql, qr):
    """R x = q_l * x * q_r (quaternion product) — never builds the matrices of eq. 8."""
    ql, qr = ql / np.linalg.norm(ql), qr / np.linalg.norm(qr)
    return np.stack([_hamilton(_hamilton(ql, e), qr) for e in np.eye(4)], axis=1)


def _one(ql, qr, ls=(0, 0, 0, 0), mean=(0, 0, 0, 0.5), t=0.5):
    sc = hand_scene([mean], [ls], [ql], [qr], t=t)
    return oracle_for(sc)


def _golden():
    rows = [list(map(float, l.split())) for l in open(GOLD) if l.strip() and not l.startswith("#")]
    return np.array(rows[0:4]), np.array(rows[4:8]), np.array(rows[8])


# ------------------------------------------------------------------ eq. 8: 4D rotation
def test_eq8_matches_hamilton_product():
    rng = np.random.default_rng(0)
    for _ in range(20):
        ql, qr = rng.normal(size=4), rng.normal(size=4)
        R, _ = _one(ql, qr).rot_cov(0)
        np.testing.assert_allclose(R, _rot_from_hamilton(ql, qr), atol=1e-14)


def test_eq8_orthogonal_det_plus_one_and_identity():
    rng = np.random.default_rng(1)
    for _ in range(10):
        R, _ = _one(rng.normal(size=4), rng.normal(size=4)).rot_cov(0)
        np.testing.assert_allclose(R.T @ R, np.eye(4), atol=1e-14)
        assert abs(np.linalg.det(R) - 1.0) < 1e-13
    # PAPER.md:L324 "initialized both q_l and q_r as unit quaternions to construct identity rotation matrix"
    R, _ = _one([1, 0, 0, 0], [1, 0, 0, 0]).rot_cov(0)
    np.testing.assert_allclose(R, np.eye(4), atol=0)
    # quaternions need not be unit: normalisation happens inside
    R2, _ = _one([3, 0, 0, 0], [0.2, 0, 0, 0]).rot_cov(0)
    np.testing.assert_allclose(R2, np.eye(4), atol=1e-15)


def test_eq8_golden_worked_example():
    Rint, Sig, sl = _golden()
    ql, qr = np.array([1.0, 2, 3, 4]), np.array([2.0, -1, 1, 3])
    # the stored integers are first re-derived independently (Hamilton product) ...
    np.testing.assert_allclose(_rot_from_hamilton(ql, qr) * np.sqrt(450.0), Rint, atol=1e-12)
    # ... then pin the oracle: eq. 8, eq. 7, eq. 9-10
    s = np.array([0.5, 1, 2, 0.25])
    o = _one(ql, qr, np.log(s), mean=(0.1, -0.2, 0.3, 0.4), t=0.6)
    R, S = o.rot_cov(0)
    np.testing.assert_allclose(R * np.sqrt(450.0), Rint, atol=1e-12)
    np.testing.assert_allclose(S, Sig, atol=1e-12)
    p = o.prims()
    got = np.concatenate([[p.sigma44[0], p.w[0]], p.mu_c[0], p.sigma_c6[0]])
    np.testing.assert_allclose(got, sl, atol=2e-12)


# ------------------------------------------------------------------ eq. 7: covariance
def test_eq7_eigenvalues_are_squared_scales():
    rng = np.random.default_rng(2)
    for _ in range(10):
        ls = rng.normal(-1, 0.7, size=4)
        _, S = _one(rng.normal(size=4), rng.normal(size=4), ls).rot_cov(0)
        np.testing.assert_allclose(S, S.T, atol=1e-15)
        np.testing.assert_allclose(np.sort(np.linalg.eigvalsh(S)), np.sort(np.exp(2 * ls)), rtol=1e-12)
        assert abs(np.linalg.det(S) / np.exp(2 * ls.sum()) - 1) < 1e-12


def test_identity_rotation_gives_diagonal_and_t_independent_mean():
    # north_star invariant: R = I => mu_c == mu_1:3 for every t, Sigma_c = diag(s^2), Sigma_44 = s_t^2
    ls = np.log([0.3, 0.5, 0.7, 0.9])
    for t in (0.1, 0.5, 1.3):
        o = _one([1, 0, 0, 0], [1, 0, 0, 0], ls, mean=(0.2, -0.1, 0.3, 0.5), t=t)
        p = o.prims()
        np.testing.assert_allclose(p.mu_c[0], [0.2, -0.1, 0.3], atol=1e-15)
        np.testing.assert_allclose(p.sigma_c(0), np.diag([0.09, 0.25, 0.49]), atol=1e-15)
        assert abs(p.sigma44[0] - 0.81) < 1e-15


def test_spatial_rotation_family_decouples_time():
    # q_r = (a,b,c,-d) with q_l = (a,b,c,d) is a pure spatial rotation (the "No-4DRot" family, L124)
    rng = np.random.default_rng(3)
    q = rng.normal(size=4)
    R, S = _one(q, q * np.array([1, 1, 1, -1]), np.log([0.3, 0.5, 0.7, 0.9])).rot_cov(0)
    np.testing.assert_allclose(R[3], [0, 0, 0, 1], atol=1e-15)
    np.testing.assert_allclose(S[:3, 3], 0, atol=1e-15)


# ------------------------------------------------------------------ eq. 9-10, 11-19: slicing
def test_factorisation_against_library_inverse():
    """exp(-1/2 d^T Sigma^-1 d) = p(t) * exp(-1/2 d3^T Sigma_c^-1 d3), brute force."""
    rng = np.random.default_rng(4)
    for _ in range(10):
        ls, mu = rng.normal(-0.5, 0.4, size=4), rng.normal(size=4)
        t = mu[3] + rng.normal() * 0.3
        o = _one(rng.normal(size=4), rng.normal(size=4), ls, mean=mu, t=t)
        _, S = o.rot_cov(0)
        p = o.prims()
        w, mu_c, Sc = p.w[0], p.mu_c[0], p.sigma_c(0)
        Sinv, Scinv = np.linalg.inv(S), np.linalg.inv(Sc)
        for _ in range(5):
            x = mu[:3] + rng.normal(size=3) * 0.5
            d = np.concatenate([x - mu[:3], [t - mu[3]]])
            joint = np.exp(-0.5 * d @ Sinv @ d)
            cond = np.exp(-0.5 * (x - mu_c) @ Scinv @ (x - mu_c))
            assert abs(joint - w * cond) < 1e-12 * max(joint, 1e-30) + 1e-15
        # eq. 15 (L165): det Sigma = Sigma_44 * det Sigma_xyz|t
        assert abs(np.linalg.det(S) / (p.sigma44[0] * np.linalg.det(Sc)) - 1) < 1e-11


def test_conditional_mean_affine_in_t_and_shift_invariance():
    rng = np.random.default_rng(5)
    ql, qr, ls, mu = rng.normal(size=4), rng.normal(size=4), rng.normal(-0.5, 0.3, size=4), rng.normal(size=4)
    res = []
    for t in (mu[3] - 0.2, mu[3], mu[3] + 0.2):
        o = _one(ql, qr, ls, mean=mu, t=t)
        p = o.prims()
        res.append((p.mu_c[0].copy(), p.sigma_c6[0].copy()))
    _, S = o.rot_cov(0)
    np.testing.assert_allclose(res[1][0], mu[:3], atol=1e-15)
    np.testing.assert_allclose((res[2][0] - res[0][0]) / 0.4, S[:3, 3] / S[3, 3], rtol=1e-12)
    np.testing.assert_allclose(res[0][1], res[2][1], atol=1e-15)          # Sigma_c independent of t
    # joint shift t -> t+d, mu_t -> mu_t+d changes nothing
    mu2 = mu.copy(); mu2[3] += 7.0
    p2 = _one(ql, qr, ls, mean=mu2, t=mu[3] + 0.2 + 7.0).prims()
    np.testing.assert_allclose(p2.mu_c[0], res[2][0], atol=1e-13)
    np.testing.assert_allclose(p2.w[0], _one(ql, qr, ls, mean=mu, t=mu[3] + 0.2).prims().w[0], rtol=1e-12)


def test_marginal_filter_threshold():
    """filter p(t) < 0.05 <=> |Delta| > sqrt(-2 ln 0.05) * sqrt(Sigma_44) = 2.44775 sigma_t."""
    st = 0.3
    edge = np.sqrt(-2 * np.log(0.05)) * st
    assert abs(edge / st - 2.44775) < 1e-5
    for dt, want in ((edge * 0.999, oracle.STATUS_VISIBLE), (edge * 1.001, oracle.STATUS_CULL_TIME)):
        p = _one([1, 0, 0, 0], [1, 0, 0, 0], np.log([0.2, 0.2, 0.2, st]), mean=(0, 0, 0, 0.5), t=0.5 + dt).prims()
        assert p.status[0] == want
        assert abs(p.w[0] - np.exp(-0.5 * dt * dt / st**2)) < 1e-14
    # marginal_min = 0 disables the filter (urban variant, L265)
    sc = hand_scene([(0, 0, 0, 0.5)], [np.log([0.2, 0.2, 0.2, st])], t=0.5 + 3 * st)
    assert oracle_for(sc, cfg=dict(marginal_min=0.0)).prims().status[0] == oracle.STATUS_VISIBLE


# ------------------------------------------------------------------ eq. 20: 4D spherindrical harmonics
def _scipy_real_sh(l, m, d):
    """Real SH from scipy's complex ones, Condon-Shortley phase kept (DESIGN reading S5)."""
    from scipy import special
    theta, phi = np.arccos(np.clip(d[2], -1, 1)), np.arctan2(d[1], d[0])      # polar, azimuth
    if hasattr(special, "sph_harm_y"):
        Y = special.sph_harm_y(l, abs(m), theta, phi)
    else:
        Y = special.sph_harm(abs(m), l, phi, theta)
    if m == 0:
        return Y.real
    return np.sqrt(2.0) * (Y.real if m > 0 else Y.imag)


def test_sh_table_against_scipy():
    rng = np.random.default_rng(6)
    for _ in range(20):
        d = rng.normal(size=3); d /= np.linalg.norm(d)
        Y = oracle.sh_basis(3, d)
        ref = np.array([_scipy_real_sh(l, m, d) for l in range(4) for m in range(-l, l + 1)])
        np.testing.assert_allclose(Y, ref, atol=1e-13)


def test_sh_orthonormal_by_quadrature():
    """'form an orthonormal basis': Gram matrix over the sphere = I (Gauss-Legendre x uniform phi)."""
    xs, ws = np.polynomial.legendre.leggauss(16)
    phis = 2 * np.pi * (np.arange(32) + 0.5) / 32
    G = np.zeros((16, 16))
    for z, wz in zip(xs, ws):
        for ph in phis:
            r = np.sqrt(1 - z * z)
            Y = oracle.sh_basis(3, np.array([r * np.cos(ph), r * np.sin(ph), z]))
            G += wz * (2 * np.pi / 32) * np.outer(Y, Y)
    np.testing.assert_allclose(G, np.eye(16), atol=1e-12)


def _colour_scene(sh, sh_degree, n_time, mu_t=0.5, t=0.5, T=1.0, pos=(0.3, -0.2, 0.1)):
    return hand_scene([(pos[0], pos[1], pos[2], mu_t)], [np.log([0.1, 0.1, 0.1, 5.0])], sh=sh, sh_degree=sh_degree,
                      n_time=n_time, t=t, T=T)


def test_colour_dc_only_and_time_independence_of_n0():
    rng = np.random.default_rng(7)
    # DC only: c = 0.5 + Y_00 * coef
    sh = np.zeros((1, 8, 3)); sh[0, 0] = [0.3, 1.0, -5.0]
    p = oracle_for(_colour_scene(sh, 1, 2)).prims()
    np.testing.assert_allclose(p.rgb[0], np.maximum(0, 0.5 + 0.28209479177387814 * sh[0, 0]), atol=1e-15)
    assert int(p.clamp_bits[0]) & 7 == 4                    # third channel clamped at 0
    # only n = 0 coefficients: colour equals ordinary SH and does not depend on t
    sh = np.zeros((1, 48, 3)); sh[0, :16] = rng.normal(0, 0.3, size=(16, 3))
    cols = [oracle_for(_colour_scene(sh, 3, 3, t=t)).prims().raw_rgb[0] for t in (0.1, 0.5, 0.77)]
    np.testing.assert_allclose(cols[0], cols[1], atol=1e-15)
    np.testing.assert_allclose(cols[0], cols[2], atol=1e-15)
    # ... and equals sum_k coef_k Y_k(dir) with dir from the camera centre (0,0,-4) to the mean
    d = np.array([0.3, -0.2, 0.1 + 4.0]); d /= np.linalg.norm(d)
    ref = 0.5 + np.array([_scipy_real_sh(l, m, d) for l in range(4) for m in range(-l, l + 1)]) @ sh[0, :16]
    np.testing.assert_allclose(cols[0], ref, atol=1e-13)


def test_fourier_basis_in_delta_t():
    """Z_nl^m = cos(2 pi n Delta/T) Y_l^m, Delta = t - mu_t (eq. 20): zero at Delta = T/(4n), period T."""
    sh = np.zeros((1, 3, 3)); sh[0, 1] = [1.0, 2.0, 3.0]     # L=0, n_time=3, only n=1
    T, mu_t = 2.0, 0.4
    raw = lambda t: oracle_for(_colour_scene(sh, 0, 3, mu_t=mu_t, t=t, T=T)).prims().raw_rgb[0]
    np.testing.assert_allclose(raw(mu_t + T / 4), 0.5, atol=1e-15)
    np.testing.assert_allclose(raw(mu_t), 0.5 + 0.28209479177387814 * sh[0, 1], atol=1e-15)
    np.testing.assert_allclose(raw(mu_t + 0.3), raw(mu_t + 0.3 + T), atol=1e-13)
    np.testing.assert_allclose(raw(mu_t + 0.3), 0.5 + np.cos(2 * np.pi * 0.3 / T) * 0.28209479177387814 * sh[0, 1], atol=1e-14)
    sh2 = np.zeros((1, 3, 3)); sh2[0, 2] = [1.0, 2.0, 3.0]   # n = 2 vanishes at T/8
    np.testing.assert_allclose(oracle_for(_colour_scene(sh2, 0, 3, mu_t=mu_t, t=mu_t + T / 8, T=T)).prims().raw_rgb[0], 0.5, atol=1e-15)


# ------------------------------------------------------------------ eq. 3-4: EWA projection
def test_ewa_against_numerical_jacobian():
    rng = np.random.default_rng(8)
    sc = scenes.fd_scene(11, 8)
    v = sc.views[0]
    o = oracle_for(sc)
    p = o.prims()
    Wm, tau = v.view[:3, :3].astype(np.float64), v.view[:3, 3].astype(np.float64)
    proj = lambda x: np.array([v.fx * (Wm @ x + tau)[0] / (Wm @ x + tau)[2] + v.cx,
                               v.fy * (Wm @ x + tau)[1] / (Wm @ x + tau)[2] + v.cy])
    for i in range(sc.N):
        assert p.status[i] == oracle.STATUS_VISIBLE
        mu_c = p.mu_c[i]
        np.testing.assert_allclose(p.uv[i], proj(mu_c), rtol=1e-13)
        Jn = np.stack([(proj(mu_c + h) - proj(mu_c - h)) / 2e-6 for h in np.eye(3) * 1e-6], axis=1)   # 2x3
        S2 = Jn @ p.sigma_c(i) @ Jn.T + 0.3 * np.eye(2)
        Q = np.linalg.inv(S2)
        np.testing.assert_allclose(p.conic[i], [Q[0, 0], Q[0, 1], Q[1, 1]], rtol=1e-7)
        lam = np.linalg.eigvalsh(S2).max()
        assert abs(p.radius[i] / (3 * np.sqrt(lam)) - 1) < 1e-7
    del rng


def test_isotropic_splat_on_axis_closed_form():
    """Lone isotropic Gaussian on the optical axis: Sigma_2d = ((f s/z)^2 + 0.3) I (north_star 'analytic footprint')."""
    s, z0 = 0.1, 4.0
    sc = hand_scene([(0, 0, 0, 0.5)], [np.log([s, s, s, 1.0])], logit=[1.0], sh=[[[2.0, 1.0, 0.5]]], bg=(0.1, 0.2, 0.3))
    v = sc.views[0]
    o = oracle_for(sc, cfg=oracle.PURE_CFG)
    p = o.prims()
    var = (v.fx * s / z0) ** 2 + 0.3
    np.testing.assert_allclose(p.sigma2d[0], [var, 0, var], rtol=1e-13, atol=1e-15)
    np.testing.assert_allclose(p.uv[0], [32, 32], atol=1e-13)
    img, fT, nc, _ = o.forward()
    ys, xs = np.mgrid[0:64, 0:64] + 0.5
    a = (1 / (1 + np.exp(-1.0))) * np.exp(-0.5 * ((xs - 32) ** 2 + (ys - 32) ** 2) / var)
    col = 0.5 + 0.28209479177387814 * np.array([2.0, 1.0, 0.5])
    ref = a[None] * col[:, None, None] + (1 - a)[None] * np.array([0.1, 0.2, 0.3])[:, None, None]
    np.testing.assert_allclose(img, ref, atol=1e-14)
    np.testing.assert_allclose(fT, 1 - a, atol=1e-15)


def test_sh_gradient_rows_against_central_differences():
    """The 48 hand-written entries dY_k/d(x,y,z), k < 16, of the polynomial extension (used by the backward of eq. 20 for
    dL/d dir) against central differences of the VALUES, which are themselves pinned by scipy and quadrature above.
    The Y_k are polynomials of degree <= 3, so a central difference with step h is exact up to h^2 * (third derivative):
    1e-5 is a loose bound; a wrong sign, factor or index in any row fails it by O(1).  Points off the unit sphere as well
    (the extension, not the restriction, is what the chain rule through dir = d / |d| needs)."""
    rng = np.random.default_rng(3)
    for trial in range(20):
        d = rng.standard_normal(3)
        if trial % 2 == 0:
            d /= np.linalg.norm(d)
        for L in (0, 1, 2, 3):
            Y, G = oracle.sh_basis_grad(L, d)
            np.testing.assert_allclose(Y, oracle.sh_basis(L, d), rtol=0, atol=0)
            h = 1e-5
            for c in range(3):
                e = np.zeros(3); e[c] = h
                fd = (oracle.sh_basis(L, d + e) - oracle.sh_basis(L, d - e)) / (2 * h)
                np.testing.assert_allclose(G[:, c], fd, rtol=1e-7, atol=1e-7)
    # Euler's theorem for homogeneous polynomials pins the rows a second, independent way: d . grad Y_k = l Y_k
    d = rng.standard_normal(3)
    Y, G = oracle.sh_basis_grad(3, d)
    deg = np.array([l for l in range(4) for _ in range(2 * l + 1)], dtype=np.float64)
    # Y_6 and the degree-3 rows are written with z^2-x^2-y^2 style terms: all homogeneous of degree l
    np.testing.assert_allclose(G @ d, deg * Y, rtol=1e-12, atol=1e-12)
