"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU, no CUDA path).

Each test names the passage it pins (P:n = PAPER.md line n, S:n = SPEC.md line n, Rk = DESIGN.md
reading k).  Nothing here re-calls the oracle to check the oracle: expected values are printed
values (tests/golden/worked_values.json), closed forms, numerical differentiation / quadrature /
sampling done in numpy, or invariants.
"""
import json
import math
import os

import numpy as np
import pytest

import oracle
from helpers import Y0, camera, level, random_rotation
from oracle import OracleScene, SKIP_THR, STOP_THR

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "worked_values.json")))


# ------------------------------------------------------------------ Eq. 3 / Eq. 4 / Eq. 1 / opacity

def test_scale_ladder_printed_values():
    """Eq. 3; printed values S:50-52."""
    for c in GOLD["scale_ladder"]["cases"]:
        assert oracle.scale_constraint(c["level"], c["tau"], c["rho"], c["l_max"]) == pytest.approx(c["s_min"], abs=1e-15)
    pc = GOLD["paper_constants"]
    ladder = [oracle.scale_constraint(l, pc["tau"], pc["rho"], pc["l_max"]) for l in range(1, pc["l_max"] + 1)]
    assert all(a > b for a, b in zip(ladder, ladder[1:])), "strictly decreasing (S:103)"
    assert ladder[-1] == 0.0 and ladder[0] == pc["tau"]
    assert math.isnan(oracle.scale_constraint(0, 0.2, 4, 5)) and math.isnan(oracle.scale_constraint(6, 0.2, 4, 5))


def test_effective_scale_printed_values():
    """Eq. 4."""
    c = GOLD["effective_scale"]["cases"]
    assert oracle.effective_scale(c[0]["s_opt"], c[0]["s_min"]) == pytest.approx(c[0]["s"], abs=1e-15)
    assert oracle.effective_scale(math.log(c[1]["s_opt_ln_of"]), c[1]["s_min"]) == pytest.approx(c[1]["s"], abs=1e-15)
    assert oracle.effective_scale(c[2]["s_opt"], c[2]["s_min"]) >= c[2]["s_lower_bound"]


def test_covariance_printed_values():
    """Eq. 1; worked matrices S:68-70."""
    for c in GOLD["covariance"]["cases"]:
        cov, _, _, _ = oracle.activate_one(np.log(np.array(c["s"], float)), c["quat_wxyz"], 0.0)
        xx, xy, xz, yy, yz, zz = cov
        np.testing.assert_allclose([xx, yy, zz], c["diag"], rtol=1e-6)
        np.testing.assert_allclose([xy, xz, yz], 0.0, atol=1e-6)


def test_covariance_eigenvalues_and_determinant():
    """Eq. 1: eigenvalues of R S S^T R^T are s^2 and det = (s1 s2 s3)^2, any quaternion norm."""
    rng = np.random.default_rng(11)
    for _ in range(50):
        s = np.exp(rng.uniform(-3, 1, 3))
        Rm, q = random_rotation(rng)
        cov, _, _, _ = oracle.activate_one(np.log(s), q * rng.uniform(0.1, 5.0), 0.0)
        xx, xy, xz, yy, yz, zz = cov.astype(np.float64)
        S = np.array([[xx, xy, xz], [xy, yy, yz], [xz, yz, zz]])
        np.testing.assert_allclose(np.sort(np.linalg.eigvalsh(S)), np.sort(s * s), rtol=2e-5)
        assert np.linalg.det(S) == pytest.approx(np.prod(s) ** 2, rel=1e-4)
        # orientation, not just spectrum: Sigma = R diag(s^2) R^T with R the textbook quaternion matrix
        np.testing.assert_allclose(S, Rm @ np.diag(s * s) @ Rm.T, rtol=1e-5, atol=1e-7 * (s * s).max())


def test_opacity_activation():
    """sigmoid(0) = 0.5; kappa = 2 ln(255 o); dead below 1/255 (R11)."""
    _, o, kappa, dead = oracle.activate_one([0, 0, 0], [1, 0, 0, 0], 0.0)
    assert o == 0.5 and not dead
    assert kappa == pytest.approx(2 * math.log(255 * 0.5), rel=1e-6)
    _, o, _, dead = oracle.activate_one([0, 0, 0], [1, 0, 0, 0], 20.0)
    assert abs(o - 1.0) < 1e-7 and not dead
    _, o, _, dead = oracle.activate_one([0, 0, 0], [1, 0, 0, 0], -20.0)
    assert o < 1e-7 and dead
    lg = math.log((1 / 255) / (1 - 1 / 255))
    assert oracle.activate_one([0, 0, 0], [1, 0, 0, 0], lg - 1e-3)[3]
    assert not oracle.activate_one([0, 0, 0], [1, 0, 0, 0], lg + 1e-3)[3]


# ------------------------------------------------------------------------------- Eq. 6 / Eq. 7

def test_d_proj_printed_values():
    """Eq. 7; 0.05*1000/1 = 50, doubling gamma halves, L_max -> 0."""
    for c in GOLD["d_proj"]["cases"]:
        assert oracle.d_proj(c["s_min"], c["gamma"], c["f"]) == pytest.approx(c["d_proj"], rel=1e-15)
    # the proportion s_min : gamma = d_proj : f
    assert oracle.d_proj(0.0125, 3.0, 700.0) * 3.0 == pytest.approx(0.0125 * 700.0)


def test_band_thresholds_overrides():
    """Eq. 7 with d_proj^(L_end) = 0 and d_proj^(L_start-1) = inf; squared, fp32."""
    lo, hi = oracle.band_thresholds([0.5, 0.05, 0.0], 1, 3, 1000.0, 1.0)
    assert lo[2] == 0.0 and hi[0] == np.inf
    assert lo[0] == np.float32(500.0 ** 2) and lo[1] == np.float32(50.0 ** 2)
    assert hi[1] == lo[0] and hi[2] == lo[1]
    # range that stops below the top uploaded level: its own s_min is overridden by 0
    lo, hi = oracle.band_thresholds([0.5, 0.05, 0.0], 1, 2, 1000.0, 1.0)
    assert lo[1] == 0.0 and hi[0] == np.inf and hi[1] == lo[0]
    assert lo[2] == 0.0 and hi[2] == 0.0   # outside the range: empty band


def _same_positions_scene(pos, level_ids, s_min):
    return OracleScene([level(l, s, pos, 0.01) for l, s in zip(level_ids, s_min)], 0)


def test_band_membership_printed_example():
    """Eq. 6; distances 10/100/1000, edges {0,50,500}, levels 5/4/3."""
    g = GOLD["band_membership"]
    pos = np.array([[0.0, 0.0, d] for d in g["distances"]])
    sc = _same_positions_scene(pos, g["levels"], g["s_min"])
    fr = sc.frame(camera(f=g["f"]), g["levels"][0], g["levels"][-1], g["gamma"])
    m = fr.mask.reshape(len(g["levels"]), -1)
    for j, lv in enumerate(g["assigned"]):
        chosen = [g["levels"][i] for i in range(len(g["levels"])) if m[i, j]]
        assert chosen == [lv]


def test_band_edge_is_half_open():
    """R1: bands are [d_proj^(l), d_proj^(l-1)); a Gaussian exactly on an edge is drawn once."""
    pos = np.array([[50.0, 0.0, 0.0], [np.nextafter(np.float32(50.0), np.float32(0.0)), 0.0, 0.0]])
    sc = _same_positions_scene(pos, [4, 5], [0.05, 0.0])
    fr = sc.frame(camera(f=1000.0), 4, 5, 1.0, ref_pos=[0.0, 0.0, 0.0])
    m = fr.mask.reshape(2, 2)
    assert m[:, 0].tolist() == [1, 0]    # d^2 = 2500 = lo^2 of level 4: level 4 only
    assert m[:, 1].tolist() == [0, 1]    # one ulp inside: level 5 only


def test_band_partition_invariant():
    """for any gamma, f and range the bands partition [0, inf): identical positions uploaded as
    every level are selected exactly once."""
    rng = np.random.default_rng(5)
    pos = rng.normal(0, 1, (400, 3)) * np.exp(rng.uniform(-3, 6, (400, 1)))
    for _ in range(40):
        L = int(rng.integers(1, 6))
        s_min = np.sort(np.exp(rng.uniform(-6, 0, L)))[::-1].copy()
        if rng.random() < 0.5:
            s_min[-1] = 0.0
        sc = _same_positions_scene(pos, list(range(1, L + 1)), s_min)
        a = int(rng.integers(1, L + 1)); b = int(rng.integers(a, L + 1))
        fr = sc.frame(camera(f=float(np.exp(rng.uniform(3, 8)))), a, b, float(np.exp(rng.uniform(-2, 3))),
                      ref_pos=rng.normal(0, 1, 3))
        m = fr.mask.reshape(L, -1).astype(int)
        assert (m[a - 1:b].sum(axis=0) == 1).all()
        assert m[:a - 1].sum() == 0 and m[b:].sum() == 0


def test_single_level_range_selects_whole_level():
    """L_start = L_end selects the entire level whatever gamma is; other levels are untouched."""
    rng = np.random.default_rng(6)
    pos = rng.normal(0, 30, (300, 3))
    sc = _same_positions_scene(pos, [1, 2, 3], [0.2, 0.05, 0.0])
    for l in (1, 2, 3):
        for gamma in (0.25, 1.0, 8.0):
            m = sc.frame(camera(), l, l, gamma).mask.reshape(3, -1)
            assert m[l - 1].all() and m.sum() == 300


def test_selection_distance_is_euclidean_to_reference():
    """R2/R3: d_G is the Euclidean distance to the camera centre c = -R^T t unless a reference is given."""
    rng = np.random.default_rng(8)
    Rm, _ = random_rotation(rng)
    eye = np.array([3.0, -2.0, 5.0])
    cam = camera(f=500.0, R=Rm, t=-Rm @ eye)
    d_edge = 0.1 * 500.0 / 2.0        # s_min f / gamma = 25
    dirs = rng.normal(size=(200, 3)); dirs /= np.linalg.norm(dirs, axis=1, keepdims=True)
    r = rng.uniform(5, 45, 200)
    r = r[np.abs(r - d_edge) > 1e-3]
    pos = eye + dirs[:len(r)] * r[:, None]
    sc = _same_positions_scene(pos, [1, 2], [0.1, 0.0])
    m = sc.frame(cam, 1, 2, 2.0).mask.reshape(2, -1)
    assert (m[0] == (r >= d_edge)).all() and (m[1] == (r < d_edge)).all()
    ref = np.array([-4.0, 1.0, 0.5])
    m = sc.frame(cam, 1, 2, 2.0, ref_pos=ref).mask.reshape(2, -1)
    dr = np.linalg.norm(pos.astype(np.float32).astype(np.float64) - ref, axis=1)
    ok = np.abs(dr - d_edge) > 1e-3
    assert (m[0][ok] == (dr >= d_edge)[ok]).all()


def test_paper_level_sanity_on_synthetic_scene():
    """selective {3,4,5} draws fewer Gaussians than level 5 alone; counts grow with level."""
    import flod_synth as fs
    g = GOLD["selective_fewer_gaussians"]
    assert g["selective_345"] < g["counts_per_level"][-1]
    assert sorted(g["counts_per_level"]) == g["counts_per_level"]
    sc = fs.make_scene(1, count_scale=0.01)
    assert [l.n for l in sc.levels] == sorted(l.n for l in sc.levels)
    osc = OracleScene(sc.levels, sc.sh_degree)
    cam = fs.make_poses(1)[0]
    n5 = osc.frame(cam, 5, 5, 1.0).counts["n_sel"]
    n345 = osc.frame(cam, 3, 5, 2.0).counts["n_sel"]
    assert n345 < n5


# ------------------------------------------------------------------------ projection (O2-O4)

def test_on_axis_projects_to_principal_point():
    """a Gaussian on the optical axis lands on (cx, cy)."""
    sc = OracleScene([level(1, 0.0, [[0, 0, 2.0], [0, 0, 7.5]], 0.1)], 0)
    fr = sc.frame(camera(width=40, height=30, f=123.0), 1, 1, 1.0)
    np.testing.assert_array_equal(fr.mu2d, [[20.0, 15.0], [20.0, 15.0]])
    np.testing.assert_array_equal(fr.depth, [2.0, 7.5])


def test_isotropic_on_axis_covariance_closed_form():
    """S:146 + R9: isotropic s at depth d on the axis has Sigma' = ((f s / d)^2 + 0.3) I."""
    f, s, d = 250.0, 0.05, 4.0
    sc = OracleScene([level(1, 0.0, [[0, 0, d]], s)], 0)
    fr = sc.frame(camera(f=f), 1, 1, 1.0)
    a, b, c = fr.cov2d[0]
    want = (f * s / d) ** 2 + 0.3
    assert a == pytest.approx(want, rel=1e-6) and c == pytest.approx(want, rel=1e-6) and abs(b) < 1e-6
    A, B, C = fr.conic[0]
    assert A == pytest.approx(1 / want, rel=1e-6) and C == pytest.approx(1 / want, rel=1e-6) and abs(B) < 1e-6


def test_near_plane_and_dead_culls():
    """z_cam <= near is absent; R11/R22: o < 1/255 is never drawn."""
    lv = level(1, 0.0, [[0, 0, 0.2], [0, 0, 0.1], [0, 0, -3.0], [0, 0, 1.0], [0, 0, 1.0]], 0.05,
               logit=[0, 0, 0, 0, -8.0])
    fr = OracleScene([lv], 0).frame(camera(z_near=0.2), 1, 1, 1.0)
    assert fr.state.tolist() == [oracle.ST_CULL_NEAR] * 3 + [oracle.ST_VISIBLE, oracle.ST_CULL_DEAD]
    assert fr.counts["n_vis"] == 1 and fr.counts["n_front"] == 2 and fr.counts["n_sel"] == 5


def _pinhole(p, cam):
    return np.array([cam.fx * p[0] / p[2] + cam.cx, cam.fy * p[1] / p[2] + cam.cy])


def test_ewa_covariance_matches_numerical_jacobian():
    """P:110 (Sigma' of the projected Gaussian): Sigma' - 0.3 I = J W Sigma W^T J^T with J the Jacobian
    of the pinhole map at mu, here obtained by central differences (independent of the analytic J)."""
    rng = np.random.default_rng(21)
    for _ in range(30):
        Rc, _ = random_rotation(rng)
        eye = rng.normal(0, 1, 3)
        cam = camera(width=200, height=160, f=180.0, R=Rc, t=-Rc @ eye)
        p_cam = np.array([rng.uniform(-0.4, 0.4), rng.uniform(-0.3, 0.3), 1.0]) * rng.uniform(1.0, 6.0)
        mu = Rc.T @ p_cam + eye
        s = np.exp(rng.uniform(-3.5, -1.5, 3))
        Rg, q = random_rotation(rng)
        fr = OracleScene([level(1, 0.0, [mu], [s], quat=[q])], 0).frame(cam, 1, 1, 1.0)
        mu32 = fr.scene and np.float32(mu).astype(np.float64)
        pc = cam.R.astype(np.float64) @ mu32 + cam.t.astype(np.float64)
        np.testing.assert_allclose(fr.mu2d[0], _pinhole(pc, cam), rtol=2e-6, atol=2e-4)
        h = 1e-5
        J = np.stack([(_pinhole(pc + h * e, cam) - _pinhole(pc - h * e, cam)) / (2 * h) for e in np.eye(3)], axis=1)
        Sigma = Rg @ np.diag(s * s) @ Rg.T
        want = J @ cam.R.astype(np.float64) @ Sigma @ cam.R.astype(np.float64).T @ J.T
        a, b, c = fr.cov2d[0].astype(np.float64)
        got = np.array([[a - 0.3, b], [b, c - 0.3]])
        np.testing.assert_allclose(got, want, rtol=2e-4, atol=2e-5 * np.abs(want).max())
        A, B, C = fr.conic[0].astype(np.float64)
        np.testing.assert_allclose(np.array([[A, B], [B, C]]) @ np.array([[a, b], [b, c]]), np.eye(2), atol=5e-4)


def test_projected_covariance_matches_sampled_points():
    """Eq. 2's Sigma': for a small Gaussian the covariance of pinhole-projected samples of
    N(mu, Sigma) equals Sigma' - 0.3 I to first order.  Catches a transposed R, M or quaternion matrix."""
    rng = np.random.default_rng(33)
    Rc, _ = random_rotation(rng)
    eye = np.array([0.5, -1.0, 2.0])
    cam = camera(width=300, height=200, f=400.0, R=Rc, t=-Rc @ eye)
    mu = Rc.T @ np.array([0.6, -0.35, 5.0]) + eye
    s = np.array([0.03, 0.008, 0.015])
    Rg, q = random_rotation(rng)
    fr = OracleScene([level(1, 0.0, [mu], [s], quat=[q])], 0).frame(cam, 1, 1, 1.0)
    pts = mu + (rng.normal(size=(400000, 3)) * s) @ Rg.T
    pc = pts @ cam.R.astype(np.float64).T + cam.t.astype(np.float64)
    uv = np.stack([cam.fx * pc[:, 0] / pc[:, 2] + cam.cx, cam.fy * pc[:, 1] / pc[:, 2] + cam.cy], axis=1)
    want = np.cov(uv.T)
    a, b, c = fr.cov2d[0].astype(np.float64)
    np.testing.assert_allclose([[a - 0.3, b], [b, c - 0.3]], want, rtol=0.02, atol=0.01 * np.abs(want).max())
    np.testing.assert_allclose(fr.mu2d[0], uv.mean(axis=0), atol=0.02)


def test_jacobian_clamp_only_beside_the_frustum():
    """R8: x/z, y/z are clamped to 1.3x the half-frustum tangent before J is formed; inside that, nothing changes;
    outside, the footprint stays bounded as if the Gaussian sat on the clamp."""
    f, W, H = 100.0, 64, 64
    lim = 1.3 * W / (2 * f)
    s, z = 0.05, 2.0
    sc = OracleScene([level(1, 0.0, [[0.9 * lim * z, 0, z], [3.0 * lim * z, 0, z]], s)], 0)
    fr = sc.frame(camera(width=W, height=H, f=f), 1, 1, 1.0)
    for g, u in ((0, 0.9 * lim), (1, lim)):
        J = np.array([[f / z, 0, -f * u / z], [0, f / z, 0]])
        want = J @ (s * s * np.eye(3)) @ J.T + 0.3 * np.eye(2)
        a, b, c = fr.cov2d[g]
        np.testing.assert_allclose([[a, b], [b, c]], want, rtol=1e-5, atol=1e-6)


def test_tile_rect_covers_the_threshold_contour():
    """R13: the rect is the padded box of the alpha = 1/255 ellipse, in 16x16 tiles, clamped to the grid."""
    rng = np.random.default_rng(44)
    cam = camera(width=200, height=120, f=150.0)
    n = 300
    pos = np.stack([rng.uniform(-3, 3, n), rng.uniform(-2, 2, n), rng.uniform(0.5, 6, n)], axis=1)
    lv = level(1, 0.0, pos, np.exp(rng.uniform(-4, -1, (n, 3))),
               quat=rng.normal(size=(n, 4)), opacity=rng.uniform(0.01, 0.99, n))
    sc = OracleScene([lv], 0)
    fr = sc.frame(cam, 1, 1, 1.0)
    TX, TY = fr.TX, fr.TY
    assert (TX, TY) == (13, 8)
    for g in np.nonzero(fr.state >= oracle.ST_EMPTY_RECT)[0]:
        a, b, c = fr.cov2d[g].astype(np.float64)
        kap = 2 * math.log(255 * float(sc.opacity[g]))
        hx, hy = math.sqrt(kap * a), math.sqrt(kap * c)       # exact half-widths of the contour's box
        mx, my = fr.mu2d[g].astype(np.float64)
        x0 = min(max(math.floor((mx - hx) / 16), 0), TX); x1 = min(max(math.floor((mx + hx) / 16) + 1, 0), TX)
        y0 = min(max(math.floor((my - hy) / 16), 0), TY); y1 = min(max(math.floor((my + hy) / 16) + 1, 0), TY)
        r = fr.rect[g]
        # the padded rect contains the exact one and exceeds it by at most one tile per side
        assert r[0] <= x0 and r[1] <= y0 and r[2] >= x1 and r[3] >= y1
        assert r[0] >= x0 - 1 and r[1] >= y0 - 1 and r[2] <= x1 + 1 and r[3] <= y1 + 1
        assert fr.n_tiles[g] == (r[2] - r[0]) * (r[3] - r[1])
        assert (fr.state[g] == oracle.ST_VISIBLE) == (fr.n_tiles[g] > 0)
    assert fr.counts["n_pairs"] == int(fr.n_tiles[fr.state == oracle.ST_VISIBLE].sum()) == int(fr.tile_counts.sum())


def _aniso_camera(rng=None, **kw):
    """fx != fy and a principal point off the image centre: every fy / cy / lim_y term of O2-O4 and R4's choice of fx
    are invisible to a camera with fx == fy, cx = W/2, cy = H/2 (a swap changes nothing there)."""
    d = dict(width=208, height=136, f=190.0, fy=127.0, cx=81.25, cy=90.5)
    d.update(kw)
    return camera(**d)


def test_anisotropic_camera_projection_and_covariance():
    """P:110, S:142-146 with fx != fy, cx != W/2, cy != H/2: on-axis point -> (cx, cy); mu' = (fx x/z + cx, fy y/z + cy);
    isotropic on-axis Sigma' = diag((fx s/d)^2, (fy s/d)^2) + 0.3 I; Sigma' against the numerical Jacobian."""
    cam = _aniso_camera()
    f, s, d = 250.0, 0.05, 4.0
    fr = OracleScene([level(1, 0.0, [[0, 0, d]], s)], 0).frame(cam, 1, 1, 1.0)
    np.testing.assert_array_equal(fr.mu2d[0], [np.float32(81.25), np.float32(90.5)])
    a, b, c = fr.cov2d[0]
    assert a == pytest.approx((cam.fx * s / d) ** 2 + 0.3, rel=1e-6) and c == pytest.approx((cam.fy * s / d) ** 2 + 0.3, rel=1e-6)
    assert abs(b) < 1e-6 and a > 1.5 * c
    rng = np.random.default_rng(211)
    for _ in range(30):
        Rc, _ = random_rotation(rng)
        eye = rng.normal(0, 1, 3)
        cam = _aniso_camera(R=Rc, t=-Rc @ eye, f=float(rng.uniform(100, 300)), fy=float(rng.uniform(100, 300)),
                            cx=float(rng.uniform(40, 160)), cy=float(rng.uniform(30, 100)))
        p_cam = np.array([rng.uniform(-0.3, 0.3), rng.uniform(-0.2, 0.2), 1.0]) * rng.uniform(1.0, 6.0)
        mu = Rc.T @ p_cam + eye
        sc3 = np.exp(rng.uniform(-3.5, -1.5, 3))
        Rg, q = random_rotation(rng)
        fr = OracleScene([level(1, 0.0, [mu], [sc3], quat=[q])], 0).frame(cam, 1, 1, 1.0)
        pc = cam.R.astype(np.float64) @ np.float32(mu).astype(np.float64) + cam.t.astype(np.float64)
        np.testing.assert_allclose(fr.mu2d[0], _pinhole(pc, cam), rtol=2e-6, atol=2e-4)
        h = 1e-5
        J = np.stack([(_pinhole(pc + h * e, cam) - _pinhole(pc - h * e, cam)) / (2 * h) for e in np.eye(3)], axis=1)
        want = J @ cam.R.astype(np.float64) @ (Rg @ np.diag(sc3 * sc3) @ Rg.T) @ cam.R.astype(np.float64).T @ J.T
        a, b, c = fr.cov2d[0].astype(np.float64)
        np.testing.assert_allclose([[a - 0.3, b], [b, c - 0.3]], want, rtol=2e-4, atol=2e-5 * np.abs(want).max())


def test_anisotropic_camera_jacobian_clamp_uses_its_own_axis():
    """R8 with fx != fy: x/z is clamped at 1.3 W / (2 fx), y/z at 1.3 H / (2 fy) -- each with its own focal length and
    image extent (a swapped pair of limits changes Sigma' of a Gaussian beside the frustum)."""
    cam = _aniso_camera(width=208, height=136, f=120.0, fy=210.0)
    limx, limy = 1.3 * cam.width / (2 * cam.fx), 1.3 * cam.height / (2 * cam.fy)
    assert abs(limx - limy) > 0.1
    s, z = 0.05, 2.0
    pos = [[3.0 * limx * z, 0, z], [0, 3.0 * limy * z, z], [0.9 * limx * z, 0.9 * limy * z, z]]
    fr = OracleScene([level(1, 0.0, pos, s)], 0).frame(cam, 1, 1, 1.0)
    for g, (u, v) in enumerate(((limx, 0.0), (0.0, limy), (0.9 * limx, 0.9 * limy))):
        J = np.array([[cam.fx / z, 0, -cam.fx * u / z], [0, cam.fy / z, -cam.fy * v / z]])
        want = J @ (s * s * np.eye(3)) @ J.T + 0.3 * np.eye(2)
        a, b, c = fr.cov2d[g]
        np.testing.assert_allclose([[a, b], [b, c]], want, rtol=1e-5, atol=1e-6)


def test_band_thresholds_use_fx_when_fx_differs_from_fy():
    """R4 (Eq. 7 "the focal length f"): f = fx.  fx = 1000, fy = 500, s_min = 0.05, gamma = 1 puts the
    edge at 50 (25 if fy were taken): a Gaussian at distance 40 belongs to the finer level, one at 60 to the coarser."""
    pos = np.array([[40.0, 0.0, 0.0], [60.0, 0.0, 0.0], [0.0, 24.0, 0.0], [0.0, 26.0, 0.0]])
    sc = _same_positions_scene(pos, [4, 5], [0.05, 0.0])
    fr = sc.frame(_aniso_camera(f=1000.0, fy=500.0), 4, 5, 1.0, ref_pos=[0.0, 0.0, 0.0])
    assert fr.mask.reshape(2, 4).tolist() == [[0, 1, 0, 0], [1, 0, 1, 1]]
    lo, hi = fr.thresholds()
    assert lo[0] == np.float32(2500.0)


def test_anisotropic_camera_tile_rect_and_footprint():
    """R13 / O4 with fx != fy and an off-centre principal point: the rect is still the padded box of the alpha = 1/255
    contour around mu' = (fx x/z + cx, fy y/z + cy); the blended pixels of one isotropic on-axis Gaussian are exactly
    those inside the axis-aligned ellipse with semi-axes sigma'_x,y sqrt(2 ln(255 o)) centred on (cx, cy)."""
    rng = np.random.default_rng(45)
    cam = _aniso_camera()
    n = 300
    pos = np.stack([rng.uniform(-3, 3, n), rng.uniform(-2, 2, n), rng.uniform(0.5, 6, n)], axis=1)
    lv = level(1, 0.0, pos, np.exp(rng.uniform(-4, -1, (n, 3))), quat=rng.normal(size=(n, 4)), opacity=rng.uniform(0.01, 0.99, n))
    sc = OracleScene([lv], 0)
    fr = sc.frame(cam, 1, 1, 1.0)
    TX, TY = fr.TX, fr.TY
    for g in np.nonzero(fr.state >= oracle.ST_EMPTY_RECT)[0]:
        a, b, c = fr.cov2d[g].astype(np.float64)
        kap = 2 * math.log(255 * float(sc.opacity[g]))
        hx, hy = math.sqrt(kap * a), math.sqrt(kap * c)
        pc = np.float32(pos[g]).astype(np.float64)
        mx, my = cam.fx * pc[0] / pc[2] + cam.cx, cam.fy * pc[1] / pc[2] + cam.cy     # from the definition, not from fr
        x0 = min(max(math.floor((mx - hx) / 16), 0), TX); x1 = min(max(math.floor((mx + hx) / 16) + 1, 0), TX)
        y0 = min(max(math.floor((my - hy) / 16), 0), TY); y1 = min(max(math.floor((my + hy) / 16) + 1, 0), TY)
        r = fr.rect[g]
        assert r[0] <= x0 and r[1] <= y0 and r[2] >= x1 and r[3] >= y1
        assert r[0] >= x0 - 1 and r[1] >= y0 - 1 and r[2] <= x1 + 1 and r[3] <= y1 + 1
    o, s, d = 0.8, 0.1, 2.0
    fr = OracleScene([level(1, 0.0, [[0, 0, d]], s, opacity=o, rgb=[1.0, 1.0, 1.0])], 0).frame(cam, 1, 1, 1.0)
    img, E, B, T = fr.composite(stats=True)
    sx2, sy2 = (cam.fx * s / d) ** 2 + 0.3, (cam.fy * s / d) ** 2 + 0.3
    jj, ii = np.mgrid[0:cam.height, 0:cam.width]
    q = 0.5 * ((ii + 0.5 - cam.cx) ** 2 / sx2 + (jj + 0.5 - cam.cy) ** 2 / sy2)
    alpha = np.minimum(0.99, float(np.float32(1 / (1 + math.exp(-math.log(o / (1 - o)))))) * np.exp(-q))
    inside = alpha >= SKIP_THR
    edge = np.abs(alpha - SKIP_THR) < 1e-6
    assert np.array_equal(B[~edge] > 0, inside[~edge]) and inside.sum() > 500
    np.testing.assert_allclose(img[0][inside & ~edge], alpha[inside & ~edge], rtol=2e-5)


# ------------------------------------------------------------------------- compositing (O7)

def test_empty_set_renders_background():
    """S:154."""
    lv = level(1, 0.0, np.zeros((0, 3)), 0.1)
    lv.quat = np.zeros((0, 4), np.float32)
    fr = OracleScene([lv], 0).frame(camera(width=20, height=10, bg=(0.25, 0.5, 0.75)), 1, 1, 1.0)
    img, E, B, T = fr.composite(stats=True)
    assert (img[0] == 0.25).all() and (img[1] == 0.5).all() and (img[2] == 0.75).all()
    assert E.sum() == 0 and (T == 1.0).all()


def test_two_layer_printed_example():
    """front red alpha 0.5 over back blue alpha 0.5 over black -> (0.5, 0, 0.25); also depth order
    does not depend on array order."""
    want = GOLD["two_layer_compositing"]["pixel"]
    for order in ((0, 1), (1, 0)):
        pos = np.array([[0, 0, 2.0], [0, 0, 3.0]])[list(order)]
        rgb = np.array([[1.0, 0, 0], [0, 0, 1.0]])[list(order)]
        fr = OracleScene([level(1, 0.0, pos, 0.2, opacity=0.5, rgb=rgb)], 0).frame(camera(33, 33, 100.0), 1, 1, 1.0)
        img = fr.composite()
        np.testing.assert_allclose(img[:, 16, 16], want, atol=1e-7)


def test_centre_pixel_alpha_is_min_o_099():
    """S:155, Eq. 2 at (x,y) = mu': alpha = min(o, 0.99); one opaque covering Gaussian gives 0.99 c + 0.01 bg."""
    bg = (0.2, 0.4, 0.6)
    for o_logit, a_want in ((0.0, 0.5), (20.0, 0.99), (math.log(0.3 / 0.7), 0.3)):
        fr = OracleScene([level(1, 0.0, [[0, 0, 2.0]], 0.3, logit=o_logit, rgb=[0.9, 0.1, 0.5])], 0).frame(
            camera(33, 33, 100.0, bg=bg), 1, 1, 1.0)
        img, E, B, T = fr.composite(stats=True)
        assert T[16, 16] == pytest.approx(1 - a_want, abs=1e-7)
        np.testing.assert_allclose(img[:, 16, 16], a_want * np.array([0.9, 0.1, 0.5]) + (1 - a_want) * np.array(bg), atol=1e-6)


def test_single_isotropic_gaussian_footprint_closed_form():
    """north_star's closed form (Eq. 2): alpha(i,j) = min(.99, o exp(-r^2 / 2 sigma'^2)) with
    sigma'^2 = (f s / d)^2 + 0.3; blended pixels are exactly those with alpha >= 1/255; their number tends to
    pi sigma'^2 2 ln(255 o) and the un-clamped sum of alpha to 2 pi sigma'^2 (o - 1/255)."""
    f, s, d, o = 200.0, 0.25, 5.0, 0.8
    W = H = 129
    col = np.array([0.7, 0.2, 0.9])
    fr = OracleScene([level(1, 0.0, [[0, 0, d]], s, opacity=o, rgb=col)], 0).frame(camera(W, H, f), 1, 1, 1.0)
    img, E, B, T = fr.composite(stats=True)
    o32 = float(np.float32(1 / (1 + math.exp(-math.log(o / (1 - o))))))
    sig2 = (f * s / d) ** 2 + 0.3
    jj, ii = np.mgrid[0:H, 0:W]
    r2 = (ii + 0.5 - W / 2) ** 2 + (jj + 0.5 - H / 2) ** 2
    alpha = np.minimum(0.99, o32 * np.exp(-r2 / (2 * sig2)))
    blended = alpha >= SKIP_THR
    margin = np.abs(alpha - SKIP_THR) < 1e-6
    assert ((B == 1) == blended)[~margin].all()
    want = np.where(blended, alpha, 0.0)
    np.testing.assert_allclose(img, col[:, None, None] * want[None], atol=2e-6)
    np.testing.assert_allclose(T, 1 - want, atol=2e-6)
    n_closed = math.pi * sig2 * 2 * math.log(255 * o32)
    assert B.sum() == pytest.approx(n_closed, rel=0.02)
    assert (1 - T).sum() == pytest.approx(2 * math.pi * sig2 * (o32 - 1 / 255), rel=0.02)
    # pixels outside the rect are never evaluated, pixels inside the contour always are
    assert (E[blended] == 1).all()


def _random_scene(rng, n, extent=1.5, two_levels=False):
    pos = np.stack([rng.uniform(-extent, extent, n), rng.uniform(-extent, extent, n), rng.uniform(0.3, 6.0, n)], axis=1)
    mk = lambda lid, smin, sl: level(lid, smin, pos[sl], np.exp(rng.uniform(-4.0, -1.0, (len(pos[sl]), 3))),
                                     quat=rng.normal(size=(len(pos[sl]), 4)), logit=rng.normal(0, 2.0, len(pos[sl])),
                                     rgb=rng.uniform(0, 1, (len(pos[sl]), 3)))
    if two_levels:
        h = n // 3
        return [mk(1, 0.02, slice(0, h)), mk(2, 0.0, slice(h, n))]
    return [mk(1, 0.0, slice(0, n))]


def test_tiled_equals_brute_force_bit_exactly():
    """S:171/S:177/S:584 and north_star's brute-force check: per pixel, compositing ALL surviving Gaussians in
    global (depth, gid) order equals compositing the tile's list.  Equality also proves the footprint rule R13
    conservative (no alpha >= 1/255 outside a rect)."""
    rng = np.random.default_rng(2024)
    for k in range(24):
        n = int(rng.integers(1, 600))
        two = bool(k % 2)
        lv = _random_scene(rng, n, two_levels=two)
        cam = camera(width=int(rng.integers(17, 90)), height=int(rng.integers(17, 70)), f=float(rng.uniform(40, 160)),
                     bg=tuple(rng.uniform(0, 1, 3)))
        fr = OracleScene(lv, 0).frame(cam, 1, 2 if two else 1, 1.0)
        t_img, tE, tB, tT = fr.composite(stats=True)
        b_img, bE, bB, bT = fr.composite(brute=True, stats=True)
        assert np.array_equal(t_img, b_img) and np.array_equal(tB, bB) and np.array_equal(tT, bT)
        assert (tE <= bE).all()


# ------------------------------------------------------------------------ pair rule 2 "ellipse" (R26)

def _needle_and_blob_scene(rng, n):
    """Footprints of every shape: blobs, large discs, needles at the dilation floor in every orientation, high and
    barely-alive opacities (kappa from 0.05 to 11)."""
    pos = np.stack([rng.uniform(-2, 2, n), rng.uniform(-1.5, 1.5, n), rng.uniform(0.4, 7.0, n)], axis=1)
    scale = np.exp(rng.uniform(-4.5, -0.5, (n, 3)))
    thin = rng.random(n) < 0.4
    scale[thin, 1:] = 1e-4
    scale[thin, 0] = np.exp(rng.uniform(-1.5, 1.0, thin.sum()))
    logit = np.where(rng.random(n) < 0.2, rng.uniform(-5.5, -5.0, n), rng.normal(0, 2.5, n))
    return [level(1, 0.0, pos, scale, quat=rng.normal(size=(n, 4)), logit=logit, rgb=rng.uniform(0, 1, (n, 3)))]


def test_ellipse_pair_rule_tiled_equals_brute_force_bit_exactly():
    """R26 keeps what R13 had to deliver (S:171 / S:177): with pair rule 2 the tiled image still equals per-pixel
    compositing over ALL Gaussians bit for bit -- no pixel with alpha >= 1/255 lies in a tile that was dropped."""
    rng = np.random.default_rng(2026)
    for k in range(30):
        n = int(rng.integers(1, 500))
        lv = _needle_and_blob_scene(rng, n) if k % 3 else _random_scene(rng, n)
        cam = camera(width=int(rng.integers(17, 150)), height=int(rng.integers(17, 110)), f=float(rng.uniform(40, 260)),
                     fy=float(rng.uniform(40, 260)), cx=float(rng.uniform(10, 90)), cy=float(rng.uniform(10, 60)),
                     bg=tuple(rng.uniform(0, 1, 3)))
        sc = OracleScene(lv, 0)
        f1, f2 = sc.frame(cam, 1, 1, 1.0), sc.frame(cam, 1, 1, 1.0, pair_rule=2)
        t_img, tE, tB, tT = f2.composite(stats=True)
        b_img, bE, bB, bT = f2.composite(brute=True, stats=True)
        assert np.array_equal(t_img, b_img) and np.array_equal(tB, bB) and np.array_equal(tT, bT)
        assert np.array_equal(t_img, f1.composite())
        # rule 2 only ever drops tiles of rule 1's rect; everything else of the frame is the same
        assert (f2.tile_counts <= f1.tile_counts).all() and (f2.n_tiles <= f1.n_tiles).all()
        assert np.array_equal(f1.rect, f2.rect) and np.array_equal(f1.state, f2.state) and f1.counts["n_vis"] == f2.counts["n_vis"]
        assert (tE <= f1.composite(stats=True)[1]).all()


def test_ellipse_pair_rule_lists_exactly_the_tiles_the_contour_reaches():
    """R26 against the definition, tile by tile (numpy, fp64, from the oracle's mu', conic and opacity): a tile is
    listed if one of its pixel centres has alpha >= 1/255 (conservative) and only if the contour grown by the pads
    reaches the box of its pixel centres (tight: the minimum of the quadratic form over that box, found by dense
    sampling of its border, is within the padded level) -- needles included."""
    rng = np.random.default_rng(909)
    cam = camera(width=208, height=136, f=150.0, fy=210.0, cx=99.0, cy=70.5)
    lv = _needle_and_blob_scene(rng, 260)
    sc = OracleScene(lv, 0)
    fr = sc.frame(cam, 1, 1, 1.0, pair_rule=2)
    tile, _, gid = fr.sorted_pairs()
    listed = {}
    for t, g in zip(tile, gid):
        listed.setdefault(int(g), set()).add(int(t))
    jj, ii = np.mgrid[0:fr.TY * 16, 0:fr.TX * 16]
    n_loose = n_listed = 0
    for g in np.nonzero(fr.state == oracle.ST_VISIBLE)[0]:
        A, B, C = fr.conic[g].astype(np.float64)
        mx, my = fr.mu2d[g].astype(np.float64)
        o = float(sc.opacity[g])
        dx, dy = mx - (ii + 0.5), my - (jj + 0.5)
        q = np.maximum(0.0, 0.5 * (A * dx * dx + C * dy * dy) + B * dx * dy)
        hit = np.minimum(0.99, o * np.exp(-q)) >= SKIP_THR
        r = fr.rect[g]
        must = {int(ty * fr.TX + tx) for ty in range(r[1], r[3]) for tx in range(r[0], r[2])
                if hit[16 * ty:16 * ty + 16, 16 * tx:16 * tx + 16].any()}
        got = listed.get(int(g), set())
        assert must <= got, f"gaussian {g}: tiles {sorted(must - got)} hold a blended pixel but are not listed"
        assert got <= {int(ty * fr.TX + tx) for ty in range(r[1], r[3]) for tx in range(r[0], r[2])}
        # tightness: min of the form over the pixel-centre box of every listed tile (dense border + centre clamp) is within
        # the padded level: E (1 + 2^-9) + 2^-16, ends moved by 2^-8 sqrt(K/A) + 2^-6 px + 2^-20 of the summed magnitudes
        # (|grad Q| <= 2 sqrt(K lambda_max))
        K0 = 2.0 * math.log(o / SKIP_THR)
        pad = math.sqrt(K0 / A) / 256 + 2.0 ** -6 + 2.0 ** -19 * (abs(mx) + 2 * abs(B / A) * (abs(my) + 16 * fr.TY))
        K = K0 * (1 + 2.0 ** -8) + 2.0 ** -14 + 2.0 * math.sqrt(K0 * (A + C)) * 2 * pad + (A + C) * (2 * pad) ** 2
        for t in got:
            ty, tx = divmod(t, fr.TX)
            xs = np.linspace(16 * tx + 0.5, 16 * tx + 15.5, 241); ys = np.linspace(16 * ty + 0.5, 16 * ty + 15.5, 241)
            bx = np.concatenate([xs, xs, np.full(241, xs[0]), np.full(241, xs[-1]), [min(max(mx, xs[0]), xs[-1])]])
            by = np.concatenate([np.full(241, ys[0]), np.full(241, ys[-1]), ys, ys, [min(max(my, ys[0]), ys[-1])]])
            qq = A * (mx - bx) ** 2 + C * (my - by) ** 2 + 2 * B * (mx - bx) * (my - by)
            n_listed += 1
            n_loose += int(qq.min() > K)
    assert n_listed > 1500 and n_loose == 0, (n_loose, n_listed)


def test_ellipse_pair_rule_closed_form_disc():
    """One isotropic Gaussian on the optical axis: the contour is the circle r = sigma' sqrt(2 ln(255 o)) around
    (cx, cy); the listed tiles are exactly those whose pixel-centre box lies within r of the centre (tiles at the
    corners of the rect are dropped: the count approaches pi/4 of the rect for large discs)."""
    f, s, d, o = 300.0, 0.25, 2.0, 0.9
    cam = camera(width=400, height=400, f=f)
    sc = OracleScene([level(1, 0.0, [[0, 0, d]], s, opacity=o)], 0)
    f1, f2 = sc.frame(cam, 1, 1, 1.0), sc.frame(cam, 1, 1, 1.0, pair_rule=2)
    o32 = float(sc.opacity[0])
    rad = math.sqrt(((f * s / d) ** 2 + 0.3) * 2 * math.log(255 * o32))
    want = np.zeros(f2.TX * f2.TY, np.uint32)
    for ty in range(f2.TY):
        for tx in range(f2.TX):
            nx = min(max(200.0, 16 * tx + 0.5), 16 * tx + 15.5); ny = min(max(200.0, 16 * ty + 0.5), 16 * ty + 15.5)
            dist = math.hypot(nx - 200.0, ny - 200.0)
            assert abs(dist - rad) > 0.05          # no tile sits on the decision edge in this construction
            want[ty * f2.TX + tx] = dist <= rad
    assert np.array_equal(f2.tile_counts, want)
    assert 0.7 < want.sum() / f1.counts["n_pairs"] < 0.86 and f1.counts["n_pairs"] > 250


def test_brute_force_in_numpy_on_tiny_input():
    """Independent restatement of P:104-111 in vectorised numpy: every pixel, every Gaussian, global depth order,
    from the oracle's projected (mu', conic) and colours.  Different code, same definition."""
    rng = np.random.default_rng(77)
    lv = _random_scene(rng, 120)
    cam = camera(width=40, height=24, f=60.0, bg=(0.1, 0.2, 0.3))
    sc = OracleScene(lv, 0)
    fr = sc.frame(cam, 1, 1, 1.0)
    ids = np.nonzero(fr.state >= oracle.ST_EMPTY_RECT)[0]
    ids = ids[np.lexsort((ids, fr.depth[ids]))]
    jj, ii = np.mgrid[0:cam.height, 0:cam.width]
    T = np.ones((cam.height, cam.width)); Cacc = np.zeros((3, cam.height, cam.width))
    alive = np.ones_like(T, dtype=bool)
    for g in ids:
        dx = float(fr.mu2d[g, 0]) - (ii + 0.5); dy = float(fr.mu2d[g, 1]) - (jj + 0.5)
        A, B, Cc = map(float, fr.conic[g])
        q = np.maximum(0.0, 0.5 * (A * dx * dx + Cc * dy * dy) + B * dx * dy)
        al = np.minimum(0.99, float(sc.opacity[g]) * np.exp(-q))
        use = alive & (al >= SKIP_THR)
        Cacc += np.where(use, T * al, 0.0)[None] * fr.rgb[g][:, None, None]
        T = np.where(use, T * (1 - al), T)
        alive &= ~(use & (T < STOP_THR))
    want = Cacc + T[None] * np.array(cam.bg)[:, None, None]
    np.testing.assert_allclose(fr.composite(), want, atol=1e-12)


def test_transmittance_and_alpha_invariants():
    """S:176 + R11: T is non-increasing in [0,1], every blended alpha lies in [1/255, 0.99], outputs finite."""
    rng = np.random.default_rng(91)
    lv = _random_scene(rng, 800, extent=1.0)
    cam = camera(width=48, height=48, f=70.0)
    fr = OracleScene(lv, 0).frame(cam, 1, 1, 1.0)
    img, E, B, T = fr.composite(stats=True)
    assert np.isfinite(img).all() and (T >= 0).all() and (T <= 1).all() and (img >= 0).all()
    seen = 0
    for (i, j) in rng.integers(0, 48, (60, 2)):
        al, Tb = fr.trace_pixel(int(i), int(j))
        assert len(al) == B[j, i]
        if len(al):
            seen += 1
            assert (al >= SKIP_THR).all() and (al <= 0.99).all()
            assert (np.diff(Tb) <= 0).all() and Tb[0] == 1.0 and (Tb > 0).all()
            assert T[j, i] == pytest.approx(Tb[-1] * (1 - al[-1]), rel=1e-12)
            assert (Tb >= STOP_THR).all(), "no blend happens after T fell below the stop threshold (R12)"
    assert seen > 30


def test_termination_is_a_small_perturbation():
    """R12: blend-then-stop makes early termination a <= 1e-4 * max colour change of the un-terminated result."""
    rng = np.random.default_rng(92)
    lv = _random_scene(rng, 1500, extent=0.8)
    for l in lv:
        l.opacity_logit[:] = np.abs(l.opacity_logit) + 1.0
    cam = camera(width=40, height=40, f=60.0, bg=(1.0, 1.0, 1.0))
    fr = OracleScene(lv, 0).frame(cam, 1, 1, 1.0)
    with_stop, E1, _, T1 = fr.composite(stats=True)
    no_stop, E0, _, T0 = fr.composite(stop_thr=-1.0, stats=True)
    assert (T1 < STOP_THR).mean() > 0.3, "scene must actually terminate"
    assert (E1 <= E0).all() and (E1 < E0).any()
    assert np.abs(with_stop - no_stop).max() <= 1.0001e-4


def test_permutation_invariance():
    """permuting the Gaussians within a level leaves the image unchanged when no two depths tie."""
    rng = np.random.default_rng(93)
    lv = _random_scene(rng, 400)[0]
    cam = camera(width=50, height=40, f=80.0)
    img = OracleScene([lv], 0).frame(cam, 1, 1, 1.0).composite()
    perm = rng.permutation(400)
    from types import SimpleNamespace
    lp = SimpleNamespace(level=1, s_min=lv.s_min, mean=lv.mean[perm], log_scale=lv.log_scale[perm], quat=lv.quat[perm],
                         opacity_logit=lv.opacity_logit[perm], sh=lv.sh[perm])
    fr = OracleScene([lp], 0).frame(cam, 1, 1, 1.0)
    assert len(np.unique(fr.depth[fr.state >= oracle.ST_EMPTY_RECT])) == (fr.state >= oracle.ST_EMPTY_RECT).sum()
    assert np.array_equal(img, fr.composite())


def test_depth_ties_break_by_gid():
    """R15 / S:151: equal depths composite in ascending global id."""
    pos = [[0, 0, 2.0], [0, 0, 2.0]]
    rgb = [[1.0, 0, 0], [0, 0, 1.0]]
    fr = OracleScene([level(1, 0.0, pos, 0.2, opacity=0.5, rgb=rgb)], 0).frame(camera(33, 33, 100.0), 1, 1, 1.0)
    for brute in (False, True):
        np.testing.assert_allclose(fr.composite(brute=brute)[:, 16, 16], [0.5, 0.0, 0.25], atol=1e-7)
    # same tie across two levels: gid is level-major
    a = level(1, 0.1, [pos[0]], 0.2, opacity=0.5, rgb=[rgb[1]])
    b = level(2, 0.0, [pos[1]], 0.2, opacity=0.5, rgb=[rgb[0]])
    fr = OracleScene([a, b], 0).frame(camera(33, 33, 100.0), 1, 2, 1.0, ref_pos=[0, 0, 2.0])
    assert fr.mask.tolist() == [0, 1]
    lo = [level(1, 0.1, [pos[0]], 0.2, opacity=0.5, rgb=[rgb[1]]), level(2, 0.05, [pos[1]], 0.2, opacity=0.5, rgb=[rgb[0]])]
    same = OracleScene([level(1, 0.0, pos, 0.2, opacity=0.5, rgb=[rgb[1], rgb[0]])], 0).frame(camera(33, 33, 100.0), 1, 1, 1.0)
    np.testing.assert_allclose(same.composite()[:, 16, 16], [0.25, 0.0, 0.5], atol=1e-7)


def test_pair_sequence_equals_one_global_sort_of_all_pairs():
    """O6 / R15: the oracle's per-tile lists, tile after tile, are the unique sequence that sorting ALL
    (tile, depth, gid) triples with a library sort gives (numpy lexsort over the pairs expanded from the rects here)."""
    import flod_synth as fs
    sc = fs.make_scene(1, count_scale=0.01)
    cam = fs.make_poses(1, 320, 208)[7]
    fr = OracleScene(sc.levels, sc.sh_degree).frame(cam, 3, 5, 2.0)
    vis = np.nonzero(fr.state == oracle.ST_VISIBLE)[0]
    rect, depth = fr.rect[vis], fr.depth[vis]
    tiles, deps, gids = [], [], []
    for g, r, d in zip(vis, rect, depth):
        ty, tx = np.mgrid[r[1]:r[3], r[0]:r[2]]
        t = (ty * fr.TX + tx).ravel()
        tiles.append(t); deps.append(np.full(t.size, d, np.float32)); gids.append(np.full(t.size, g, np.uint32))
    tiles, deps, gids = np.concatenate(tiles).astype(np.uint32), np.concatenate(deps), np.concatenate(gids)
    order = np.lexsort((gids, deps, tiles))
    tile, dep, gid = fr.sorted_pairs()
    assert tile.size == fr.counts["n_pairs"] > 10000
    assert np.array_equal(tile, tiles[order]) and np.array_equal(dep, deps[order]) and np.array_equal(gid, gids[order])
    assert np.array_equal(fr.tile_counts, np.bincount(tiles, minlength=fr.TX * fr.TY).astype(np.uint32))


def test_rigid_motion_invariance():
    """Moving scene and camera together changes nothing beyond rounding."""
    rng = np.random.default_rng(94)
    lv = _random_scene(rng, 300)[0]
    cam = camera(width=48, height=48, f=70.0)
    img = OracleScene([lv], 0).frame(cam, 1, 1, 1.0).composite()
    Rw, qw = random_rotation(rng)
    tw = np.array([3.0, -1.0, 0.5])
    from types import SimpleNamespace

    def qmul(a, b):
        w1, x1, y1, z1 = a; w2, x2, y2, z2 = b.T
        return np.stack([w1 * w2 - x1 * x2 - y1 * y2 - z1 * z2, w1 * x2 + x1 * w2 + y1 * z2 - z1 * y2,
                         w1 * y2 - x1 * z2 + y1 * w2 + z1 * x2, w1 * z2 + x1 * y2 - y1 * x2 + z1 * w2], axis=1)
    moved = SimpleNamespace(level=1, s_min=0.0, mean=(lv.mean.astype(np.float64) @ Rw.T + tw).astype(np.float32),
                            log_scale=lv.log_scale, quat=qmul(qw, lv.quat.astype(np.float64)).astype(np.float32),
                            opacity_logit=lv.opacity_logit, sh=lv.sh)
    cam2 = camera(width=48, height=48, f=70.0, R=Rw.T, t=-(Rw.T @ tw))
    img2 = OracleScene([moved], 0).frame(cam2, 1, 1, 1.0).composite()
    d = np.abs(img - img2)
    assert d.mean() < 2e-5 and np.quantile(d, 0.999) < 1e-3


# --------------------------------------------------------------------------------- SH (O5)

def test_sh_basis_is_orthonormal_by_quadrature():
    """R16: the 16 basis functions are orthonormal on the sphere (Gauss-Legendre in cos(theta), uniform in phi).
    Pins every normalisation constant and polynomial; the sign convention stays unpinned."""
    xs, ws = np.polynomial.legendre.leggauss(24)
    phis = (np.arange(48) + 0.5) * (2 * math.pi / 48)
    G = np.zeros((16, 16))
    for ct, w in zip(xs, ws):
        st = math.sqrt(1 - ct * ct)
        for ph in phis:
            Y = oracle.sh_basis(3, [st * math.cos(ph), st * math.sin(ph), ct])
            G += w * (2 * math.pi / 48) * np.outer(Y, Y)
    np.testing.assert_allclose(G, np.eye(16), atol=1e-10)


def test_sh_degree0_colour_and_view_dependence():
    """R16/R17: degree-0 colour = 0.5 + Y0 dc, clamped at 0; higher bands use the direction from the TRUE camera centre."""
    fr = OracleScene([level(1, 0.0, [[0, 0, 2.0], [0.3, 0.1, 3.0]], 0.1, rgb=[[0.2, 0.6, 1.0], [-0.5, 0.5, 2.0]])], 0).frame(
        camera(), 1, 1, 1.0)
    np.testing.assert_allclose(fr.rgb, [[0.2, 0.6, 1.0], [0.0, 0.5, 2.0]], atol=1e-7)
    rng = np.random.default_rng(3)
    sh = rng.normal(0, 0.3, (1, 16, 3))
    eye = np.array([1.0, 0.5, -1.0])
    Rc, _ = random_rotation(rng)
    mu = Rc.T @ np.array([0.4, -0.2, 3.0]) + eye
    cam = camera(f=80.0, R=Rc, t=-Rc @ eye)
    fr = OracleScene([level(1, 0.0, [mu], 0.05, sh=sh)], 3).frame(cam, 1, 1, 1.0, ref_pos=[9.0, 9.0, 9.0])
    d = np.float32(mu).astype(np.float64) - fr.centre.astype(np.float64)
    d /= np.linalg.norm(d)
    Y = oracle.sh_basis(3, d)
    want = np.maximum(0.0, 0.5 + np.einsum("k,kc->c", Y, sh[0].astype(np.float32).astype(np.float64)))
    got = fr.rgb[0] if fr.state[0] >= oracle.ST_EMPTY_RECT else None
    assert got is not None
    np.testing.assert_allclose(got, want, atol=1e-12)
    np.testing.assert_allclose(fr.centre, eye, atol=1e-6)
    # low-order bands against their textbook Cartesian forms: Y1 ~ (-y, z, -x), Y2[2] ~ 2z^2 - x^2 - y^2
    assert Y[1] == pytest.approx(-math.sqrt(3 / (4 * math.pi)) * d[1])
    assert Y[6] == pytest.approx(0.25 * math.sqrt(5 / math.pi) * (3 * d[2] ** 2 - 1))


def test_sh_basis_equals_library_spherical_harmonics():
    """R16 against a library routine: the 16 basis functions are the real combinations of scipy's complex spherical
    harmonics Y_l^m (which carry the Condon-Shortley phase): sqrt(2) Im Y_l^|m| for m < 0, Y_l^0, sqrt(2) Re Y_l^m for
    m > 0, in the order (l, m = -l..l).  This pins every sign of R16 to that stated definition (which sign convention a
    trained model uses stays a convention)."""
    from scipy.special import sph_harm_y
    rng = np.random.default_rng(11)
    for _ in range(50):
        d = rng.normal(size=3)
        d /= np.linalg.norm(d)
        theta, phi = math.acos(d[2]), math.atan2(d[1], d[0])            # polar angle from +z, azimuth from +x
        want = []
        for l in range(4):
            for m in range(-l, l + 1):
                y = complex(sph_harm_y(l, abs(m), theta, phi))
                want.append(math.sqrt(2) * y.imag if m < 0 else (y.real if m == 0 else math.sqrt(2) * y.real))
        np.testing.assert_allclose(oracle.sh_basis(3, d), want, atol=1e-12)


# ------------------------------------------------------------------------ variant O64

def test_fp32_pipeline_sits_on_the_fp64_result():
    """O32 (canonical fp32 geometry, the parity target) against O64 (every step in fp64, nothing rounded on the way) on
    config 0: same masks and cull states, O64's exact rect never sticks out of O32's padded one (the pad covers the fp32
    rounding: R13's conservativeness does not rest on fp32 luck), images within 1e-5 -- two orders below north_star's
    1e-3, so the tolerance is spent on the kernel's fp32 compositing, not on the geometry's precision."""
    import flod_synth as fs
    sc = fs.make_scene(0)
    cam = fs.make_poses(0)[0]
    osc = OracleScene(sc.levels, sc.sh_degree)
    for (ls, le) in ((2, 2), (1, 2)):
        a, b = osc.frame(cam, ls, le, 1.0), osc.frame(cam, ls, le, 1.0, fp64=True)
        assert np.array_equal(a.mask, b.mask) and np.array_equal(a.state, b.state)
        vis = a.state == oracle.ST_VISIBLE
        ra, rb = a.rect[vis], b.rect[vis]
        assert (rb[:, :2] >= ra[:, :2]).all() and (rb[:, 2:] <= ra[:, 2:]).all()
        assert (ra != rb).any(axis=1).mean() < 0.02            # the pad costs under 2 % of the rects one more tile row/column
        np.testing.assert_allclose(a.mu2d[vis], b.mu2d[vis], rtol=1e-5, atol=1e-4)
        np.testing.assert_allclose(a.conic[vis], b.conic[vis], rtol=2e-4, atol=1e-7)
        assert np.abs(a.composite() - b.composite()).max() < 1e-5
