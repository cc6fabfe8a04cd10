"""The rasterizer's backward pass (Alg. 1): pins of the oracle (CPU), then the CUDA
kernels against the oracle (GPU, through the C ABI)."""
import numpy as np
import pytest
import torch

import oracle
from helpers import camera, level
from oracle import OracleScene
from oracle import backward as ob


def _scene(rng, n=(6, 9), sh_degree=1, extent=0.8):
    out = []
    K = (sh_degree + 1) ** 2
    for i, m in enumerate(n):
        pos = np.stack([rng.uniform(-extent, extent, m), rng.uniform(-extent, extent, m), rng.uniform(1.5, 4.0, m)], axis=1)
        sh = rng.normal(0, 0.3, (m, K, 3)); sh[:, 0, :] += 0.6
        out.append(level(i + 1, (0.05, 0.0)[i] if len(n) == 2 else 0.0, pos, np.exp(rng.uniform(-2.6, -1.2, (m, 3))),
                         quat=rng.normal(size=(m, 4)), logit=rng.normal(0.5, 1.5, m), sh=sh))
    return out


# ------------------------------------------------------------------------------------ pins of the oracle (CPU)

def test_differentiable_forward_equals_the_c_oracle_image():
    """The restated forward (fp64, PyTorch) draws the image of oracle/flod_oracle.c's brute-force compositing: same
    definition, other code (their geometry differs by fp32 rounding only)."""
    rng = np.random.default_rng(3)
    for deg in (0, 2, 3):
        lv = _scene(rng, (40, 60), sh_degree=deg)
        cam = camera(width=40, height=28, f=55.0, fy=47.0, cx=18.5, cy=15.25, bg=(0.2, 0.3, 0.1))
        fr = OracleScene(lv, deg).frame(cam, 1, 2, 1.0)
        ids, order = ob.frame_selection(fr)
        img = ob.forward(ob.scene_params(lv, False), cam, deg, torch.as_tensor(ids), order).numpy()
        ref = fr.composite(brute=True)
        d = np.abs(img - ref)
        assert np.quantile(d, 0.99) < 2e-5 and d.max() < 5e-3      # (a 1/255-marginal pixel may differ by one skipped term)


def test_gradients_match_central_finite_differences():
    """S:161 / S:586: analytic gradient vs central finite differences (fp64) for every parameter: relative error < 1e-3
    (mean, scale, rotation), < 1e-5 (colour, opacity)."""
    rng = np.random.default_rng(11)
    for trial in range(4):
        lv = _scene(rng, (5, 6), sh_degree=trial % 3 + 1)
        deg = trial % 3 + 1
        cam = camera(width=16, height=16, f=22.0, fy=19.0, cx=7.5, cy=8.25, bg=(0.1, 0.2, 0.3))
        fr = OracleScene(lv, deg).frame(cam, 1, 2, 1.0)
        ids, order = ob.frame_selection(fr)
        up = rng.normal(size=(3, 16, 16))
        grads, _ = ob.backward(lv, deg, cam, fr, up)
        base = ob.scene_params(lv, False)
        upt = torch.as_tensor(up)
        f = lambda prm: float((ob.forward(prm, cam, deg, torch.as_tensor(ids), order) * upt).sum())
        for name, h, tol in (("mean", 1e-6, 1e-3), ("log_scale", 1e-6, 1e-3), ("quat", 1e-6, 1e-3), ("logit", 1e-6, 1e-5), ("sh", 1e-6, 1e-5)):
            g = grads["logit" if name == "logit" else name]
            flat = base[name].reshape(-1)
            scale = np.abs(g).max() + 1e-12
            for idx in rng.choice(flat.numel(), size=min(12, flat.numel()), replace=False):
                keep = float(flat[idx])
                flat[idx] = keep + h; fp = f(base)
                flat[idx] = keep - h; fm = f(base)
                flat[idx] = keep
                fd = (fp - fm) / (2 * h)
                assert abs(fd - g.reshape(-1)[idx]) <= tol * scale + 1e-9, (name, idx, fd, g.reshape(-1)[idx])


def test_zero_upstream_and_dead_gaussians():
    """upstream 0 -> every gradient exactly 0; logit = -20 -> colour gradient below 1e-7."""
    rng = np.random.default_rng(2)
    lv = _scene(rng, (8,), sh_degree=0)
    lv[0].opacity_logit[3] = -5.0                       # alive (o = 0.0067 > 1/255) but faint
    cam = camera(width=16, height=16, f=22.0)
    fr = OracleScene(lv, 0).frame(cam, 1, 1, 1.0)
    g0, _ = ob.backward(lv, 0, cam, fr, np.zeros((3, 16, 16)))
    assert all((v == 0).all() for v in g0.values())
    g1, _ = ob.backward(lv, 0, cam, fr, np.ones((3, 16, 16)))
    assert np.abs(g1["sh"]).max() > 1e-3
    lv[0].opacity_logit[3] = -20.0                      # dead: culled, no gradient at all
    fr = OracleScene(lv, 0).frame(cam, 1, 1, 1.0)
    g2, _ = ob.backward(lv, 0, cam, fr, np.ones((3, 16, 16)))
    assert np.abs(g2["sh"][3]).max() < 1e-7 and np.abs(g2["mean"][3]).max() == 0.0


# ------------------------------------------------------------------------------------ the CUDA kernels (GPU)

def _gpu_vs_oracle(lv, deg, cam, ls, le, gamma, up, tol=1e-4):
    from paper_2408_12894_b200 import build
    build.build()
    import paper_2408_12894_b200 as pkg
    r = pkg.Renderer(0)
    r.upload_levels(lv, deg)
    r.set_workspace(cam.width, cam.height, 1 << 22)
    r.set_options(pkg.FLOD_OPT_FULL_SORT)             # the backward pass walks the lists of the forward pass: all of them in order
    img = r.render(cam, ls, le, gamma).cpu().numpy()
    got = {k: v.cpu().numpy() for k, v in r.render_backward(cam, torch.from_numpy(up.astype(np.float32)).cuda(), deg).items()}
    fr = OracleScene(lv, deg).frame(cam, ls, le, gamma, pair_rule=r.pair_rule)
    want, ref_img = ob.backward(lv, deg, cam, fr, up)
    assert np.abs(img - ref_img).max() < 5e-3
    worst = {}
    for k in ("mean", "log_scale", "quat", "logit", "sh"):
        scale = np.abs(want[k]).max()
        err = np.abs(got[k] - want[k]).max()
        worst[k] = err / (scale + 1e-30)
        assert err <= tol * scale + 1e-7, (k, err, scale)
    # Gaussians the frame does not draw have zero gradients on both sides
    drawn = fr.state >= oracle.ST_EMPTY_RECT
    assert all((got[k][~drawn] == 0).all() for k in got)
    r.close()
    return worst, got, want


@pytest.mark.gpu
@pytest.mark.parametrize("seed,deg", [(0, 0), (1, 1), (2, 2), (3, 3), (4, 3), (5, 1)])
def test_kernel_gradients_match_the_oracle(seed, deg):
    """Every parameter's gradient within 1e-4 of the array's largest gradient (fp32 kernels, sums in atomic order, against
    the fp64 oracle), on scenes that span several tiles, ragged images, off-centre anisotropic cameras, both level modes."""
    rng = np.random.default_rng(100 + seed)
    lv = _scene(rng, (60, 90), sh_degree=deg, extent=1.2)
    cam = camera(width=int(rng.integers(30, 70)), height=int(rng.integers(30, 60)), f=float(rng.uniform(25, 60)), fy=float(rng.uniform(25, 60)),
                 cx=float(rng.uniform(15, 30)), cy=float(rng.uniform(15, 30)), bg=tuple(rng.uniform(0, 1, 3)))
    up = rng.normal(size=(3, cam.height, cam.width))
    worst, _, _ = _gpu_vs_oracle(lv, deg, cam, 1, 2, 1.0, up)
    print("single frame, levels {1,2}:", {k: f"{v:.1e}" for k, v in worst.items()})
    _gpu_vs_oracle(lv, deg, cam, 2, 2, 1.0, up)


@pytest.mark.gpu
def test_kernel_saturated_pixels_clamps_and_early_stop():
    """Opaque, large, overlapping Gaussians: alpha clamped at 0.99 (zero slope there), pixels that stop early (entries
    behind the stop get nothing), a Gaussian beside the frustum (R8's clamp), a non-zero background."""
    rng = np.random.default_rng(77)
    n = 80
    pos = np.stack([rng.uniform(-1.5, 1.5, n), rng.uniform(-1.0, 1.0, n), rng.uniform(1.0, 5.0, n)], axis=1)
    pos[0] = [4.5, 0.2, 1.5]                                      # far beside the frustum, large: the Jacobian clamp is active
    sc = np.exp(rng.uniform(-1.8, -0.3, (n, 3))); sc[0] = 1.2
    sh = rng.normal(0, 0.2, (n, 4, 3)); sh[:, 0, :] += 0.9
    lv = [level(1, 0.0, pos, sc, quat=rng.normal(size=(n, 4)), logit=rng.normal(4.0, 2.0, n), sh=sh)]
    cam = camera(width=48, height=40, f=40.0, bg=(0.7, 0.1, 0.4))
    up = rng.normal(size=(3, 40, 48))
    worst, got, want = _gpu_vs_oracle(lv, 1, cam, 1, 1, 1.0, up, tol=5e-4)
    print('saturated:', {k: f'{v:.1e}' for k, v in worst.items()})
    fr = OracleScene(lv, 1).frame(cam, 1, 1, 1.0)
    _, E, B, T = fr.composite(stats=True)
    assert (T < 1e-4).mean() > 0.3                                 # many pixels stop early


@pytest.mark.gpu
def test_kernel_contract_and_zero_upstream():
    from paper_2408_12894_b200 import build
    build.build()
    import paper_2408_12894_b200 as pkg
    rng = np.random.default_rng(9)
    lv = _scene(rng, (30,), sh_degree=2)
    cam = camera(width=32, height=32, f=30.0)
    r = pkg.Renderer(0)
    r.upload_levels(lv, 2)
    r.set_workspace(32, 32, 1 << 20)
    z = torch.zeros((3, 32, 32), device="cuda")
    r.set_options(pkg.FLOD_OPT_FULL_SORT)                           # (a frame whose long lists were ordered lazily is refused)
    with pytest.raises(pkg.FlodError):                              # nothing rendered yet
        r.render_backward(cam, z, 2)
    r.render(cam, 1, 1, 1.0)
    g = r.render_backward(cam, z, 2)
    assert all((v == 0).all().item() for v in g.values())
    with pytest.raises(pkg.FlodError):                              # not the camera of the forward pass
        r.render_backward(camera(width=32, height=32, f=31.0), z, 2)
    r.render_rows(cam, 1, 1, 1.0, 0, 1)
    with pytest.raises(pkg.FlodError):                              # the last frame was a strip
        r.render_backward(cam, z, 2)
    r.close()


@pytest.mark.gpu
def test_kernel_on_long_lists_over_many_tiles():
    """1000 Gaussians (degree 3, two levels, selective rendering) on a ragged 110 x 70 image: 35 tiles whose lists hold
    hundreds of entries -- several batches of the backward walk, many entries per pixel behind the early stop."""
    rng = np.random.default_rng(21)
    lv = _scene(rng, (400, 600), sh_degree=3, extent=1.6)
    cam = camera(width=110, height=70, f=62.0, fy=55.0, cx=52.0, cy=37.5, bg=(0.2, 0.4, 0.6))
    up = rng.normal(size=(3, 70, 110))
    fr = OracleScene(lv, 3).frame(cam, 2, 2, 1.0)
    assert fr.tile_counts.max() > 3 * 64 and fr.counts["n_vis"] > 400
    _gpu_vs_oracle(lv, 3, cam, 1, 2, 1.0, up, tol=2e-4)
    worst, got, want = _gpu_vs_oracle(lv, 3, cam, 2, 2, 1.0, up, tol=2e-4)
    print("long lists:", {k: f"{v:.1e}" for k, v in worst.items()}, "longest list", int(fr.tile_counts.max()))
