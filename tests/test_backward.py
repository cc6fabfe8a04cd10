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
