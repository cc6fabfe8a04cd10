"""Gradients of the rendered image with respect to every learnable parameter -- TEST INFRASTRUCTURE (see oracle/__init__.py).

Alg. 1 of the paper: I <- Rasterize(M, S^(l), R, C, A); L <- Loss(I, I^); M, S_opt, R, C, A <- Adam(grad L).
The rasterizer's backward pass is the gradient of <G, I> for an upstream image-shaped G = dL/dI.  The oracle is
the DEFINITION: the forward pass written out once more as a plain differentiable function in PyTorch CPU ops, fp64 --
Eq. 1, the pinhole projection and the projected covariance (R8, R9), Eq. 2, front-to-back
compositing (R11, R12), SH colour (R16) -- over ALL selected, un-culled Gaussians in (depth, gid) order, no tiles;
autograd differentiates it.  The discrete decisions (which Gaussians are selected and survive the culls, their order, the
1/255 skip, the stop at T < 1e-4) are constants of the differentiation, taken from the oracle's fp32 frame (oracle/
flod_oracle.c) so that they are the forward pass's own; min(0.99, .) and max(0, .) have their mathematical derivative
(zero on the clamped side).
Pins (tests/test_backward.py): its image equals the C oracle's brute-force image; central finite differences of its own
forward for every parameter; zero upstream gradient -> zero gradients; logit -20 -> no colour gradient.
"""
from __future__ import annotations

import math

import numpy as np
import torch

from . import ST_EMPTY_RECT, SKIP_THR, STOP_THR


def _sh_basis(deg, d):
    """Real SH of DESIGN R16 at unit directions d [n, 3] -> [n, K] (the same polynomials as orc_sh_basis)."""
    x, y, z = d[:, 0], d[:, 1], d[:, 2]
    pi = math.pi
    Y = [torch.full_like(x, 0.5 * math.sqrt(1.0 / pi))]
    if deg >= 1:
        c1 = math.sqrt(3.0 / (4.0 * pi))
        Y += [-c1 * y, c1 * z, -c1 * x]
    if deg >= 2:
        xx, yy, zz = x * x, y * y, z * z
        Y += [0.5 * math.sqrt(15.0 / pi) * x * y, -0.5 * math.sqrt(15.0 / pi) * y * z,
              0.25 * math.sqrt(5.0 / pi) * (2.0 * zz - xx - yy), -0.5 * math.sqrt(15.0 / pi) * x * z,
              0.25 * math.sqrt(15.0 / pi) * (xx - yy)]
    if deg >= 3:
        Y += [-0.25 * math.sqrt(35.0 / (2.0 * pi)) * y * (3.0 * xx - yy), 0.5 * math.sqrt(105.0 / pi) * x * y * z,
              -0.25 * math.sqrt(21.0 / (2.0 * pi)) * y * (4.0 * zz - xx - yy),
              0.25 * math.sqrt(7.0 / pi) * z * (2.0 * zz - 3.0 * xx - 3.0 * yy),
              -0.25 * math.sqrt(21.0 / (2.0 * pi)) * x * (4.0 * zz - xx - yy), 0.25 * math.sqrt(105.0 / pi) * z * (xx - yy),
              -0.25 * math.sqrt(35.0 / (2.0 * pi)) * x * (xx - 3.0 * yy)]
    return torch.stack(Y, dim=1)


def forward(params, cam, sh_degree, ids, order, skip_thr=SKIP_THR, stop_thr=STOP_THR):
    """The image [3, H, W] (fp64) of the Gaussians `ids` (indices into the concatenated parameter arrays) composited in the
    order `order` (a permutation of range(len(ids))).  params: dict of fp64 tensors mean [n,3], log_scale [n,3], quat [n,4],
    logit [n], sh [n,K,3]."""
    f64 = torch.float64
    mean, ls, q, logit, sh = (params[k][ids] for k in ("mean", "log_scale", "quat", "logit", "sh"))
    Rc = torch.tensor(np.asarray(cam.R, np.float64).reshape(3, 3), dtype=f64)
    t = torch.tensor(np.asarray(cam.t, np.float64).reshape(3), dtype=f64)
    W, H = cam.width, cam.height
    # Eq. 1
    s = torch.exp(ls)
    qn = q / q.norm(dim=1, keepdim=True)
    w, x, y, z = qn[:, 0], qn[:, 1], qn[:, 2], qn[:, 3]
    Rg = torch.stack([1 - 2 * (y * y + z * z), 2 * (x * y - w * z), 2 * (x * z + w * y),
                      2 * (x * y + w * z), 1 - 2 * (x * x + z * z), 2 * (y * z - w * x),
                      2 * (x * z - w * y), 2 * (y * z + w * x), 1 - 2 * (x * x + y * y)], dim=1).reshape(-1, 3, 3)
    Mg = Rg * s[:, None, :]
    Sigma = Mg @ Mg.transpose(1, 2)
    # projection (O2, O3)
    p = mean @ Rc.T + t
    px, py, pz = p[:, 0], p[:, 1], p[:, 2]
    ix, iy = px / pz, py / pz
    mu2 = torch.stack([cam.fx * ix + cam.cx, cam.fy * iy + cam.cy], dim=1)
    limx, limy = 1.3 * W / (2.0 * cam.fx), 1.3 * H / (2.0 * cam.fy)
    u, v = torch.clamp(ix, -limx, limx), torch.clamp(iy, -limy, limy)
    zero = torch.zeros_like(pz)
    J = torch.stack([cam.fx / pz, zero, -(cam.fx * u) / pz, zero, cam.fy / pz, -(cam.fy * v) / pz], dim=1).reshape(-1, 2, 3)
    M = J @ Rc
    cov = M @ Sigma @ M.transpose(1, 2)
    a, b, c = cov[:, 0, 0] + 0.3, cov[:, 0, 1], cov[:, 1, 1] + 0.3
    det = a * c - b * b
    A, B, C = c / det, -b / det, a / det
    o = torch.sigmoid(logit)
    # colour (O5)
    centre = -(Rc.T @ t)
    d = mean - centre
    rgb = torch.clamp_min(0.5 + torch.einsum("nk,nkc->nc", _sh_basis(sh_degree, d / d.norm(dim=1, keepdim=True)), sh), 0.0)
    # compositing (O7) in the given order
    ordt = torch.as_tensor(np.asarray(order, np.int64))
    mu2, A, B, C, o, rgb = mu2[ordt], A[ordt], B[ordt], C[ordt], o[ordt], rgb[ordt]
    jj, ii = torch.meshgrid(torch.arange(H, dtype=f64) + 0.5, torch.arange(W, dtype=f64) + 0.5, indexing="ij")
    dx = mu2[:, 0, None, None] - ii[None]
    dy = mu2[:, 1, None, None] - jj[None]
    qf = torch.clamp_min(0.5 * (A[:, None, None] * dx * dx + C[:, None, None] * dy * dy) + B[:, None, None] * dx * dy, 0.0)
    alpha = torch.clamp_max(o[:, None, None] * torch.exp(-qf), 0.99)
    alpha = alpha * (alpha.detach() >= skip_thr)                                   # the 1/255 skip (a constant mask)
    one_minus = 1.0 - alpha
    T_before = torch.cat([torch.ones_like(alpha[:1]), torch.cumprod(one_minus, dim=0)[:-1]], dim=0)
    active = (T_before.detach() >= stop_thr).to(f64)                                # processed: the pixel had not stopped yet
    weight = active * T_before * alpha
    T_final = torch.prod(1.0 - alpha * active, dim=0)
    bg = torch.tensor([float(v) for v in cam.bg], dtype=f64)
    return torch.einsum("nhw,nc->chw", weight, rgb) + T_final[None] * bg[:, None, None]


def frame_selection(frame):
    """ids (ascending gid) and compositing order of the oracle frame's un-culled Gaussians: (depth as fp32, gid)."""
    state, depth = frame.state, frame.depth
    ids = np.nonzero(state >= ST_EMPTY_RECT)[0]
    order = np.lexsort((ids, depth[ids]))
    return ids, order


def scene_params(levels, requires_grad=True):
    cat = lambda name: torch.tensor(np.concatenate([np.asarray(getattr(lv, name), np.float64) for lv in levels]),
                                    dtype=torch.float64, requires_grad=requires_grad)
    return {"mean": cat("mean"), "log_scale": cat("log_scale"), "quat": cat("quat"), "logit": cat("opacity_logit"), "sh": cat("sh")}


def backward(levels, sh_degree, cam, frame, upstream):
    """Gradients of <upstream, image> w.r.t. (mean, log_scale, quat, logit, sh), as numpy fp64 arrays over ALL Gaussians
    of the scene (zero for those the frame does not draw), plus the image."""
    params = scene_params(levels)
    ids, order = frame_selection(frame)
    img = forward(params, cam, sh_degree, torch.as_tensor(ids), order)
    loss = (img * torch.as_tensor(np.asarray(upstream, np.float64))).sum()
    grads = torch.autograd.grad(loss, [params[k] for k in ("mean", "log_scale", "quat", "logit", "sh")], allow_unused=True)
    out = {k: (g if g is not None else torch.zeros_like(params[k])).numpy() for k, g in zip(("mean", "log_scale", "quat", "logit", "sh"), grads)}
    return out, img.detach().numpy()
