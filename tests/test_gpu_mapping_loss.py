"""GPU parity of sgs_mapping_loss (Eq. 23-26 without SSIM) against oracle.mapping_loss: the loss value and
all upstream gradients, on a synthetic bumpy frame (every branch of the stencil) and on the oracle's own C3 render."""
import numpy as np
import pytest
import torch

import oracle
import scenegen
from scenegen import Camera

pytestmark = pytest.mark.gpu

sgs = pytest.importorskip("paper_2506_00970_b200")
from gpu_common import camera, planes  # noqa: E402


def run(ren, cam, img, trgb, tdep, lam, wd, wn, sign):
    H, W = cam.height, cam.width
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()
    r = dict(rgb=t(img[0:3]), depth=t(img[3:4]), normal=t(img[4:7]), alpha=t(img[7:8]))
    up = {k: torch.full_like(v, 5.0) for k, v in r.items()}
    loss = torch.zeros(1, device="cuda")
    ren.mapping_loss(camera(cam), r, t(trgb), t(tdep[None]), lam, wd, wn, sign, up, loss)
    img32 = np.concatenate([v.cpu().numpy() for v in (r["rgb"], r["depth"], r["normal"], r["alpha"])], 0).astype(np.float64)
    return float(loss.item()), planes(up), img32


def check(cam, img, trgb, tdep, lam, wd, wn, sign, ren):
    L, up, img32 = run(ren, cam, img, trgb, tdep, lam, wd, wn, sign)
    camv = oracle.make_cam(cam)
    L_ref, up_ref = oracle.mapping_loss(img32, trgb.astype(np.float32), tdep.astype(np.float32), camv, lam, wd, wn, sign)
    assert abs(L - L_ref) <= 2e-5 * abs(L_ref), (L, L_ref)
    # colour / depth-L1 signs are exact; the N_D chain is fp32 stencil arithmetic: 1e-4 relative to the plane's scale
    for ch in range(8):
        scale = np.abs(up_ref[ch]).max() + 1e-30
        bad = np.abs(up[ch] - up_ref[ch]) > 2e-4 * np.abs(up_ref[ch]) + 2e-5 * scale
        assert bad.mean() <= 1e-3, (ch, bad.sum(), np.abs(up[ch] - up_ref[ch]).max(), scale)
    assert (up[7] == 0).all()


def test_mapping_loss_synthetic_frame():
    cam = Camera(203, 131, 180.0, 175.0, 100.5, 64.0)        # ragged against the 32x8 thread tiles
    g = scenegen.SplitMix(21)
    H, W = cam.height, cam.width
    X, Y = np.meshgrid(np.arange(W) + 0.5, np.arange(H) + 0.5)
    img = np.zeros((8, H, W))
    img[3] = 2.0 + 0.3 * np.sin(X / 17.0) * np.cos(Y / 11.0) + 0.01 * g.normal(H * W).reshape(H, W)
    img[3, 40:44, 50:60] = 0.0                                # holes: zero depth -> degenerate cross products
    img[4:7] = g.normal(3 * H * W).reshape(3, H, W)
    img[0:3] = g.uniform(3 * H * W).reshape(3, H, W)
    img[7] = g.uniform(H * W).reshape(H, W)
    trgb = g.uniform(3 * H * W).reshape(3, H, W)
    tdep = img[3] + 0.05 * g.normal(H * W).reshape(H, W)
    ren = sgs.Renderer()
    for sign in (1.0, -1.0):
        check(cam, img, trgb, tdep, 0.875, 0.5, 0.02, sign, ren)
    check(cam, img, trgb, tdep, 1.0, 0.0, 0.0, 1.0, ren)      # colour only
    ren.close()


def test_mapping_loss_on_c3_render():
    """The oracle's own C3 view (1200x680, un-normalised depth, blended normals) as the rendered frame."""
    sc, cams, _ = scenegen.make_config("C3")
    cam = cams[2]
    cfg = oracle.make_cfg()
    img = oracle.render(sc, oracle.make_cam(cam), cfg, counters=False)["img"]
    T_tgt = scenegen.perturb_pose(cam.T_cw, np.array([0.02, 0.0, 0.0, 0.0, 0.01, 0.0]))
    tgt = oracle.render(sc, oracle.make_cam(cam, T_tgt), cfg, counters=False)["img"]
    ren = sgs.Renderer()
    check(cam, img, tgt[0:3], tgt[3], 0.875, 0.5, 0.02, -1.0, ren)
    ren.close()
