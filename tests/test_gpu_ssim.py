"""GPU parity of sgs_ssim_loss (SSIM term of PAPER.md Eq. 24) against oracle.ssim_loss: loss and gradient, on a ragged
synthetic image pair and on the oracle's C3 render vs its perturbed-pose target; accumulation semantics; bandwidth."""
import numpy as np
import pytest
import torch

import oracle
import scenegen

pytestmark = pytest.mark.gpu

sgs = pytest.importorskip("paper_2506_00970_b200")


def check(ren, x, y, weight):
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()
    xd, yd = t(x), t(y)
    up = torch.zeros_like(xd)
    loss = torch.zeros(1, device="cuda")
    ren.ssim_loss(xd, yd, weight, up, loss)
    L_ref, g_ref = oracle.ssim_loss(xd.cpu().numpy(), yd.cpu().numpy(), weight)
    L = float(loss.item())
    up2 = up.clone()
    ren.ssim_loss(xd, yd, weight, up2, loss)             # both outputs ACCUMULATE
    assert torch.allclose(up2, 2 * up, rtol=1e-5, atol=1e-12)
    assert abs(float(loss.item()) - 2 * L) <= 1e-5 * abs(L) + 1e-9
    g = up.cpu().numpy().astype(np.float64)
    assert abs(L - L_ref) <= 5e-5 * abs(L_ref) + 1e-6, (L, L_ref)
    scale = np.abs(g_ref).max()
    bad = np.abs(g - g_ref) > 1e-3 * np.abs(g_ref) + 2e-4 * scale + 1e-4 * weight / g.size   # fp32 window sums; the floor is 1e-4 of one pixel's share
    assert bad.mean() <= 1e-3, (bad.sum(), np.abs(g - g_ref).max(), scale)


def test_ssim_synthetic_pair():
    g = scenegen.SplitMix(3)
    H, W = 75, 131                                       # ragged against the 16 x 16 tiles, smaller than a halo in places
    X, Y = np.meshgrid(np.arange(W), np.arange(H))
    base = 0.5 + 0.4 * np.sin(X / 9.0) * np.cos(Y / 7.0)
    x = np.clip(np.stack([base, base[::-1], base.T[:H, :W] if base.T.shape == base.shape else base * 0.8]) +
                0.05 * g.normal(3 * H * W).reshape(3, H, W), 0, 1)
    y = np.clip(x + 0.1 * g.normal(3 * H * W).reshape(3, H, W), 0, 1)
    ren = sgs.Renderer()
    check(ren, x, y, 0.125)
    check(ren, x, x, 1.0)                               # identical images: loss 0, gradient 0
    check(ren, np.zeros((3, 5, 7)), np.ones((3, 5, 7)) * 0.5, 0.3)     # image smaller than the window
    ren.close()


def test_ssim_on_c3_render_and_bandwidth():
    sc, cams, _ = scenegen.make_config("C3")
    cam = cams[1]
    cfg = oracle.make_cfg()
    img = oracle.render(sc, oracle.make_cam(cam), cfg, counters=False)["img"]
    T_tgt = scenegen.perturb_pose(cam.T_cw, np.array([0.01, 0.0, 0.0, 0.0, 0.005, 0.0]))
    tgt = oracle.render(sc, oracle.make_cam(cam, T_tgt), cfg, counters=False)["img"]
    ren = sgs.Renderer()
    check(ren, img[0:3], tgt[0:3], 0.125)
    xd = torch.from_numpy(img[0:3].astype(np.float32)).cuda(); yd = torch.from_numpy(tgt[0:3].astype(np.float32)).cuda()
    up = torch.zeros_like(xd); loss = torch.zeros(1, device="cuda")
    for _ in range(3):
        ren.ssim_loss(xd, yd, 0.125, up, loss)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(10):
        ren.ssim_loss(xd, yd, 0.125, up, loss)
    e1.record(); torch.cuda.synchronize()
    us = e0.elapsed_time(e1) * 100.0
    px = xd.shape[1] * xd.shape[2]
    print(f"ssim_loss: {us:.1f} us at {xd.shape[2]}x{xd.shape[1]} = {px * 3 * 4 * (2 + 3 + 3 + 2 + 2) / (us * 1e-6) / 1e9:.0f} GB/s algorithmic")
    ren.close()
