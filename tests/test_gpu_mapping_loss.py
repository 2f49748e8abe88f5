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


def test_holes_in_the_sensor_depth_carry_no_depth_term():
    """Reading R25: where the target depth is 0, negative, inf or NaN (how RGB-D sensors encode "no measurement") the
    depth terms of Eq. 19 and Eq. 26 vanish, loss and gradient; the colour terms stay.  sgs_mapping_loss and
    sgs_tracking_loss against the oracle on a synthetic frame with holes; the two fused tracking paths
    (sgs_backward_tracking, sgs_track_iter) against the unfused sequence on a rendered frame with the same holes."""
    from scenegen import Scene
    from gpu_common import to_device, alloc_images
    cam = Camera(70, 50, 60.0, 60.0, 35.0, 25.0)
    camv = oracle.make_cam(cam)
    g = scenegen.SplitMix(31)
    H, W = cam.height, cam.width
    img = np.zeros((8, H, W))
    img[0:3] = g.uniform(3 * H * W).reshape(3, H, W)
    img[3] = 2.0 + 0.2 * g.normal(H * W).reshape(H, W)
    img[6] = 1.0
    img[7] = 0.99
    trgb = g.uniform(3 * H * W).reshape(3, H, W)
    tdep = img[3] + 0.05 * g.normal(H * W).reshape(H, W)
    holes = np.zeros((H, W), bool)
    for k, v in enumerate((0.0, -1.0, np.inf, -np.inf, np.nan)):
        tdep[5 + 8 * k: 10 + 8 * k, 10:50] = v
        holes[5 + 8 * k: 10 + 8 * k, 10:50] = True
    ren = sgs.Renderer()
    # mapping loss (Eq. 26's depth term) and tracking loss (Eq. 16, 19) kernels vs the oracle
    L, up, img32 = run(ren, cam, img, trgb, tdep, 0.875, 0.5, 0.0, 1.0)
    L_ref, up_ref = oracle.mapping_loss(img32, trgb.astype(np.float32), tdep.astype(np.float32), camv, 0.875, 0.5, 0.0, 1.0)
    assert np.isfinite(L) and abs(L - L_ref) <= 2e-5 * abs(L_ref)
    assert (up[3][holes] == 0).all() and (up[3][~holes] != 0).all() and np.array_equal(np.sign(up[0:4]), np.sign(up_ref[0:4]))
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()
    r = dict(rgb=t(img[0:3]), depth=t(img[3:4]), normal=t(img[4:7]), alpha=t(img[7:8]))
    upt = {k: torch.full_like(v, 5.0) for k, v in r.items()}
    loss = torch.zeros(1, device="cuda")
    ren.tracking_loss(camera(cam), r, t(trgb), t(tdep[None]), 0.5, 1.0, upt, loss)
    Lt_ref, upt_ref = oracle.tracking_loss(img32, trgb.astype(np.float32), tdep.astype(np.float32), camv, 0.5, 1.0)
    assert np.isfinite(float(loss.item())) and abs(float(loss.item()) - Lt_ref) <= 2e-5 * abs(Lt_ref)
    gup = planes(upt)
    assert (gup[3][holes] == 0).all() and np.abs(gup - upt_ref).max() <= 1e-6 * np.abs(upt_ref).max()
    # fused paths on a rendered frame: same numbers as loss kernel + backward, all finite
    sc = scenegen.tiny_scene(7, 6000)
    sc.opacity[:] = 0.9
    tt, sf = to_device(sc)
    c = camera(cam)
    im, upi = alloc_images(cam), alloc_images(cam)
    ren.render(sf, c, **im)
    tgt_rgb = (im["rgb"] * 0.9 + 0.01).contiguous()
    tgt_dep = (im["depth"] * 1.02).contiguous()
    hm = torch.from_numpy(holes).cuda()[None]
    assert float(((im["alpha"] > 0.95) & hm).float().sum()) > 50        # holes fall on pixels that pass M_o
    tgt_dep[hm] = t(tdep[None])[hm]
    lu, pu = torch.zeros(1, device="cuda"), torch.zeros(6, device="cuda")
    ren.tracking_loss(c, im, tgt_rgb, tgt_dep, 0.5, 1.0, upi, lu)
    ren.backward(d_rgb=upi["rgb"], d_depth=upi["depth"], d_normal=upi["normal"], d_alpha=upi["alpha"], d_pose6=pu)
    assert (upi["depth"][hm] == 0).all() and np.isfinite(pu.cpu().numpy()).all() and float(pu.abs().max()) > 0
    pf, lf = torch.zeros(6, device="cuda"), torch.zeros(1, device="cuda")
    ren.backward_tracking(tgt_rgb, tgt_dep, 0.5, 1.0, pf, lf)
    pt, lt = torch.zeros(6, device="cuda"), torch.zeros(1, device="cuda")
    ren.track_iter(sf, c, tgt_rgb, tgt_dep, 0.5, 1.0, pt, lt)
    for p, l in ((pf, lf), (pt, lt)):
        np.testing.assert_allclose(l.cpu().numpy(), lu.cpu().numpy(), rtol=1e-5)
        np.testing.assert_allclose(p.cpu().numpy(), pu.cpu().numpy(), rtol=1e-4, atol=1e-6 * float(pu.abs().max()))
    ren.close()
