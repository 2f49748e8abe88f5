"""GPU parity of SGS_FLAG_LOWPASS (reading R28: rho^2 = min(u^2 + v^2, 2 |x - x_c|^2), centre depth where
the screen term wins) against the oracle's lowpass mode (pinned by P19): binning bit-exact (footprint = ellipse AABB united
with the filter's disc), images, every surfel gradient, the pose gradient in full and pose-only mode, the fused tracking
backward, on scenes where the screen term matters (sub-pixel and edge-on splats) and on C1 / C2."""
import numpy as np
import pytest
import torch

import oracle
import scenegen
from scenegen import Scene, Camera

pytestmark = pytest.mark.gpu

sgs = pytest.importorskip("paper_2506_00970_b200")
from gpu_common import (to_device, camera, alloc_images, planes, alloc_grads, split_upstream, image_check,  # noqa: E402
                        assert_image_check, assert_grads, assert_pose, tracking_reference, tracking_flips, tracking_slack,
                        GROUPS, C_EXPO)


def run(ren, sc, cam, up, T=None, full=True):
    t, sf = to_device(sc)
    c = camera(cam, T)
    im = alloc_images(cam)
    ren.render(sf, c, **im)
    tiles = ((cam.width + 15) // 16) * ((cam.height + 15) // 16)
    out = dict(img=planes(im), bin=ren.get_binning(sc.n, tiles))
    g = alloc_grads(sc.n) if full else None
    p6 = torch.full((6,), 3.0, device="cuda")
    ren.backward(**split_upstream(up), grads=g, d_pose6=p6)
    torch.cuda.synchronize()
    if full:
        out["grads"] = {k: v.cpu().numpy() for k, v in g.items()}
    out["pose"] = p6.cpu().numpy()
    return out


def check(sc, cam, T=None, seed=1, min_2d_share=0.0, max_fragile=None):
    cfg = oracle.make_cfg(lowpass=True)
    camv = oracle.make_cam(cam, T)
    up = scenegen.upstream_normal(seed, cam.height, cam.width)
    ren = sgs.Renderer(lowpass=True)
    out = run(ren, sc, cam, up, T)
    ob = oracle.binning(sc, camv, cfg)
    for k in ("culled", "keys", "idx", "ranges"):
        assert np.array_equal(out["bin"][k], ob[k]), k
    o = oracle.render(sc, camv, cfg)
    plain = oracle.render(sc, camv, oracle.make_cfg(), counters=False)["img"]
    assert np.abs(o["img"][7] - plain[7]).sum() >= min_2d_share * o["img"][7].sum()     # the filter matters on this scene
    chk = image_check(out["img"], o["img"], o["fragile"], oracle.pixel_bounds(sc, camv, cfg))
    if max_fragile is None:
        assert_image_check(chk)
    else:   # (the stress scene is BUILT of edge-on splats and slivers: its fragile fraction is the scene's; the bounds are the derived ones)
        assert chk["n_bad"] == 0 and chk["n_bad_fragile"] == 0 and chk["fragile_frac"] < max_fragile, chk
    og, ex = oracle.backward(sc, camv, cfg, up), oracle.exposure(sc, camv, cfg, up)
    assert_grads(out["grads"], og, ex)
    assert_pose(out["pose"], og["pose"], ex["pose"], max_slack=0.2)
    out2 = run(ren, sc, cam, up, T, full=False)                                          # pose-only mode (per-pixel Eq. 11-13)
    assert_pose(out2["pose"], og["pose"], ex["pose"], max_slack=0.2)
    ren.close()


@pytest.mark.parametrize("tau", [None, [0.1, -0.2, 0.15, 0.2, -0.1, 0.3]])
def test_c1_with_the_filter(tau):
    sc, cams, _ = scenegen.make_config("C1")
    cam = cams[0]
    check(sc, cam, None if tau is None else scenegen.perturb_pose(cam.T_cw, tau))


def test_sub_pixel_and_edge_on_splats():
    """C1's splats shrunk to 0.5 - 2.5 mm (most of them below a pixel: nearly all alpha comes from the screen term), plus
    the stress scene (slivers, edge-on splats) at two poses."""
    sc, cams, _ = scenegen.make_config("C1")
    small = Scene(sc.mean, sc.scale * np.float32(0.05), sc.quat, sc.opacity, sc.rgb)
    check(small, cams[0], seed=2, min_2d_share=0.5)
    st, scam = scenegen.stress_scene(), scenegen.stress_camera()
    check(st, scam, seed=3, max_fragile=0.08)
    check(st, scam, scenegen.perturb_pose(scam.T_cw, [0.05, -0.08, 0.1, 0.3, -0.2, 0.4]), seed=3, max_fragile=0.08)


def test_c2_tracking_with_the_filter():
    """C2 at full size: images, then the Eq. 15-19 tracking iteration; sgs_track_iter takes the unfused sequence under
    the flag and must agree with sgs_render + sgs_backward_tracking and, within the flip slack, with the oracle."""
    sc, cams, info = scenegen.make_config("C2")
    cam = cams[0]
    cfg = oracle.make_cfg(lowpass=True)
    camv, c = oracle.make_cam(cam), camera(cam)
    g = scenegen.SplitMix(info["tau0_seed"])
    d = np.stack([g.normal(3), g.normal(3)])
    tau0 = np.concatenate([0.02 * d[0] / np.linalg.norm(d[0]), np.deg2rad(1.0) * d[1] / np.linalg.norm(d[1])])
    tgt = oracle.render(sc, oracle.make_cam(cam, scenegen.perturb_pose(cam.T_cw, tau0)), cfg, counters=False)["img"]
    tgt = tgt.astype(np.float32).astype(np.float64)
    ren = sgs.Renderer(lowpass=True)
    t, sf = to_device(sc)
    im, upi = alloc_images(cam), alloc_images(cam)
    ren.render(sf, c, **im)
    o = oracle.render(sc, camv, cfg)
    assert_image_check(image_check(planes(im), o["img"], o["fragile"], oracle.pixel_bounds(sc, camv, cfg)))
    tr = tracking_reference(sc, camv, cfg, o, tgt, 0.5, -1.0, oracle)
    trgb = torch.from_numpy(tgt[0:3].astype(np.float32)).cuda()
    tdep = torch.from_numpy(tgt[3:4].astype(np.float32)).cuda()
    loss = torch.zeros(1, device="cuda")
    ren.tracking_loss(c, im, trgb, tdep, 0.5, -1.0, upi, loss)
    D = tracking_flips(tr, planes(upi))
    pose_slack, loss_slack = tracking_slack(sc, camv, cfg, tr, D, oracle)
    p6f, lf = torch.zeros(6, device="cuda"), torch.zeros(1, device="cuda")
    ren.backward_tracking(trgb, tdep, 0.5, -1.0, p6f, lf)
    assert abs(float(lf.item()) - tr["L"]) <= tr["loss_tol"] + loss_slack
    assert_pose(p6f.cpu().numpy(), tr["og"]["pose"], tr["ex"]["pose"] + pose_slack / C_EXPO)
    p6t, lt = torch.zeros(6, device="cuda"), torch.zeros(1, device="cuda")
    ren.track_iter(sf, c, trgb, tdep, 0.5, -1.0, p6t, lt)
    np.testing.assert_allclose(lt.cpu().numpy(), lf.cpu().numpy(), rtol=1e-5)
    np.testing.assert_allclose(p6t.cpu().numpy(), p6f.cpu().numpy(), rtol=1e-4, atol=1e-6 * float(p6f.abs().max()))
    with pytest.raises(sgs.SgsError):
        ren.render_contrib(sf, c, torch.zeros(sc.n, device="cuda"), **im)
    with pytest.raises(sgs.SgsError):
        sgs.Renderer(lowpass=True, tight_binning=True)
    ren.close()
