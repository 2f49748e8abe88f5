"""GPU parity of SGS_FLAG_NORMALISED_DEPTH (depth image D_n = D / O) against the oracle's
normalise_depth / normalised_depth_upstream (pinned by P16): images, full and pose-only backward, the tracking
iteration (k_track<NDEPTH>, and its equality with render + sgs_backward_tracking) and the degenerate cases."""
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


@pytest.fixture(scope="module")
def ren():
    r = sgs.Renderer(normalised_depth=True)
    yield r
    r.close()


def check_images(gimg, o, sc, camv, cfg):
    assert_image_check(image_check(gimg, o["img"], o["fragile"], oracle.pixel_bounds(sc, camv, cfg), raw=o["img_raw"]))


@pytest.mark.parametrize("tau", [None, [0.1, -0.2, 0.15, 0.2, -0.1, 0.3]])
def test_c1_images_and_all_gradients(ren, tau):
    sc, cams, _ = scenegen.make_config("C1")
    cam = cams[0]
    T = None if tau is None else scenegen.perturb_pose(cam.T_cw, tau)
    camv, cfg = oracle.make_cam(cam, T), oracle.make_cfg()
    up = scenegen.upstream_normal(1, cam.height, cam.width)
    t, sf = to_device(sc)
    c = camera(cam, T)
    im = alloc_images(cam)
    ren.render(sf, c, **im)
    o = oracle.render_normalised(sc, camv, cfg)
    gimg = planes(im)
    check_images(gimg, o, sc, camv, cfg)
    m = o["img"][7] > 0.05
    assert np.abs(gimg[3][m] - o["img_raw"][3][m]).max() > 0.1      # it is not the Eq. 8 depth any more
    ob = oracle.binning(sc, camv, cfg)
    gb = ren.get_binning(sc.n, 12)
    assert np.array_equal(gb["keys"], ob["keys"]) and np.array_equal(gb["idx"], ob["idx"])
    og = oracle.backward_normalised(sc, camv, cfg, up)
    ex = oracle.exposure(sc, camv, cfg, oracle.normalised_depth_upstream(o["img_raw"], up))
    g, p6 = alloc_grads(sc.n), torch.full((6,), 3.0, device="cuda")
    ren.backward(**split_upstream(up), grads=g, d_pose6=p6)
    torch.cuda.synchronize()
    assert_grads({k: g[k].cpu().numpy() for k in GROUPS}, og, ex)
    assert_pose(p6.cpu().numpy(), og["pose"], ex["pose"], max_slack=0.5)
    # the normalisation matters to the gradients: the plain backward of the same upstream is far away
    plain = oracle.backward(sc, camv, cfg, up)
    assert np.abs(plain["pose"] - og["pose"]).max() > 0.05 * np.abs(og["pose"]).max()
    # pose-only mode, depth upstream alone (dL/dO comes from the depth term only)
    up_d = np.zeros_like(up); up_d[3] = up[3]
    ren.render(sf, c, **im)
    p6b = torch.zeros(6, device="cuda")
    ren.backward(**split_upstream(up_d), d_pose6=p6b)
    ogd = oracle.backward_normalised(sc, camv, cfg, up_d)
    exd = oracle.exposure(sc, camv, cfg, oracle.normalised_depth_upstream(o["img_raw"], up_d))
    # (D_n = D / O amplifies the upstream by 1 / O exactly at the faint pixels whose single splat sits on the alpha_min edge,
    # so on this 3072-pixel frame the fragile pixels' exposure is a larger share of the gradient than anywhere else)
    assert_pose(p6b.cpu().numpy(), ogd["pose"], exd["pose"], max_slack=0.5)


def test_c2_tracking_iteration_at_full_size(ren):
    """C2 (200k surfels, 640x480): images, then sgs_track_iter (loss Eq. 15-19 on D_n, pose gradient) against the
    oracle's loss on ITS OWN normalised images and its analytic backward through the division; masks / signs the renderer
    evaluates differently on its own image may only sit inside the image bar, and bound the allowed difference."""
    sc, cams, info = scenegen.make_config("C2")
    cam = cams[0]
    camv, cfg = oracle.make_cam(cam), oracle.make_cfg()
    g = scenegen.SplitMix(info["tau0_seed"])
    d = np.stack([g.normal(3), g.normal(3)])
    tau0 = np.concatenate([0.02 * d[0] / np.linalg.norm(d[0]), np.deg2rad(1.0) * d[1] / np.linalg.norm(d[1])])
    tgt = oracle.render_normalised(sc, oracle.make_cam(cam, scenegen.perturb_pose(cam.T_cw, tau0)), cfg, counters=False)["img"]
    tgt = tgt.astype(np.float32).astype(np.float64)       # the frame both sides see
    t, sf = to_device(sc)
    c = camera(cam)
    im, upi = alloc_images(cam), alloc_images(cam)
    trgb = torch.from_numpy(tgt[0:3].astype(np.float32)).cuda()
    tdep = torch.from_numpy(tgt[3:4].astype(np.float32)).cuda()
    p6, loss = torch.zeros(6, device="cuda"), torch.zeros(1, device="cuda")
    ren.track_iter(sf, c, trgb, tdep, 0.5, -1.0, p6, loss, **im)
    torch.cuda.synchronize()
    o = oracle.render_normalised(sc, camv, cfg)
    gimg = planes(im)
    check_images(gimg, o, sc, camv, cfg)
    tr = tracking_reference(sc, camv, cfg, o, tgt, 0.5, -1.0, oracle, normalised=True)
    assert (tr["up"][3] != 0).mean() > 0.05
    l2 = torch.zeros(1, device="cuda")
    ren.tracking_loss(c, im, trgb, tdep, 0.5, -1.0, upi, l2)
    D = tracking_flips(tr, planes(upi))
    assert D.any(0).mean() < 2e-4
    pose_slack, loss_slack = tracking_slack(sc, camv, cfg, tr, D, oracle)
    assert abs(float(loss.item()) - tr["L"]) <= tr["loss_tol"] + loss_slack
    assert_pose(p6.cpu().numpy(), tr["og"]["pose"], tr["ex"]["pose"] + pose_slack / C_EXPO)
    # render + backward_tracking gives the same numbers as track_iter
    im2 = alloc_images(cam)
    ren.render(sf, c, **im2)
    p6b, lb = torch.zeros(6, device="cuda"), torch.zeros(1, device="cuda")
    ren.backward_tracking(trgb, tdep, 0.5, -1.0, p6b, lb)
    torch.cuda.synchronize()
    assert np.array_equal(planes(im2), gimg)
    np.testing.assert_allclose(p6b.cpu().numpy(), p6.cpu().numpy(), rtol=1e-4, atol=1e-6 * float(p6.abs().max()))
    np.testing.assert_allclose(lb.cpu().numpy(), loss.cpu().numpy(), rtol=1e-5)


def test_degenerate_cases(ren):
    cam = Camera(40, 24, 30.0, 30.0, 20.0, 12.0)
    # no surfels: O = 0 everywhere -> D_n = 0, gradients zero, nothing non-finite
    z = lambda *s: np.zeros(s, np.float32)
    sc0 = Scene(z(0, 3), z(0, 2), z(0, 4), z(0), z(0, 3))
    t, sf = to_device(sc0)
    im = alloc_images(cam)
    for v in im.values():
        v.fill_(5.0)
    ren.render(sf, camera(cam), **im)
    assert float(planes(im)[3].max()) == 0.0 and float(planes(im)[7].max()) == 0.0
    # one small splat: most pixels empty (D_n = 0 there), covered pixels carry the plane's depth
    sc1 = Scene(np.float32([[0, 0, 2.0]]), np.float32([[0.1, 0.1]]), np.float32([[1, 0, 0, 0]]), np.float32([0.3]),
                np.float32([[0.2, 0.4, 0.6]]))
    t, sf = to_device(sc1)
    ren.render(sf, camera(cam), **im)
    gi = planes(im)
    cov = gi[7] > 0
    assert 0 < cov.sum() < cov.size
    assert np.abs(gi[3][cov] - 2.0).max() < 1e-5 and (gi[3][~cov] == 0).all()
    up = scenegen.upstream_normal(3, cam.height, cam.width)
    g, p6 = alloc_grads(1), torch.zeros(6, device="cuda")
    ren.backward(**split_upstream(up), grads=g, d_pose6=p6)
    og = oracle.backward_normalised(sc1, oracle.make_cam(cam), oracle.make_cfg(), up)
    for k in ("mean", "scale", "quat", "opacity", "rgb"):
        a = g[k].cpu().numpy().astype(np.float64)
        assert np.isfinite(a).all()
        assert np.abs(a - og[k]).max() <= 1e-3 * np.abs(og[k]).max() + 1e-6, (k, a, og[k])
    assert np.abs(p6.cpu().numpy() - og["pose"]).max() <= 1e-3 * np.abs(og["pose"]).max()


def test_track_iter_long_lists_and_reuse():
    """k_track<NDEPTH> == render + sgs_backward_tracking on C1 and on tile lists of ~900 entries (several 256-entry batches)
    and ~6000 entries (pre-sorted path), with and without the kept survivor list."""
    cases = []
    sc, cams, _ = scenegen.make_config("C1")
    cases.append((sc, cams[0]))
    g = scenegen.SplitMix(11)
    for n in (900, 6000):
        mean = np.stack([g.uniform(n, -0.05, 0.05), g.uniform(n, -0.05, 0.05), g.uniform(n, 1.0, 3.0)], 1).astype(np.float32)
        cases.append((Scene(mean, np.full((n, 2), 0.01, np.float32), np.tile(np.float32([1, 0.1, 0, 0]), (n, 1)),
                            np.full(n, 0.03 if n > 2000 else 0.2, np.float32),
                            np.stack([g.uniform(n) for _ in range(3)], 1).astype(np.float32)),
                      Camera(64, 48, 60.0, 60.0, 32.0, 24.0)))
    for reuse in (False, True):
        for sc, cam in cases:
            r = sgs.Renderer(normalised_depth=True, track_reuse=reuse)
            t, sf = to_device(sc)
            c = camera(cam)
            im, im2 = alloc_images(cam), alloc_images(cam)
            r.render(sf, c, **im)
            tgt_rgb = (im["rgb"] * 0.9 + 0.01).contiguous()
            tgt_dep = (im["depth"] * 1.02).contiguous()
            p6a, la = torch.zeros(6, device="cuda"), torch.zeros(1, device="cuda")
            r.backward_tracking(tgt_rgb, tgt_dep, 0.5, 1.0, p6a, la)
            for _ in range(2):   # second call: from the kept list under reuse
                p6b, lb = torch.zeros(6, device="cuda"), torch.zeros(1, device="cuda")
                r.track_iter(sf, c, tgt_rgb, tgt_dep, 0.5, 1.0, p6b, lb, **im2)
                torch.cuda.synchronize()
                assert np.array_equal(planes(im), planes(im2))
                assert float(la.abs().item()) > 0 and np.abs(p6a.cpu().numpy()).max() > 0
                np.testing.assert_allclose(lb.cpu().numpy(), la.cpu().numpy(), rtol=1e-5)
                np.testing.assert_allclose(p6b.cpu().numpy(), p6a.cpu().numpy(), rtol=1e-4, atol=1e-6 * float(p6a.abs().max()))
            r.close()


def test_flag_through_async_prepare_and_host_calls(ren):
    """The same D_n images and gradients through SGS_FLAG_ASYNC, sgs_prepare + sgs_render, sgs_render_contrib and the
    HOST-buffer calls (sgs_render_host, sgs_backward_host, sgs_track_iter_host) as through the plain device calls."""
    sc, cams, _ = scenegen.make_config("C1")
    cam = cams[0]
    up = scenegen.upstream_normal(6, cam.height, cam.width)
    t, sf = to_device(sc)
    c = camera(cam)

    def full(r, prep=False, contrib=False):
        im, g, p6 = alloc_images(cam), alloc_grads(sc.n), torch.zeros(6, device="cuda")
        if prep:
            r.prepare(sf, c)
        if contrib:
            r.render_contrib(sf, c, torch.zeros(sc.n, device="cuda"), **im)
        else:
            r.render(sf, c, **im)
        r.backward(**split_upstream(up), grads=g, d_pose6=p6)
        torch.cuda.synchronize()
        return planes(im), {k: v.cpu().numpy() for k, v in g.items()}, p6.cpu().numpy()

    ref = full(ren)
    a = sgs.Renderer(async_mode=True, normalised_depth=True)
    for kw in (dict(), dict(prep=True), dict(contrib=True)):
        for _ in range(2):
            img, g, p6 = full(a, **kw)
        assert np.array_equal(img, ref[0]), kw
        for k in g:
            np.testing.assert_allclose(g[k], ref[1][k], rtol=2e-4, atol=1e-5 * np.abs(ref[1][k]).max())
        np.testing.assert_allclose(p6, ref[2], rtol=1e-4, atol=1e-5 * np.abs(ref[2]).max())
    pin = lambda x, dt=torch.float32: torch.from_numpy(np.ascontiguousarray(x)).to(dt).pin_memory()
    a.upload_surfels(pin(sc.mean), pin(sc.scale), pin(sc.quat), pin(sc.opacity), pin(sc.rgb))
    H, W = cam.height, cam.width
    h = dict(rgb=torch.zeros(3, H, W).pin_memory(), depth=torch.zeros(1, H, W).pin_memory(),
             normal=torch.zeros(3, H, W).pin_memory(), alpha=torch.zeros(1, H, W).pin_memory())
    a.render_host(c, **h)
    himg = torch.cat([h["rgb"], h["depth"], h["normal"], h["alpha"]], 0).numpy().astype(np.float64)
    assert np.array_equal(himg, ref[0])
    u = torch.from_numpy(up)
    hg = {k: torch.zeros(v.shape).pin_memory() for k, v in ref[1].items()}
    hp = torch.zeros(6).pin_memory()
    a.backward_host(d_rgb=u[0:3].contiguous(), d_depth=u[3:4].contiguous(), d_normal=u[4:7].contiguous(),
                    d_alpha=u[7:8].contiguous(), grads=hg, d_pose6=hp)
    for k in hg:
        np.testing.assert_allclose(hg[k].numpy(), ref[1][k], rtol=2e-4, atol=1e-4 * np.abs(ref[1][k]).max())
    np.testing.assert_allclose(hp.numpy(), ref[2], rtol=1e-4, atol=1e-5 * np.abs(ref[2]).max())
    # resident tracking iteration == the device-buffer iteration on the same target
    trgb, tdep = (h["rgb"] * 0.9).contiguous(), (h["depth"] * 1.01).contiguous()
    a.upload_target(c, trgb.pin_memory(), tdep.pin_memory())
    loss_h, p6_h = a.track_iter_host(c, 0.5, 1.0)
    p6d, ld = torch.zeros(6, device="cuda"), torch.zeros(1, device="cuda")
    ren.track_iter(sf, c, trgb.cuda(), tdep.cuda(), 0.5, 1.0, p6d, ld)
    torch.cuda.synchronize()
    assert abs(loss_h - float(ld.item())) <= 1e-5 * abs(float(ld.item())) and abs(loss_h) > 0
    np.testing.assert_allclose(p6_h, p6d.cpu().numpy(), rtol=1e-4, atol=1e-6 * float(p6d.abs().max()))
    a.close()
