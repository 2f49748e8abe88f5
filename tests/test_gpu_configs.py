"""GPU parity at BASELINE.json's FULL sizes (C2-C5), in the launch configuration bench.py times
(SGS_FLAG_ASYNC renderer, same scenes, same views): binning bit-exact, whole images, the Eq. 15-19 loss,
and the backward the config asks for (pose-only for the tracking-shaped C2/C5, full + pose for the
mapping-shaped C3/C4) against the oracle on WHOLE images -- the fp64 oracle finishes a view in seconds.
Every pixel and every gradient element is bounded (gpu_common: the strict bars, plus oracle-derived allowances on
fragile pixels only); the benchmarked tracking path is held to north_star's 1e-3 plus an oracle-computed flip slack.
Every oracle input comes from scenegen/ or from the oracle itself (target frame, upstream gradients);
nothing the CUDA path produced is fed to it."""
import numpy as np
import pytest
import torch

import oracle
import scenegen

pytestmark = pytest.mark.gpu

sgs = pytest.importorskip("paper_2506_00970_b200")
from gpu_common import (to_device, camera, alloc_images, planes, alloc_grads, image_check, assert_image_check,  # noqa: E402
                        assert_grads, assert_pose, tracking_reference, tracking_flips, tracking_slack, GROUPS, C_EXPO)

LAMBDA_D, NSIGN = 0.5, -1.0


def tau0(seed):
    g = scenegen.SplitMix(seed)
    d = np.stack([g.normal(3), g.normal(3)])
    return np.concatenate([0.02 * d[0] / np.linalg.norm(d[0]), np.deg2rad(1.0) * d[1] / np.linalg.norm(d[1])])


def render_settled(ren, sf, cam, im):
    """Async mode reports a bucket overflow on the NEXT call (after growing the workspace): retry."""
    for _ in range(6):
        try:
            ren.render(sf, cam, **im)
            ren.stats()
            ren.render(sf, cam, **im)
            ren.stats()
            return
        except sgs.SgsError as e:
            if e.status != sgs.SGS_WORKSPACE_OVERFLOW:
                raise
    raise AssertionError("workspace did not settle")


def assert_binning(gb, ob):
    assert gb["E"] == ob["E"]
    assert np.array_equal(gb["culled"], ob["culled"])
    assert np.array_equal(gb["keys"], ob["keys"])
    assert np.array_equal(gb["idx"], ob["idx"])
    assert np.array_equal(gb["ranges"], ob["ranges"])


def check_config(name, views, full, tight=False):
    """tight: SGS_FLAG_TIGHT_BINNING against the oracle's tight mode (readings R26, R27): the same checks, shorter lists."""
    sc, cams, info = scenegen.make_config(name)
    cfg = oracle.make_cfg(tight=tight)
    ren = sgs.Renderer(async_mode=True, tight_binning=tight)
    t, sf = to_device(sc)
    try:
        for v in views:
            cam = cams[v]
            camv, c = oracle.make_cam(cam), camera(cam)
            tiles = ((cam.width + 15) // 16) * ((cam.height + 15) // 16)
            im, upi = alloc_images(cam), alloc_images(cam)
            render_settled(ren, sf, c, im)
            # ---- binning: bit-exact
            ob = oracle.binning(sc, camv, cfg)
            assert_binning(ren.get_binning(sc.n, tiles), ob)
            if tight:
                assert ob["E"] < 0.95 * oracle.binning(sc, camv, oracle.make_cfg())["E"]
            # ---- images: every pixel (fragile ones within the oracle-derived allowance)
            o = oracle.render(sc, camv, cfg)
            gimg = planes(im)
            assert_image_check(image_check(gimg, o["img"], o["fragile"], oracle.pixel_bounds(sc, camv, cfg)), (name, v))
            # ---- Eq. 15-19 against a target frame rendered BY THE ORACLE at the perturbed pose (as binary32: the frame
            # both sides see)
            T_tgt = scenegen.perturb_pose(cam.T_cw, tau0(info.get("tau0_seed", 2000 + v)))
            tgt = oracle.render(sc, oracle.make_cam(cam, T_tgt), cfg, counters=False)["img"].astype(np.float32).astype(np.float64)
            tr = tracking_reference(sc, camv, cfg, o, tgt, LAMBDA_D, NSIGN, oracle)
            L_ref, up_ref = tr["L"], tr["up"]
            assert (up_ref != 0).mean() > 0.02
            trgb = torch.from_numpy(tgt[0:3].astype(np.float32)).cuda()
            tdep = torch.from_numpy(tgt[3:4].astype(np.float32)).cuda()
            loss = torch.zeros(1, device="cuda")
            ren.tracking_loss(c, im, trgb, tdep, LAMBDA_D, NSIGN, upi, loss)
            # the loss's gradient is +-1/|Omega| per pixel: it may differ from the oracle's only where a mask or a sign
            # sits inside the image bar (asserted), and those pixels bound what the fused paths may differ by
            D = tracking_flips(tr, planes(upi))
            assert D.any(0).mean() < 2e-4, D.sum(axis=(1, 2))
            pose_slack, loss_slack = tracking_slack(sc, camv, cfg, tr, D, oracle)
            assert abs(float(loss.item()) - L_ref) <= tr["loss_tol"] + loss_slack, (float(loss.item()), L_ref)
            # ---- backward on the ORACLE's upstream gradients (same array to both sides)
            u = torch.from_numpy(up_ref.astype(np.float32)).cuda()
            up32 = u.cpu().numpy().astype(np.float64)
            og, ex = oracle.backward(sc, camv, cfg, up32), oracle.exposure(sc, camv, cfg, up32)
            kw = dict(d_rgb=u[0:3].contiguous(), d_depth=u[3:4].contiguous(), d_normal=u[4:7].contiguous(),
                      d_alpha=u[7:8].contiguous())
            p6 = torch.full((6,), 3.0, device="cuda")
            if full:
                # the mapping-shaped configs: EVERY element of every surfel gradient, under the mapping loss of Eq. 24-26
                # (dense upstream on all channels), then under the tracking loss's masked upstream
                _, upm = oracle.mapping_loss(o["img"], tgt[0:3], tgt[3], camv, 0.875, 0.5, 0.02, NSIGN)
                for upx in (upm, up32):
                    ux = torch.from_numpy(upx.astype(np.float32)).cuda()
                    ux64 = ux.cpu().numpy().astype(np.float64)
                    ogx, exx = oracle.backward(sc, camv, cfg, ux64), oracle.exposure(sc, camv, cfg, ux64)
                    g = alloc_grads(sc.n)
                    ren.backward(d_rgb=ux[0:3].contiguous(), d_depth=ux[3:4].contiguous(), d_normal=ux[4:7].contiguous(),
                                 d_alpha=ux[7:8].contiguous(), grads=g, d_pose6=p6)
                    torch.cuda.synchronize()
                    gn = {k: g[k].cpu().numpy() for k in GROUPS}
                    assert_grads(gn, ogx, exx, (name, v))
                    for k in GROUPS:
                        assert (gn[k][ob["culled"].astype(bool)] == 0).all()
                    assert_pose(p6.cpu().numpy(), ogx["pose"], exx["pose"], (name, v))
            else:
                ren.backward(**kw, d_pose6=p6)
                assert_pose(p6.cpu().numpy(), og["pose"], ex["pose"], (name, v))
            if not full:
                # the launch bench.py times: Eq. 15-19 evaluated inside the pose-only backward on the GPU's own images:
                # north_star's 1e-3 plus what the masks / signs that came out differently (D) can change
                allow = tr["ex"]["pose"] + pose_slack / C_EXPO
                p6f, lossf = torch.zeros(6, device="cuda"), torch.zeros(1, device="cuda")
                ren.backward_tracking(trgb, tdep, LAMBDA_D, NSIGN, p6f, lossf)
                assert abs(float(lossf.item()) - L_ref) <= tr["loss_tol"] + loss_slack
                posef = p6f.cpu().numpy().astype(np.float64)
                assert_pose(posef, tr["og"]["pose"], allow, (name, v, "backward_tracking"))
                # ... and the single-launch iteration (sgs_track_iter: sort + render + loss + backward in one kernel)
                im2 = alloc_images(cam)
                p6t, losst = torch.zeros(6, device="cuda"), torch.zeros(1, device="cuda")
                for _ in range(2):
                    ren.track_iter(sf, c, trgb, tdep, LAMBDA_D, NSIGN, p6t, losst, **im2)
                    ren.stats()
                assert np.array_equal(planes(im2), gimg)                      # same images, bit for bit
                assert_binning(ren.get_binning(sc.n, tiles), ob)
                assert abs(float(losst.item()) - float(lossf.item())) <= 1e-6 * abs(L_ref)
                poset = p6t.cpu().numpy().astype(np.float64)
                assert np.abs(poset - posef).max() <= 1e-5 * np.abs(posef).max(), (poset, posef)
                assert_pose(poset, tr["og"]["pose"], allow, (name, v, "track_iter"))
                ren.track_iter(sf, c, trgb, tdep, LAMBDA_D, NSIGN, p6t, losst)   # no image outputs
                np.testing.assert_allclose(p6t.cpu().numpy(), poset, rtol=1e-5, atol=1e-7 * np.abs(poset).max())
    finally:
        ren.close()


def test_c2_full_size():
    check_config("C2", [0], full=False)


def test_c3_full_size():
    check_config("C3", [0, 7], full=True)


def test_c4_full_size():
    check_config("C4", [0, 6], full=True)


def test_c5_full_size():
    check_config("C5", [0], full=False)


@pytest.mark.parametrize("name,views,full", [("C2", [0], False), ("C3", [0], True), ("C4", [6], True), ("C5", [0], False)])
def test_tight_binning_full_size(name, views, full):
    """SGS_FLAG_TIGHT_BINNING (opacity-aware cutoff + tile-exact culling) on every full-size config: the shorter lists are
    bit-identical to the oracle's tight mode; images, losses and gradients meet the same bars as with the default binning."""
    check_config(name, views, full, tight=True)


@pytest.mark.parametrize("name", ["C2", "C5"])
def test_tracking_launch_configuration_with_the_kept_survivor_list(name):
    """What bench.py times on the tracking configs: SGS_FLAG_ASYNC + SGS_FLAG_TRACK_REUSE, the survivor list built once per
    frame (sgs_track_new_frame) and kept while the pose moves inside its margin.  Three poses of one frame (the keyframe's,
    then two steps of 8 mm / 0.3 deg): at each, binning bit-exact, images and the pose gradient / loss of sgs_track_iter
    against the oracle at THAT pose (1e-3 + the oracle-computed flip slack)."""
    sc, cams, info = scenegen.make_config(name)
    cfg = oracle.make_cfg()
    cam = cams[0]
    ren = sgs.Renderer(async_mode=True, track_reuse=True)
    t, sf = to_device(sc)
    tiles = ((cam.width + 15) // 16) * ((cam.height + 15) // 16)
    T_tgt = scenegen.perturb_pose(cam.T_cw, tau0(info.get("tau0_seed", 2000)))
    tgt = oracle.render(sc, oracle.make_cam(cam, T_tgt), cfg, counters=False)["img"].astype(np.float32).astype(np.float64)
    trgb = torch.from_numpy(tgt[0:3].astype(np.float32)).cuda()
    tdep = torch.from_numpy(tgt[3:4].astype(np.float32)).cuda()
    step = np.array([0.004, -0.005, 0.004, 0.003, 0.002, -0.003])
    try:
        ren.track_new_frame()
        for it in range(3):
            T = scenegen.perturb_pose(cam.T_cw, it * step) if it else cam.T_cw
            camv, c = oracle.make_cam(cam, T), camera(cam, T)
            im, upi = alloc_images(cam), alloc_images(cam)
            p6, loss = torch.zeros(6, device="cuda"), torch.zeros(1, device="cuda")
            for _ in range(4):   # (async mode: an overflow of the first iteration is reported by the next call)
                try:
                    ren.track_iter(sf, c, trgb, tdep, LAMBDA_D, NSIGN, p6, loss, **im)
                    ren.stats()
                    ren.track_iter(sf, c, trgb, tdep, LAMBDA_D, NSIGN, p6, loss, **im)
                    break
                except sgs.SgsError as e:
                    if e.status != sgs.SGS_WORKSPACE_OVERFLOW:
                        raise
            torch.cuda.synchronize()
            ob = oracle.binning(sc, camv, cfg)
            assert_binning(ren.get_binning(sc.n, tiles), ob)
            o = oracle.render(sc, camv, cfg)
            assert_image_check(image_check(planes(im), o["img"], o["fragile"], oracle.pixel_bounds(sc, camv, cfg)), (name, it))
            tr = tracking_reference(sc, camv, cfg, o, tgt, LAMBDA_D, NSIGN, oracle)
            l2 = torch.zeros(1, device="cuda")
            ren.tracking_loss(c, im, trgb, tdep, LAMBDA_D, NSIGN, upi, l2)     # which masks / signs came out differently
            D = tracking_flips(tr, planes(upi))
            assert D.any(0).mean() < 2e-4
            pose_slack, loss_slack = tracking_slack(sc, camv, cfg, tr, D, oracle)
            assert abs(float(loss.item()) - tr["L"]) <= tr["loss_tol"] + loss_slack
            assert_pose(p6.cpu().numpy().astype(np.float64), tr["og"]["pose"], tr["ex"]["pose"] + pose_slack / C_EXPO, (name, it))
    finally:
        ren.close()
