"""GPU parity: the CUDA path (through the C ABI binding) against the CPU oracle, element by element,
on the same seeded inputs.  Bars (BASELINE.json north_star): binning bit-exact; images
1e-4 rel / 1e-5 abs on every non-fragile pixel, fragile pixels within the oracle-derived allowance
(oracle.pixel_bounds); EVERY gradient element within 1e-3 rel (+1e-3 RMS(group) floor) plus the oracle-derived
exposure of the fragile pixels (oracle.exposure), which is zero for most elements and asserted small in total.
Nothing the CUDA path produced is ever an input of the oracle."""
import numpy as np
import pytest
import torch

import oracle
import scenegen
from scenegen import Scene, Camera

pytestmark = pytest.mark.gpu

sgs = pytest.importorskip("paper_2506_00970_b200")
from gpu_common import (to_device, camera, alloc_images, planes, alloc_grads, split_upstream, image_check,  # noqa: E402
                        assert_image_check, assert_grads, assert_pose, tracking_reference, tracking_flips, tracking_slack, C_EXPO)


@pytest.fixture(scope="module")
def ren():
    r = sgs.Renderer()
    yield r
    r.close()


def run_gpu(ren, sc, cam, up=None, full=True, pose=True, T_cw=None):
    t, sf = to_device(sc)
    c = camera(cam, T_cw)
    im = alloc_images(cam)
    ren.render(sf, c, **im)
    tiles = ((cam.width + 15) // 16) * ((cam.height + 15) // 16)
    out = dict(img=planes(im), bin=ren.get_binning(sc.n, tiles), stats=ren.stats())
    if up is not None:
        g = alloc_grads(sc.n) if full else None
        p6 = torch.full((6,), 3.0, device="cuda") if pose else None
        ren.backward(**split_upstream(up), grads=g, d_pose6=p6)
        torch.cuda.synchronize()
        if g is not None:
            out["grads"] = {k: v.cpu().numpy() for k, v in g.items()}
        if p6 is not None:
            out["pose"] = p6.cpu().numpy().astype(np.float64)
    return out


def assert_binning(gb, ob):
    assert gb["E"] == ob["E"]
    assert np.array_equal(gb["culled"], ob["culled"])
    assert np.array_equal(gb["keys"], ob["keys"])
    assert np.array_equal(gb["idx"], ob["idx"])
    assert np.array_equal(gb["ranges"], ob["ranges"])


def assert_images(gpu_img, o, sc, camv, cfg, ctx=None):
    assert_image_check(image_check(gpu_img, o["img"], o["fragile"], oracle.pixel_bounds(sc, camv, cfg)), ctx)


POSES = [None, [0.1, -0.2, 0.15, 0.2, -0.1, 0.3]]


@pytest.mark.parametrize("tau", POSES)
def test_c1_full(ren, tau):
    """Config 1: binning bit-exact, images, all surfel gradients and the pose gradient."""
    sc, cams, _ = scenegen.make_config("C1")
    cam = cams[0]
    T = None if tau is None else scenegen.perturb_pose(cam.T_cw, tau)
    camv, cfg = oracle.make_cam(cam, T), oracle.make_cfg()
    up = scenegen.upstream_normal(1, cam.height, cam.width)
    out = run_gpu(ren, sc, cam, up, T_cw=T)
    assert_binning(out["bin"], oracle.binning(sc, camv, cfg))
    o = oracle.render(sc, camv, cfg)
    assert_images(out["img"], o, sc, camv, cfg)
    og, ex = oracle.backward(sc, camv, cfg, up), oracle.exposure(sc, camv, cfg, up)
    assert_grads(out["grads"], og, ex)
    assert_pose(out["pose"], og["pose"], ex["pose"])
    # pose-only mode (per-pixel Eq. 11-13) against the same oracle
    out2 = run_gpu(ren, sc, cam, up, full=False, T_cw=T)
    assert_pose(out2["pose"], og["pose"], ex["pose"])


@pytest.mark.parametrize("tau", POSES)
def test_c1_tight_binning(tau):
    """SGS_FLAG_TIGHT_BINNING on C1 (opacities 0.1 .. 0.99, so the opacity-aware cutoff bites): the list is the oracle's tight
    list bit for bit and a strict subset of the default one; images are BIT-IDENTICAL to the default binning's on the GPU too
    (the dropped entries composite nothing); gradients and pose against the oracle."""
    sc, cams, _ = scenegen.make_config("C1")
    cam = cams[0]
    T = None if tau is None else scenegen.perturb_pose(cam.T_cw, tau)
    camv, cfgt = oracle.make_cam(cam, T), oracle.make_cfg(tight=True)
    up = scenegen.upstream_normal(1, cam.height, cam.width)
    rt, rd = sgs.Renderer(tight_binning=True), sgs.Renderer()
    out, ref = run_gpu(rt, sc, cam, up, T_cw=T), run_gpu(rd, sc, cam, up, T_cw=T)
    ob = oracle.binning(sc, camv, cfgt)
    assert_binning(out["bin"], ob)
    assert out["bin"]["E"] < 0.9 * ref["bin"]["E"]
    assert np.array_equal(out["img"], ref["img"])
    o = oracle.render(sc, camv, cfgt)
    assert_images(out["img"], o, sc, camv, cfgt)
    og, ex = oracle.backward(sc, camv, cfgt, up), oracle.exposure(sc, camv, cfgt, up)
    assert_grads(out["grads"], og, ex)
    assert_pose(out["pose"], og["pose"], ex["pose"])
    # a splat below alpha_min is culled by the tight binning and composites nothing under the default one
    faint = Scene(sc.mean[:50], sc.scale[:50], sc.quat[:50], np.full(50, 0.003, np.float32), sc.rgb[:50])
    a, b = run_gpu(rt, faint, cam), run_gpu(rd, faint, cam)
    assert a["bin"]["E"] == 0 and a["bin"]["culled"].all() and b["bin"]["E"] > 0 and (a["img"] == 0).all() and (b["img"] == 0).all()
    with pytest.raises(sgs.SgsError):
        sgs.Renderer(tight_binning=True, radix_binning=True)
    rt.close(); rd.close()


def test_c2_tracking_shape(ren):
    """Config 2 (200k surfels, 640x480): binning, images, tracking loss (Eq. 15-19), pose-only backward -- each stage on
    the ORACLE's inputs: the loss kernel is run on the oracle's image (rounded to binary32), the backward on the oracle's
    upstream gradients; the fused paths, which evaluate the loss on the renderer's own image, may differ from the oracle only
    through masks / signs that sit inside the image bar (tracking_flips asserts that), by at most tracking_slack."""
    sc, cams, info = scenegen.make_config("C2")
    cam = cams[0]
    camv, cfg = oracle.make_cam(cam), oracle.make_cfg()
    # target frame: the oracle's own render at the perturbed pose Exp(tau0) T, as binary32 (what the C ABI carries)
    g = scenegen.SplitMix(info["tau0_seed"])
    d = np.stack([g.normal(3), g.normal(3)])
    tau0 = np.concatenate([0.02 * d[0] / np.linalg.norm(d[0]), np.deg2rad(1.0) * d[1] / np.linalg.norm(d[1])])
    T_tgt = scenegen.perturb_pose(cam.T_cw, tau0)
    tgt = oracle.render(sc, oracle.make_cam(cam, T_tgt), cfg, counters=False)["img"].astype(np.float32).astype(np.float64)
    t, sf = to_device(sc)
    c = camera(cam)
    im, upi = alloc_images(cam), alloc_images(cam)
    ren.render(sf, c, **im)
    tiles = ((cam.width + 15) // 16) * ((cam.height + 15) // 16)
    assert_binning(ren.get_binning(sc.n, tiles), oracle.binning(sc, camv, cfg))
    o = oracle.render(sc, camv, cfg)
    gimg = planes(im)
    assert_images(gimg, o, sc, camv, cfg)
    tr = tracking_reference(sc, camv, cfg, o, tgt, 0.5, -1.0, oracle)
    L_ref, up_ref, og = tr["L"], tr["up"], tr["og"]
    assert (up_ref != 0).mean() > 0.05
    trgb = torch.from_numpy(tgt[0:3].astype(np.float32)).cuda()
    tdep = torch.from_numpy(tgt[3:4].astype(np.float32)).cuda()
    # loss kernel on the ORACLE's image as binary32: same masks and signs except where the rounding of the image itself
    # crosses a threshold (candidates only), same loss
    o32 = o["img"].astype(np.float32)
    oim = dict(rgb=torch.from_numpy(o32[0:3]).cuda(), depth=torch.from_numpy(o32[3:4]).cuda(),
               normal=torch.from_numpy(o32[4:7]).cuda(), alpha=torch.from_numpy(o32[7:8]).cuda())
    loss = torch.zeros(1, device="cuda")
    ren.tracking_loss(c, oim, trgb, tdep, 0.5, -1.0, upi, loss)
    D0 = tracking_flips(tr, planes(upi))
    assert D0.sum() <= 1e-4 * D0[0].size and abs(float(loss.item()) - L_ref) <= 1e-5 * abs(L_ref) + tracking_slack(sc, camv, cfg, tr, D0, oracle)[1]
    same = ~D0.any(0)
    assert np.abs(planes(upi) - up_ref)[:, same].max() <= 1e-6 * np.abs(up_ref).max()
    # pose-only backward on the oracle's upstream gradients vs the oracle's analytic backward
    u = torch.from_numpy(up_ref.astype(np.float32)).cuda()
    og32 = oracle.backward(sc, camv, cfg, u.cpu().numpy().astype(np.float64))
    p6 = torch.zeros(6, device="cuda")
    ren.backward(d_rgb=u[0:3].contiguous(), d_depth=u[3:4].contiguous(), d_normal=u[4:7].contiguous(),
                 d_alpha=u[7:8].contiguous(), d_pose6=p6)
    assert_pose(p6.cpu().numpy(), og32["pose"], tr["ex"]["pose"])
    # the renderer's own loss on its own image: which masks / signs came out differently, and what that may change
    ren.tracking_loss(c, im, trgb, tdep, 0.5, -1.0, upi, loss.zero_())
    D = tracking_flips(tr, planes(upi))
    pose_slack, loss_slack = tracking_slack(sc, camv, cfg, tr, D, oracle)
    assert abs(float(loss.item()) - L_ref) <= tr["loss_tol"] + loss_slack
    # fused loss + backward (sgs_backward_tracking) == loss kernel followed by backward, and == the oracle
    p6f, lossf = torch.zeros(6, device="cuda"), torch.zeros(1, device="cuda")
    ren.backward_tracking(trgb, tdep, 0.5, -1.0, p6f, lossf)
    assert abs(float(lossf.item()) - L_ref) <= tr["loss_tol"] + loss_slack
    assert_pose(p6f.cpu().numpy(), og["pose"], tr["ex"]["pose"] + pose_slack / C_EXPO)
    p6u = torch.zeros(6, device="cuda")
    ren.backward(d_rgb=upi["rgb"], d_depth=upi["depth"], d_normal=upi["normal"], d_alpha=upi["alpha"], d_pose6=p6u)
    np.testing.assert_allclose(p6f.cpu().numpy(), p6u.cpu().numpy(), rtol=1e-4, atol=1e-6 * float(p6u.abs().max()))


def test_backward_is_repeatable_and_overwrites(ren):
    sc, cams, _ = scenegen.make_config("C1")
    cam = cams[0]
    up = scenegen.upstream_normal(4, cam.height, cam.width)
    t, sf = to_device(sc)
    ren.render(sf, camera(cam), **alloc_images(cam))
    res = []
    for _ in range(2):
        g, p6 = alloc_grads(sc.n), torch.full((6,), 9.0, device="cuda")
        ren.backward(**split_upstream(up), grads=g, d_pose6=p6)
        res.append(({k: v.cpu().numpy() for k, v in g.items()}, p6.cpu().numpy()))
    for k in res[0][0]:
        np.testing.assert_allclose(res[0][0][k], res[1][0][k], rtol=1e-4, atol=1e-4 * np.abs(res[0][0][k]).max())
    np.testing.assert_allclose(res[0][1], res[1][1], rtol=1e-4)
    culled = ren.get_binning(sc.n, 12)["culled"].astype(bool)
    assert culled.any()
    for k in res[0][0]:
        assert (res[0][0][k][culled] == 0).all()     # exactly zero for culled surfels


def test_mask_equals_compacted_subset(ren):
    """L204/L161: inactive splats contribute nothing -- render(all, mask) == render(active subset) bit for bit."""
    sc, cams, _ = scenegen.make_config("C1")
    cam = cams[0]
    act = (scenegen.SplitMix(99).uniform(sc.n) < 0.3).astype(np.uint8)
    m = act.astype(bool)
    masked = Scene(sc.mean, sc.scale, sc.quat, sc.opacity, sc.rgb, act)
    sub = Scene(sc.mean[m], sc.scale[m], sc.quat[m], sc.opacity[m], sc.rgb[m])
    up = scenegen.upstream_normal(5, cam.height, cam.width)
    a, b = run_gpu(ren, masked, cam, up), run_gpu(ren, sub, cam, up)
    assert np.array_equal(a["img"], b["img"])
    assert np.array_equal(a["bin"]["keys"], b["bin"]["keys"])
    assert np.array_equal(a["bin"]["idx"], np.nonzero(m)[0][b["bin"]["idx"]])
    for k in a["grads"]:
        assert (a["grads"][k][~m] == 0).all()
    assert_binning(a["bin"], oracle.binning(masked, oracle.make_cam(cam), oracle.make_cfg()))


def test_edge_cases(ren):
    cam = Camera(70, 50, 60.0, 60.0, 35.0, 25.0)     # ragged: 70 = 4.375 tiles, 50 = 3.125 tiles
    cfg = oracle.make_cfg()
    # empty map
    empty = Scene(*[np.zeros(s, np.float32) for s in ((0, 3), (0, 2), (0, 4), (0,), (0, 3))])
    out = run_gpu(ren, empty, cam, scenegen.upstream_normal(1, 50, 70), full=True)
    assert out["bin"]["E"] == 0 and (out["img"] == 0).all() and (out["pose"] == 0).all()
    # everything behind the camera / off-screen -> all culled
    sc = scenegen.tiny_scene(3, 500)
    behind = Scene(sc.mean * np.float32([1, 1, -1]), sc.scale, sc.quat, sc.opacity, sc.rgb)
    out = run_gpu(ren, behind, cam, scenegen.upstream_normal(1, 50, 70))
    assert out["bin"]["E"] == 0 and out["bin"]["culled"].all() and (out["img"] == 0).all()
    assert all((v == 0).all() for v in out["grads"].values())
    # ragged image, degenerate inputs: zero quaternion, NaN mean, huge and tiny scales, opacity 1 (clamp)
    sc = scenegen.tiny_scene(7, 3000)
    sc.quat[5] = 0; sc.mean[6] = np.nan; sc.scale[7] = 5.0; sc.scale[8] = 1e-5; sc.opacity[:50] = 1.0
    sc.mean[9] = [0.0, 0.0, 0.25]; sc.scale[9] = 0.5   # disk crossing the camera plane
    camv = oracle.make_cam(cam)
    up = scenegen.upstream_normal(2, 50, 70)
    out = run_gpu(ren, sc, cam, up)
    ob = oracle.binning(sc, camv, cfg)
    assert_binning(out["bin"], ob)
    assert ob["culled"][5] and ob["culled"][6]
    assert_images(out["img"], oracle.render(sc, camv, cfg), sc, camv, cfg)
    og, ex = oracle.backward(sc, camv, cfg, up), oracle.exposure(sc, camv, cfg, up)
    assert_grads(out["grads"], og, ex)
    assert_pose(out["pose"], og["pose"], ex["pose"])


def test_invalid_arguments(ren):
    sc, cams, _ = scenegen.make_config("C1")
    t, sf = to_device(sc)
    bad = sgs.make_camera(0, 48, 60, 60, 32, 24, np.eye(4)[:3])
    with pytest.raises(sgs.SgsError) as e:
        ren.render(sf, bad)
    assert e.value.status == sgs.SGS_INVALID_ARGUMENT
    fresh = sgs.Renderer()
    with pytest.raises(sgs.SgsError) as e:
        fresh.backward(d_pose6=torch.zeros(6, device="cuda"))
    assert e.value.status == sgs.SGS_NO_FORWARD_STATE
    # the other documented refusals: a map of 2^24 or more splats (the tile keys hold 24 index bits), an image beyond 16384
    # pixels on a side, non-finite pose entries, accumulate without gradient arrays, a window fetch / staging probe without
    # the state they need
    import ctypes as C
    big = sgs.sgs_surfels()
    C.memmove(C.byref(big), C.byref(sf), C.sizeof(big))
    big.n = 1 << 24
    cam_ok = sgs.make_camera(64, 48, 60, 60, 32, 24, np.eye(4)[:3])
    for bad_sf, bad_cam in ((big, cam_ok), (sf, sgs.make_camera(20000, 48, 60, 60, 32, 24, np.eye(4)[:3])),
                            (sf, sgs.make_camera(64, 48, 60, 60, 32, 24, np.full((3, 4), np.nan)))):
        with pytest.raises(sgs.SgsError) as e:
            fresh.render(bad_sf, bad_cam)
        assert e.value.status == sgs.SGS_INVALID_ARGUMENT
    fresh.render(sf, cam_ok)
    with pytest.raises(sgs.SgsError) as e:
        fresh.backward(d_pose6=torch.zeros(6, device="cuda"), accumulate=True)          # no gradient arrays to add to
    assert e.value.status == sgs.SGS_INVALID_ARGUMENT
    other = sgs.Renderer()
    for call in (lambda: other.probe_staging(0), lambda: other.fetch_grads_host({"mean": torch.zeros(sc.n, 3).pin_memory()})):
        with pytest.raises(sgs.SgsError) as e:
            call()
        assert e.value.status == sgs.SGS_NO_FORWARD_STATE
    with pytest.raises(sgs.SgsError) as e:
        other.probe_staging(2)
    assert e.value.status == sgs.SGS_INVALID_ARGUMENT
    other.close()
    fresh.close()


def test_async_mode_and_host_path():
    """SGS_FLAG_ASYNC gives the same result without a host sync; the HOST-buffer calls equal the device calls."""
    sc, cams, _ = scenegen.make_config("C1")
    cam = cams[0]
    up = scenegen.upstream_normal(6, cam.height, cam.width)
    sync = sgs.Renderer()
    ref = run_gpu(sync, sc, cam, up)
    a = sgs.Renderer(async_mode=True)
    for _ in range(3):
        out = run_gpu(a, sc, cam, up)
    assert np.array_equal(out["img"], ref["img"]) and np.array_equal(out["bin"]["keys"], ref["bin"]["keys"])
    # host path
    pin = lambda x, dt=torch.float32: torch.from_numpy(np.ascontiguousarray(x)).to(dt).pin_memory()
    a.upload_surfels(pin(sc.mean), pin(sc.scale), pin(sc.quat), pin(sc.opacity), pin(sc.rgb))
    c = camera(cam)
    H, W = cam.height, cam.width
    h = dict(rgb=torch.zeros(3, H, W).pin_memory(), depth=torch.zeros(1, H, W).pin_memory(),
             normal=torch.zeros(3, H, W).pin_memory(), alpha=torch.zeros(1, H, W).pin_memory())
    a.render_host(c, **h)
    himg = torch.cat([h["rgb"], h["depth"], h["normal"], h["alpha"]], 0).numpy().astype(np.float64)
    assert np.array_equal(himg, ref["img"])
    u = torch.from_numpy(up)
    hg = {k: torch.zeros(v.shape).pin_memory() for k, v in ref["grads"].items()}
    hp = torch.zeros(6).pin_memory()
    a.backward_host(d_rgb=u[0:3].contiguous(), d_depth=u[3:4].contiguous(), d_normal=u[4:7].contiguous(),
                    d_alpha=u[7:8].contiguous(), grads=hg, d_pose6=hp)
    for k in hg:
        np.testing.assert_allclose(hg[k].numpy(), ref["grads"][k], rtol=1e-4, atol=1e-4 * np.abs(ref["grads"][k]).max())
    np.testing.assert_allclose(hp.numpy(), ref["pose"], rtol=1e-4)
    # tracking iteration on resident map/target
    a.upload_target(c, h["rgb"] * 0.9, h["depth"] * 1.01)
    loss, p6 = a.track_iter_host(c, 0.5, 1.0)
    assert np.isfinite(loss) and np.isfinite(p6).all()
    sync.close(); a.close()


@pytest.mark.parametrize("name,n_override", [("C2", 60000), ("C3", None)])
def test_radix_binning_path_gives_the_same_list(name, n_override):
    """SGS_FLAG_RADIX_BINNING (global LSD radix sort of the 64-bit tile|depth keys) and the default
    per-tile buckets + in-tile sort produce the identical sorted list, images and gradients -- on a small map and on C3
    view 0 at full size (3225 tiles = 12 tile bits, E = 0.74 M: multi-tile look-back chains in every pass)."""
    sc, cams, _ = scenegen.make_config(name, n_override=n_override) if n_override else scenegen.make_config(name)
    cam = cams[0]
    up = scenegen.upstream_normal(8, cam.height, cam.width)
    a, b = sgs.Renderer(), sgs.Renderer(radix_binning=True)
    ra, rb = run_gpu(a, sc, cam, up), run_gpu(b, sc, cam, up)
    assert_binning(ra["bin"], rb["bin"])
    assert_binning(rb["bin"], oracle.binning(sc, oracle.make_cam(cam), oracle.make_cfg()))
    assert np.array_equal(ra["img"], rb["img"])
    np.testing.assert_allclose(ra["pose"], rb["pose"], rtol=1e-4)
    for k in ra["grads"]:
        np.testing.assert_allclose(ra["grads"][k], rb["grads"][k], rtol=1e-3, atol=1e-4 * np.abs(ra["grads"][k]).max())
    a.close(); b.close()


def test_track_helpers_wait_for_their_owner(monkeypatch):
    """K-track's helper blocks (second half of the walk back of the 32 longest tile lists) read the tile's bucket only
    after the owner block has published the SORTED keys, and the hand-over flags are built from a device-side epoch.  With
    every helper delayed by 0.2 ms (SGS_DEBUG_HELPER_DELAY_NS: the owners are long past their sort, mid-way through their
    walks) and over several back-to-back iterations the pose gradient, loss, images and binning equal those of an
    undelayed context -- a helper that ranked a half-permuted bucket, or met a stale flag, would not."""
    sc, cams, info = scenegen.make_config("C2")
    cam = cams[0]
    camv, cfg = oracle.make_cam(cam), oracle.make_cfg()
    ob = oracle.binning(sc, camv, cfg)
    lens = ob["ranges"][:, 1].astype(np.int64) - ob["ranges"][:, 0]
    assert (lens > 160).sum() >= 4 and lens.max() <= 384          # tiles that split between owner and helper exist
    t, sf = to_device(sc)
    c = camera(cam)
    tiles = ((cam.width + 15) // 16) * ((cam.height + 15) // 16)
    ref = sgs.Renderer()
    im0 = alloc_images(cam)
    ref.render(sf, c, **im0)
    tgt_rgb, tgt_dep = (im0["rgb"] * 0.9 + 0.01).contiguous(), (im0["depth"] * 1.02).contiguous()
    pr, lr = torch.zeros(6, device="cuda"), torch.zeros(1, device="cuda")
    for _ in range(3):
        ref.track_iter(sf, c, tgt_rgb, tgt_dep, 0.5, -1.0, pr, lr)
    monkeypatch.setenv("SGS_DEBUG_HELPER_DELAY_NS", "200000")
    slow = sgs.Renderer()
    monkeypatch.delenv("SGS_DEBUG_HELPER_DELAY_NS")
    for it in range(4):
        im = alloc_images(cam)
        p6, loss = torch.zeros(6, device="cuda"), torch.zeros(1, device="cuda")
        slow.track_iter(sf, c, tgt_rgb, tgt_dep, 0.5, -1.0, p6, loss, **im)
        torch.cuda.synchronize()
        assert np.array_equal(planes(im), planes(im0))
        np.testing.assert_allclose(loss.cpu().numpy(), lr.cpu().numpy(), rtol=1e-5)
        np.testing.assert_allclose(p6.cpu().numpy(), pr.cpu().numpy(), rtol=1e-4, atol=1e-6 * float(pr.abs().max()))
    assert_binning(slow.get_binning(sc.n, tiles), ob)
    ref.close(); slow.close()


def test_tile_bucket_overflow_grows(ren):
    """Many surfels stacked on one tile overflow the initial per-tile capacity: the sync path regrows and
    re-emits; the async path reports SGS_WORKSPACE_OVERFLOW on the next call and then succeeds."""
    g = scenegen.SplitMix(5)
    n = 6000
    mean = np.stack([g.uniform(n, -0.02, 0.02), g.uniform(n, -0.02, 0.02), g.uniform(n, 1.0, 3.0)], 1).astype(np.float32)
    sc = Scene(mean, np.full((n, 2), 0.01, np.float32), np.tile(np.float32([1, 0, 0, 0]), (n, 1)),
               np.full(n, 0.05, np.float32), np.full((n, 3), 0.5, np.float32))
    cam = Camera(64, 48, 60.0, 60.0, 32.0, 24.0)
    camv, cfg = oracle.make_cam(cam), oracle.make_cfg()
    out = run_gpu(sgs.Renderer(), sc, cam)
    ob = oracle.binning(sc, camv, cfg)
    assert (ob["ranges"][:, 1] - ob["ranges"][:, 0]).max() > 2048
    assert_binning(out["bin"], ob)
    assert_images(out["img"], oracle.render(sc, camv, cfg), sc, camv, cfg)
    a = sgs.Renderer(async_mode=True)
    t, sf = to_device(sc)
    im = alloc_images(cam)
    a.render(sf, camera(cam), **im)
    with pytest.raises(sgs.SgsError) as e:
        a.render(sf, camera(cam), **im)
    assert e.value.status == sgs.SGS_WORKSPACE_OVERFLOW
    a.render(sf, camera(cam), **im)
    a.stats()
    assert np.array_equal(planes(im), out["img"])
    a.close()
    # the same through sgs_prepare: the render that follows reports the overflow of the prepared binning before it
    # composites anything; rendering again bins in line with the grown buckets
    b = sgs.Renderer(async_mode=True)
    c = camera(cam)
    im.update(alloc_images(cam))
    b.prepare(sf, c)
    with pytest.raises(sgs.SgsError) as e:
        b.render(sf, c, **im)
    assert e.value.status == sgs.SGS_WORKSPACE_OVERFLOW
    assert float(im["alpha"].abs().max()) == 0.0   # nothing was composited
    b.render(sf, c, **im)
    b.stats()
    assert np.array_equal(planes(im), out["img"])
    b.close()


@pytest.mark.parametrize("crowded", [False, True])
def test_fused_sort_of_long_buckets(ren, crowded):
    """Buckets of 129..2048 keys take the counting sort of histsort.cuh inside k_forward; a bucket whose depths crowd into
    one bin (here 400 splats at exactly the same depth beside a wide depth range) is declined by it and takes the bitonic
    networks.  Either way the exported lists equal the oracle's bit for bit and the images meet the image bar."""
    g = scenegen.SplitMix(11)
    n = 1500
    z = g.uniform(n, 1.0, 3.0)
    if crowded:
        z[:400] = 2.0
    x = g.uniform(n, -0.02, 0.02)
    x[1100:] += 0.35 * z[1100:]               # 400 of them project 21 px to the right: a tile of their own
    mean = np.stack([x, g.uniform(n, -0.02, 0.02), z], 1).astype(np.float32)
    sc = Scene(mean, np.full((n, 2), 0.01, np.float32), np.tile(np.float32([1, 0, 0, 0]), (n, 1)),
               np.full(n, 0.05, np.float32), np.full((n, 3), 0.5, np.float32))
    cam = Camera(64, 48, 60.0, 60.0, 32.0, 24.0)
    camv, cfg = oracle.make_cam(cam), oracle.make_cfg()
    ob = oracle.binning(sc, camv, cfg)
    ln = ob["ranges"][:, 1] - ob["ranges"][:, 0]
    assert ln.max() <= 2048 and (ln > 512).any() and ((ln > 128) & (ln <= 512)).any()
    if crowded:   # the 400 equal depths share a tile: more than HS_MAX_BIN = 96 keys in one depth bin
        s0, e0 = ob["ranges"][int(np.argmax(ln))]
        d = ob["keys"][s0:e0] & 0xffffffff
        assert np.bincount((d - d.min()).astype(np.int64) >> max(0, int(d.max() - d.min()).bit_length() - 10)).max() > 96
    out = run_gpu(ren, sc, cam)
    assert_binning(out["bin"], ob)
    assert_images(out["img"], oracle.render(sc, camv, cfg), sc, camv, cfg)


def test_track_iter_matches_unfused_sequence():
    """sgs_track_iter == sgs_render + sgs_backward_tracking on C1 (short lists) and on a tile list longer than one
    256-entry batch and longer than the in-kernel sort bound (bucket regrowth -> pre-sorted path)."""
    cases = []
    sc, cams, _ = scenegen.make_config("C1")
    cases.append((sc, cams[0]))
    g = scenegen.SplitMix(11)
    # ~n entries on the central tiles: multi-batch (ordered inside k_track by the counting sort of histsort.cuh; the second 900
    # has 400 splats at one depth, which that sort declines: the bitonic network); > 2048 -> tilesort pre-pass
    for n, crowded in ((900, False), (900, True), (6000, False)):
        z = g.uniform(n, 1.0, 3.0)
        if crowded:
            z[:400] = 2.0
        mean = np.stack([g.uniform(n, -0.05, 0.05), g.uniform(n, -0.05, 0.05), z], 1).astype(np.float32)
        cases.append((Scene(mean, np.full((n, 2), 0.01, np.float32), np.tile(np.float32([1, 0.1, 0, 0]), (n, 1)),
                            np.full(n, 0.03 if n > 2000 else 0.2, np.float32),
                            np.stack([g.uniform(n) for _ in range(3)], 1).astype(np.float32)),
                      Camera(64, 48, 60.0, 60.0, 32.0, 24.0)))
    for sc, cam in cases:
        ren = sgs.Renderer()
        t, sf = to_device(sc)
        c = camera(cam)
        im, im2 = alloc_images(cam), alloc_images(cam)
        ren.render(sf, c, **im)
        tgt_rgb = (im["rgb"] * 0.9 + 0.01).contiguous()
        tgt_dep = (im["depth"] * 1.02).contiguous()
        p6a, la = torch.zeros(6, device="cuda"), torch.zeros(1, device="cuda")
        ren.backward_tracking(tgt_rgb, tgt_dep, 0.5, 1.0, p6a, la)
        p6b, lb = torch.zeros(6, device="cuda"), torch.zeros(1, device="cuda")
        ren.track_iter(sf, c, tgt_rgb, tgt_dep, 0.5, 1.0, p6b, lb, **im2)
        torch.cuda.synchronize()
        assert np.array_equal(planes(im), planes(im2))
        assert float(la.abs().item()) > 0 and np.abs(p6a.cpu().numpy()).max() > 0
        np.testing.assert_allclose(lb.cpu().numpy(), la.cpu().numpy(), rtol=1e-5)
        np.testing.assert_allclose(p6b.cpu().numpy(), p6a.cpu().numpy(), rtol=1e-4, atol=1e-6 * float(p6a.abs().max()))
        with pytest.raises(sgs.SgsError) as e:   # track_iter leaves no state for sgs_backward
            ren.backward(d_pose6=p6a)
        assert e.value.status == sgs.SGS_NO_FORWARD_STATE
        ren.close()


def test_random_poses_binning_and_images(ren):
    """Eight seeded random camera poses inside a 30 k-surfel room (looking at every wall, rolled, close to
    surfaces): binning bit-exact and images within the bar at each -- guards the conservative binary32 pre-cull
    and the two-kernel preprocess against view-dependent mistakes."""
    sc, _, _ = scenegen.make_config("C2", n_override=30000)
    g = scenegen.SplitMix(4242)
    cfg = oracle.make_cfg()
    t, sf = to_device(sc)
    for k in range(8):
        eye = np.array([g.uniform(1, 0.3, 4.7)[0], g.uniform(1, 0.3, 3.7)[0], g.uniform(1, 0.3, 2.7)[0]])
        tgt = np.array([g.uniform(1, -1.0, 6.0)[0], g.uniform(1, -1.0, 5.0)[0], g.uniform(1, -1.0, 4.0)[0]])
        T = scenegen.look_at(eye, tgt).astype(np.float64)
        roll = scenegen.se3_exp(np.array([0, 0, 0, 0, 0, g.uniform(1, -np.pi, np.pi)[0]]))[:3, :3]
        T = np.concatenate([roll @ T[:, :3], (roll @ T[:, 3])[:, None]], axis=1)
        cam = Camera(200 + 16 * k + (k % 3), 150 + 7 * k, 180.0 + 10 * k, 175.0 + 9 * k, 100.0 + 3 * k, 75.0 - 2 * k,
                     T.astype(np.float32))
        camv = oracle.make_cam(cam)
        im = alloc_images(cam)
        ren.render(sf, camera(cam), **im)
        tiles = ((cam.width + 15) // 16) * ((cam.height + 15) // 16)
        ob = oracle.binning(sc, camv, cfg)
        assert ob["E"] > 1000
        assert_binning(ren.get_binning(sc.n, tiles), ob)
        assert_images(planes(im), oracle.render(sc, camv, cfg), sc, camv, cfg, k)


@pytest.mark.parametrize("reuse", [False, True])
def test_track_iter_edge_cases(reuse):
    """sgs_track_iter on an empty map, an all-culled map and a ragged image (70x50: partial tiles); with and without
    SGS_FLAG_TRACK_REUSE (each case twice in a row, so that the second call runs from the kept list)."""
    cam = Camera(70, 50, 60.0, 60.0, 35.0, 25.0)
    c = camera(cam)
    tgt_rgb = torch.full((3, 50, 70), 0.3, device="cuda")
    tgt_dep = torch.full((1, 50, 70), 1.5, device="cuda")
    ren = sgs.Renderer(track_reuse=reuse)
    empty = Scene(*[np.zeros(s, np.float32) for s in ((0, 3), (0, 2), (0, 4), (0,), (0, 3))])
    sc = scenegen.tiny_scene(3, 500)
    behind = Scene(sc.mean * np.float32([1, 1, -1]), sc.scale, sc.quat, sc.opacity, sc.rgb)
    for scene in (empty, behind):
        t, sf = to_device(scene)
        im = alloc_images(cam)
        im["rgb"].fill_(9.0)
        for _ in range(2):
            im["rgb"].fill_(9.0)
            p6, loss = torch.full((6,), 3.0, device="cuda"), torch.full((1,), 3.0, device="cuda")
            ren.track_iter(sf, c, tgt_rgb, tgt_dep, 0.5, 1.0, p6, loss, **im)
            torch.cuda.synchronize()
            assert (planes(im) == 0).all() and (p6 == 0).all() and float(loss.item()) == 0.0
    # ragged image, dense enough that many pixels pass M_o: fused == unfused
    sc = scenegen.tiny_scene(7, 6000)
    sc.opacity[:] = 0.9
    t, sf = to_device(sc)
    im, im2 = alloc_images(cam), alloc_images(cam)
    ren.render(sf, c, **im)
    assert float((im["alpha"] > 0.95).float().mean()) > 0.05
    pa, la = torch.zeros(6, device="cuda"), torch.zeros(1, device="cuda")
    ren.backward_tracking(tgt_rgb, tgt_dep, 0.5, 1.0, pa, la)
    for _ in range(2):
        pb, lb = torch.zeros(6, device="cuda"), torch.zeros(1, device="cuda")
        ren.track_iter(sf, c, tgt_rgb, tgt_dep, 0.5, 1.0, pb, lb, **im2)
        assert np.array_equal(planes(im), planes(im2))
        np.testing.assert_allclose(lb.cpu().numpy(), la.cpu().numpy(), rtol=1e-5)
        np.testing.assert_allclose(pb.cpu().numpy(), pa.cpu().numpy(), rtol=1e-4, atol=1e-6 * float(pa.abs().max()))
    ren.close()


def test_stress_scene_masks_stay_conservative(ren):
    """Splats built to strain the culling and the two-stage warp-patch masks (slivers of 200:1, edge-on splats,
    sub-pixel and screen-filling splats, opacities around 1/255, splats at the near plane, splats reaching in from
    far outside the frustum): binning bit-exact, images, every gradient and both pose paths against the oracle, and
    the fused tracking kernel against the unfused sequence.  A mask that dropped one pair that eval_pair() accepts
    would show as an image error of a whole blending weight."""
    sc, cam = scenegen.stress_scene(), scenegen.stress_camera()
    for tau in (None, [0.05, -0.08, 0.1, 0.3, -0.2, 0.4]):
        T = None if tau is None else scenegen.perturb_pose(cam.T_cw, tau)
        camv, cfg = oracle.make_cam(cam, T), oracle.make_cfg()
        up = scenegen.upstream_normal(3, cam.height, cam.width)
        out = run_gpu(ren, sc, cam, up, T_cw=T)
        assert_binning(out["bin"], oracle.binning(sc, camv, cfg))
        o = oracle.render(sc, camv, cfg)
        chk = image_check(out["img"], o["img"], o["fragile"], oracle.pixel_bounds(sc, camv, cfg))
        # (this scene is BUILT of edge-on splats and slivers: 5-6 % of its pixels hold a pair with kappa > 32, so the
        # fragile fraction is the scene's, not the renderer's; the bound on those pixels is still the derived one)
        assert chk["n_bad"] == 0 and chk["n_bad_fragile"] == 0 and chk["fragile_frac"] < 0.08, chk
        og, ex = oracle.backward(sc, camv, cfg, up), oracle.exposure(sc, camv, cfg, up)
        assert_grads(out["grads"], og, ex)
        assert_pose(out["pose"], og["pose"], ex["pose"])
        out2 = run_gpu(ren, sc, cam, up, full=False, T_cw=T)
        assert_pose(out2["pose"], og["pose"], ex["pose"])
    r2 = sgs.Renderer()
    t, sf = to_device(sc)
    c = camera(cam)
    im, im2 = alloc_images(cam), alloc_images(cam)
    r2.render(sf, c, **im)
    tgt_rgb, tgt_dep = (im["rgb"] * 0.9 + 0.01).contiguous(), (im["depth"] * 1.02).contiguous()
    p6a, la = torch.zeros(6, device="cuda"), torch.zeros(1, device="cuda")
    r2.backward_tracking(tgt_rgb, tgt_dep, 0.5, 1.0, p6a, la)
    p6b, lb = torch.zeros(6, device="cuda"), torch.zeros(1, device="cuda")
    r2.track_iter(sf, c, tgt_rgb, tgt_dep, 0.5, 1.0, p6b, lb, **im2)
    torch.cuda.synchronize()
    assert np.array_equal(planes(im), planes(im2))
    np.testing.assert_allclose(lb.cpu().numpy(), la.cpu().numpy(), rtol=1e-5)
    np.testing.assert_allclose(p6b.cpu().numpy(), p6a.cpu().numpy(), rtol=1e-4, atol=1e-6 * float(p6a.abs().max()))
    r2.close()


def test_prepare_then_render_equals_render():
    """sgs_prepare (binning only, on a side stream) followed by sgs_render of the same view == plain sgs_render:
    binning and images bit-identical, gradients equal up to the order of the atomic sums; a render of ANOTHER view
    after a prepare bins again; two contexts alternating over a window of views reproduce the in-line sequence."""
    sc, cams, _ = scenegen.make_config("C1")
    cam = cams[0]
    t, sf = to_device(sc)
    tiles = ((cam.width + 15) // 16) * ((cam.height + 15) // 16)
    up = scenegen.upstream_normal(5, cam.height, cam.width)
    taus = [None, [0.05, 0.02, -0.04, 0.1, -0.05, 0.2], [-0.1, 0.05, 0.02, -0.2, 0.1, 0.05]]
    cs = [camera(cam, None if tau is None else scenegen.perturb_pose(cam.T_cw, tau)) for tau in taus]
    side = torch.cuda.Stream()

    def full(ren, c, prepared_on=None):
        im, g, p6 = alloc_images(cam), alloc_grads(sc.n), torch.zeros(6, device="cuda")
        if prepared_on is not None:
            ren.prepare(sf, prepared_on, stream=side)
        ren.render(sf, c, **im)
        b = ren.get_binning(sc.n, tiles)
        ren.backward(**split_upstream(up), grads=g, d_pose6=p6)
        torch.cuda.synchronize()
        return planes(im), b, {k: v.cpu().numpy() for k, v in g.items()}, p6.cpu().numpy()

    ref_ren = sgs.Renderer()
    refs = [full(ref_ren, c) for c in cs]
    ra, rb = sgs.Renderer(), sgs.Renderer()
    # same view prepared; another view prepared (the render must bin again)
    for c_prep, k in ((cs[1], 1), (cs[2], 1)):
        img, b, g, p6 = full(ra, cs[k], prepared_on=c_prep)
        assert np.array_equal(img, refs[k][0])
        assert_binning(b, refs[k][1])
        for name in g:
            np.testing.assert_allclose(g[name], refs[k][2][name], rtol=2e-4, atol=1e-5 * np.abs(refs[k][2][name]).max())
        np.testing.assert_allclose(p6, refs[k][3], rtol=1e-4, atol=1e-5 * np.abs(refs[k][3]).max())
    # a window of views over two contexts: binning of view v+1 enqueued on the side stream before view v is rendered
    rens = [ra, rb]
    ims = [alloc_images(cam) for _ in cs]
    p6s = [torch.zeros(6, device="cuda") for _ in cs]
    main = torch.cuda.current_stream()
    side.wait_stream(main)
    rens[0].prepare(sf, cs[0], stream=side)
    for v, c in enumerate(cs):
        if v + 1 < len(cs):
            rens[(v + 1) % 2].prepare(sf, cs[v + 1], stream=side)
        rens[v % 2].render(sf, c, **ims[v])
        rens[v % 2].backward(**split_upstream(up), grads=None, d_pose6=p6s[v])
    torch.cuda.synchronize()
    for v in range(len(cs)):
        assert np.array_equal(planes(ims[v]), refs[v][0])
        np.testing.assert_allclose(p6s[v].cpu().numpy(), refs[v][3], rtol=1e-4, atol=1e-5 * np.abs(refs[v][3]).max())
    for r in (ref_ren, ra, rb):
        r.close()


def test_track_reuse_keeps_the_binning_exact():
    """SGS_FLAG_TRACK_REUSE: along a pose trajectory (steps inside the survivor list's 3 cm / 0.02 rad margin, a step
    that leaves it, another map, a new frame) every iteration's binning is bit-identical to the oracle's and images,
    loss and pose gradient equal those of a context without the flag; the list is rebuilt exactly when it has to be
    (kernel launch counts: 6 launches when K-pre-A and the gather of the listed splats run, 4 otherwise: K-pre-B, the one-warp
    kernel that publishes the counters to the host, K-track and the one-block tile-order kernel)."""
    sc, _, _ = scenegen.make_config("C2", n_override=30000)
    sc2 = Scene(sc.mean + np.float32(0.01), sc.scale, sc.quat, sc.opacity, sc.rgb, sc.active)
    cfg = oracle.make_cfg()
    t, sf = to_device(sc)
    t2, sf2 = to_device(sc2)
    T0 = scenegen.look_at(np.array([2.4, 0.6, 1.5]), np.array([2.6, 3.9, 1.2])).astype(np.float32)
    base = Camera(208, 150, 150.0, 150.0, 104.0, 75.0, T0)
    ra, rb = sgs.Renderer(track_reuse=True), sgs.Renderer()
    im0 = alloc_images(base)
    rb.render(sf, camera(base), **im0)
    tgt_rgb, tgt_dep = (im0["rgb"] * 0.9 + 0.01).contiguous(), (im0["depth"] * 1.02).contiguous()
    tiles = ((base.width + 15) // 16) * ((base.height + 15) // 16)
    p0, l0_ = torch.zeros(6, device="cuda"), torch.zeros(1, device="cuda")
    ra.track_iter(sf, camera(base), tgt_rgb, tgt_dep, 0.5, -1.0, p0, l0_)   # first call: workspace + tile order set up
    ra.track_new_frame()
    # (tau relative to T0, which map, new frame first?, expected number of kernel launches of the iteration)
    steps = [([0, 0, 0, 0, 0, 0], 0, False, 6),
             ([0.01, -0.005, 0.008, 0.004, -0.006, 0.005], 0, False, 4),        # inside the margin: list reused
             ([-0.015, 0.01, 0.005, -0.008, 0.004, -0.007], 0, False, 4),
             ([0.05, 0.0, 0.02, 0.0, 0.03, 0.0], 0, False, 6),                   # outside: rebuilt around this pose
             ([0.055, 0.004, 0.018, 0.003, 0.033, -0.004], 0, False, 4),        # inside the NEW list's margin
             ([0.055, 0.004, 0.018, 0.003, 0.033, -0.004], 1, False, 6),        # another map
             ([0.055, 0.004, 0.018, 0.003, 0.033, -0.004], 1, False, 4),
             ([0.055, 0.004, 0.018, 0.003, 0.033, -0.004], 1, True, 6)]         # new frame
    for tau, which, new_frame, want_launches in steps:
        T = scenegen.perturb_pose(T0, tau)
        cam = Camera(base.width, base.height, base.fx, base.fy, base.cx, base.cy, T)
        c = camera(cam)
        scene, s_dev = (sc, sf) if which == 0 else (sc2, sf2)
        if new_frame:
            ra.track_new_frame()
        ima, imb = alloc_images(cam), alloc_images(cam)
        pa, la = torch.zeros(6, device="cuda"), torch.zeros(1, device="cuda")
        pb, lb = torch.zeros(6, device="cuda"), torch.zeros(1, device="cuda")
        l0 = ra.stats()["kernel_launches"]
        ra.track_iter(s_dev, c, tgt_rgb, tgt_dep, 0.5, -1.0, pa, la, **ima)
        assert ra.stats()["kernel_launches"] - l0 == want_launches, (tau, which, new_frame)
        rb.track_iter(s_dev, c, tgt_rgb, tgt_dep, 0.5, -1.0, pb, lb, **imb)
        torch.cuda.synchronize()
        ob = oracle.binning(scene, oracle.make_cam(cam), cfg)
        assert ob["E"] > 1000
        assert_binning(ra.get_binning(scene.n, tiles), ob)
        assert np.array_equal(planes(ima), planes(imb))
        np.testing.assert_allclose(la.cpu().numpy(), lb.cpu().numpy(), rtol=1e-5)
        np.testing.assert_allclose(pa.cpu().numpy(), pb.cpu().numpy(), rtol=1e-4, atol=1e-6 * float(pb.abs().max()))
    ra.close(); rb.close()


def test_lazy_grads_equal_after_wait():
    """SGS_FLAG_LAZY_GRADS: after sgs_wait_grads the surfel and pose gradients equal those of a context without the
    flag (same kernels; sums of atomics differ in order only), also when the next view is rendered on another context
    in between and when the same context is reused for a later view (its own calls order themselves)."""
    sc, cams, _ = scenegen.make_config("C1")
    cam = cams[0]
    t, sf = to_device(sc)
    up = scenegen.upstream_normal(9, cam.height, cam.width)
    taus = [None, [0.05, 0.02, -0.04, 0.1, -0.05, 0.2], [-0.1, 0.05, 0.02, -0.2, 0.1, 0.05], [0.02, 0.0, 0.01, 0.0, 0.03, 0.0]]
    cs = [camera(cam, None if tau is None else scenegen.perturb_pose(cam.T_cw, tau)) for tau in taus]
    ref = sgs.Renderer()
    refs = []
    for c in cs:
        im, g, p6 = alloc_images(cam), alloc_grads(sc.n), torch.zeros(6, device="cuda")
        ref.render(sf, c, **im)
        ref.backward(**split_upstream(up), grads=g, d_pose6=p6)
        torch.cuda.synchronize()
        refs.append(({k: v.cpu().numpy() for k, v in g.items()}, p6.cpu().numpy()))
    rens = [sgs.Renderer(lazy_grads=True), sgs.Renderer(lazy_grads=True)]
    outs = []
    for v, c in enumerate(cs):   # two contexts alternate; nothing waits until the end
        im, g, p6 = alloc_images(cam), alloc_grads(sc.n), torch.full((6,), 7.0, device="cuda")
        rens[v % 2].render(sf, c, **im)
        rens[v % 2].backward(**split_upstream(up), grads=g, d_pose6=p6)
        outs.append((g, p6))
    for r in rens:
        r.wait_grads()
    res = [({k: x.cpu().numpy() for k, x in g.items()}, p6.cpu().numpy()) for g, p6 in outs]   # on the waited stream
    for (g, p6), (rg, rp6) in zip(res, refs):
        for name in g:
            np.testing.assert_allclose(g[name], rg[name], rtol=2e-4, atol=1e-5 * np.abs(rg[name]).max())
        np.testing.assert_allclose(p6, rp6, rtol=1e-4, atol=1e-5 * np.abs(rp6).max())
    for r in rens + [ref]:
        r.close()
