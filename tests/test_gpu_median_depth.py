"""GPU parity of sgs_render_median (reading R9m) against oracle.median_depth (pinned by P17).  The
median picks ONE splat per pixel, a decision on T against 1/2: both sides take it on their own T (fp32 / fp64), and the
pixels where the oracle's T passes within 1e-4 of 1/2 -- or where the oracle flags an image-affecting decision as
fragile -- may legitimately pick a neighbouring splat; everywhere else the depth agrees to the image tolerance."""
import numpy as np
import pytest
import torch

import oracle
import scenegen
from scenegen import Scene, Camera

pytestmark = pytest.mark.gpu

sgs = pytest.importorskip("paper_2506_00970_b200")
from gpu_common import to_device, camera, alloc_images, planes  # noqa: E402


def check(r, sc, cam, T=None, min_frac=0.02):
    camv, cfg = oracle.make_cam(cam, T), oracle.make_cfg()
    t, sf = to_device(sc)
    im, im2 = alloc_images(cam), alloc_images(cam)
    med = torch.full((cam.height, cam.width), -7.0, device="cuda")
    r.render_median(sf, camera(cam, T), med, **im)
    r.render(sf, camera(cam, T), **im2)
    torch.cuda.synchronize()
    assert np.array_equal(planes(im), planes(im2))          # the other outputs are those of sgs_render
    want, mf = oracle.median_depth(sc, camv, cfg)
    o = oracle.render(sc, camv, cfg, counters=False)
    good = (mf == 0) & ((o["fragile"] & 5) == 0)
    got = med.cpu().numpy().astype(np.float64)
    assert good.mean() > 0.97, good.mean()
    err = np.abs(got - want)
    assert (err[good] <= 1e-4 * np.abs(want[good]) + 1e-5).all(), (err[good].max(), int((err[good] > 1e-4).sum()))
    assert ((want > 0) & good).mean() >= min_frac
    # where the pixel stays below half opacity both say 0
    low = good & (o["img"][7] < 0.5 - 1e-3)
    assert (got[low] == 0).all()
    return got, want


def test_c1_two_poses_and_flag_combination():
    sc, cams, _ = scenegen.make_config("C1")
    cam = cams[0]
    for nd in (False, True):
        r = sgs.Renderer(normalised_depth=nd)
        check(r, sc, cam)
        check(r, sc, cam, scenegen.perturb_pose(cam.T_cw, [0.1, -0.2, 0.15, 0.2, -0.1, 0.3]))
        r.close()


def test_c2_full_size_and_long_lists():
    sc, cams, _ = scenegen.make_config("C2")
    r = sgs.Renderer(async_mode=True)
    got, want = check(r, sc, cams[0], min_frac=0.2)
    assert len(np.unique(np.round(want[want > 0], 2))) > 50      # a real depth image, not one plane
    # ~900 entries on the central tiles (several staged batches), low opacity: the crossing happens deep in the list
    g = scenegen.SplitMix(11)
    n = 900
    mean = np.stack([g.uniform(n, -0.05, 0.05), g.uniform(n, -0.05, 0.05), g.uniform(n, 1.0, 3.0)], 1).astype(np.float32)
    scl = Scene(mean, np.full((n, 2), 0.01, np.float32), np.tile(np.float32([1, 0.1, 0, 0]), (n, 1)),
                np.full(n, 0.05, np.float32), np.stack([g.uniform(n) for _ in range(3)], 1).astype(np.float32))
    check(r, scl, Camera(64, 48, 60.0, 60.0, 32.0, 24.0), min_frac=0.003)
    r.close()


def test_degenerate_and_arguments():
    cam = Camera(40, 24, 30.0, 30.0, 20.0, 12.0)
    r = sgs.Renderer()
    z = lambda *s: np.zeros(s, np.float32)
    t, sf = to_device(Scene(z(0, 3), z(0, 2), z(0, 4), z(0), z(0, 3)))
    med = torch.full((cam.height, cam.width), 3.0, device="cuda")
    r.render_median(sf, camera(cam), med)
    assert float(med.abs().max()) == 0.0
    # one opaque fronto-parallel splat: covered pixels with a >= 1/2 carry its depth, the rest 0
    sc1 = Scene(np.float32([[0, 0, 2.0]]), np.float32([[0.2, 0.2]]), np.float32([[1, 0, 0, 0]]), np.float32([0.9]),
                np.float32([[0.2, 0.4, 0.6]]))
    t, sf = to_device(sc1)
    im = alloc_images(cam)
    r.render_median(sf, camera(cam), med, **im)
    a = planes(im)[7]
    m = med.cpu().numpy()
    assert (np.abs(m[a > 0.501] - 2.0) < 1e-5).all() and (a > 0.501).sum() > 10 and (m[a < 0.499] == 0).all()
    with pytest.raises(sgs.SgsError) as e:
        r.render_median(sf, camera(cam), None)
    assert e.value.status == sgs.SGS_INVALID_ARGUMENT
    r.close()
