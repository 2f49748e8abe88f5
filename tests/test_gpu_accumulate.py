"""Gradient accumulation over a mapping window (one optimiser step on the summed loss of N_a + N_i
views): sgs_backward_accumulate against the SUM of the oracle's per-view gradients, element by element (each view
contributes its own strict bar and its own fragile-pixel exposure to the bound), and the HOST-buffer window calls
(sgs_map_view_host / sgs_fetch_grads_host / sgs_sync_host) against the device-buffer sequence they wrap."""
import ctypes

import numpy as np
import pytest
import torch

import oracle
import scenegen

pytestmark = pytest.mark.gpu

sgs = pytest.importorskip("paper_2506_00970_b200")
from gpu_common import (to_device, camera, alloc_images, alloc_grads, split_upstream, assert_pose, GROUPS, C_EXPO)  # noqa: E402


def window_against_oracle(sc, cam_views, ups, async_mode=False):
    """cam_views: [(Camera, T_cw or None)], ups: upstream (8,H,W) per view."""
    cfg = oracle.make_cfg()
    ren = sgs.Renderer(async_mode=async_mode)
    t, sf = to_device(sc)
    g = alloc_grads(sc.n)                     # poisoned with 7.0: zero_grads must clear it
    ren.zero_grads(g)
    ref = {k: 0.0 for k in GROUPS}
    bound = {k: 0.0 for k in GROUPS}
    seen = np.zeros(sc.n, bool)
    for (cam, T), up in zip(cam_views, ups):
        camv, c = oracle.make_cam(cam, T), camera(cam, T)
        im = alloc_images(cam)
        for _ in range(3 if async_mode else 1):
            try:
                ren.render(sf, c, **im); ren.stats(); ren.render(sf, c, **im)
                break
            except sgs.SgsError as e:
                if e.status != sgs.SGS_WORKSPACE_OVERFLOW:
                    raise
        u = torch.from_numpy(up.astype(np.float32)).cuda()
        up32 = u.cpu().numpy().astype(np.float64)
        p6 = torch.full((6,), 5.0, device="cuda")
        ren.backward(**split_upstream(up32), grads=g, d_pose6=p6, accumulate=True)
        og, ex = oracle.backward(sc, camv, cfg, up32), oracle.exposure(sc, camv, cfg, up32)
        assert_pose(p6.cpu().numpy(), og["pose"], ex["pose"])      # the pose gradient is per view: overwritten, not summed
        for k in GROUPS:
            ref[k] = ref[k] + og[k]
            bound[k] = bound[k] + 1e-3 * np.abs(og[k]) + 1e-3 * np.sqrt(np.mean(og[k] ** 2)) + C_EXPO * ex[k]
        seen |= oracle.binning(sc, camv, cfg)["culled"] == 0
    torch.cuda.synchronize()
    for k in GROUPS:
        got = g[k].cpu().numpy().astype(np.float64)
        err = np.abs(got - ref[k])
        assert (err <= bound[k]).all(), (k, int((err > bound[k]).sum()), float((err / bound[k]).max()))
        assert (got[~seen] == 0).all()         # splats no view of the window saw keep the window's zero
    ren.close()


def test_three_view_window_on_c1():
    sc, cams, _ = scenegen.make_config("C1")
    cam = cams[0]
    taus = [None, [0.05, 0.02, -0.04, 0.1, -0.05, 0.2], [-0.1, 0.05, 0.02, -0.2, 0.1, 0.05]]
    views = [(cam, None if tau is None else scenegen.perturb_pose(cam.T_cw, tau)) for tau in taus]
    ups = [scenegen.upstream_normal(20 + i, cam.height, cam.width) for i in range(3)]
    window_against_oracle(sc, views, ups)


def test_two_view_window_on_c3_at_full_size():
    """C3 views 0 and 7 (500 k surfels, 1200 x 680) under the mapping loss of Eq. 24-26 (dense upstream)."""
    sc, cams, _ = scenegen.make_config("C3")
    cfg = oracle.make_cfg()
    views, ups = [], []
    for v in (0, 7):
        cam = cams[v]
        camv = oracle.make_cam(cam)
        img = oracle.render(sc, camv, cfg, counters=False)["img"]
        T_tgt = scenegen.perturb_pose(cam.T_cw, np.array([0.02, 0.0, -0.01, 0.0, 0.01, 0.005]))
        tgt = oracle.render(sc, oracle.make_cam(cam, T_tgt), cfg, counters=False)["img"]
        _, up = oracle.mapping_loss(img, tgt[0:3], tgt[3], camv, 0.875, 0.5, 0.02, -1.0)
        views.append((cam, None)); ups.append(up)
    window_against_oracle(sc, views, ups, async_mode=True)


def test_host_window_calls_equal_the_device_sequence():
    """sgs_map_view_host x 3 + sgs_fetch_grads_host, twice in a row (both accumulators of the double buffer, the re-zeroing
    behind the copy-out), against render + mapping_loss + ssim_loss + backward_accumulate on device buffers."""
    sc, cams, _ = scenegen.make_config("C1")
    cam = cams[0]
    H, W = cam.height, cam.width
    t, sf = to_device(sc)
    taus = [None, [0.05, 0.02, -0.04, 0.1, -0.05, 0.2], [-0.1, 0.05, 0.02, -0.2, 0.1, 0.05]]
    cs = [camera(cam, None if tau is None else scenegen.perturb_pose(cam.T_cw, tau)) for tau in taus]
    g0 = scenegen.SplitMix(77)
    tgts = [(torch.from_numpy(g0.uniform(3 * H * W).reshape(3, H, W).astype(np.float32)),
             torch.from_numpy((1.5 + g0.uniform(H * W)).reshape(1, H, W).astype(np.float32))) for _ in range(6)]
    dev = sgs.Renderer()
    host = sgs.Renderer()
    pin = lambda x, dt=torch.float32: torch.from_numpy(np.ascontiguousarray(x)).to(dt).pin_memory()
    host.upload_surfels(pin(sc.mean), pin(sc.scale), pin(sc.quat), pin(sc.opacity), pin(sc.rgb))
    hg = [{k: torch.full(v.shape, 9.0).pin_memory() for k, v in alloc_grads(sc.n).items()} for _ in range(2)]
    hl = [torch.zeros(1).pin_memory() for _ in range(6)]
    hp = [torch.zeros(6).pin_memory() for _ in range(6)]
    want = []
    for w in range(2):
        g = alloc_grads(sc.n)
        dev.zero_grads(g)
        for v in range(3):
            trgb, tdep = tgts[3 * w + v]
            im, up = alloc_images(cam), alloc_images(cam)
            loss, p6 = torch.zeros(1, device="cuda"), torch.zeros(6, device="cuda")
            dev.render(sf, cs[v], **im)
            dev.mapping_loss(cs[v], im, trgb.cuda(), tdep.cuda(), 0.875, 0.5, 0.02, -1.0, up, loss)
            dev.ssim_loss(im["rgb"], trgb.cuda(), 0.125, up["rgb"], loss)
            dev.backward(d_rgb=up["rgb"], d_depth=up["depth"], d_normal=up["normal"], d_alpha=up["alpha"], grads=g, d_pose6=p6,
                         accumulate=True)
            want.append((float(loss.item()), p6.cpu().numpy()))
            host.map_view_host(cs[v], trgb.pin_memory(), tdep.pin_memory(), 0.875, 0.5, 0.02, 0.125, -1.0, hl[3 * w + v], hp[3 * w + v])
        host.fetch_grads_host(hg[w])            # no wait: the second window is enqueued behind it
        want.append({k: x.cpu().numpy() for k, x in g.items()})
    host.sync_host()
    for w in range(2):
        ref = want[4 * w + 3]
        for k in ref:
            assert np.abs(ref[k]).max() > 0
            np.testing.assert_allclose(hg[w][k].numpy(), ref[k], rtol=2e-4, atol=1e-5 * np.abs(ref[k]).max())
        for v in range(3):
            L, p = want[4 * w + v]
            assert abs(float(hl[3 * w + v].item()) - L) <= 1e-5 * abs(L) and L > 0
            np.testing.assert_allclose(hp[3 * w + v].numpy(), p, rtol=1e-4, atol=1e-5 * np.abs(p).max())
    dev.close(); host.close()


def test_sparse_window_fetch_delivers_exactly_the_touched_rows():
    """sgs_fetch_grads_sparse_host against sgs_fetch_grads_host on the same views: two windows in a row (both accumulators,
    the re-zeroing behind the read), the map padded with surfels behind the camera so that most rows stay zero.  The listed
    ids ascend, are exactly the rows the dense fetch has non-zero, and carry its values (the two runs differ by the order
    of the atomic adds inside a view only); the rows past `count` are not written.  The second window's arrays are pageable memory."""
    sc, cams, _ = scenegen.make_config("C1")
    cam = cams[0]
    H, W = cam.height, cam.width
    n0, pad = sc.n, 3000                       # ragged against the 1024-surfel blocks and the 32-surfel flag words
    back = np.linalg.inv(np.vstack([cam.T_cw[:3], [0, 0, 0, 1]]))[:3] @ np.array([0.0, 0.0, -2.0, 1.0])
    mean = np.vstack([np.tile(back, (pad // 2, 1)), sc.mean, np.tile(back, (pad - pad // 2, 1))])
    rep = lambda a: np.concatenate([np.repeat(a[:1], pad // 2, 0), a, np.repeat(a[:1], pad - pad // 2, 0)])
    n = n0 + pad
    pin = lambda x, dt=torch.float32: torch.from_numpy(np.ascontiguousarray(x)).to(dt).pin_memory()
    taus = [None, [0.05, 0.02, -0.04, 0.1, -0.05, 0.2], [-0.1, 0.05, 0.02, -0.2, 0.1, 0.05]]
    cs = [camera(cam, None if tau is None else scenegen.perturb_pose(cam.T_cw, tau)) for tau in taus]
    g0 = scenegen.SplitMix(78)
    tgts = [(pin(g0.uniform(3 * H * W).reshape(3, H, W)), pin((1.5 + g0.uniform(H * W)).reshape(1, H, W))) for _ in range(6)]
    shapes = dict(mean=3, scale=2, quat=4, opacity=1, rgb=3)
    res = {}
    for mode in ("dense", "sparse"):
        ren = sgs.Renderer()
        ren.upload_surfels(pin(mean), pin(rep(sc.scale)), pin(rep(sc.quat)), pin(rep(sc.opacity)), pin(rep(sc.rgb)))
        out = []
        for w in range(2):
            for v in range(3):
                ren.map_view_host(cs[v], *tgts[3 * w + v], 0.875, 0.5, 0.02, 0.125, -1.0)
            if mode == "dense":
                hg = {k: torch.full((n, d), 9.0).pin_memory() for k, d in shapes.items()}
                ren.fetch_grads_host(hg)
                out.append(hg)
            else:
                pm = (lambda x: x.pin_memory()) if w == 0 else (lambda x: x)
                rows = {k: pm(torch.full((n, d), 9.0)) for k, d in shapes.items()}
                ids, cnt = pm(torch.full((n,), -7, dtype=torch.int32)), torch.full((1,), -1, dtype=torch.int64).pin_memory()
                ren.fetch_grads_sparse_host(ids, rows, cnt)
                out.append((ids, rows, cnt))
        ren.sync_host()
        res[mode] = out
        if mode == "sparse":   # a third, empty window: nothing is listed (the accumulator was zeroed behind the reads)
            ids, cnt = torch.full((n,), -7, dtype=torch.int32).pin_memory(), torch.full((1,), -1, dtype=torch.int64).pin_memory()
            rows = {k: torch.full((n, d), 9.0).pin_memory() for k, d in shapes.items()}
            ren.fetch_grads_sparse_host(ids, rows, cnt); ren.fetch_grads_sparse_host(ids, rows, cnt)
            ren.sync_host()
            assert int(cnt.item()) == 0 and (ids.numpy() == -7).all() and all((r.numpy() == 9.0).all() for r in rows.values())
            assert ren.lib.sgs_fetch_grads_sparse_host(ren._ctx, None, None, ctypes.c_int64(-1), None, None) == sgs.SGS_INVALID_ARGUMENT
        ren.close()
    for w in range(2):
        dense = {k: v.numpy() for k, v in res["dense"][w].items()}
        ids, rows, cnt = res["sparse"][w]
        k = int(cnt.item())
        i = ids.numpy()[:k].astype(np.int64)
        nz = np.zeros(n, bool)
        for a in dense.values():
            nz |= (a != 0).any(axis=1)
        assert 0 < k < n0 + 1 and (np.diff(i) > 0).all() and i.min() >= pad // 2 and i.max() < pad // 2 + n0
        assert np.array_equal(i, np.nonzero(nz)[0])
        assert (ids.numpy()[k:] == -7).all()
        for name, a in dense.items():
            r = rows[name].numpy()
            assert (r[k:] == 9.0).all()
            np.testing.assert_allclose(r[:k], a[i], rtol=2e-4, atol=1e-5 * np.abs(a).max())


def test_sparse_window_fetch_with_too_little_room_delivers_the_first_rows():
    """cap < count: the first cap rows (ascending ids) arrive, *count is the true number of touched surfels, nothing is
    written past cap, and the accumulator is clean for the next window all the same."""
    sc, cams, _ = scenegen.make_config("C1")
    cam = cams[0]
    H, W = cam.height, cam.width
    pin = lambda x, dt=torch.float32: torch.from_numpy(np.ascontiguousarray(x)).to(dt).pin_memory()
    g0 = scenegen.SplitMix(79)
    tgt = (pin(g0.uniform(3 * H * W).reshape(3, H, W)), pin((1.5 + g0.uniform(H * W)).reshape(1, H, W)))
    shapes = dict(mean=3, scale=2, quat=4, opacity=1, rgb=3)
    ren = sgs.Renderer()
    ren.upload_surfels(pin(sc.mean), pin(sc.scale), pin(sc.quat), pin(sc.opacity), pin(sc.rgb))
    c = camera(cam)
    full = {k: torch.full((sc.n, d), 9.0).pin_memory() for k, d in shapes.items()}
    ids_f, cnt_f = torch.full((sc.n,), -7, dtype=torch.int32).pin_memory(), torch.zeros(1, dtype=torch.int64).pin_memory()
    ren.map_view_host(c, *tgt, 0.875, 0.5, 0.02, 0.125, -1.0)
    ren.fetch_grads_sparse_host(ids_f, full, cnt_f)
    ren.sync_host()
    k = int(cnt_f.item())
    cap = k // 3
    assert cap > 10
    part = {kk: torch.full((cap + 5, d), 9.0).pin_memory() for kk, d in shapes.items()}
    ids_p, cnt_p = torch.full((cap + 5,), -7, dtype=torch.int32).pin_memory(), torch.zeros(1, dtype=torch.int64).pin_memory()
    ren.map_view_host(c, *tgt, 0.875, 0.5, 0.02, 0.125, -1.0)
    g = ren._grads(part, "cpu")    # (the binding takes cap from the tensors: call the C entry with an explicit smaller one)
    C = ctypes
    assert ren.lib.sgs_fetch_grads_sparse_host(ren._ctx, C.c_void_p(ids_p.data_ptr()), C.byref(g), C.c_int64(cap),
                                               C.c_void_p(cnt_p.data_ptr()),
                                               C.c_void_p(torch.cuda.current_stream().cuda_stream)) == sgs.SGS_OK
    ren.sync_host()
    assert int(cnt_p.item()) == k
    assert np.array_equal(ids_p.numpy()[:cap], ids_f.numpy()[:cap]) and (ids_p.numpy()[cap:] == -7).all()
    for name in shapes:
        assert (part[name].numpy()[cap:] == 9.0).all()
        np.testing.assert_allclose(part[name].numpy()[:cap], full[name].numpy()[:cap], rtol=2e-4,
                                   atol=1e-5 * np.abs(full[name].numpy()[:k]).max())
    ren.fetch_grads_sparse_host(ids_f, full, cnt_f)      # nothing accumulated since: the lost rows were zeroed too
    ren.sync_host()
    assert int(cnt_f.item()) == 0
    ren.close()


def test_bench_launch_configuration_on_c4():
    """The configuration bench.py times on the mapping configs, at C4's full size (2 M surfels, 1200 x 680): two contexts
    (async, lazy gradients), the binning of the next view prepared on a side stream while the current view composites, each
    context ADDING its views' gradients to its own accumulator.  Views 0 and 6 under the Eq. 24-26 upstream (the oracle's);
    every gradient element of each view against the oracle with the strict bar + the exposure of fragile pixels."""
    from gpu_common import assert_grads
    sc, cams, _ = scenegen.make_config("C4")
    cfg = oracle.make_cfg()
    t, sf = to_device(sc)
    rens = [sgs.Renderer(async_mode=True, lazy_grads=True) for _ in range(2)]
    side = torch.cuda.Stream()
    views = (0, 6)
    ccams = [camera(cams[v]) for v in views]
    ups = []
    for v in views:
        camv = oracle.make_cam(cams[v])
        img = oracle.render(sc, camv, cfg, counters=False)["img"]
        T_tgt = scenegen.perturb_pose(cams[v].T_cw, np.array([0.02, 0.0, -0.01, 0.0, 0.01, 0.005]))
        tgt = oracle.render(sc, oracle.make_cam(cams[v], T_tgt), cfg, counters=False)["img"]
        _, up = oracle.mapping_loss(img, tgt[0:3], tgt[3], camv, 0.875, 0.5, 0.02, -1.0)
        ups.append(torch.from_numpy(up.astype(np.float32)).cuda())
    for k in range(2):   # workspaces at size: an overflowing first render regrows and is reported once (async mode)
        im = alloc_images(cams[views[k]])
        for _ in range(3):
            try:
                rens[k].render(sf, ccams[k], **im); rens[k].stats(); rens[k].render(sf, ccams[k], **im)
                break
            except sgs.SgsError as e:
                if e.status != sgs.SGS_WORKSPACE_OVERFLOW:
                    raise
    torch.cuda.synchronize()
    grads = [alloc_grads(sc.n) for _ in range(2)]
    p6 = [torch.zeros(6, device="cuda") for _ in range(2)]
    main = torch.cuda.current_stream()
    side.wait_stream(main)
    for k in range(2):
        rens[k].zero_grads(grads[k])
    rens[0].prepare(sf, ccams[0], stream=side)
    ims = [alloc_images(cams[v]) for v in views]
    for k in range(2):
        if k + 1 < 2:
            rens[k + 1].prepare(sf, ccams[k + 1], stream=side)      # next view's binning under this view's kernels
        rens[k].render(sf, ccams[k], **ims[k])                      # finds its binning prepared, orders itself behind it
        u = ups[k]
        rens[k].backward(d_rgb=u[0:3].contiguous(), d_depth=u[3:4].contiguous(), d_normal=u[4:7].contiguous(),
                         d_alpha=u[7:8].contiguous(), grads=grads[k], d_pose6=p6[k], accumulate=True)
    main.wait_stream(side)
    for r in rens:
        r.wait_grads()
    torch.cuda.synchronize()
    for k, v in enumerate(views):
        camv = oracle.make_cam(cams[v])
        up32 = ups[k].cpu().numpy().astype(np.float64)
        og, ex = oracle.backward(sc, camv, cfg, up32), oracle.exposure(sc, camv, cfg, up32)
        assert_grads({kk: x.cpu().numpy() for kk, x in grads[k].items()}, og, ex, ("C4", v))
        assert_pose(p6[k].cpu().numpy(), og["pose"], ex["pose"], ("C4", v))
    for r in rens:
        r.close()


def test_sparse_window_fetch_at_c4_size_equals_the_dense_fetch():
    """2 M surfels: the compaction's block scan runs over more than 1024 blocks of 1024 surfels (its carry path).  Two views of
    C4 through sgs_map_view_host on two contexts, one fetched dense, one sparse: same rows (ids = the dense fetch's non-zero
    rows, ascending), same values up to the order of the atomic adds inside a view."""
    sc, cams, _ = scenegen.make_config("C4")
    H, W = cams[0].height, cams[0].width
    pin = lambda x, dt=torch.float32: torch.from_numpy(np.ascontiguousarray(x)).to(dt).pin_memory()
    g0 = scenegen.SplitMix(80)
    tgts = [(pin(g0.uniform(3 * H * W).reshape(3, H, W)), pin((1.5 + g0.uniform(H * W)).reshape(1, H, W))) for _ in range(2)]
    shapes = dict(mean=3, scale=2, quat=4, opacity=1, rgb=3)
    host = dict(mean=pin(sc.mean), scale=pin(sc.scale), quat=pin(sc.quat), opacity=pin(sc.opacity), rgb=pin(sc.rgb))
    out = {}
    for mode in ("dense", "sparse"):
        ren = sgs.Renderer()
        ren.upload_surfels(host["mean"], host["scale"], host["quat"], host["opacity"], host["rgb"])
        for k, v in enumerate((0, 6)):
            ren.map_view_host(camera(cams[v]), *tgts[k], 0.875, 0.5, 0.02, 0.125, -1.0)
        rows = {k: torch.full((sc.n, d), 9.0).pin_memory() for k, d in shapes.items()}
        if mode == "dense":
            ren.fetch_grads_host(rows)
            ren.sync_host()
            out[mode] = {k: v.numpy() for k, v in rows.items()}
        else:
            ids, cnt = torch.full((sc.n,), -7, dtype=torch.int32).pin_memory(), torch.zeros(1, dtype=torch.int64).pin_memory()
            ren.fetch_grads_sparse_host(ids, rows, cnt)
            ren.sync_host()
            out[mode] = (ids.numpy(), {k: v.numpy() for k, v in rows.items()}, int(cnt.item()))
        ren.close()
    dense = out["dense"]
    ids, rows, k = out["sparse"]
    nz = np.zeros(sc.n, bool)
    for a in dense.values():
        nz |= (a != 0).any(axis=1)
    assert 100_000 < k < sc.n // 2 and k == int(nz.sum())
    assert np.array_equal(ids[:k].astype(np.int64), np.nonzero(nz)[0]) and (ids[k:] == -7).all()
    for name, a in dense.items():
        assert (rows[name][k:] == 9.0).all()
        np.testing.assert_allclose(rows[name][:k], a[ids[:k]], rtol=2e-4, atol=1e-5 * np.abs(a).max())
