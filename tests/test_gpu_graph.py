"""SGS_FLAG_GRAPH makes the calls capturable: sgs_render + sgs_backward (full, with the pose) and sgs_track_iter recorded
into a CUDA graph once the workspace has its size, replayed, give the results of the eager calls -- also after the
inputs (map colours, target) were changed in place between replays."""
import numpy as np
import pytest
import torch

import scenegen

pytestmark = pytest.mark.gpu

sgs = pytest.importorskip("paper_2506_00970_b200")
from gpu_common import to_device, camera, alloc_images, planes, alloc_grads, split_upstream  # noqa: E402


def test_render_backward_and_track_iter_in_a_cuda_graph():
    sc, cams, _ = scenegen.make_config("C1")
    cam = cams[0]
    up = split_upstream(scenegen.upstream_normal(4, cam.height, cam.width))
    t, sf = to_device(sc)
    c = camera(cam)
    r = sgs.Renderer(graph=True)
    im, g, p6 = alloc_images(cam), alloc_grads(sc.n), torch.zeros(6, device="cuda")
    p6t, lt = torch.zeros(6, device="cuda"), torch.zeros(1, device="cuda")
    tgt_rgb, tgt_dep = torch.rand(3, cam.height, cam.width, device="cuda"), torch.rand(1, cam.height, cam.width, device="cuda") + 1.0

    def step():
        r.render(sf, c, **im)
        r.backward(**up, grads=g, d_pose6=p6)
        r.track_iter(sf, c, tgt_rgb, tgt_dep, 0.5, 1.0, p6t, lt)

    def snapshot():
        torch.cuda.synchronize()
        return (planes(im), {k: v.cpu().numpy() for k, v in g.items()}, p6.cpu().numpy(), p6t.cpu().numpy(), lt.cpu().numpy())

    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        for _ in range(3):      # workspace reaches its size; nothing is allocated during capture
            step()
    torch.cuda.current_stream().wait_stream(s)
    eager = snapshot()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=s):
        step()
    for round_ in range(2):
        for v in list(im.values()) + list(g.values()) + [p6, p6t, lt]:
            v.fill_(-3.0)
        graph.replay()
        got = snapshot()
        assert np.array_equal(got[0], eager[0])
        for k in got[1]:
            np.testing.assert_allclose(got[1][k], eager[1][k], rtol=2e-4, atol=1e-5 * np.abs(eager[1][k]).max())
        np.testing.assert_allclose(got[2], eager[2], rtol=1e-4, atol=1e-5 * np.abs(eager[2]).max())
        np.testing.assert_allclose(got[3], eager[3], rtol=1e-4, atol=1e-6 * np.abs(eager[3]).max())
        np.testing.assert_allclose(got[4], eager[4], rtol=1e-5)
        if round_ == 0:         # new inputs in the same buffers: the replay must follow them
            t["rgb"].mul_(0.5)
            tgt_rgb.mul_(0.7)
            with torch.cuda.stream(s):
                step()
            torch.cuda.current_stream().wait_stream(s)
            eager2 = snapshot()
            assert not np.array_equal(eager2[0], eager[0])
            eager = eager2
    st = r.stats()
    assert st["overflow"] == 0 and st["n_entries"] > 0
    with pytest.raises(sgs.SgsError):
        r.prepare(sf, c)
    r.close()


def test_mapping_iteration_in_a_cuda_graph():
    """render -> Eq. 23-26 mapping loss -> SSIM term -> full backward, recorded once and replayed, equals the eager calls."""
    sc, cams, _ = scenegen.make_config("C1")
    cam = cams[0]
    t, sf = to_device(sc)
    c = camera(cam)
    r = sgs.Renderer(graph=True)
    im, upi, g, p6 = alloc_images(cam), alloc_images(cam), alloc_grads(sc.n), torch.zeros(6, device="cuda")
    loss = torch.zeros(1, device="cuda")
    trgb = torch.rand(3, cam.height, cam.width, device="cuda")
    tdep = torch.rand(1, cam.height, cam.width, device="cuda") + 1.5

    def step():
        loss.zero_()
        r.render(sf, c, **im)
        r.mapping_loss(c, im, trgb, tdep, 0.875, 0.5, 0.02, -1.0, upi, loss)
        r.ssim_loss(im["rgb"], trgb, 0.125, upi["rgb"], loss)
        r.backward(d_rgb=upi["rgb"], d_depth=upi["depth"], d_normal=upi["normal"], d_alpha=upi["alpha"], grads=g, d_pose6=p6)

    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        for _ in range(3):
            step()
    torch.cuda.current_stream().wait_stream(s)
    torch.cuda.synchronize()
    eager = ({k: v.cpu().numpy() for k, v in g.items()}, p6.cpu().numpy(), float(loss.item()), planes(upi))
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=s):
        step()
    for v in list(g.values()) + list(upi.values()) + [p6, loss]:
        v.fill_(-3.0)
    graph.replay()
    torch.cuda.synchronize()
    assert np.array_equal(planes(upi), eager[3]) and eager[2] > 0
    assert abs(float(loss.item()) - eager[2]) <= 1e-5 * eager[2]
    for k in g:
        np.testing.assert_allclose(g[k].cpu().numpy(), eager[0][k], rtol=2e-4, atol=1e-5 * np.abs(eager[0][k]).max())
    np.testing.assert_allclose(p6.cpu().numpy(), eager[1], rtol=1e-4, atol=1e-5 * np.abs(eager[1]).max())
    r.close()


def test_track_iter_graph_replays_back_to_back_with_split_tiles():
    """C2 at full size has tile lists of 161-384 entries, which K-track splits between an owner and a helper block; their
    hand-over flags carry a DEVICE-side epoch, so a graph -- whose kernel arguments are frozen at capture -- can be replayed
    back to back (no eager call in between) with the target changed in place, and every replay equals the eager result."""
    sc, cams, _ = scenegen.make_config("C2")
    cam = cams[0]
    t, sf = to_device(sc)
    c = camera(cam)
    r = sgs.Renderer(graph=True)
    im = alloc_images(cam)
    r.render(sf, c, **im)
    base_rgb, base_dep = im["rgb"].clone(), im["depth"].clone()
    tgt_rgb, tgt_dep = (base_rgb * 0.9 + 0.01).contiguous(), (base_dep * 1.02).contiguous()
    p6, loss = torch.zeros(6, device="cuda"), torch.zeros(1, device="cuda")

    def frame():
        for _ in range(3):   # three iterations per graph: flags written by one are met by the next inside a replay too
            r.track_iter(sf, c, tgt_rgb, tgt_dep, 0.5, -1.0, p6, loss)

    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        for _ in range(2):
            frame()
    torch.cuda.current_stream().wait_stream(s)
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=s):
        frame()
    eager = sgs.Renderer()
    pe, le = torch.zeros(6, device="cuda"), torch.zeros(1, device="cuda")
    for k, (a, b) in enumerate([(0.9, 1.02), (0.8, 1.05), (1.1, 0.97), (0.95, 1.0)]):
        tgt_rgb.copy_(base_rgb * a + 0.01); tgt_dep.copy_(base_dep * b)
        p6.fill_(-3.0); loss.fill_(-3.0)
        graph.replay()                       # replays follow one another directly
        eager.track_iter(sf, c, tgt_rgb, tgt_dep, 0.5, -1.0, pe, le)
        torch.cuda.synchronize()
        np.testing.assert_allclose(loss.cpu().numpy(), le.cpu().numpy(), rtol=1e-5)
        np.testing.assert_allclose(p6.cpu().numpy(), pe.cpu().numpy(), rtol=1e-4, atol=1e-6 * float(pe.abs().max()))
    assert r.stats()["overflow"] == 0
    r.close(); eager.close()


def test_track_iter_dev_pose_changes_inside_one_graph():
    """sgs_track_iter_dev reads T_cw from device memory when the kernels run: a frame of 10 iterations at 10 DIFFERENT poses
    (a device-to-device copy stands for the tracker's pose update between iterations), captured as ONE graph with a kept
    survivor list, equals 10 eager host-pose calls -- and follows new poses written into the same device tensor before a
    replay.  A pose that leaves the kept list's margin turns that iteration's loss and gradient into NaN (the host cannot
    see it; the device check does), and so does a tile-bucket overflow."""
    from scenegen import Camera, Scene
    sc, cams, _ = scenegen.make_config("C2", n_override=60000)
    cam = cams[0]
    t, sf = to_device(sc)
    c = camera(cam)
    g = scenegen.SplitMix(123)

    def pose_set(scale):
        Ts = []
        for k in range(10):
            tau = np.concatenate([scale * 0.012 * g.normal(3) / 3, scale * 0.007 * g.normal(3) / 3])
            Ts.append(scenegen.perturb_pose(cam.T_cw, tau).astype(np.float32))
        return Ts

    ref = sgs.Renderer()
    im = alloc_images(cam)
    ref.render(sf, c, **im)
    tgt_rgb, tgt_dep = (im["rgb"] * 0.9 + 0.01).contiguous(), (im["depth"] * 1.02).contiguous()

    def eager(Ts):
        out = []
        pe, le = torch.zeros(6, device="cuda"), torch.zeros(1, device="cuda")
        for T in Ts:
            ref.track_iter(sf, camera(cam, T), tgt_rgb, tgt_dep, 0.5, -1.0, pe, le)
            out.append((pe.cpu().numpy().copy(), float(le.item())))
        return out

    r = sgs.Renderer(graph=True, track_reuse=True)
    T_all = torch.zeros(10, 12, device="cuda")
    T_cur = torch.zeros(12, device="cuda")
    p6_all, loss_all = torch.zeros(10, 6, device="cuda"), torch.zeros(10, device="cuda")

    def frame():
        r.track_new_frame()
        for k in range(10):
            T_cur.copy_(T_all[k])                 # "the tracker's update kernel"
            r.track_iter_dev(sf, c, T_cur, tgt_rgb, tgt_dep, 0.5, -1.0, p6_all[k], loss_all[k:k + 1])

    Ts = pose_set(1.0)
    T_all.copy_(torch.from_numpy(np.stack([T.reshape(12) for T in Ts])))
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        for _ in range(2):
            frame()
    torch.cuda.current_stream().wait_stream(s)
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=s):
        frame()
    for round_ in range(2):
        want = eager(Ts)
        p6_all.fill_(-3.0); loss_all.fill_(-3.0)
        graph.replay()
        torch.cuda.synchronize()
        for k in range(10):
            assert abs(float(loss_all[k]) - want[k][1]) <= 1e-5 * abs(want[k][1])
            np.testing.assert_allclose(p6_all[k].cpu().numpy(), want[k][0], rtol=1e-4, atol=1e-6 * np.abs(want[k][0]).max())
        assert len({round(w[1], 9) for w in want}) == 10          # the ten iterations really differ
        Ts = pose_set(0.7)                                        # new poses, same device tensor
        T_all.copy_(torch.from_numpy(np.stack([T.reshape(12) for T in Ts])))
    # iterations 6.. leave the margin of the list built at iteration 0: NaN, not numbers from an incomplete list
    far = scenegen.perturb_pose(cam.T_cw, [0.2, 0.0, 0.1, 0.0, 0.05, 0.0]).astype(np.float32).reshape(12)
    T_all[6:] = torch.from_numpy(far).cuda()
    graph.replay()
    torch.cuda.synchronize()
    assert torch.isfinite(loss_all[:6]).all() and torch.isfinite(p6_all[:6]).all()
    assert torch.isnan(loss_all[6:]).all() and torch.isnan(p6_all[6:]).all()
    r.close(); ref.close()
    # a tile-bucket overflow in async mode: that iteration's results are NaN at once; the NEXT call reports it
    n = 6000
    mean = np.stack([g.uniform(n, -0.02, 0.02), g.uniform(n, -0.02, 0.02), g.uniform(n, 1.0, 3.0)], 1).astype(np.float32)
    dense = Scene(mean, np.full((n, 2), 0.01, np.float32), np.tile(np.float32([1, 0, 0, 0]), (n, 1)),
                  np.full(n, 0.05, np.float32), np.full((n, 3), 0.5, np.float32))
    small = Camera(64, 48, 60.0, 60.0, 32.0, 24.0)
    td, sfd = to_device(dense)
    a = sgs.Renderer(async_mode=True)
    pa, la = torch.zeros(6, device="cuda"), torch.zeros(1, device="cuda")
    trgb, tdep = torch.full((3, 48, 64), 0.3, device="cuda"), torch.full((1, 48, 64), 1.5, device="cuda")
    a.track_iter(sfd, camera(small), trgb, tdep, 0.5, 1.0, pa, la)
    torch.cuda.synchronize()
    assert torch.isnan(la).all() and torch.isnan(pa).all()
    with pytest.raises(sgs.SgsError) as e:
        a.stats(); a.track_iter(sfd, camera(small), trgb, tdep, 0.5, 1.0, pa, la)
    assert e.value.status == sgs.SGS_WORKSPACE_OVERFLOW
    a.track_iter(sfd, camera(small), trgb, tdep, 0.5, 1.0, pa, la)
    torch.cuda.synchronize()
    assert torch.isfinite(la).all() and torch.isfinite(pa).all()
    a.close()
