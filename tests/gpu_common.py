"""Helpers shared by the GPU parity tests: move a scenegen.Scene to the device, run the CUDA
path through the binding, and the comparison rules of DESIGN.md §6."""
import numpy as np
import torch

import paper_2506_00970_b200 as sgs


def to_device(sc):
    d = lambda a, dt=torch.float32: None if a is None else torch.from_numpy(np.ascontiguousarray(a)).to("cuda", dt)
    t = dict(mean=d(sc.mean), scale=d(sc.scale), quat=d(sc.quat), opacity=d(sc.opacity), rgb=d(sc.rgb),
             active=d(sc.active, torch.uint8))
    return t, sgs.Renderer.surfels(t["mean"], t["scale"], t["quat"], t["opacity"], t["rgb"], t["active"])


def camera(cam, T_cw=None):
    return sgs.make_camera(cam.width, cam.height, cam.fx, cam.fy, cam.cx, cam.cy, cam.T_cw if T_cw is None else T_cw)


def alloc_images(cam):
    H, W = cam.height, cam.width
    z = lambda c: torch.zeros((c, H, W), device="cuda", dtype=torch.float32)
    return dict(rgb=z(3), depth=z(1), normal=z(3), alpha=z(1))


def planes(im):
    return torch.cat([im["rgb"], im["depth"], im["normal"], im["alpha"]], 0).cpu().numpy().astype(np.float64)


def alloc_grads(n):
    z = lambda *s: torch.full(s, 7.0, device="cuda", dtype=torch.float32)  # poisoned: must be overwritten
    return dict(mean=z(n, 3), scale=z(n, 2), quat=z(n, 4), opacity=z(n), rgb=z(n, 3))


def split_upstream(up):
    u = torch.from_numpy(np.ascontiguousarray(up, dtype=np.float32)).cuda()
    return dict(d_rgb=u[0:3].contiguous(), d_depth=u[3:4].contiguous(), d_normal=u[4:7].contiguous(), d_alpha=u[7:8].contiguous())


def image_check(gpu, ref, fragile, rtol=1e-4, atol=1e-5):
    """|d| <= rtol |ref| + atol on non-fragile pixels; fragile pixels (a decision within 1e-4 of its
    threshold in the fp64 oracle) may differ by one flipped decision: bounded loosely."""
    good = (fragile & 5) == 0
    err = np.abs(gpu - ref)
    bound = rtol * np.abs(ref) + atol
    bad = (err > bound) & good[None]
    loose = err[:, ~good] <= 0.05 * (1.0 + np.abs(ref[:, ~good]))
    return dict(n_bad=int(bad.sum()), max_excess=float((err - bound)[:, good].max()) if good.any() else 0.0,
                fragile_frac=float(1 - good.mean()), fragile_ok=bool(loose.all()),
                worst=float((err / (np.abs(ref) + atol / rtol))[:, good].max()) if good.any() else 0.0)


def grad_check(gpu, ref, rtol=1e-3):
    """Per parameter group: |d| <= rtol |ref| + rtol RMS(ref group)."""
    gpu = np.asarray(gpu, dtype=np.float64); ref = np.asarray(ref, dtype=np.float64)
    rms = np.sqrt(np.mean(ref ** 2)) if ref.size else 0.0
    bound = rtol * np.abs(ref) + rtol * rms
    err = np.abs(gpu - ref)
    return dict(frac_bad=float((err > bound).mean()) if ref.size else 0.0,
                worst=float((err / (bound + 1e-300)).max()) if ref.size else 0.0, rms=float(rms))
