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


EPS32 = 2.0 ** -23     # unit roundoff scale of binary32
C_ROUND = 8.0          # roundings of the intersection's inputs counted in the kappa bound (payload 7 coefficients rounded
                       # to binary32, re-basing, the pair's FMAs, rcp.approx: <= 16 half-ulp errors = 8 ulp); fixed a priori
C_FLIP = 2.0           # a flipped decision moves a blended value by at most 2 vmax x (weight at stake), see orc_pixel_bounds
MAX_FRAGILE = 0.02     # largest fragile-pixel fraction accepted (measured <= 1.5 %)


def image_check(gpu, ref, fragile, pb, rtol=1e-4, atol=1e-5, raw=None):
    """Images against the oracle.  Non-fragile pixels: |d| <= rtol |ref| + atol, no exception.  Fragile
    pixels (a decision of the fp64 oracle within 1e-4 of its threshold, or a composited pair with kappa > 32; reading
    R21) get the oracle-DERIVED allowance on top (oracle.pixel_bounds):
        C_FLIP vmax flip_w            one flipped decision moves a blend by at most twice the weight at stake
      + 2 vmax C_ROUND 2^-23 kerr     binary32 rounding of the intersection's inputs, amplified by kappa rho^2
      + C_ROUND 2^-23 kerr_z          (depth plane only) the same for the depth values themselves
    with vmax = 1 for colour, normal and alpha and the pixel's largest intersection depth for the depth plane.
    raw: the oracle's un-normalised images when `ref` holds the normalised depth D_n = D / O (reading R9n): the depth
    plane's allowance then follows from the quotient, (allowance(D) + |D_n| allowance(O)) / O."""
    good = (fragile & 5) == 0
    err = np.abs(gpu - ref)
    strict = rtol * np.abs(ref) + atol
    vmax = np.ones_like(ref)
    vmax[3] = np.maximum(pb["zmax"], 1e-3)
    allow = C_FLIP * vmax * pb["flip_w"][None] + 2.0 * vmax * C_ROUND * EPS32 * pb["kerr"][None]
    allow[3] += C_ROUND * EPS32 * pb["kerr_z"]
    if raw is not None:
        allow[3] = (allow[3] + np.abs(ref[3]) * allow[7]) / np.maximum(raw[7], 1e-12)
    loose = strict + allow
    bad = (err > strict) & good[None]
    bad_f = (err > loose) & ~good[None]
    return dict(n_bad=int(bad.sum()), n_bad_fragile=int(bad_f.sum()),
                max_excess=float((err - strict)[:, good].max()) if good.any() else 0.0,
                fragile_frac=float(1 - good.mean()),
                worst=float((err / strict)[:, good].max()) if good.any() else 0.0,
                worst_fragile=float((err / loose)[:, ~good].max()) if (~good).any() else 0.0,
                median_allowance=float(np.median((loose - strict)[:, ~good])) if (~good).any() else 0.0)


def assert_image_check(chk, ctx=None):
    assert chk["n_bad"] == 0 and chk["n_bad_fragile"] == 0 and chk["fragile_frac"] < MAX_FRAGILE, (ctx, chk)


C_EXPO = 2.0           # gradient allowance: this multiple of the exposed pixels' summed |contribution| (oracle.exposure)


def grad_check(gpu, ref, expo, rtol=1e-3):
    """Per parameter group, EVERY element: |d| <= rtol |ref| + rtol RMS(ref group) + C_EXPO expo, where expo is the oracle's
    summed |contribution| of the exposed (fragile) pixels to that element, on the oracle's list and on the list with the
    pixel's fragile decisions inverted: a renderer that decides differently there moves the element by at most that much.
    Elements of surfels that touch no fragile pixel have expo = 0 and meet north_star's bar with no exception."""
    gpu = np.asarray(gpu, dtype=np.float64); ref = np.asarray(ref, dtype=np.float64); expo = np.asarray(expo, dtype=np.float64)
    rms = np.sqrt(np.mean(ref ** 2)) if ref.size else 0.0
    strict = rtol * np.abs(ref) + rtol * rms
    bound = strict + C_EXPO * expo
    err = np.abs(gpu - ref)
    clean = expo == 0
    return dict(n_bad=int((err > bound).sum()), worst=float((err / (bound + 1e-300)).max()) if ref.size else 0.0,
                worst_clean=float((err / (strict + 1e-300))[clean].max()) if clean.any() else 0.0,
                frac_over_strict=float((err > strict).mean()) if ref.size else 0.0,
                clean_frac=float(clean.mean()) if ref.size else 1.0,
                expo_share=float(expo.sum() / (np.abs(ref).sum() + 1e-300)), rms=float(rms))


GROUPS = ("mean", "scale", "quat", "opacity", "rgb")
MAX_EXPO_SHARE = 0.15  # the exposed pixels' |contribution| must stay a small part of the gradient mass


def assert_grads(g, og, ex, ctx=None):
    for k in GROUPS:
        chk = grad_check(g[k], og[k], ex[k])
        assert chk["n_bad"] == 0 and chk["expo_share"] < MAX_EXPO_SHARE, (ctx, k, chk)


def pose_check(p, ref, expo_pose, rtol=1e-3):
    """|d| <= rtol ||ref||_inf + C_EXPO expo_pose per component."""
    p = np.asarray(p, dtype=np.float64); ref = np.asarray(ref, dtype=np.float64)
    bound = rtol * np.abs(ref).max() + C_EXPO * np.asarray(expo_pose, dtype=np.float64)
    err = np.abs(p - ref)
    return dict(ok=bool((err <= bound).all()), worst=float((err / bound).max()), worst_strict=float(err.max() / (rtol * np.abs(ref).max())),
                slack_share=float(np.max(C_EXPO * np.asarray(expo_pose) / (np.abs(ref).max() + 1e-300))))


def assert_pose(p, ref, expo_pose, ctx=None, max_slack=0.05):
    chk = pose_check(p, ref, expo_pose)
    assert chk["ok"] and chk["slack_share"] < max_slack, (ctx, chk, p, ref)


def tracking_reference(sc, camv, cfg, o, tgt, lambda_d, nsign, oracle, normalised=False):
    """Oracle side of a tracking iteration (Eq. 15-19): loss L, upstream gradients `up`, gradients `og`, the exposure `ex`
    of the render's fragile pixels under that upstream -- and, per loss channel (r, g, b, depth), the CANDIDATE pixels
    `cand[ch]` at which a binary32 renderer may legitimately evaluate a mask (M_o, M_n) or the sign of Eq. 15-16
    differently: it evaluates them on ITS images, which may differ from the oracle's by the image bar (1e-4 |v| + 1e-5), so
    only pixels whose margin is inside that bar (or that are fragile in the render) qualify.
    normalised: o is oracle.render_normalised's result and the loss sees D_n = D / O (reading R9n); gradients and exposure then
    go through the division's Jacobian (oracle.normalised_depth_upstream)."""
    img = o["img"]
    W, H = int(camv[0]), int(camv[1])
    fx, fy, cx, cy = camv[2:6]
    HW = W * H
    L, up = oracle.tracking_loss(img, tgt[0:3], tgt[3], camv, lambda_d, nsign)
    to_raw = (lambda u: oracle.normalised_depth_upstream(o["img_raw"], u)) if normalised else (lambda u: u)
    og = oracle.backward(sc, camv, cfg, to_raw(up))
    ex = oracle.exposure(sc, camv, cfg, to_raw(up))
    tol = 1e-4 * np.abs(img) + 1e-5
    X, Y = np.meshgrid(np.arange(W) + 0.5, np.arange(H) + 0.5)
    rx, ry = (X - cx) / fx, (Y - cy) / fy
    nr = img[4] * rx + img[5] * ry + img[6]
    nr_tol = tol[4] * np.abs(rx) + tol[5] * np.abs(ry) + tol[6] + 4 * EPS32 * (np.abs(img[4] * rx) + np.abs(img[5] * ry) + np.abs(img[6]))
    d = np.concatenate([img[0:3] - tgt[0:3], oracle._depth_residual(img[3], tgt[3])[None]], 0)
    dtol = tol[0:4] + EPS32 * np.abs(tgt[0:4])
    fragile = (o["fragile"] & 5) != 0
    m_flip = (np.abs(img[7] - 0.95) <= tol[7] + EPS32) | (np.abs(nr) <= nr_tol) | fragile
    could_pass = ((nsign * nr > -nr_tol) & (img[7] > 0.95 - tol[7] - EPS32)) | fragile
    cand = ((np.abs(d) <= dtol) | m_flip[None] | fragile[None]) & could_pass[None]
    w = np.array([1.0, 1.0, 1.0, lambda_d]) / HW
    # loss: the image bar on every term that can be in the sum; flipped masks are added by the caller (loss_slack_of)
    loss_tol = float((dtol * w[:, None, None] * could_pass[None]).sum())
    return dict(L=L, up=up, og=og, ex=ex, cand=cand, d=d, w=w, loss_tol=loss_tol, cand_frac=float(cand.any(0).mean()),
                to_raw=to_raw)


def tracking_flips(tr, up_gpu):
    """Pixels at which the renderer's loss (its upstream gradients `up_gpu`, (8,H,W)) decided differently from the oracle, per
    loss channel; every one of them must be a candidate."""
    D = np.sign(up_gpu[0:4]) != np.sign(tr["up"][0:4])
    assert not (D & ~tr["cand"]).any(), ("a mask or sign differs at a pixel whose margin is outside the image bar",
                                         int((D & ~tr["cand"]).sum()))
    return D


def tracking_slack(sc, camv, cfg, tr, D, oracle):
    """What the flips D (tracking_flips) may change: pose 6-vector (twice the |contribution| of the flipped pixel under the
    unmasked upstream of that channel: a mask flip adds or removes the term, a sign flip changes it by twice itself) and loss."""
    pose = np.zeros(6)
    for ch in range(4):
        if D[ch].any():
            u1 = np.zeros_like(tr["up"]); u1[ch] = tr["w"][ch] * D[ch]
            pose += 2.0 * oracle.exposure(sc, camv, cfg, tr["to_raw"](u1), extra_mask=D[ch])["pose"]
    loss = float((np.abs(tr["d"]) * tr["w"][:, None, None] * D).sum())
    return pose, loss
