"""Pins of the CPU oracle (P1-P10) against what PAPER.md and the mathematics fix.
None of these retypes the oracle's formula: they use closed forms, a hand-evaluated fixture, a
library matrix inverse, scipy rotations, invariants, finite differences and symmetries."""
import os
import numpy as np
import pytest
from scipy.spatial.transform import Rotation

import oracle
import scenegen
from scenegen import Scene, Camera

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def one_surfel(mu, s, q, o=0.8, rgb=(0.2, 0.5, 0.9)):
    f = lambda a, sh: np.asarray(a, np.float32).reshape(sh)
    return Scene(f(mu, (1, 3)), f(s, (1, 2)), f(q, (1, 4)), f([o], (1,)), f(rgb, (1, 3)))


def cat(*scs):
    return Scene(*[np.concatenate([getattr(s, k) for s in scs]) for k in ("mean", "scale", "quat", "opacity", "rgb")])


CAM = Camera(64, 48, 60.0, 60.0, 32.0, 24.0)


def pix_grid(cam):
    x = np.arange(cam.width) + 0.5
    y = np.arange(cam.height) + 0.5
    return np.meshgrid(x, y)  # (H,W) each


# ---------------------------------------------------------------- P1: closed-form footprint (Eq. 1-4, 8)
@pytest.mark.parametrize("mu", [(0.0, 0.0, 2.0), (0.31, -0.17, 1.5)])
def test_p1_fronto_parallel_footprint(mu):
    su, sv, o = 0.11, 0.07, 0.8
    sc = one_surfel(mu, (su, sv), (1, 0, 0, 0), o)
    r = oracle.render(sc, oracle.make_cam(CAM), oracle.make_cfg())
    X, Y = pix_grid(CAM)
    mu32 = np.float32(mu).astype(np.float64); su, sv, o = [float(np.float32(v)) for v in (su, sv, o)]
    z0 = mu32[2]
    u = ((X - CAM.cx) * z0 / CAM.fx - mu32[0]) / su
    v = ((Y - CAM.cy) * z0 / CAM.fy - mu32[1]) / sv
    a = o * np.exp(-(u * u + v * v) / 2)
    a[(u * u + v * v > 9.0) | (a < float(np.float32(1 / 255)))] = 0.0
    assert np.abs(a).max() > 0.5
    np.testing.assert_allclose(r["img"][7], a, rtol=0, atol=1e-12)
    np.testing.assert_allclose(r["img"][3], a * z0, rtol=0, atol=1e-12)       # depth plane = a * z0
    np.testing.assert_allclose(r["img"][0], a * float(np.float32(0.2)), atol=1e-12)
    np.testing.assert_allclose(r["img"][6], a * 1.0, atol=1e-12)              # normal = +z for R = I


# ---------------------------------------------------------------- P2: depth = ray-plane intersection depth
def test_p2_tilted_plane_depth():
    rot = Rotation.from_euler("xyz", [25, -35, 10], degrees=True)
    qx, qy, qz, qw = rot.as_quat()
    mu = np.array([0.1, -0.05, 1.8])
    sc = one_surfel(mu, (0.3, 0.2), (qw, qx, qy, qz), 0.9)
    r = oracle.render(sc, oracle.make_cam(CAM), oracle.make_cfg())
    q32 = sc.quat[0].astype(np.float64)
    n = Rotation.from_quat([q32[1], q32[2], q32[3], q32[0]]).as_matrix()[:, 2]
    X, Y = pix_grid(CAM)
    d = np.stack([(X - CAM.cx) / CAM.fx, (Y - CAM.cy) / CAM.fy, np.ones_like(X)], axis=-1)
    z = (n @ sc.mean[0].astype(np.float64)) / (d @ n)
    O = r["img"][7]
    m = O > 0
    assert m.sum() > 100
    np.testing.assert_allclose(r["img"][3][m] / O[m], z[m], rtol=1e-12)
    # normal plane = O * t_n in camera space (identity pose)
    for ch in range(3):
        np.testing.assert_allclose(r["img"][4 + ch][m], O[m] * n[ch], atol=1e-12)


# ---------------------------------------------------------------- P3: hand-evaluated stacks (golden fixture)
def _read_stack():
    rows, exp = [], {}
    for line in open(os.path.join(GOLDEN, "eq8_stack.txt")):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        a, b = line.split()
        if a.startswith("expected"):
            exp[a] = float(b)
        else:
            rows.append((float(a), float(b)))
    return rows, exp


def _stack_scene(rows, depths):
    i, j = 40, 13  # pixel whose centre the surfels project onto
    scs = []
    for (o, val), z in zip(rows, depths):
        mu = ((i + 0.5 - CAM.cx) / CAM.fx * z, (j + 0.5 - CAM.cy) / CAM.fy * z, z)
        scs.append(one_surfel(mu, (0.2, 0.2), (1, 0, 0, 0), o, (val, 0, 0)))
    return cat(*scs), i, j


def test_p3_hand_computed_stack():
    rows, exp = _read_stack()
    cfg = oracle.make_cfg(alpha_max=1.0)
    sc, i, j = _stack_scene(rows, (1.0, 2.0, 3.0))
    r = oracle.render(sc, oracle.make_cam(CAM), cfg)
    assert abs(r["img"][0][j, i] - exp["expected_V"]) < 1e-6
    assert abs(r["img"][7][j, i] - exp["expected_O"]) < 1e-6
    assert abs(r["T_final"][j, i] - exp["expected_T"]) < 1e-6
    sc, i, j = _stack_scene(rows, (2.0, 1.0, 3.0))  # first two swapped in depth
    r = oracle.render(sc, oracle.make_cam(CAM), cfg)
    assert abs(r["img"][0][j, i] - exp["expected_V_swapped"]) < 1e-6
    assert abs(r["img"][7][j, i] - exp["expected_O"]) < 1e-6


def test_p3_depth_ties_break_by_index():
    """Equal depth bits: order is the surfel index (R2), so listing order decides the blend."""
    rows = [(0.5, 1.0), (0.5, 3.0)]
    sc, i, j = _stack_scene(rows, (2.0, 2.0))
    r = oracle.render(sc, oracle.make_cam(CAM), oracle.make_cfg())
    assert abs(r["img"][0][j, i] - (0.5 * 1.0 + 0.25 * 3.0)) < 1e-6


# ---------------------------------------------------------------- P4: invariants
@pytest.fixture(scope="module")
def c1():
    sc, cams, _ = scenegen.make_config("C1")
    camv, cfg = oracle.make_cam(cams[0]), oracle.make_cfg()
    return sc, cams[0], camv, cfg, oracle.render(sc, camv, cfg)


def test_p4_invariants(c1):
    sc, cam, camv, cfg, r = c1
    O, T = r["img"][7], r["T_final"]
    np.testing.assert_allclose(O, 1.0 - T, atol=1e-13)
    assert O.max() <= 1.0 and O.min() >= 0.0 and T.min() >= float(cfg[4])
    assert r["counters"]["Q_c"] == r["n_comp"].sum() and r["counters"]["Q_c"] > 5000
    assert (r["img"][3] >= 0).all()


def test_brute_force_equals_skipping_bitwise(c1):
    sc, cam, camv, cfg, r = c1
    rb = oracle.render(sc, camv, cfg, brute=True)
    assert np.array_equal(r["img"], rb["img"]) and np.array_equal(r["T_final"], rb["T_final"])
    up = scenegen.upstream_normal(1, cam.height, cam.width)
    g, gb = oracle.backward(sc, camv, cfg, up), oracle.backward(sc, camv, cfg, up, brute=True)
    for k in ("mean", "scale", "quat", "opacity", "rgb", "pose"):
        np.testing.assert_allclose(g[k], gb[k], rtol=1e-10, atol=1e-9)  # atomics reorder fp64 sums


# ---------------------------------------------------------------- P5: channels are the same blend (L118-120)
def test_p5_channel_consistency(c1):
    sc, cam, camv, cfg, r = c1
    ones = Scene(sc.mean, sc.scale, sc.quat, sc.opacity, np.ones_like(sc.rgb))
    r1 = oracle.render(ones, camv, cfg)
    for ch in range(3):
        np.testing.assert_allclose(r1["img"][ch], r["img"][7], atol=1e-13)
    q = sc.quat.astype(np.float64)
    n_c = Rotation.from_quat(q[:, [1, 2, 3, 0]]).as_matrix()[:, :, 2]  # identity pose: t_nc = t_n
    rn = oracle.render(Scene(sc.mean, sc.scale, sc.quat, sc.opacity, n_c.astype(np.float32)), camv, cfg)
    np.testing.assert_allclose(rn["img"][0:3], r["img"][4:7], atol=2e-7)  # rgb carries f32-rounded normals


# ---------------------------------------------------------------- P6: truncation constants -> plain Eq. 8
def test_p6_truncation_limit(c1):
    sc, cam, camv, cfg, r = c1
    smooth = oracle.render(sc, camv, oracle.smooth_cfg())["img"]
    errs = []
    for c, amin, tmin in [(2.0, 1 / 64, 1e-2), (3.0, 1 / 255, 1e-4), (4.0, 1e-4, 1e-6), (6.0, 1e-8, 1e-10), (9.0, 0.0, 0.0)]:
        cc = oracle.make_cfg(cutoff=c, alpha_min=amin, alpha_max=1.0, t_min=tmin, z_near=0.0)
        errs.append(np.abs(oracle.render(sc, camv, cc)["img"] - smooth).max())
    assert all(a > b for a, b in zip(errs, errs[1:])), errs
    assert errs[-1] < 1e-12


# ---------------------------------------------------------------- P7: binning (list structure + conservativeness)
def _numpy_uv(M, X, Y):
    """(u,v) by the textbook route the paper avoids: invert the 3x3 homography with a library
    routine, (u,v,1) ~ M^-1 (x,y,1).  Independent of the oracle's cross-product formula (R1)."""
    Minv = np.linalg.inv(M)
    p = np.stack([X, Y, np.ones_like(X)], axis=-1) @ Minv.T
    return p[..., 0] / p[..., 2], p[..., 1] / p[..., 2]


def test_p7_binning_structure_and_conservativeness(c1):
    sc, cam, camv, cfg, r = c1
    b = oracle.binning(sc, camv, cfg)
    E, keys, idx, ranges = b["E"], b["keys"], b["idx"], b["ranges"]
    assert E == int(b["count"].sum()) == len(keys)
    assert (np.diff(keys.astype(np.uint64)) >= 0).all() if E > 1 else True
    # ranges partition the list in tile order
    nz = ranges[ranges[:, 1] > ranges[:, 0]]
    assert nz[0, 0] == 0 and nz[-1, 1] == E and (nz[1:, 0] == nz[:-1, 1]).all()
    for t, (s, e) in enumerate(ranges):
        assert ((keys[s:e] >> np.uint64(32)) == t).all()
        same = keys[s:e][1:] == keys[s:e][:-1]
        assert (idx[s:e][1:][same] > idx[s:e][:-1][same]).all()      # stable: ties by surfel index
    # depth bits are those of float32(mu_c.z); identity pose => mu_c.z = mean z
    vis = b["culled"] == 0
    assert np.array_equal(b["depth_bits"][vis], sc.mean[vis, 2].view(np.uint32))
    # conservativeness: every covering pair (rho^2 <= c^2 via library inverse) is in the pixel's tile list
    X, Y = pix_grid(cam)
    tile = int(cfg[0])
    tid = (np.arange(cam.height)[:, None] // tile) * b["tiles_x"] + (np.arange(cam.width)[None, :] // tile)
    members = [set(idx[s:e].tolist()) for s, e in ranges]
    n_cover = 0
    tt = np.linspace(0, 2 * np.pi, 20001)
    for k in np.nonzero(vis)[0]:
        u, v = _numpy_uv(b["M"][k].reshape(3, 3), X, Y)
        cover = (u * u + v * v <= 9.0)
        n_cover += cover.sum()
        for t in np.unique(tid[cover]):
            assert k in members[t]
        # the AABB is exact: forward-map the cutoff circle with Eq. 4, x = (M0.p)/(M2.p), p = (3cos t, 3sin t, 1)
        xmin, xmax, ymin, ymax = b["aabb"][k]
        pc = np.stack([3 * np.cos(tt), 3 * np.sin(tt), np.ones_like(tt)], axis=0)
        Mk = b["M"][k].reshape(3, 3)
        ex, ey = (Mk[0] @ pc) / (Mk[2] @ pc), (Mk[1] @ pc) / (Mk[2] @ pc)
        tol = 1e-5 * max(1.0, xmax - xmin, ymax - ymin)
        assert abs(ex.min() - xmin) < tol and abs(ex.max() - xmax) < tol
        assert abs(ey.min() - ymin) < tol and abs(ey.max() - ymax) < tol
    assert n_cover >= r["counters"]["cover"] > 0   # z>z_near and culling only remove pairs


def test_p7b_tile_rect_is_tight_and_conservative():
    """P7b.  The tile rectangle is exactly the set of tiles the screen AABB touches: floor(aabb / 16) clamped to the grid
    (O2 (iv)), checked (i) against that definition recomputed here from the exported AABB (itself pinned against the
    forward-mapped cutoff circle in P7), and (ii) geometrically without any floor: every listed tile's square meets the AABB,
    and no tile next to the rectangle does.  A ceil-for-floor, an off-by-one or a missing clamp fails here.  C1 seen by a
    200 x 120 camera: 13 x 8 tiles, ragged on both axes (200 = 12.5, 120 = 7.5 tiles), many splats crossing the border."""
    sc, _, _ = scenegen.make_config("C1")
    cam = Camera(200, 120, 150.0, 150.0, 97.0, 63.0, scenegen.perturb_pose(np.eye(4)[:3], [0.05, -0.02, 0.1, 0.03, 0.05, -0.2]))
    camv, cfg = oracle.make_cam(cam), oracle.make_cfg()
    b = oracle.binning(sc, camv, cfg)
    tx, ty = b["tiles_x"], b["tiles_y"]
    assert (tx, ty) == (13, 8)
    vis = np.nonzero(b["culled"] == 0)[0]
    assert len(vis) > 500
    aabb, rect = b["aabb"][vis], b["rect"][vis]
    want = np.stack([np.clip(np.floor(aabb[:, 0] / 16), 0, tx - 1), np.clip(np.floor(aabb[:, 2] / 16), 0, ty - 1),
                     np.clip(np.floor(aabb[:, 1] / 16), 0, tx - 1), np.clip(np.floor(aabb[:, 3] / 16), 0, ty - 1)], 1)
    np.testing.assert_array_equal(rect, want.astype(np.int32))
    assert np.array_equal(b["count"][vis], (rect[:, 2] - rect[:, 0] + 1) * (rect[:, 3] - rect[:, 1] + 1))
    clipped = 0
    for (x0, x1, y0, y1), (rx0, ry0, rx1, ry1) in zip(aabb, rect):
        meets_x = lambda t: 16 * t <= x1 and 16 * (t + 1) > x0        # tile column [16 t, 16 t + 16) meets [x0, x1]
        meets_y = lambda t: 16 * t <= y1 and 16 * (t + 1) > y0
        assert all(meets_x(t) for t in range(rx0, rx1 + 1)) and all(meets_y(t) for t in range(ry0, ry1 + 1))
        assert not any(meets_x(t) for t in (rx0 - 1, rx1 + 1) if 0 <= t < tx)      # tight: the neighbours do not
        assert not any(meets_y(t) for t in (ry0 - 1, ry1 + 1) if 0 <= t < ty)
        clipped += (x0 < 0) or (y0 < 0) or (x1 >= 200) or (y1 >= 120)
    assert clipped > 20                                   # the clamp is exercised
    # the list is the rectangles, written out: per tile, exactly the splats whose rectangle holds the tile
    for t in (0, 5, tx - 1, tx * 3 + 6, tx * ty - 1):
        s0, e0 = b["ranges"][t]
        inside = vis[(rect[:, 0] <= t % tx) & (t % tx <= rect[:, 2]) & (rect[:, 1] <= t // tx) & (t // tx <= rect[:, 3])]
        assert sorted(b["idx"][s0:e0].tolist()) == sorted(inside.tolist())


def test_p7_full_forward_against_library_inverse(c1):
    """Whole forward against an independent numpy render: library matrix inverse for (u,v),
    cumulative product for the transmittance (Eq. 8 written as array ops)."""
    sc, cam, camv, cfg, r = c1
    b = oracle.binning(sc, camv, cfg)
    X, Y = pix_grid(cam)
    order = np.lexsort((np.arange(sc.n), b["depth_bits"]))
    order = order[b["culled"][order] == 0]
    amin, amax, tmin, znear = cfg[2], cfg[3], cfg[4], cfg[5]
    T = np.ones_like(X); done = np.zeros_like(X, bool); img = np.zeros((8,) + X.shape)
    n_c = Rotation.from_quat(sc.quat.astype(np.float64)[:, [1, 2, 3, 0]]).as_matrix()[:, :, 2]
    for k in order:
        M = b["M"][k].reshape(3, 3)
        u, v = _numpy_uv(M, X, Y)
        z = M[2, 0] * u + M[2, 1] * v + M[2, 2]
        a = np.minimum(amax, float(sc.opacity[k]) * np.exp(-(u * u + v * v) / 2))
        ok = (u * u + v * v <= 9.0) & (z > znear) & (a >= amin) & ~done
        stop = ok & (T * (1 - a) < tmin)
        done |= stop
        ok &= ~stop
        w = np.where(ok, a * T, 0.0)
        vals = list(sc.rgb[k].astype(np.float64)) + [z] + list(n_c[k]) + [1.0]
        for ch in range(8):
            img[ch] += w * vals[ch]
        T = np.where(ok, T * (1 - a), T)
    good = r["fragile"] == 0
    assert good.mean() > 0.99
    np.testing.assert_allclose(img[:, good], r["img"][:, good], rtol=1e-9, atol=1e-11)


# ---------------------------------------------------------------- P8: finite differences of every gradient
def _tiny(seed=7, n=6):
    g = scenegen.SplitMix(seed)
    mean = np.stack([g.uniform(n, -0.25, 0.25), g.uniform(n, -0.2, 0.2), g.uniform(n, 0.8, 1.6)], 1)
    scale = np.exp(np.stack([g.uniform(n, np.log(0.08), np.log(0.2)) for _ in range(2)], 1))
    quat = np.stack([g.normal(n) for _ in range(4)], 1) * g.uniform(n, 0.5, 2.0)[:, None]   # NOT unit
    quat[:, 0] += 2.0 * np.sign(quat[:, 0])  # mostly camera-facing
    sc = Scene(mean.astype(np.float32), scale.astype(np.float32), quat.astype(np.float32),
               g.uniform(n, 0.3, 0.95).astype(np.float32), np.stack([g.uniform(n) for _ in range(3)], 1).astype(np.float32))
    cam = Camera(16, 12, 14.0, 15.0, 8.3, 5.6, scenegen.perturb_pose(np.eye(4)[:3], [0.02, -0.03, 0.05, 0.04, -0.03, 0.06]))
    return sc, cam


_NORMALISED = [False]   # _loss / _fd_check differentiate the normalised-depth images (P16) when set


def _loss(sc, camv, cfg, up):
    r = oracle.render_normalised if _NORMALISED[0] else oracle.render
    return float((r(sc, camv, cfg, counters=False)["img"] * up).sum())


def _decisions(sc, camv, cfg):
    r = oracle.render(sc, camv, cfg, counters=False)
    return r["n_comp"]


def _fd_check(cfg, rtol, scene=None, guard=False, hexp=-12):
    """guard: the truncation rules make the image piecewise smooth; a central difference is the derivative of the current
    piece only if no discrete decision changes between the two evaluations -- asserted through the per-pixel count of
    composited splats (a skip <-> composite or a stop flip changes it)."""
    sc, cam = scene if scene is not None else _tiny()
    camv = oracle.make_cam(cam, widen_from_f32=False)
    n0 = _decisions(sc, camv, cfg) if guard else None
    up = scenegen.upstream_normal(11, cam.height, cam.width).astype(np.float64)
    g = (oracle.backward_normalised if _NORMALISED[0] else oracle.backward)(sc, camv, cfg, up)
    worst = 0.0
    for name in ("mean", "scale", "quat", "opacity", "rgb"):
        arr = getattr(sc, name)
        flat = arr.reshape(-1)
        ga = g[name].reshape(-1)
        scale_ref = np.abs(ga).max() + 1e-30
        for e in range(flat.size):
            x0 = flat[e]
            h = np.float32(max(abs(float(x0)), 0.05) * 2.0 ** hexp)
            xp, xm = np.float32(x0 + h), np.float32(x0 - h)
            flat[e] = xp; lp = _loss(sc, camv, cfg, up)
            if guard: assert np.array_equal(_decisions(sc, camv, cfg), n0), (name, e, "+h crosses a decision")
            flat[e] = xm; lm = _loss(sc, camv, cfg, up)
            if guard: assert np.array_equal(_decisions(sc, camv, cfg), n0), (name, e, "-h crosses a decision")
            flat[e] = x0
            fd = (lp - lm) / (float(xp) - float(xm))          # exact step between two float32 inputs
            err = abs(fd - ga[e]) / scale_ref
            worst = max(worst, err)
            assert err < rtol, (name, e, fd, ga[e])
    # SE(3) pose: central differences of L(Exp(+-eps e_i) o T_cw)   (Eq. 12)
    eps = 1e-6
    for i in range(6):
        tau = np.zeros(6); tau[i] = eps
        cp, cm = (oracle.make_cam(cam, scenegen.perturb_pose(cam.T_cw, s_ * tau), False) for s_ in (1, -1))
        lp, lm = _loss(sc, cp, cfg, up), _loss(sc, cm, cfg, up)
        if guard: assert np.array_equal(_decisions(sc, cp, cfg), n0) and np.array_equal(_decisions(sc, cm, cfg), n0), i
        fd = (lp - lm) / (2 * eps)
        assert abs(fd - g["pose"][i]) < rtol * np.abs(g["pose"]).max(), (i, fd, g["pose"])
    return worst


def test_p8_finite_differences_smooth():
    """Plain Eq. 8 (no truncation): every surfel gradient and the SE(3) pose gradient."""
    _fd_check(oracle.smooth_cfg(), 2e-6)


def test_p8_finite_differences_alpha_clamp():
    """alpha_max clamp active (true derivative = 0 when clamped, R5), other truncations off."""
    cfg = oracle.make_cfg(cutoff=np.inf, alpha_min=0.0, alpha_max=0.6, t_min=0.0, z_near=0.0)
    sc, cam = _tiny()
    r = oracle.render(sc, oracle.make_cam(cam, widen_from_f32=False), cfg)
    assert (r["fragile"] & 2).sum() == 0, "pick another seed: a pixel sits on the clamp boundary"
    _fd_check(cfg, 2e-6)


def _stacked(seed=3):
    """A tiny scene on which EVERY truncation rule of Eq. 8 (R3-R7) acts: three nearly opaque splats stacked on the axis
    (pixels behind them stop: T (1 - a) < 1e-4), splats behind the stack (cut off by the stop), a faint splat (o = 0.2: the
    a >= 1/255 test bites inside the cutoff), splat rims inside the image (rho^2 = 9), opacities above alpha_max = 0.99's
    reach (o G clamped), and a small tilted splat whose near side dips under z_near = 0.2."""
    g = scenegen.SplitMix(seed)
    n = 9
    mean = np.array([[0.02, 0.01, 0.9], [-0.03, 0.02, 1.0], [0.01, -0.02, 1.1], [0.05, 0.03, 1.3], [-0.2, 0.1, 1.4],
                     [0.25, -0.12, 1.2], [-0.1, -0.15, 0.8], [0.03, 0.02, 0.27], [0.15, 0.12, 1.6]])
    scale = np.array([[0.12, 0.1], [0.11, 0.13], [0.14, 0.1], [0.2, 0.18], [0.1, 0.08], [0.09, 0.12], [0.07, 0.1], [0.05, 0.045],
                      [0.16, 0.2]])
    opac = np.array([0.995, 0.985, 0.98, 0.9, 0.2, 0.7, 0.5, 0.6, 0.95])
    quat = np.stack([g.normal(n) for _ in range(4)], 1) * 0.25
    quat[:, 0] += 1.5
    quat[7] = [0.55, 0.8, 0.15, 0.1]       # the near splat: tilted ~ 110 deg about x, so its far side rises and its near side dips
    rgb = np.stack([g.uniform(n) for _ in range(3)], 1)
    sc = Scene(mean.astype(np.float32), scale.astype(np.float32), quat.astype(np.float32), opac.astype(np.float32),
               rgb.astype(np.float32))
    cam = Camera(16, 12, 14.0, 15.0, 8.3, 5.6, scenegen.perturb_pose(np.eye(4)[:3], [0.01, -0.02, 0.02, 0.02, -0.015, 0.03]))
    # the front splat is fully opaque and centred on pixel (8, 6): there o G = 1 > alpha_max, the clamp acts
    T = np.asarray(cam.T_cw, dtype=np.float64)
    Xc = np.array([(8.5 - 8.3) / 14.0 * 0.9, (6.5 - 5.6) / 15.0 * 0.9, 0.9])
    sc.mean[0] = (T[:, :3].T @ (Xc - T[:, 3])).astype(np.float32)
    sc.opacity[0] = 1.0
    return sc, cam


def test_p8b_finite_differences_with_every_truncation_rule_active():
    """P8b.  Central finite differences of every surfel gradient and of the SE(3) pose gradient under the DEFAULT config
    (cutoff 3, alpha_min, alpha_max, T_min stop, z_near): pins the backward's replay loop -- which pairs it revisits, that the
    stopping splat and everything behind it get nothing, the clamp's zero derivative.  The scene is checked to exercise
    each rule (switching the rule off changes the image), to have pixels that stop, and to have no fragile pixel; the
    guard in _fd_check asserts that no decision flips inside a difference."""
    sc, cam = _stacked()
    camv = oracle.make_cam(cam, widen_from_f32=False)
    cfg = oracle.make_cfg()
    r = oracle.render(sc, camv, cfg)
    assert (r["fragile"] != 0).sum() == 0, "a pixel sits within 1e-4 of a threshold: move a splat"
    assert (r["T_final"] < 1e-2).sum() >= 4 and r["counters"]["Q_t"] > r["counters"]["Q_tb"]   # pixels that stop early
    base = r["img"]
    for name, kw in (("cutoff", dict(cutoff=12.0)), ("alpha_min", dict(alpha_min=0.0)), ("alpha_max", dict(alpha_max=0.99999)),
                     ("t_min", dict(t_min=0.0)), ("z_near", dict(z_near=1e-3))):
        other = oracle.render(sc, camv, oracle.make_cfg(**kw), counters=False)["img"]
        assert np.abs(other - base).max() > 1e-6, name + " never acts on this scene"
    # the stop is not a no-op for the gradient either: splats behind the stack get less than without it
    up = scenegen.upstream_normal(11, cam.height, cam.width).astype(np.float64)
    g1, g0 = oracle.backward(sc, camv, cfg, up), oracle.backward(sc, camv, oracle.make_cfg(t_min=0.0), up)
    assert np.abs(g1["rgb"] - g0["rgb"]).max() > 1e-9
    _fd_check(cfg, 1e-5, scene=(sc, cam), guard=True, hexp=-19)


def test_comparison_support_is_pinned_to_the_backward(c1):
    """oracle.exposure / oracle.pixel_bounds only feed the tolerance of the GPU parity tests, but a wrong bound would hide
    errors.  (i) signed_all: the exposure's own pair-by-pair chain recomputes the whole gradient and must equal
    oracle.backward.  (ii) With every pixel handed in as `extra_mask` the result dominates |backward| (sum of |.| >= |sum|).
    (iii) A pixel is exposed iff the forward marks it fragile (or the mask names it); zero upstream there gives zero.
    (iv) A constructed flip: one fronto-parallel splat and alpha_min set 5e-5 below the closed-form alpha of ONE pixel:
    that pixel is the only exposed one, inverting its decision removes its whole contribution, so the exposure of the
    colour gradient is |g| a and of the opacity gradient |g . v| G there -- hand values.  (v) pixel_bounds: flip_w is
    positive only on decision-fragile pixels and equals a T of the pair at stake in (iv); kappa = 1 for a fronto-parallel
    splat, so kerr = w rho^2 in closed form; zmax >= the blended depth."""
    sc, cam, camv, cfg, r = c1
    up = scenegen.upstream_normal(1, cam.height, cam.width)
    g = oracle.backward(sc, camv, cfg, up)
    e = oracle.exposure(sc, camv, cfg, up, signed_all=True)
    for k in ("mean", "scale", "quat", "opacity", "rgb", "pose"):
        np.testing.assert_allclose(e[k], g[k], rtol=1e-9, atol=1e-9 * np.abs(g[k]).max())
    full = oracle.exposure(sc, camv, cfg, up, extra_mask=np.ones((cam.height, cam.width), np.uint8))
    for k in ("mean", "scale", "quat", "opacity", "rgb"):
        assert (full[k] >= np.abs(g[k]) * (1 - 1e-9) - 1e-12).all(), k
    a = oracle.exposure(sc, camv, cfg, up)
    assert np.array_equal(a["pix_exposed"] != 0, r["fragile"] != 0) and (r["fragile"] != 0).sum() > 3
    assert all((a[k] <= full[k] * (1 + 1e-9) + 1e-12).all() for k in ("mean", "scale", "quat", "opacity", "rgb"))
    none = oracle.exposure(sc, camv, cfg, up * (a["pix_exposed"] == 0)[None])    # zero upstream on every exposed pixel
    assert all(np.abs(none[k]).max() == 0 for k in ("mean", "scale", "quat", "opacity", "rgb", "pose"))
    extra = np.zeros((cam.height, cam.width), np.uint8); extra[10:20, 10:30] = 1
    b = oracle.exposure(sc, camv, cfg, up, extra_mask=extra)
    assert ((b["pix_exposed"] != 0) == ((r["fragile"] != 0) | (extra != 0))).all() and b["rgb"].sum() > a["rgb"].sum()
    pb = oracle.pixel_bounds(sc, camv, cfg)
    assert ((pb["flip_w"] > 0) <= ((r["fragile"] & 1) != 0)).all() and (pb["flip_w"] > 0).sum() > 0
    assert (pb["flip_w"] <= 2.0 + 1e-12).all() and (pb["kerr"] >= 0).all() and (pb["kerr_z"] >= 0).all()
    comp = r["n_comp"] > 0
    assert (pb["zmax"][comp] >= (r["img"][3][comp] / r["img"][7][comp]) * (1 - 1e-12)).all()   # max depth >= mean depth
    # (iv), (v) on one fronto-parallel splat with closed-form alpha (P1)
    mu, su, sv, o = (0.31, -0.17, 1.5), float(np.float32(0.11)), float(np.float32(0.07)), float(np.float32(0.8))
    one = one_surfel(mu, (su, sv), (1, 0, 0, 0), o)
    mu32 = np.float32(mu).astype(np.float64)
    X, Y = pix_grid(CAM)
    u = ((X - CAM.cx) * mu32[2] / CAM.fx - mu32[0]) / su; v = ((Y - CAM.cy) * mu32[2] / CAM.fy - mu32[1]) / sv
    G = np.exp(-(u * u + v * v) / 2); al = o * G
    jj, ii = np.unravel_index(np.argmin(np.abs(al - 0.05)), al.shape)       # a pixel on the splat's flank
    cfg1 = oracle.make_cfg(alpha_min=al[jj, ii] / (1 + 5e-5))
    camv1 = oracle.make_cam(CAM)
    up1 = scenegen.upstream_normal(5, CAM.height, CAM.width)
    r1 = oracle.render(one, camv1, cfg1)
    assert (r1["fragile"] != 0).sum() == 1 and r1["fragile"][jj, ii] == 1 and r1["img"][7][jj, ii] > 0
    x1 = oracle.exposure(one, camv1, cfg1, up1)
    gpix = up1[:, jj, ii]
    np.testing.assert_allclose(x1["rgb"][0], np.abs(gpix[0:3]) * al[jj, ii], rtol=1e-9)
    rgb1 = one.rgb[0].astype(np.float64)
    gv = gpix[0:3] @ rgb1 + gpix[3] * mu32[2] + gpix[6] * 1.0 + gpix[7]      # v = (rgb, z0, n = +z, 1); T = 1, no suffix
    np.testing.assert_allclose(x1["opacity"][0], abs(gv) * G[jj, ii], rtol=1e-9)
    pb1 = oracle.pixel_bounds(one, camv1, cfg1)
    assert (pb1["flip_w"] > 0).sum() == 1 and abs(pb1["flip_w"][jj, ii] - al[jj, ii]) < 1e-12
    w1 = r1["img"][7]
    np.testing.assert_allclose(pb1["kerr"], w1 * (u * u + v * v), atol=1e-9)
    np.testing.assert_allclose(pb1["kerr_z"], 0.0, atol=1e-12)               # fronto-parallel: M20 = M21 = 0


# ---------------------------------------------------------------- P9: rigid-motion identity (no FD)
def test_p9_rigid_motion_identity():
    sc, cams, _ = scenegen.make_config("C1")
    cam = Camera(64, 48, 60.0, 60.0, 32.0, 24.0, scenegen.perturb_pose(np.eye(4)[:3], [0.1, -0.2, 0.15, 0.2, -0.1, 0.3]))
    camv, cfg = oracle.make_cam(cam), oracle.make_cfg()
    up = scenegen.upstream_normal(3, cam.height, cam.width)
    g = oracle.backward(sc, camv, cfg, up)
    T = camv[6:].reshape(3, 4); R, t = T[:, :3], T[:, 3]
    c_cam = -R.T @ t
    gm, gq = g["mean"], g["quat"]
    q = sc.quat.astype(np.float64); w, v = q[:, :1], q[:, 1:]
    gw, gv = gq[:, :1], gq[:, 1:]
    rot_term = 0.5 * (-gw * v + w * gv + np.cross(v, gv))
    d_rho = R @ gm.sum(0)
    d_theta = R @ (np.cross(sc.mean.astype(np.float64) - c_cam, gm) + rot_term).sum(0)
    s = np.abs(g["pose"]).max()
    np.testing.assert_allclose(g["pose"][:3], d_rho, atol=1e-9 * s)
    np.testing.assert_allclose(g["pose"][3:], d_theta, atol=1e-9 * s)
    # scale gradient is invisible to a rigid motion but the quaternion gradient must be tangent to |q|
    assert np.abs((q * gq).sum(1)).max() < 1e-9 * np.abs(gq).max()


# ---------------------------------------------------------------- P10: symmetries
def test_p10_swap_tangents(c1):
    sc, cam, camv, cfg, r = c1
    q = sc.quat.astype(np.float64)
    s = np.sqrt(0.5)
    qs = np.array([0.0, s, s, 0.0])  # 180 deg about (1,1,0): t_u <-> t_v, t_n -> -t_n
    w1, v1 = q[:, :1], q[:, 1:]
    q2 = np.concatenate([w1 * qs[0] - v1 @ qs[1:, None], w1 * qs[1:] + qs[0] * v1 + np.cross(v1, qs[1:])], axis=1)
    sw = Scene(sc.mean, sc.scale[:, ::-1].copy(), q2.astype(np.float32), sc.opacity, sc.rgb)
    r2 = oracle.render(sw, camv, cfg)
    good = (r["fragile"] == 0) & (r2["fragile"] == 0)
    np.testing.assert_allclose(r2["img"][[0, 1, 2, 3, 7]][:, good], r["img"][[0, 1, 2, 3, 7]][:, good], rtol=1e-4, atol=2e-5)
    np.testing.assert_allclose(r2["img"][4:7][:, good], -r["img"][4:7][:, good], rtol=1e-4, atol=2e-5)


def test_p10_mask_equals_subset():
    sc, cams, _ = scenegen.make_config("C1")
    act = (scenegen.SplitMix(99).uniform(sc.n) < 0.3).astype(np.uint8)
    camv, cfg = oracle.make_cam(cams[0]), oracle.make_cfg()
    masked = Scene(sc.mean, sc.scale, sc.quat, sc.opacity, sc.rgb, act)
    m = act.astype(bool)
    sub = Scene(sc.mean[m], sc.scale[m], sc.quat[m], sc.opacity[m], sc.rgb[m])
    ra, rs = oracle.render(masked, camv, cfg), oracle.render(sub, camv, cfg)
    assert np.array_equal(ra["img"], rs["img"])
    ba, bs = oracle.binning(masked, camv, cfg), oracle.binning(sub, camv, cfg)
    remap = np.nonzero(m)[0]
    assert np.array_equal(ba["keys"], bs["keys"]) and np.array_equal(ba["idx"], remap[bs["idx"]])
    up = scenegen.upstream_normal(5, 48, 64)
    ga, gs = oracle.backward(masked, camv, cfg, up), oracle.backward(sub, camv, cfg, up)
    assert (ga["mean"][~m] == 0).all() and (ga["quat"][~m] == 0).all() and (ga["opacity"][~m] == 0).all()
    np.testing.assert_allclose(ga["mean"][m], gs["mean"], rtol=1e-10, atol=1e-9)
    np.testing.assert_allclose(ga["pose"], gs["pose"], rtol=1e-10)


def test_no_view_dependence_of_colour():
    """L128: no spherical harmonics -- rotating the camera about its centre leaves a surfel's
    blended colour / alpha ratio at its own centre pixel unchanged."""
    sc = one_surfel((0.0, 0.0, 2.0), (0.3, 0.3), (1, 0, 0, 0), 0.7, (0.3, 0.6, 0.9))
    for ang in (0.0, 0.1, -0.2):
        T = scenegen.perturb_pose(np.eye(4)[:3], [0, 0, 0, 0, ang, 0])
        r = oracle.render(sc, oracle.make_cam(CAM, T), oracle.make_cfg())
        m = r["img"][7] > 0.05
        for ch, c in enumerate((0.3, 0.6, 0.9)):
            np.testing.assert_allclose(r["img"][ch][m] / r["img"][7][m], float(np.float32(c)), rtol=1e-12)


# ---------------------------------------------------------------- P11: per-splat contribution and covisibility (Eq. 20-22)
def _footprint_alpha(mu, su, sv, o, cam=CAM):
    """Closed-form alpha image of a fronto-parallel surfel (as P1), fp64, with the truncation conventions."""
    X, Y = pix_grid(cam)
    mu32 = np.float32(mu).astype(np.float64); su, sv, o = [float(np.float32(v)) for v in (su, sv, o)]
    u = ((X - cam.cx) * mu32[2] / cam.fx - mu32[0]) / su
    v = ((Y - cam.cy) * mu32[2] / cam.fy - mu32[1]) / sv
    a = np.minimum(o * np.exp(-(u * u + v * v) / 2), float(np.float32(0.99)))
    a[(u * u + v * v > 9.0) | (a < float(np.float32(1 / 255)))] = 0.0
    return a


def test_p11_contribution_sums_to_the_alpha_image(c1):
    """Eq. 21 summed over k is Eq. 8's accumulated opacity summed over the pixels: sum_k C_k = sum_p O(p)."""
    sc, cam, camv, cfg, r = c1
    C = oracle.contribution(sc, camv, cfg)
    assert abs(C.sum() - r["img"][7].sum()) <= 1e-10 * C.sum()
    assert (C >= 0).all() and (C[oracle.binning(sc, camv, cfg)["culled"].astype(bool)] == 0).all()
    assert np.abs(C - oracle.contribution(sc, camv, cfg, brute=True)).max() <= 1e-12 * C.max()


def test_p11_single_surfel_and_occlusion_closed_forms():
    """C of a lone fronto-parallel splat is the sum of its closed-form footprint; behind a second splat with the same
    footprint every coefficient is scaled by that pixel's (1 - a_front) (Eq. 20)."""
    a_front = _footprint_alpha((0.1, -0.05, 1.5), 0.09, 0.06, 0.7)
    sc1 = one_surfel((0.1, -0.05, 1.5), (0.09, 0.06), (1, 0, 0, 0), 0.7)
    camv, cfg = oracle.make_cam(CAM), oracle.make_cfg()
    np.testing.assert_allclose(oracle.contribution(sc1, camv, cfg), [a_front.sum()], rtol=1e-12)
    a_back = _footprint_alpha((0.0, 0.0, 2.5), 0.2, 0.2, 0.9)
    sc2 = cat(one_surfel((0.0, 0.0, 2.5), (0.2, 0.2), (1, 0, 0, 0), 0.9), sc1)   # index order != depth order
    C = oracle.contribution(sc2, camv, cfg)
    np.testing.assert_allclose(C, [(a_back * (1 - a_front)).sum(), a_front.sum()], rtol=1e-12)


def test_p11_contribution_approaches_the_footprint_integral():
    """"How many pixels the splat contributes to" (L214): for a footprint of many pixels C tends to the integral of
    o exp(-rho^2/2) over the cutoff ellipse, 2 pi o sx sy (1 - exp(-c^2/2)) with s = f s_world / z pixels."""
    cam = Camera(400, 300, 300.0, 300.0, 200.0, 150.0)
    su, sv, o, z0 = 0.12, 0.08, 0.6, 2.0
    sc = one_surfel((0.0, 0.0, z0), (su, sv), (1, 0, 0, 0), o)
    C = oracle.contribution(sc, oracle.make_cam(cam), oracle.make_cfg())[0]
    sx, sy = 300.0 * float(np.float32(su)) / z0, 300.0 * float(np.float32(sv)) / z0
    expect = 2 * np.pi * float(np.float32(o)) * sx * sy * (1 - np.exp(-4.5))
    assert abs(C - expect) <= 2e-3 * expect


def test_p11_covisibility_hand_example():
    """Eq. 22 on a hand example: G_A = {0,1,2}, G_B = {1,2,3} -> 2/4; identical views -> 1; disjoint -> 0."""
    CA = np.array([0.9, 3.0, 0.51, 0.5, 0.0]); CB = np.array([0.2, 0.6, 7.0, 0.7, 0.5])
    assert oracle.covisibility(CA, CB) == (0.5, 2, 4)
    assert oracle.covisibility(CA, CA)[0] == 1.0
    assert oracle.covisibility(CA, np.zeros(5)) == (0.0, 0, 3)
    act = np.array([1, 0, 1, 1, 1], np.uint8)                       # only splats of the active map count (L216)
    assert oracle.covisibility(CA, CB, active=act) == (1 / 3, 1, 3)
    assert oracle.covisibility(np.zeros(3), np.zeros(3)) == (0.0, 0, 0)


# ---------------------------------------------------------------- P12: tracking loss harness (Eq. 15-19)
def test_p12_tracking_loss_hand_example_masks_and_gradient():
    """Eq. 15-19 on a 2x2 frame evaluated by hand: pixel (0,0) passes both masks, (1,0) fails M_o (alpha 0.9),
    (0,1) fails M_n (normal faces away), (1,1) passes.  L_t = (1/4) sum M_n M_o (|dI|_1 + lambda_d |dD|)."""
    cam = Camera(2, 2, 1.0, 1.0, 1.0, 1.0)
    camv = oracle.make_cam(cam)
    img = np.zeros((8, 2, 2))
    img[0:3] = [[[0.5, 0.2], [0.3, 0.9]], [[0.1, 0.2], [0.3, 0.4]], [[0.0, 0.2], [0.3, 0.6]]]
    img[3] = [[2.0, 1.0], [1.5, 3.0]]
    img[6] = [[1.0, 1.0], [-1.0, 1.0]]                  # N_r = (0, 0, +-1): N.r = +-1 for every ray (r_z = 1)
    img[7] = [[0.99, 0.9], [0.99, 0.96]]
    trgb = np.zeros((3, 2, 2)); trgb[:, 0, 0] = [0.4, 0.3, 0.0]; trgb[:, 1, 1] = [1.0, 0.1, 0.6]
    tdep = np.array([[2.5, 0.0], [3.0, 2.0]])
    L, up = oracle.tracking_loss(img, trgb, tdep, camv, 0.5, 1.0)
    # (0,0): |0.1| + |-0.2| + 0 + 0.5 |-0.5| = 0.55 ; (1,1): |-0.1| + |0.3| + 0 + 0.5 |1.0| = 0.9
    assert abs(L - (0.55 + 0.9) / 4) < 1e-15
    assert (up[:, 0, 1] == 0).all() and (up[:, 1, 0] == 0).all() and (up[4:] == 0).all()
    np.testing.assert_allclose(up[0:4, 0, 0], np.array([1, -1, 0, -0.5]) / 4)
    np.testing.assert_allclose(up[0:4, 1, 1], np.array([-1, 1, 0, 0.5]) / 4)
    # the other sign convention (R19) swaps which pixels pass M_n
    L2, _ = oracle.tracking_loss(img, trgb, tdep, camv, 0.5, -1.0)
    assert abs(L2 - (0.3 + 0.3 + 0.3 + 0.5 * 1.5) / 4) < 1e-15     # only (0,1): rgb 0.3 each, depth |1.5 - 3.0|


def test_p12_p13_holes_in_the_sensor_depth_carry_no_depth_term():
    """Reading R25: a pixel whose target depth is a hole (0, negative, inf, NaN -- how RGB-D sensors encode "no
    measurement", L350) contributes its colour term only: hand values on a 2x2 frame, for Eq. 19 and for Eq. 26."""
    cam = Camera(2, 2, 1.0, 1.0, 1.0, 1.0)
    camv = oracle.make_cam(cam)
    img = np.zeros((8, 2, 2))
    img[0] = [[0.5, 0.25], [0.75, 1.0]]                   # only the red channel differs from the (zero) target
    img[3] = [[2.0, 1.0], [1.5, 3.0]]
    img[6] = 1.0; img[7] = 0.99                           # every pixel passes M_n and M_o
    trgb = np.zeros((3, 2, 2))
    for hole in (0.0, -1.0, np.inf, np.nan):
        tdep = np.array([[2.5, hole], [hole, 2.0]])
        L, up = oracle.tracking_loss(img, trgb, tdep, camv, 0.5, 1.0)
        # colour: 0.5 + 0.25 + 0.75 + 1.0 = 2.5; depth only at (0,0) and (1,1): 0.5 (0.5 + 1.0)
        assert abs(L - (2.5 + 0.5 * 1.5) / 4) < 1e-15, hole
        np.testing.assert_array_equal(up[3], np.array([[-0.5, 0.0], [0.0, 0.5]]) / 4)
        np.testing.assert_array_equal(up[0], np.full((2, 2), 0.25))
        Lm, upm = oracle.mapping_loss(img, trgb, tdep, camv, 0.875, 0.5, 0.0, 1.0)   # w_n = 0: no normal term
        assert abs(Lm - (0.875 * 2.5 + 0.5 * 1.5) / 4) < 1e-15, hole
        np.testing.assert_array_equal(upm[3], np.array([[-0.5, 0.0], [0.0, 0.5]]) / 4)
        assert np.isfinite(up).all() and np.isfinite(upm).all()


def test_p12_tracking_loss_gradient_is_its_finite_difference(c1):
    """`up` is dL_t/d(image) wherever L_t is differentiable (central differences on the C1 render)."""
    sc, cam, camv, cfg, r = c1
    img = r["img"].copy()
    img[7] = np.where(img[7] > 0.5, 0.97, img[7])       # let a good share of pixels pass M_o = [O > 0.95]
    g = scenegen.SplitMix(5)
    trgb = img[0:3] + 0.05 * g.normal(img[0:3].size).reshape(img[0:3].shape)
    tdep = img[3] + 0.1 * g.normal(img[3].size).reshape(img[3].shape)
    for nsign in (1.0, -1.0):
        L, up = oracle.tracking_loss(img, trgb, tdep, camv, 0.5, nsign)
        nz = np.argwhere(up != 0)
        assert len(nz) > 50
        for ch, j, i in nz[:: max(1, len(nz) // 40)]:
            d = np.zeros_like(img); d[ch, j, i] = 1e-6
            fd = (oracle.tracking_loss(img + d, trgb, tdep, camv, 0.5, nsign)[0] -
                  oracle.tracking_loss(img - d, trgb, tdep, camv, 0.5, nsign)[0]) / 2e-6
            assert abs(fd - up[ch, j, i]) <= 1e-6 * abs(up[ch, j, i]) + 1e-12
    assert oracle.tracking_loss(img, img[0:3], img[3], camv, 0.5, 1.0)[0] == 0.0


# ---------------------------------------------------------------- P13: normal from depth and the mapping loss (Eq. 23-26)
def _plane_depth(cam, n, d):
    """Depth image of the plane n.X = d seen by `cam` (closed form: z = d / (n . ray))."""
    X, Y = pix_grid(cam)
    ray = np.stack([(X - cam.cx) / cam.fx, (Y - cam.cy) / cam.fy, np.ones_like(X)], 0)
    return d / (n[:, None, None] * ray).sum(0), ray


def test_p13_normal_from_depth_of_a_plane_is_the_plane_normal():
    """Differences of points of a plane lie in the plane: Eq. 23 returns the plane's unit normal exactly (interior)."""
    cam = Camera(40, 30, 50.0, 45.0, 19.0, 16.0)
    camv = oracle.make_cam(cam)
    for n in ([0.0, 0.0, 1.0], [0.3, -0.2, 0.9], [-0.5, 0.4, 0.6]):
        n = np.array(n) / np.linalg.norm(n)
        D, _ = _plane_depth(cam, n, 2.0)
        assert (D > 0).all()
        N = oracle.normal_from_depth(D, camv)
        np.testing.assert_allclose(N[:, 1:-1, 1:-1], np.broadcast_to(n[:, None, None], (3, 28, 38)), atol=1e-10)
        assert (N[:, 0] == 0).all() and (N[:, :, -1] == 0).all()      # border: undefined -> 0


def test_p13_mapping_loss_values_and_gradient():
    """Eq. 24-26 (no SSIM): exact values on a plane (L_n = 0 where N_r = N_D, 2 where N_r = -N_D), and `up` equals
    central finite differences of L on a bumpy depth image."""
    cam = Camera(24, 18, 30.0, 28.0, 12.5, 8.0)
    camv = oracle.make_cam(cam)
    n = np.array([0.2, -0.3, 0.93]); n /= np.linalg.norm(n)
    D, _ = _plane_depth(cam, n, 1.7)
    img = np.zeros((8, 18, 24)); img[3] = D; img[4:7] = n[:, None, None]
    HW = 24 * 18
    L, _ = oracle.mapping_loss(img, img[0:3], D, camv, 0.875, 0.5, 0.02, 1.0)
    border = HW - 22 * 16
    assert abs(L - 0.02 * border / HW) < 1e-12                       # interior consistent; the border keeps L_n = 1
    L, _ = oracle.mapping_loss(img, img[0:3], D, camv, 0.875, 0.5, 0.02, -1.0)
    assert abs(L - 0.02 * (border + 2 * 22 * 16) / HW) < 1e-12
    L, _ = oracle.mapping_loss(img, img[0:3] + 0.1, D - 0.25, camv, 0.875, 0.5, 0.0)
    assert abs(L - (0.875 * 0.3 + 0.5 * 0.25)) < 1e-12
    # gradient check on a generic image
    g = scenegen.SplitMix(9)
    img[3] = D + 0.05 * g.normal(HW).reshape(18, 24)
    img[4:7] = g.normal(3 * HW).reshape(3, 18, 24)
    img[0:3] = g.uniform(3 * HW).reshape(3, 18, 24)
    trgb, tdep = g.uniform(3 * HW).reshape(3, 18, 24), D
    args = (trgb, tdep, camv, 0.875, 0.5, 0.3, -1.0)
    L, up = oracle.mapping_loss(img, *args)
    assert (up[7] == 0).all()
    for ch, j, i in [(3, 5, 7), (3, 1, 1), (3, 0, 4), (3, 9, 23), (3, 16, 12), (4, 6, 6), (5, 3, 20), (6, 10, 2), (0, 2, 2),
                     (2, 17, 23), (3, 8, 11), (3, 2, 21)]:
        d = np.zeros_like(img); d[ch, j, i] = 1e-6
        fd = (oracle.mapping_loss(img + d, *args)[0] - oracle.mapping_loss(img - d, *args)[0]) / 2e-6
        assert abs(fd - up[ch, j, i]) <= 2e-6 * abs(up[ch, j, i]) + 1e-11, (ch, j, i, fd, up[ch, j, i])


# ---------------------------------------------------------------- P14: map correction (Eq. 31-32)
def _rand_poses(g, k, scale=1.0):
    rot = Rotation.from_rotvec(scale * np.stack([g.normal(3) for _ in range(k)]))
    T = np.zeros((k, 3, 4)); T[:, :, :3] = rot.as_matrix(); T[:, :, 3] = 2.0 * np.stack([g.normal(3) for _ in range(k)])
    return T


def test_p14_map_correction_moves_splats_rigidly_with_their_keyframe():
    """A splat expressed in its keyframe's frame keeps those coordinates: T_o^{-1} (mu', R') = T^{-1} (mu, R) (what Eq.
    31-32 mean), checked with scipy rotations; identity increments leave the map unchanged; two splats of one keyframe
    keep their distance."""
    g = scenegen.SplitMix(31)
    n, K = 200, 7
    To, Tn = _rand_poses(g, K), _rand_poses(g, K)
    mean = np.stack([g.normal(n) for _ in range(3)], 1)
    quat = np.stack([g.normal(n) for _ in range(4)], 1) * 1.7          # not unit
    fid = (g.uniform(n) * K).astype(np.int32)
    mu2, R2 = oracle.map_correction(mean, quat, fid, To, Tn)
    qx = quat / np.linalg.norm(quat, axis=1, keepdims=True)
    R = Rotation.from_quat(np.stack([qx[:, 1], qx[:, 2], qx[:, 3], qx[:, 0]], 1)).as_matrix()   # scipy: (x,y,z,w)
    np.testing.assert_allclose(oracle.quat_to_matrix(quat), R, atol=1e-12)
    for k in range(n):
        Ro, to, Rn, tn = To[fid[k], :, :3], To[fid[k], :, 3], Tn[fid[k], :, :3], Tn[fid[k], :, 3]
        np.testing.assert_allclose(Rn.T @ (mu2[k] - tn), Ro.T @ (mean[k] - to), atol=1e-10)   # same local coordinates
        np.testing.assert_allclose(Rn.T @ R2[k], Ro.T @ R[k], atol=1e-10)                      # same local orientation
        assert abs(np.linalg.det(R2[k]) - 1) < 1e-10
    mu3, R3 = oracle.map_correction(mean, quat, fid, To, To)
    np.testing.assert_allclose(mu3, mean, atol=1e-12); np.testing.assert_allclose(R3, R, atol=1e-12)
    a, b = np.nonzero(fid == fid[0])[0][:2]
    assert abs(np.linalg.norm(mu2[a] - mu2[b]) - np.linalg.norm(mean[a] - mean[b])) < 1e-10


# ---------------------------------------------------------------- P15: SSIM term of Eq. 24
def test_p15_ssim_closed_forms_brute_force_and_gradient():
    g = scenegen.SplitMix(15)
    H, W = 17, 23
    x = g.uniform(3 * H * W).reshape(3, H, W); y = np.clip(x + 0.1 * g.normal(3 * H * W).reshape(3, H, W), 0, 1)
    # identical images: SSIM = 1 everywhere -> loss 0, gradient 0
    L, gr = oracle.ssim_loss(x, x, 0.125)
    assert abs(L) < 1e-14 and np.abs(gr).max() < 1e-12
    # constant images (far from the zero-padded border): SSIM = (2 c1 c2 + C1) / (c1^2 + c2^2 + C1), variances are 0
    c1, c2 = 0.3, 0.7
    Lc, _ = oracle.ssim_loss(np.full((1, 41, 41), c1), np.full((1, 41, 41), c2), 1.0)
    s_int = (2 * c1 * c2 + 1e-4) / (c1 * c1 + c2 * c2 + 1e-4)
    big = np.full((1, 41, 41), c1); bigy = np.full((1, 41, 41), c2)
    # interior pixel value through the brute-force definition below
    def ssim_at(xx, yy, j, i):
        w1 = oracle.ssim_window(); acc = dict(m1=0, m2=0, e11=0, e22=0, e12=0)
        for dj in range(-5, 6):
            for di in range(-5, 6):
                jj, ii = j + dj, i + di
                if 0 <= jj < xx.shape[0] and 0 <= ii < xx.shape[1]:
                    ww = w1[dj + 5] * w1[di + 5]; a, b = xx[jj, ii], yy[jj, ii]
                    acc["m1"] += ww * a; acc["m2"] += ww * b; acc["e11"] += ww * a * a; acc["e22"] += ww * b * b; acc["e12"] += ww * a * b
        m1, m2 = acc["m1"], acc["m2"]; s1, s2, s12 = acc["e11"] - m1 * m1, acc["e22"] - m2 * m2, acc["e12"] - m1 * m2
        return (2 * m1 * m2 + 1e-4) * (2 * s12 + 9e-4) / ((m1 * m1 + m2 * m2 + 1e-4) * (s1 + s2 + 9e-4))
    assert abs(ssim_at(big[0], bigy[0], 20, 20) - s_int) < 1e-12
    # loss = mean over pixels and channels of 1 - SSIM, against the brute-force window sums (incl. border pixels)
    L, gr = oracle.ssim_loss(x, y, 0.2)
    brute = np.mean([[1 - ssim_at(x[c], y[c], j, i) for j in range(H) for i in range(W)] for c in range(3)])
    assert abs(L - 0.2 * brute) < 1e-12
    # gradient = central finite differences
    for c, j, i in [(0, 0, 0), (1, 8, 11), (2, 16, 22), (0, 5, 1), (1, 3, 19), (2, 10, 4)]:
        d = np.zeros_like(x); d[c, j, i] = 1e-6
        fd = (oracle.ssim_loss(x + d, y, 0.2)[0] - oracle.ssim_loss(x - d, y, 0.2)[0]) / 2e-6
        assert abs(fd - gr[c, j, i]) <= 1e-6 * abs(gr[c, j, i]) + 1e-11


# ---------------------------------------------------------------- P16: normalised depth D_n = D / O
def test_p16_normalised_depth_of_coplanar_splats_is_the_ray_plane_depth():
    """Five partly transparent splats on ONE tilted plane: whatever their weights, the expected depth of a pixel is
    the ray-plane intersection depth (closed form), while the plain Eq. 8 depth is O times it."""
    rot = Rotation.from_euler("xyz", [20, -30, 15], degrees=True)
    qx, qy, qz, qw = rot.as_quat()
    R = rot.as_matrix()
    mu0 = np.array([0.05, -0.02, 1.7])
    scs = []
    for k, (a, b, o) in enumerate([(0, 0, 0.3), (0.2, 0.1, 0.6), (-0.15, 0.2, 0.9), (0.1, -0.2, 0.45), (-0.2, -0.1, 0.75)]):
        scs.append(one_surfel(mu0 + a * R[:, 0] + b * R[:, 1], (0.12 + 0.02 * k, 0.1), (qw, qx, qy, qz), o))
    sc = cat(*scs)
    r = oracle.render_normalised(sc, oracle.make_cam(CAM), oracle.make_cfg())
    # the plane through the float32 centres with the float32 quaternion's normal (centres are coplanar up to 1e-7)
    q32 = sc.quat[0].astype(np.float64)
    n = Rotation.from_quat([q32[1], q32[2], q32[3], q32[0]]).as_matrix()[:, 2]
    X, Y = pix_grid(CAM)
    d = np.stack([(X - CAM.cx) / CAM.fx, (Y - CAM.cy) / CAM.fy, np.ones_like(X)], axis=-1)
    z = (n @ mu0) / (d @ n)
    O = r["img"][7]
    m = O > 0
    assert m.sum() > 300 and (r["n_comp"] >= 2).sum() > 50
    np.testing.assert_allclose(r["img"][3][m], z[m], rtol=1e-6)          # float32 rounding of the five centres
    np.testing.assert_allclose(r["img_raw"][3][m], O[m] * z[m], rtol=1e-6)
    assert np.abs(r["img_raw"][3][m] - z[m]).max() > 0.5                   # the un-normalised image is far from metric
    assert (r["img"][3][~m] == 0).all()
    for ch in (0, 1, 2, 4, 5, 6, 7):                                       # every other plane untouched
        assert (r["img"][ch] == r["img_raw"][ch]).all()


def test_p16_normalised_depth_two_layers_hand_value():
    """Two fronto-parallel splats at z1 < z2 on the optical axis: at the principal pixel G = 1 for both (centre pixel
    ray through both centres), so a1 = o1, a2 = o2 and D_n = (o1 z1 + o2 (1 - o1) z2) / (o1 + o2 (1 - o1))."""
    cam = Camera(9, 9, 20.0, 20.0, 4.5, 4.5)
    o1, o2, z1, z2 = 0.5, 0.25, 1.0, 3.0
    sc = cat(one_surfel((0, 0, z1), (0.2, 0.2), (1, 0, 0, 0), o1), one_surfel((0, 0, z2), (0.5, 0.5), (1, 0, 0, 0), o2))
    r = oracle.render_normalised(sc, oracle.make_cam(cam), oracle.make_cfg())
    want = (o1 * z1 + o2 * (1 - o1) * z2) / (o1 + o2 * (1 - o1))            # = 0.875 / 0.625 = 1.4
    assert abs(want - 1.4) < 1e-15
    assert abs(r["img"][3][4, 4] - 1.4) < 1e-12
    assert abs(r["img_raw"][3][4, 4] - 0.875) < 1e-12 and abs(r["img"][7][4, 4] - 0.625) < 1e-12


def test_p16_normalised_depth_gradients_are_finite_differences():
    """Surfel and SE(3) pose gradients of a loss on (rgb, D_n, normal, O) against central differences (smooth Eq. 8:
    O > 0 at every pixel, D_n smooth), and with the alpha clamp active."""
    _NORMALISED[0] = True
    try:
        _fd_check(oracle.smooth_cfg(), 2e-6)
        _fd_check(oracle.make_cfg(cutoff=np.inf, alpha_min=0.0, alpha_max=0.6, t_min=0.0, z_near=0.0), 2e-6)
    finally:
        _NORMALISED[0] = False


def test_p16_upstream_map_is_the_jacobian_transpose_of_the_division():
    """normalised_depth_upstream against a direct numerical Jacobian of (D, O) -> D / O at random pixels."""
    g = np.random.default_rng(5)
    img = g.uniform(0.2, 1.0, (8, 3, 4)); img[7, 0, 0] = 0.0; img[3, 0, 0] = 0.0
    up = g.normal(size=(8, 3, 4))
    got = oracle.normalised_depth_upstream(img, up)
    L = lambda im: float((oracle.normalise_depth(im) * up).sum())
    for ch in (3, 7):
        for (i, j) in [(1, 2), (2, 3), (0, 1)]:
            p, m_ = img.copy(), img.copy()
            p[ch, i, j] += 1e-6; m_[ch, i, j] -= 1e-6
            assert abs((L(p) - L(m_)) / 2e-6 - got[ch, i, j]) < 1e-7
    assert got[3, 0, 0] == 0.0 and got[7, 0, 0] == up[7, 0, 0]               # O = 0: only the opacity upstream survives
    for ch in (0, 1, 2, 4, 5, 6):
        assert (got[ch] == up[ch]).all()


# ---------------------------------------------------------------- P17: median depth (DESIGN R9m)
def test_p17_median_depth_hand_stacks():
    """Fronto-parallel splats on the optical axis, principal pixel (G = 1, a_i = o_i): T runs 1 -> 0.7 -> 0.35 for
    o = (0.3, 0.5, 0.9), so the median is the SECOND splat's depth; o = (0.6, ..) crosses at the first; o = (0.3, 0.2)
    never reaches 1/2 (T_final = 0.56) and gives 0.  Listed out of depth order on purpose."""
    cam = Camera(9, 9, 20.0, 20.0, 4.5, 4.5)
    camv, cfg = oracle.make_cam(cam), oracle.make_cfg()
    mk = lambda z, o: one_surfel((0, 0, z), (0.3, 0.3), (1, 0, 0, 0), o)
    med, _ = oracle.median_depth(cat(mk(3.0, 0.9), mk(1.0, 0.3), mk(2.0, 0.5)), camv, cfg)
    assert med[4, 4] == 2.0
    med, _ = oracle.median_depth(cat(mk(2.0, 0.5), mk(1.0, 0.6)), camv, cfg)
    assert med[4, 4] == 1.0
    med, _ = oracle.median_depth(cat(mk(2.0, 0.2), mk(1.0, 0.3)), camv, cfg)
    assert med[4, 4] == 0.0


def test_p17_median_depth_against_numpy_on_closed_form_footprints():
    """Six fronto-parallel splats at distinct depths: per pixel, the closed-form alphas (P1) in depth order, a
    cumulative product, and the first index with T <= 1/2 -- numpy against the oracle at every pixel that is not within
    1e-4 of the threshold; brute force and skipping traversal agree; a tilted plane's median is the ray-plane depth."""
    specs = [((0.10, -0.05, 1.5), 0.25, 0.20, 0.45), ((-0.20, 0.10, 2.0), 0.40, 0.30, 0.60), ((0.0, 0.0, 2.5), 0.50, 0.50, 0.35),
             ((0.15, 0.12, 1.2), 0.12, 0.15, 0.30), ((-0.1, -0.1, 3.0), 0.9, 0.9, 0.95), ((0.3, -0.2, 1.8), 0.2, 0.25, 0.80)]
    sc = cat(*[one_surfel(mu, (su, sv), (1, 0, 0, 0), o) for mu, su, sv, o in specs])
    camv, cfg = oracle.make_cam(CAM), oracle.make_cfg()
    med, mf = oracle.median_depth(sc, camv, cfg)
    order = np.argsort([s[0][2] for s in specs])
    T = np.ones((CAM.height, CAM.width)); want = np.zeros_like(T); near = np.zeros(T.shape, bool)
    for k in order:
        mu, su, sv, o = specs[k]
        a = _footprint_alpha(mu, float(np.float32(su)), float(np.float32(sv)), float(np.float32(o)))
        Tn = T * (1 - a)
        cross = (a > 0) & (T > 0.5) & (Tn <= 0.5)
        want[cross] = float(np.float32(mu[2]))
        near |= (a > 0) & (np.abs(Tn - 0.5) < 2e-4)
        T = Tn
    ok = ~near
    assert (mf.astype(bool) & ok).sum() == 0 and ok.mean() > 0.99
    assert (want[ok] > 0).sum() > 500 and len(np.unique(want[ok])) >= 4
    np.testing.assert_allclose(med[ok], want[ok], rtol=0, atol=1e-12)
    assert np.array_equal(med, oracle.median_depth(sc, camv, cfg, brute=True)[0])
    # one opaque tilted splat: the median is that splat's intersection depth = the ray-plane depth (P2's closed form)
    rot = Rotation.from_euler("xyz", [25, -35, 10], degrees=True)
    qx, qy, qz, qw = rot.as_quat()
    s1 = one_surfel((0.1, -0.05, 1.8), (0.3, 0.2), (qw, qx, qy, qz), 0.9)
    med1, _ = oracle.median_depth(s1, camv, cfg)
    r1 = oracle.render(s1, camv, cfg)
    q32 = s1.quat[0].astype(np.float64)
    nrm = Rotation.from_quat([q32[1], q32[2], q32[3], q32[0]]).as_matrix()[:, 2]
    X, Y = pix_grid(CAM)
    d = np.stack([(X - CAM.cx) / CAM.fx, (Y - CAM.cy) / CAM.fy, np.ones_like(X)], axis=-1)
    z = (nrm @ s1.mean[0].astype(np.float64)) / (d @ nrm)
    m = r1["img"][7] >= 0.5 + 1e-3
    assert m.sum() > 50
    np.testing.assert_allclose(med1[m], z[m], rtol=1e-12)
    assert (med1[r1["img"][7] < 0.5 - 1e-3] == 0).all()


# ---------------------------------------------------------------- P18: tight binning (readings R26, R27)
def test_p18_two_ln_upper_is_a_tight_upper_bound():
    """R26's logarithm from +, -, x, / alone: never below 2 ln r (conservative), never more than 3e-9 (rel + abs) above."""
    rs = np.concatenate([[1.0, 1.0 + 2.0 ** -40, 2.0, 4.0, 255.0, 255.0 * 0.1, 1e6], np.exp(np.linspace(0, 14, 400)),
                         255.0 * np.linspace(1 / 255, 1, 200), 2.0 ** np.arange(0, 20) * (1 - 2.0 ** -52)])
    rs = rs[rs >= 1.0]
    got = np.array([oracle.two_ln_upper(float(r)) for r in rs])
    ref = 2.0 * np.log(rs)
    assert (got >= ref).all()
    assert (got <= ref * (1 + 3e-9) + 3e-9).all()


def _tight_pair(sc, cam, T=None):
    camv = oracle.make_cam(cam, T)
    return camv, oracle.make_cfg(), oracle.make_cfg(tight=True)


def test_p18_tight_binning_leaves_the_rendered_function_unchanged(c1):
    """The variant only shortens the tile lists: images, transmittance, composited counts are bit-identical to the default
    binning in fp64 (brute force and skipping mode) and the gradients agree to the order of the fp64 sums."""
    sc, cam, camv, cfg, r = c1
    _, _, cfgt = _tight_pair(sc, cam)
    for brute in (False, True):
        rt = oracle.render(sc, camv, cfgt, brute=brute)
        assert np.array_equal(rt["img"], r["img"]) and np.array_equal(rt["T_final"], r["T_final"])
        assert np.array_equal(rt["n_comp"], r["n_comp"])
    assert oracle.render(sc, camv, cfgt)["counters"]["Q_t"] < 0.9 * r["counters"]["Q_t"]      # ... but fewer pairs are tested
    up = scenegen.upstream_normal(1, cam.height, cam.width)
    g, gt = oracle.backward(sc, camv, cfg, up), oracle.backward(sc, camv, cfgt, up)
    for k in ("mean", "scale", "quat", "opacity", "rgb", "pose"):
        np.testing.assert_allclose(gt[k], g[k], rtol=1e-10, atol=1e-9)


def test_p18_tight_lists_are_conservative_and_shorter(c1):
    """Every pair that can be composited -- rho^2 <= min(c^2, 2 ln(o / alpha_min)) with (u, v) from a LIBRARY matrix inverse
    and numpy's log -- lies in its pixel's tile list; the list is a subset of the default one; counts add up."""
    sc, cam, camv, cfg, r = c1
    cam2 = Camera(200, 120, 150.0, 150.0, 97.0, 63.0, scenegen.perturb_pose(np.eye(4)[:3], [0.05, -0.02, 0.1, 0.03, 0.05, -0.2]))
    for cm in (cam, cam2):
        cv, cfg0, cfgt = _tight_pair(sc, cm)
        b0, bt = oracle.binning(sc, cv, cfg0), oracle.binning(sc, cv, cfgt)
        assert bt["E"] == int(bt["count"].sum()) == len(bt["keys"]) and bt["E"] < 0.9 * b0["E"]
        assert (np.diff(bt["keys"].astype(np.uint64)) >= 0).all()
        assert set(zip(bt["keys"].tolist(), bt["idx"].tolist())) <= set(zip(b0["keys"].tolist(), b0["idx"].tolist()))
        assert ((bt["culled"] == 0) <= (b0["culled"] == 0)).all()
        X, Y = pix_grid(cm)
        tid = (np.arange(cm.height)[:, None] // 16) * bt["tiles_x"] + (np.arange(cm.width)[None, :] // 16)
        members = [set(bt["idx"][s:e].tolist()) for s, e in bt["ranges"]]
        amin = cfg0[2]
        n_pairs = 0
        for k in np.nonzero(b0["culled"] == 0)[0]:
            u, v = _numpy_uv(b0["M"][k].reshape(3, 3), X, Y)
            c2k = min(9.0, 2.0 * np.log(float(sc.opacity[k]) / amin))
            cover = (u * u + v * v <= c2k)
            n_pairs += int(cover.sum())
            for t in np.unique(tid[cover]):
                assert k in members[t], (k, t)
        assert n_pairs > 2000


def test_p18_lone_splat_lists_exactly_the_tiles_its_support_reaches():
    """A large faint splat (o = 0.1: support rho^2 <= 2 ln(25.5) = 6.48 < 9), tilted: the tight list is the set of tiles
    whose pixel-centre rectangle the support ellipse reaches, found here by dense sampling of rho^2 (0.1 px grid, library
    inverse) -- a tile the sampling finds must be listed; a listed tile the sampling misses must be a corner graze."""
    rot = Rotation.from_euler("xyz", [40, -30, 20], degrees=True)
    qx, qy, qz, qw = rot.as_quat()
    cam = Camera(160, 112, 140.0, 140.0, 80.0, 56.0)
    sc = one_surfel((0.05, -0.02, 1.6), (0.22, 0.12), (qw, qx, qy, qz), 0.1)
    camv, cfg0, cfgt = _tight_pair(sc, cam)
    b0, bt = oracle.binning(sc, camv, cfg0), oracle.binning(sc, camv, cfgt)
    assert bt["E"] < b0["E"] and bt["E"] > 8
    listed = set((bt["keys"] >> np.uint64(32)).astype(int).tolist())
    M = b0["M"][0].reshape(3, 3)
    c2k = oracle.two_ln_upper(float(np.float32(0.1)) / cfg0[2])
    assert abs(c2k - 2 * np.log(25.5)) < 1e-6
    hit, near = set(), set()
    for ty in range(bt["tiles_y"]):
        for tx in range(bt["tiles_x"]):
            xs = np.linspace(16 * tx + 0.5, min(16 * tx + 15.5, cam.width - 0.5), 151)
            ys = np.linspace(16 * ty + 0.5, min(16 * ty + 15.5, cam.height - 0.5), 151)
            Xs, Ys = np.meshgrid(xs, ys)
            u, v = _numpy_uv(M, Xs, Ys)
            m = (u * u + v * v).min()
            if m <= c2k:
                hit.add(ty * bt["tiles_x"] + tx)
            if m <= c2k * 1.02:
                near.add(ty * bt["tiles_x"] + tx)
    assert hit <= listed <= near, (sorted(listed - hit), sorted(hit - listed))
    assert len(hit) >= 10
    # o < alpha_min: the splat has no support at all and is culled
    faint = one_surfel((0.05, -0.02, 1.6), (0.22, 0.12), (qw, qx, qy, qz), 0.003)
    assert oracle.binning(faint, camv, cfgt)["culled"][0] == 1 and oracle.binning(faint, camv, cfg0)["culled"][0] == 0
    assert oracle.render(faint, camv, cfg0)["img"].max() == 0.0


# ---------------------------------------------------------------- P19: screen-space low-pass filter (reading R28)
def test_p19_lowpass_closed_forms():
    """R28: rho^2 = min(u^2 + v^2, 2 |x - x_c|^2).  (i) A splat far smaller than a pixel, centred between pixel centres,
    renders nothing without the filter and the closed form o exp(-|x - x_c|^2) (depth plane: that times the centre depth)
    with it.  (ii) A splat several pixels wide is untouched: its own Gaussian is the larger one everywhere (sigma_px^2 > 1/2),
    images bit-identical.  (iii) An edge-on splat (its plane contains the viewing ray) is invisible without the filter and
    a blob at its centre depth with it."""
    cfg0, cfgf = oracle.make_cfg(), oracle.make_cfg(lowpass=True)
    camv = oracle.make_cam(CAM)
    X, Y = pix_grid(CAM)
    z0 = 2.0
    xc, yc = 30.3, 20.8                                  # projected centre, between pixel centres
    mu = ((xc - CAM.cx) / CAM.fx * z0, (yc - CAM.cy) / CAM.fy * z0, z0)
    tiny = one_surfel(mu, (1e-4, 1e-4), (1, 0, 0, 0), 0.9)
    assert oracle.render(tiny, camv, cfg0)["img"].max() == 0.0
    r = oracle.render(tiny, camv, cfgf)
    mu32 = np.float32(mu).astype(np.float64)
    xc32, yc32 = CAM.fx * mu32[0] / mu32[2] + CAM.cx, CAM.fy * mu32[1] / mu32[2] + CAM.cy
    d2 = (X - xc32) ** 2 + (Y - yc32) ** 2
    a = float(np.float32(0.9)) * np.exp(-d2)
    a[(2 * d2 > 9.0) | (a < float(np.float32(1 / 255)))] = 0.0
    assert (a > 0).sum() >= 9
    np.testing.assert_allclose(r["img"][7], a, atol=1e-12)
    np.testing.assert_allclose(r["img"][3], a * mu32[2], atol=1e-12)
    b = oracle.binning(tiny, camv, cfgf)
    np.testing.assert_allclose(b["aabb"][0], [xc32 - 3 / np.sqrt(2), xc32 + 3 / np.sqrt(2), yc32 - 3 / np.sqrt(2), yc32 + 3 / np.sqrt(2)], atol=1e-9)
    big = one_surfel((0.31, -0.17, 1.5), (0.11, 0.07), (1, 0, 0, 0), 0.8)       # sigma_px = 60 * 0.07 / 1.5 = 2.8 px
    assert np.array_equal(oracle.render(big, camv, cfg0)["img"], oracle.render(big, camv, cfgf)["img"])
    # edge-on: the splat's plane contains the ray through its centre (normal t_n = x axis, centre on the optical axis)
    rot = Rotation.from_euler("y", 90, degrees=True)
    qx, qy, qz, qw = rot.as_quat()
    edge = one_surfel((0.0, 0.0, 1.5), (0.1, 0.1), (qw, qx, qy, qz), 0.9)
    r0, rf = oracle.render(edge, camv, cfg0), oracle.render(edge, camv, cfgf)
    col = int(CAM.cx)                                                              # the pixel columns next to the axis
    assert r0["img"][7][:, col - 3:col + 3].max() < 0.9 * rf["img"][7][:, col - 3:col + 3].max()
    m = rf["img"][7] > 0.2
    assert m.sum() >= 4
    np.testing.assert_allclose(rf["img"][3][m] / rf["img"][7][m], 1.5, rtol=0.05)   # depth ~ the centre's (exactly where the screen term wins)


def _filter_scene():
    """_tiny's six splats plus a sub-pixel one, a one-pixel one and a nearly edge-on one: pairs of both kinds exist."""
    sc, cam = _tiny()
    extra_mu = np.float32([[0.05, 0.03, 1.0], [-0.1, -0.05, 1.2], [0.12, -0.08, 0.9]])
    extra_s = np.float32([[2e-3, 2e-3], [0.03, 0.04], [0.15, 0.12]])
    rot = Rotation.from_euler("xyz", [5, 86, 10], degrees=True).as_quat()
    extra_q = np.float32([[1, 0.1, 0.05, 0.02], [0.9, -0.2, 0.1, 0.3], [rot[3], rot[0], rot[1], rot[2]]])
    cat2 = lambda a, b: np.concatenate([a, b])
    sc2 = Scene(cat2(sc.mean, extra_mu), cat2(sc.scale, extra_s), cat2(sc.quat, extra_q), cat2(sc.opacity, np.float32([0.8, 0.7, 0.9])),
                cat2(sc.rgb, np.float32([[0.9, 0.1, 0.2], [0.2, 0.8, 0.3], [0.3, 0.3, 0.9]])))
    return sc2, cam


def test_p19_lowpass_gradients_are_finite_differences():
    """Every surfel gradient and the SE(3) pose gradient with the filter on: plain Eq. 8 + filter, and the default
    truncation rules + filter.  The min() of R28 is a kink like the other decisions: no pixel may sit on it (fragile
    mask empty) and the guard of _fd_check watches the composited counts."""
    sc, cam = _filter_scene()
    camv = oracle.make_cam(cam, widen_from_f32=False)
    for cfg, guard in ((oracle.smooth_cfg(lowpass=True), False), (oracle.make_cfg(lowpass=True), True)):
        r = oracle.render(sc, camv, cfg)
        plain = oracle.render(sc, camv, oracle.smooth_cfg() if not guard else oracle.make_cfg())
        assert (r["fragile"] & 1).sum() == 0, "a pixel sits on a decision: move a splat"
        assert np.abs(r["img"] - plain["img"]).max() > 1e-3          # the screen term does win somewhere
        _fd_check(cfg, 1e-5, scene=(sc, cam), guard=guard, hexp=-19)


def test_p19_lowpass_lists_are_conservative(c1):
    """Every pair with min(rho_3d^2, rho_2d^2) <= c^2 (library inverse; 2 |x - x_c|^2 from M) is in its pixel's tile list."""
    sc, cam, camv, cfg, r = c1
    small = Scene(sc.mean, (sc.scale * np.float32(0.05)), sc.quat, sc.opacity, sc.rgb)    # 0.5 - 2.5 mm: mostly sub-pixel
    cfgf = oracle.make_cfg(lowpass=True)
    b = oracle.binning(small, camv, cfgf)
    X, Y = pix_grid(cam)
    tid = (np.arange(cam.height)[:, None] // 16) * b["tiles_x"] + (np.arange(cam.width)[None, :] // 16)
    members = [set(b["idx"][s:e].tolist()) for s, e in b["ranges"]]
    n2d = 0
    for k in np.nonzero(b["culled"] == 0)[0]:
        M = b["M"][k].reshape(3, 3)
        u, v = _numpy_uv(M, X, Y)
        r2 = 2 * ((X - M[0, 2] / M[2, 2]) ** 2 + (Y - M[1, 2] / M[2, 2]) ** 2)
        cover = np.minimum(u * u + v * v, r2) <= 9.0
        n2d += int((cover & (r2 < u * u + v * v)).sum())
        for t in np.unique(tid[cover]):
            assert k in members[t]
    assert n2d > 1000
    rf, r0 = oracle.render(small, camv, cfgf), oracle.render(small, camv, oracle.make_cfg())
    assert rf["img"][7].sum() > 3 * r0["img"][7].sum()                # the filter is what makes these splats visible
