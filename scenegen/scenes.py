"""Scene / camera generators for BASELINE.json's five configs.

Only generator math lives here (sampling on rectangles, quaternion composition to orient a
splat, look-at camera frames, an SE(3) exponential to perturb a pose).  Nothing here
projects, bins or blends."""
from dataclasses import dataclass, field
import json
import os
import numpy as np

from .rng import SplitMix

CONFIG_NAMES = ("C1", "C2", "C3", "C4", "C5")
_CALIB_PATH = os.path.join(os.path.dirname(__file__), "calibration.json")


@dataclass
class Scene:
    mean: np.ndarray      # (n,3) f32 world-space centres
    scale: np.ndarray     # (n,2) f32 activated scales s_u, s_v in metres
    quat: np.ndarray      # (n,4) f32 (w,x,y,z), not necessarily unit
    opacity: np.ndarray   # (n,)  f32 activated opacity in (0,1]
    rgb: np.ndarray       # (n,3) f32
    active: np.ndarray = None  # (n,) u8 or None (= all active)

    @property
    def n(self):
        return self.mean.shape[0]


@dataclass
class Camera:
    width: int
    height: int
    fx: float
    fy: float
    cx: float
    cy: float
    T_cw: np.ndarray = field(default_factory=lambda: np.eye(4)[:3].astype(np.float32))  # (3,4) f32


# ----------------------------------------------------------------------------- helpers
def _quat_mul(a, b):
    aw, ax, ay, az = a[..., 0], a[..., 1], a[..., 2], a[..., 3]
    bw, bx, by, bz = b[..., 0], b[..., 1], b[..., 2], b[..., 3]
    return np.stack([aw * bw - ax * bx - ay * by - az * bz,
                     aw * bx + ax * bw + ay * bz - az * by,
                     aw * by - ax * bz + ay * bw + az * bx,
                     aw * bz + ax * by - ay * bx + az * bw], axis=-1)


def _quat_axis_angle(axis, angle):
    axis = axis / np.linalg.norm(axis, axis=-1, keepdims=True)
    h = 0.5 * angle
    return np.concatenate([np.cos(h)[..., None], axis * np.sin(h)[..., None]], axis=-1)


def _quat_from_frame(ex, ey, ez):
    """Unit quaternion of the rotation whose columns are (ex, ey, ez); few frames only."""
    R = np.stack([ex, ey, ez], axis=-1)
    out = np.zeros(R.shape[:-2] + (4,))
    for i in np.ndindex(R.shape[:-2]):
        m = R[i]
        t = np.trace(m)
        if t > 0:
            s = np.sqrt(t + 1.0) * 2
            q = [0.25 * s, (m[2, 1] - m[1, 2]) / s, (m[0, 2] - m[2, 0]) / s, (m[1, 0] - m[0, 1]) / s]
        elif m[0, 0] > m[1, 1] and m[0, 0] > m[2, 2]:
            s = np.sqrt(1.0 + m[0, 0] - m[1, 1] - m[2, 2]) * 2
            q = [(m[2, 1] - m[1, 2]) / s, 0.25 * s, (m[0, 1] + m[1, 0]) / s, (m[0, 2] + m[2, 0]) / s]
        elif m[1, 1] > m[2, 2]:
            s = np.sqrt(1.0 + m[1, 1] - m[0, 0] - m[2, 2]) * 2
            q = [(m[0, 2] - m[2, 0]) / s, (m[0, 1] + m[1, 0]) / s, 0.25 * s, (m[1, 2] + m[2, 1]) / s]
        else:
            s = np.sqrt(1.0 + m[2, 2] - m[0, 0] - m[1, 1]) * 2
            q = [(m[1, 0] - m[0, 1]) / s, (m[0, 2] + m[2, 0]) / s, (m[1, 2] + m[2, 1]) / s, 0.25 * s]
        out[i] = q
    return out


def look_at(eye, target, up=(0.0, 0.0, 1.0)):
    """World->camera (3,4) f32: camera z forward, x right, y down (image convention)."""
    eye = np.asarray(eye, dtype=np.float64)
    fwd = np.asarray(target, dtype=np.float64) - eye
    fwd /= np.linalg.norm(fwd)
    right = np.cross(fwd, np.asarray(up, dtype=np.float64))
    right /= np.linalg.norm(right)
    down = np.cross(fwd, right)
    R = np.stack([right, down, fwd], axis=0)
    t = -R @ eye
    return np.concatenate([R, t[:, None]], axis=1).astype(np.float32)


def se3_exp(tau):
    """Exp: se(3) -> SE(3), tau = (rho, theta), translation block first (Eq. 12-13)."""
    tau = np.asarray(tau, dtype=np.float64)
    rho, th = tau[:3], tau[3:]
    a = np.linalg.norm(th)
    K = np.array([[0, -th[2], th[1]], [th[2], 0, -th[0]], [-th[1], th[0], 0]])
    if a < 1e-10:
        R = np.eye(3) + K + 0.5 * K @ K
        V = np.eye(3) + 0.5 * K + K @ K / 6.0
    else:
        R = np.eye(3) + np.sin(a) / a * K + (1 - np.cos(a)) / a**2 * K @ K
        V = np.eye(3) + (1 - np.cos(a)) / a**2 * K + (a - np.sin(a)) / a**3 * K @ K
    T = np.eye(4)
    T[:3, :3] = R
    T[:3, 3] = V @ rho
    return T


def perturb_pose(T_cw, tau):
    """Left perturbation Exp(tau) o T_cw, returned as (3,4) float64."""
    T = np.eye(4)
    T[:3] = np.asarray(T_cw, dtype=np.float64)
    return (se3_exp(tau) @ T)[:3]


def upstream_normal(seed, height, width, channels=8):
    """Seeded N(0,1) upstream gradients, channel-planar (8,H,W) f32:
    rgb(3), depth(1), normal(3), alpha(1)."""
    g = SplitMix(seed ^ 0x5EED).normal(channels * height * width, stream=0)
    return g.reshape(channels, height, width).astype(np.float32)


# ----------------------------------------------------------------------------- C1
def tiny_scene(seed=1, n=2000):
    """C1: means uniform in a 2 m cube, z in [1,3]; scales log-uniform 1-5 cm; q uniform on S^3;
    opacity U(0.1,0.99); rgb U[0,1]."""
    g = SplitMix(seed)
    mean = np.stack([g.uniform(n, -1.0, 1.0), g.uniform(n, -1.0, 1.0), g.uniform(n, 1.0, 3.0)], axis=1)
    ls = np.stack([g.uniform(n, np.log(0.01), np.log(0.05)), g.uniform(n, np.log(0.01), np.log(0.05))], axis=1)
    quat = np.stack([g.normal(n) for _ in range(4)], axis=1)
    quat /= np.linalg.norm(quat, axis=1, keepdims=True)
    opacity = g.uniform(n, 0.1, 0.99)
    rgb = np.stack([g.uniform(n) for _ in range(3)], axis=1)
    return Scene(mean.astype(np.float32), np.exp(ls).astype(np.float32), quat.astype(np.float32),
                 opacity.astype(np.float32), rgb.astype(np.float32))


def tiny_camera():
    return Camera(64, 48, 60.0, 60.0, 32.0, 24.0)


def stress_scene(seed=11, n=1600):
    """Splats chosen to strain the renderer's conservative culling and masking, not to look like a room (camera at the
    origin looking down +z, `stress_camera`): slivers (axis ratio up to 200:1), edge-on splats (normal within a few
    degrees of perpendicular to the view ray), sub-pixel splats, splats larger than the screen, opacities around the
    1/255 threshold, and splats close to the near plane.  Eight equal groups, parameters only (no method arithmetic)."""
    g = SplitMix(seed)
    k = n // 8
    n = 8 * k
    grp = np.repeat(np.arange(8), k)
    mean = np.stack([g.uniform(n, -1.2, 1.2), g.uniform(n, -1.0, 1.0), g.uniform(n, 1.0, 3.0)], axis=1)
    ls = np.stack([g.uniform(n, np.log(0.01), np.log(0.05)), g.uniform(n, np.log(0.01), np.log(0.05))], axis=1)
    quat = np.stack([g.normal(n) for _ in range(4)], axis=1)
    quat /= np.linalg.norm(quat, axis=1, keepdims=True)
    opacity = g.uniform(n, 0.1, 0.99)
    rgb = np.stack([g.uniform(n) for _ in range(3)], axis=1)
    m = grp == 0                                   # slivers: 5-40 cm by 0.2-2 mm
    ls[m, 0] = g.uniform(n, np.log(0.05), np.log(0.4))[m]; ls[m, 1] = g.uniform(n, np.log(0.0002), np.log(0.002))[m]
    m = grp == 1                                   # edge-on: t_u along the view ray to the centre, tilted by < 3 degrees
    ang = g.uniform(n, -0.05, 0.05); roll = g.uniform(n, 0.0, 2 * np.pi)
    for i in np.nonzero(m)[0]:
        ez0 = mean[i] / np.linalg.norm(mean[i])                      # view ray
        a = np.cross(ez0, [0.0, 1.0, 0.0]); a /= np.linalg.norm(a)
        b = np.cross(ez0, a)
        side = np.cos(roll[i]) * a + np.sin(roll[i]) * b             # in-plane axis perpendicular to the ray
        tn = np.cos(ang[i]) * np.cross(ez0, side) + np.sin(ang[i]) * ez0   # normal: almost perpendicular to the ray
        tn /= np.linalg.norm(tn)
        tu = np.cross(side, tn)
        quat[i] = _quat_from_frame(tu, side, tn)
    m = grp == 2                                   # sub-pixel: 0.1-2 mm
    ls[m] = np.stack([g.uniform(n, np.log(0.0001), np.log(0.002)), g.uniform(n, np.log(0.0001), np.log(0.002))], axis=1)[m]
    m = grp == 3                                   # larger than the screen: 1-3 m
    ls[m] = np.stack([g.uniform(n, np.log(1.0), np.log(3.0)), g.uniform(n, np.log(1.0), np.log(3.0))], axis=1)[m]
    opacity[m] = g.uniform(n, 0.02, 0.2)[m]
    m = grp == 4                                   # opacity around 1/255
    opacity[m] = g.uniform(n, 0.002, 0.02)[m]
    ls[m] = np.stack([g.uniform(n, np.log(0.03), np.log(0.2)), g.uniform(n, np.log(0.03), np.log(0.2))], axis=1)[m]
    m = grp == 5                                   # close to the near plane (z_near = 0.2)
    mean[m, 2] = g.uniform(n, 0.15, 0.45)[m]; mean[m, 0] *= 0.2; mean[m, 1] *= 0.2
    m = grp == 6                                   # far outside the frustum sideways, large enough to reach in
    mean[m, 0] = (np.sign(mean[m, 0]) + (mean[m, 0] == 0)) * g.uniform(n, 2.0, 6.0)[m]
    ls[m] = np.stack([g.uniform(n, np.log(0.3), np.log(2.0)), g.uniform(n, np.log(0.02), np.log(0.3))], axis=1)[m]
    # group 7: plain splats (the C1 recipe) as filler
    return Scene(mean.astype(np.float32), np.exp(ls).astype(np.float32), quat.astype(np.float32),
                 opacity.astype(np.float32), rgb.astype(np.float32))


def stress_camera():
    """104 x 72 (7 x 5 tiles, both edges ragged), f = 70 px."""
    return Camera(104, 72, 70.0, 70.0, 51.3, 36.7)


# ----------------------------------------------------------------------------- rooms
ROOM = np.array([5.0, 4.0, 3.0])


def _room_rects(g, n_patches, patch_lo, patch_hi):
    """Rectangles as (origin, edge_u, edge_v, normal). Six walls with inward normals, then
    n_patches random planar patches inside the room."""
    X, Y, Z = ROOM
    o, eu, ev, nn = [], [], [], []

    def add(org, u, v):
        u = np.asarray(u, float); v = np.asarray(v, float)
        nrm = np.cross(u, v)
        o.append(np.asarray(org, float)); eu.append(u); ev.append(v); nn.append(nrm / np.linalg.norm(nrm))

    add([0, 0, 0], [X, 0, 0], [0, Y, 0])      # floor, normal +z
    add([0, 0, Z], [0, Y, 0], [X, 0, 0])      # ceiling, normal -z
    add([0, 0, 0], [0, Y, 0], [0, 0, Z])      # x=0 wall, normal +x
    add([X, 0, 0], [0, 0, Z], [0, Y, 0])      # x=X wall, normal -x
    add([0, 0, 0], [0, 0, Z], [X, 0, 0])      # y=0 wall, normal +y
    add([0, Y, 0], [X, 0, 0], [0, 0, Z])      # y=Y wall, normal -y
    if n_patches > 0:
        c = np.stack([g.uniform(n_patches, 0.5, X - 0.5), g.uniform(n_patches, 0.5, Y - 0.5),
                      g.uniform(n_patches, 0.3, Z - 0.3)], axis=1)
        nv = np.stack([g.normal(n_patches) for _ in range(3)], axis=1)
        nv /= np.linalg.norm(nv, axis=1, keepdims=True)
        a = np.stack([g.normal(n_patches) for _ in range(3)], axis=1)
        a -= nv * np.sum(a * nv, axis=1, keepdims=True)
        a /= np.linalg.norm(a, axis=1, keepdims=True)
        b = np.cross(nv, a)
        wu = g.uniform(n_patches, patch_lo, patch_hi)
        wv = g.uniform(n_patches, patch_lo, patch_hi)
        for i in range(n_patches):
            add(c[i] - 0.5 * wu[i] * a[i] - 0.5 * wv[i] * b[i], wu[i] * a[i], wv[i] * b[i])
    return np.array(o), np.array(eu), np.array(ev), np.array(nn)


def _smooth_rgb(g, p):
    """Seeded smooth noise texture: per channel a sum of 4 sinusoids of position, mapped to [0,1]."""
    out = np.zeros((p.shape[0], 3))
    for ch in range(3):
        acc = np.zeros(p.shape[0])
        k = np.stack([g.uniform(4, -4.0, 4.0) for _ in range(3)], axis=1)   # (4,3) wave vectors
        ph = g.uniform(4, 0.0, 2 * np.pi)
        for j in range(4):
            acc += np.sin(p @ k[j] + ph[j])
        out[:, ch] = 0.5 + 0.125 * acc
    return out


def room_scene(seed, n, n_patches=20, patch_lo=0.5, patch_hi=1.5, scale_lo=0.005, scale_hi=0.03,
               scale_mult=1.0, patch_area_boost=1.0, active_frac=None):
    """C2-C5 style: n surfels area-uniform on 6 walls + random rectangles; normals follow the
    surface with U(0,5 deg) jitter about a random axis; tangents at a random in-plane angle;
    scales log-uniform; opacity U(0.5,1); colour from a smooth texture.
    patch_area_boost > 1 puts proportionally more surfels on the clutter patches (C4)."""
    g = SplitMix(seed)
    o, eu, ev, nn = _room_rects(g, n_patches, patch_lo, patch_hi)
    area = np.linalg.norm(np.cross(eu, ev), axis=1)
    area[6:] *= patch_area_boost
    cdf = np.cumsum(area) / np.sum(area)
    ridx = np.minimum(np.searchsorted(cdf, g.uniform(n), side="right"), len(cdf) - 1)
    a, b = g.uniform(n), g.uniform(n)
    mean = o[ridx] + a[:, None] * eu[ridx] + b[:, None] * ev[ridx]
    # orientation: surface frame (e_u, n x e_u, n), in-plane spin, then small jitter
    fu = eu / np.linalg.norm(eu, axis=1, keepdims=True)
    fv = np.cross(nn, fu)
    q_surf = _quat_from_frame(fu, fv, nn)[ridx]
    spin = _quat_axis_angle(np.tile([0.0, 0.0, 1.0], (n, 1)), g.uniform(n, 0.0, 2 * np.pi))
    jax = np.stack([g.normal(n) for _ in range(3)], axis=1)
    jit = _quat_axis_angle(jax, np.deg2rad(g.uniform(n, 0.0, 5.0)))
    quat = _quat_mul(jit, _quat_mul(q_surf, spin))
    ls = np.stack([g.uniform(n, np.log(scale_lo), np.log(scale_hi)),
                   g.uniform(n, np.log(scale_lo), np.log(scale_hi))], axis=1)
    scale = np.exp(ls) * scale_mult
    opacity = g.uniform(n, 0.5, 1.0)
    rgb = np.clip(_smooth_rgb(g, mean), 0.0, 1.0)
    active = None
    if active_frac is not None:
        active = (g.uniform(n) < active_frac).astype(np.uint8)
    return Scene(mean.astype(np.float32), scale.astype(np.float32), quat.astype(np.float32),
                 opacity.astype(np.float32), rgb.astype(np.float32), active)


def _room_camera(g, width, height, f):
    X, Y, Z = ROOM
    eye = np.array([g.uniform(1, 0.5, X - 0.5)[0], g.uniform(1, 0.5, Y - 0.5)[0], g.uniform(1, 0.5, Z - 0.5)[0]])
    # far-wall point: on the x-wall farther from the eye
    wx = X if eye[0] < X / 2 else 0.0
    tgt = np.array([wx, g.uniform(1, 0.5, Y - 0.5)[0], g.uniform(1, 0.5, Z - 0.5)[0]])
    return Camera(width, height, f, f, width / 2.0, height / 2.0, look_at(eye, tgt))


def _calibration():
    if os.path.exists(_CALIB_PATH):
        with open(_CALIB_PATH) as fh:
            return json.load(fh)
    return {}


def make_config(name, n_override=None):
    """Returns (scene, [cameras], info) for BASELINE.json config `name` in C1..C5.
    n_override shrinks the surfel count (same recipe) for quick tests."""
    cal = _calibration()
    if name == "C1":
        sc = tiny_scene(1, n_override or 2000)
        return sc, [tiny_camera()], {"mode": "full", "iters": 1}
    if name == "C2":
        sc = room_scene(2, n_override or 200_000)
        cam = _room_camera(SplitMix(1002), 640, 480, 525.0)
        return sc, [cam], {"mode": "pose", "iters": 100, "tau0_seed": 2002}
    if name == "C3":
        sc = room_scene(3, n_override or 500_000)
        cams = _path_cameras(SplitMix(1003), 8, 1200, 680, 600.0, circle=False)
        return sc, cams, {"mode": "full", "iters": 1}
    if name == "C4":
        c = cal.get("C4", {})
        sc = room_scene(4, n_override or 2_000_000, n_patches=c.get("n_patches", 400), patch_lo=0.2,
                        patch_hi=1.0, scale_mult=c.get("scale_mult", 1.0),
                        patch_area_boost=c.get("patch_area_boost", 4.0))
        cams = _path_cameras(SplitMix(1004), 16, 1200, 680, 600.0, circle=True)
        return sc, cams, {"mode": "full+pose", "iters": 1}
    if name == "C5":
        c = cal.get("C5", {})
        sc = room_scene(5, n_override or 5_000_000, scale_mult=c.get("scale_mult", 1.0), active_frac=0.2)
        cam = _room_camera(SplitMix(1005), 640, 480, 525.0)
        return sc, [cam], {"mode": "pose", "iters": 200, "tau0_seed": 2005}
    raise ValueError(name)


def _path_cameras(g, k, width, height, f, circle):
    X, Y, Z = ROOM
    cams = []
    if circle:
        ctr = np.array([X / 2, Y / 2, 1.5])
        for i in range(k):
            ang = 2 * np.pi * i / k
            eye = ctr + np.array([1.0 * np.cos(ang), 0.8 * np.sin(ang), 0.0])
            tgt = ctr + np.array([2.4 * np.cos(ang + 0.6), 1.9 * np.sin(ang + 0.6), -0.3])
            cams.append(Camera(width, height, f, f, width / 2.0, height / 2.0, look_at(eye, tgt)))
    else:
        start = np.array([1.0, g.uniform(1, 1.0, Y - 1.0)[0], g.uniform(1, 1.0, 2.0)[0]])
        tgt = np.array([X, g.uniform(1, 1.0, Y - 1.0)[0], g.uniform(1, 0.8, 2.2)[0]])
        for i in range(k):
            eye = start + np.array([0.0, 1.0, 0.0]) * (2.0 * i / (k - 1) - 1.0) * 0.0 + \
                np.array([2.0 * i / (k - 1), 0.0, 0.0])
            cams.append(Camera(width, height, f, f, width / 2.0, height / 2.0, look_at(eye, tgt)))
    return cams
