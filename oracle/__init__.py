"""CPU oracle of the 2DGS surfel renderer (fp64, written from PAPER.md).  TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It never imports the CUDA path (paper_2506_00970_b200) and shares no code
with it.  The arithmetic lives in oracle/sgs_oracle.c (plain C, OpenMP over pixel rows); this file
only marshals numpy arrays through ctypes.

Parity unpinned: absolute image values on the paper's datasets (the paper prints none; the
datasets are not available).  Everything else is pinned by tests/test_oracle_pins.py (P1-P10).
"""
import ctypes
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sgs_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None

C_F32 = ctypes.POINTER(ctypes.c_float)
C_F64 = ctypes.POINTER(ctypes.c_double)
C_U8 = ctypes.POINTER(ctypes.c_uint8)
C_U32 = ctypes.POINTER(ctypes.c_uint32)
C_I32 = ctypes.POINTER(ctypes.c_int32)
C_U64 = ctypes.POINTER(ctypes.c_uint64)
C_I64 = ctypes.POINTER(ctypes.c_int64)


def build(force=False):
    """gcc -O2 -fopenmp -ffp-contract=off (no FMA contraction: the binning stage is a bit-exact
    contract).  Building the checker is not using it."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.orc_preprocess.restype = ctypes.c_int64
        _lib.orc_num_threads.restype = ctypes.c_int
    return _lib


def _p(a, t):
    return None if a is None else a.ctypes.data_as(t)


def make_cfg(tile=16, cutoff=3.0, alpha_min=1.0 / 255.0, alpha_max=0.99, t_min=1e-4, z_near=0.2, tight=False, lowpass=False):
    """Truncation constants (readings R3-R7).  Values pass through float32 first because the C-ABI
    config struct holds floats: both sides then use the identical real numbers.  tight: the binning variant of
    readings R26 + R27 (opacity-aware cutoff, tile-exact culling) -- the rendered function is the
    same, the tile lists are shorter.  lowpass: the compositing variant of reading R28 (screen-space low-pass filter:
    rho^2 = min(u^2 + v^2, 2 |x - x_c|^2), centre depth where the screen term wins)."""
    f = lambda v: float(np.float32(v))
    return np.array([tile, f(cutoff), f(alpha_min), f(alpha_max), f(t_min), f(z_near), 1.0 if tight else 0.0,
                     1.0 if lowpass else 0.0], dtype=np.float64)


def smooth_cfg(tile=16, lowpass=False):
    """Plain Eq. 8: no cutoff, no alpha bounds, no stop, no near plane (used for finite differences)."""
    return np.array([tile, np.inf, 0.0, 1.0, 0.0, 0.0, 0.0, 1.0 if lowpass else 0.0], dtype=np.float64)


def make_cam(cam, T_cw=None, widen_from_f32=True):
    """Camera vector [W,H,fx,fy,cx,cy,T_cw(12)].  By default intrinsics and pose are rounded to
    float32 first (what the C-ABI carries); pass widen_from_f32=False for fp64 finite differences."""
    T = np.asarray(cam.T_cw if T_cw is None else T_cw, dtype=np.float64)[:3].reshape(12)
    k = np.array([cam.fx, cam.fy, cam.cx, cam.cy], dtype=np.float64)
    if widen_from_f32:
        T = T.astype(np.float32).astype(np.float64)
        k = k.astype(np.float32).astype(np.float64)
    return np.concatenate([[cam.width, cam.height], k, T]).astype(np.float64)


def _scene_arrays(sc):
    f = lambda a: np.ascontiguousarray(a, dtype=np.float32)
    act = None if sc.active is None else np.ascontiguousarray(sc.active, dtype=np.uint8)
    return f(sc.mean), f(sc.scale), f(sc.quat), f(sc.opacity), f(sc.rgb), act


def two_ln_upper(r):
    """The upper bound of 2 ln r the tight binning uses for the opacity-aware cutoff (reading R26)."""
    f = lib().orc_two_ln_upper
    f.restype = ctypes.c_double
    return float(f(ctypes.c_double(r)))


def preprocess(sc, camv, cfgv):
    mean, scale, quat, opac, _, act = _scene_arrays(sc)
    n = mean.shape[0]
    out = dict(culled=np.zeros(n, np.uint8), depth_bits=np.zeros(n, np.uint32), rect=np.zeros((n, 4), np.int32),
               count=np.zeros(n, np.uint32), M=np.zeros((n, 9)), aabb=np.zeros((n, 4)))
    E = lib().orc_preprocess(ctypes.c_int64(n), _p(mean, C_F32), _p(scale, C_F32), _p(quat, C_F32), _p(opac, C_F32), _p(act, C_U8),
                             _p(camv, C_F64), _p(cfgv, C_F64), _p(out["culled"], C_U8), _p(out["depth_bits"], C_U32),
                             _p(out["rect"], C_I32), _p(out["count"], C_U32), _p(out["M"], C_F64), _p(out["aabb"], C_F64))
    out["E"] = int(E)
    return out


def binning(sc, camv, cfgv):
    """Stage O2: culled flags, sorted (key, idx) list and per-tile ranges -- the bit-exact contract."""
    pre = preprocess(sc, camv, cfgv)
    W, H, tile = int(camv[0]), int(camv[1]), int(cfgv[0])
    tx, ty = (W + tile - 1) // tile, (H + tile - 1) // tile
    E = pre["E"]
    keys = np.zeros(max(E, 1), np.uint64)
    idx = np.zeros(max(E, 1), np.uint32)
    ranges = np.zeros((tx * ty, 2), np.uint32)
    mean, scale, quat, opac, _, act = _scene_arrays(sc)
    lib().orc_bin(ctypes.c_int64(sc.n), _p(mean, C_F32), _p(scale, C_F32), _p(quat, C_F32), _p(opac, C_F32), _p(act, C_U8),
                  _p(camv, C_F64), _p(cfgv, C_F64), ctypes.c_int64(E), _p(keys, C_U64), _p(idx, C_U32), _p(ranges, C_U32))
    pre.update(keys=keys[:E], idx=idx[:E], ranges=ranges, tiles_x=tx, tiles_y=ty)
    return pre


def render(sc, camv, cfgv, brute=False, counters=True):
    """Forward (O3-O4).  Returns dict: img (8,H,W) f64 [rgb, depth, normal, alpha], T_final, n_comp,
    fragile (bit0: image-affecting decision within 1e-4; bit1: alpha_max clamp within 1e-4;
    bit2: a composited pair whose intersection has condition number > 32, i.e. tilt > 88.2 deg), counters."""
    mean, scale, quat, opac, rgb, act = _scene_arrays(sc)
    W, H = int(camv[0]), int(camv[1])
    img = np.zeros((8, H, W)); T = np.zeros((H, W)); nc = np.zeros((H, W), np.int32)
    frag = np.zeros((H, W), np.uint8); cnt = np.zeros(6, np.int64); qtb = np.zeros((H, W), np.int32)
    lib().orc_render(ctypes.c_int64(sc.n), _p(mean, C_F32), _p(scale, C_F32), _p(quat, C_F32), _p(opac, C_F32),
                     _p(rgb, C_F32), _p(act, C_U8), _p(camv, C_F64), _p(cfgv, C_F64), ctypes.c_int(int(brute)),
                     _p(img, C_F64), _p(T, C_F64), _p(nc, C_I32), _p(frag, C_U8), _p(cnt if counters else None, C_I64),
                     _p(qtb if counters else None, C_I32))
    return dict(img=img, T_final=T, n_comp=nc, fragile=frag, qtb_pix=qtb,
                counters=dict(Q_t=int(cnt[0]), Q_c=int(cnt[1]), cover=int(cnt[2]), n_vis=int(cnt[3]), n_fragile=int(cnt[4]), Q_tb=int(cnt[5])))


def contribution(sc, camv, cfgv, brute=False):
    """Eq. 20-21 (L208-214): C_k^V = sum_p w_k(p), the sum of splat k's blending coefficients over the pixels of
    the view (fp64, (n,)); zero for inactive, culled or never-composited splats."""
    mean, scale, quat, opac, rgb, act = _scene_arrays(sc)
    W, H = int(camv[0]), int(camv[1])
    img = np.zeros((8, H, W))
    contrib = np.zeros(sc.n)
    lib().orc_render_ex(ctypes.c_int64(sc.n), _p(mean, C_F32), _p(scale, C_F32), _p(quat, C_F32), _p(opac, C_F32),
                        _p(rgb, C_F32), _p(act, C_U8), _p(camv, C_F64), _p(cfgv, C_F64), ctypes.c_int(int(brute)),
                        _p(img, C_F64), None, None, None, None, None, _p(contrib, C_F64))
    return contrib


def median_depth(sc, camv, cfgv, brute=False):
    """Median depth image (DESIGN R9m): the intersection depth of the composited splat at which the pixel's transmittance
    first falls to <= 1/2; 0 where T_final > 1/2.  Returns (median (H,W) f64, fragile (H,W) u8: a composited splat left T
    within 1e-4 of 1/2)."""
    mean, scale, quat, opac, rgb, act = _scene_arrays(sc)
    W, H = int(camv[0]), int(camv[1])
    img = np.zeros((8, H, W)); med = np.zeros((H, W)); mf = np.zeros((H, W), np.uint8)
    lib().orc_render_ex2(ctypes.c_int64(sc.n), _p(mean, C_F32), _p(scale, C_F32), _p(quat, C_F32), _p(opac, C_F32),
                         _p(rgb, C_F32), _p(act, C_U8), _p(camv, C_F64), _p(cfgv, C_F64), ctypes.c_int(int(brute)),
                         _p(img, C_F64), None, None, None, None, None, None, _p(med, C_F64), _p(mf, C_U8))
    return med, mf


def covisibility(contrib_a, contrib_b, active=None, threshold=0.5):
    """Eq. 22 (L216-221): |G_A n G_B| / |G_A u G_B| with G_V = {k in M_A : C_k^V > 0.5}.  Returns
    (score, n_intersection, n_union); the score of two empty sets is 0."""
    a = np.asarray(contrib_a) > threshold
    b = np.asarray(contrib_b) > threshold
    if active is not None:
        m = np.asarray(active).astype(bool)
        a, b = a & m, b & m
    inter, union = int((a & b).sum()), int((a | b).sum())
    return (inter / union if union else 0.0), inter, union


def backward(sc, camv, cfgv, upstream, brute=False, debug=False):
    """Analytic backward (O5-O7).  upstream: (8,H,W).  Returns fp64 grads for mean, scale, quat,
    opacity, rgb, and pose (6,) = (rho, theta) under T <- Exp(tau) o T_cw (Eq. 11-13)."""
    mean, scale, quat, opac, rgb, act = _scene_arrays(sc)
    n = sc.n
    up = np.ascontiguousarray(upstream, dtype=np.float64)
    g = dict(mean=np.zeros((n, 3)), scale=np.zeros((n, 2)), quat=np.zeros((n, 4)), opacity=np.zeros(n),
             rgb=np.zeros((n, 3)), pose=np.zeros(6), surfel_fragile=np.zeros(n, np.uint8))
    dM = np.zeros((n, 9)) if debug else None
    dnc = np.zeros((n, 3)) if debug else None
    lib().orc_backward(ctypes.c_int64(n), _p(mean, C_F32), _p(scale, C_F32), _p(quat, C_F32), _p(opac, C_F32),
                       _p(rgb, C_F32), _p(act, C_U8), _p(camv, C_F64), _p(cfgv, C_F64), ctypes.c_int(int(brute)),
                       _p(up, C_F64), _p(g["mean"], C_F64), _p(g["scale"], C_F64), _p(g["quat"], C_F64),
                       _p(g["opacity"], C_F64), _p(g["rgb"], C_F64), _p(g["pose"], C_F64), _p(dM, C_F64), _p(dnc, C_F64),
                       _p(g["surfel_fragile"], C_U8))
    if debug:
        g["dM"] = dM; g["dnc"] = dnc
    return g


def pixel_bounds(sc, camv, cfgv):
    """Comparison support (not part of the rendered function): per-pixel bounds for pixels where a binary32 renderer may
    legitimately differ from this oracle -- see orc_pixel_bounds in sgs_oracle.c.  Returns dict of (H,W) fp64 arrays:
    flip_w (blending weight at stake in the pixel's fragile decisions), kerr / kerr_z (first-order sensitivity of the
    blend / of the depth values to the relative rounding of the intersection's inputs), zmax."""
    mean, scale, quat, opac, rgb, act = _scene_arrays(sc)
    W, H = int(camv[0]), int(camv[1])
    out = {k: np.zeros((H, W)) for k in ("flip_w", "kerr", "kerr_z", "zmax")}
    lib().orc_pixel_bounds(ctypes.c_int64(sc.n), _p(mean, C_F32), _p(scale, C_F32), _p(quat, C_F32), _p(opac, C_F32),
                           _p(rgb, C_F32), _p(act, C_U8), _p(camv, C_F64), _p(cfgv, C_F64), _p(out["flip_w"], C_F64),
                           _p(out["kerr"], C_F64), _p(out["kerr_z"], C_F64), _p(out["zmax"], C_F64))
    return out


def exposure(sc, camv, cfgv, upstream, extra_mask=None, signed_all=False, round_eps=8.0 * 2.0 ** -23):
    """Comparison support: what a renderer that decides differently at the EXPOSED pixels (the oracle's fragile pixels,
    plus `extra_mask`) can change in every gradient element: sum over those pixels of |contribution with the pixel's
    fragile decisions inverted - the oracle's contribution| + phi |contribution| (phi: rounding of ill-conditioned
    intersections, round_eps kappa (1 + rho^2)) + the whole |contribution| on `extra_mask` pixels (orc_exposure in
    sgs_oracle.c).  Returns dict: mean (n,3), scale (n,2), quat (n,4), opacity (n,), rgb (n,3), pose (6,), pix_exposed
    (H,W) u8.  signed_all=True: signed contributions of the oracle's own list over all pixels instead, i.e. backward()
    recomputed pair by pair (the self-check of this function)."""
    mean, scale, quat, opac, rgb, act = _scene_arrays(sc)
    n = sc.n
    W, H = int(camv[0]), int(camv[1])
    up = np.ascontiguousarray(upstream, dtype=np.float64)
    em = None if extra_mask is None else np.ascontiguousarray(extra_mask, dtype=np.uint8)
    ex = np.zeros((max(n, 1), 13)); pose = np.zeros(6); pe = np.zeros((H, W), np.uint8)
    lib().orc_exposure(ctypes.c_int64(n), _p(mean, C_F32), _p(scale, C_F32), _p(quat, C_F32), _p(opac, C_F32),
                       _p(rgb, C_F32), _p(act, C_U8), _p(camv, C_F64), _p(cfgv, C_F64), _p(up, C_F64), _p(em, C_U8),
                       ctypes.c_int(int(signed_all)), ctypes.c_double(round_eps), _p(ex, C_F64), _p(pose, C_F64), _p(pe, C_U8))
    ex = ex[:n]
    return dict(mean=ex[:, 0:3].copy(), scale=ex[:, 3:5].copy(), quat=ex[:, 5:9].copy(), opacity=ex[:, 9].copy(),
                rgb=ex[:, 10:13].copy(), pose=pose, pix_exposed=pe)


def normalise_depth(img):
    """Expected depth D_n = D / O (DESIGN R9n; D = sum w z and O = sum w are the depth and opacity
    images of Eq. 8): the blend weights renormalised to sum to one.  0 where O = 0 (no splat composited).
    img: (8,H,W) [rgb, depth, normal, alpha]; returns a copy with the depth plane replaced."""
    out = np.array(img, dtype=np.float64, copy=True)
    D, O = out[3], out[7]
    out[3] = np.divide(D, O, out=np.zeros_like(D), where=O > 0)
    return out


def normalised_depth_upstream(img_raw, upstream_n):
    """Chain rule of D_n = D / O: an upstream gradient on (.., D_n, .., O) becomes one on the raw images of Eq. 8,
    dL/dD = g_Dn / O and dL/dO = g_O - g_Dn D / O^2 (both contributions of g_Dn vanish where O = 0)."""
    up = np.array(upstream_n, dtype=np.float64, copy=True)
    D, O = img_raw[3], img_raw[7]
    m = O > 0
    gD = np.divide(up[3], O, out=np.zeros_like(D), where=m)
    up[7] = up[7] - np.where(m, gD * np.divide(D, O, out=np.zeros_like(D), where=m), 0.0)
    up[3] = gD
    return up


def render_normalised(sc, camv, cfgv, brute=False, counters=True):
    """render() with the depth plane normalised; the raw images of Eq. 8 stay under "img_raw"."""
    r = render(sc, camv, cfgv, brute=brute, counters=counters)
    r["img_raw"] = r["img"]
    r["img"] = normalise_depth(r["img"])
    return r


def backward_normalised(sc, camv, cfgv, upstream_n, brute=False):
    """backward() of a loss on the normalised-depth images: upstream_n[3] is dL/dD_n."""
    raw = render(sc, camv, cfgv, brute=brute, counters=False)["img"]
    return backward(sc, camv, cfgv, normalised_depth_upstream(raw, upstream_n), brute=brute)


def num_threads():
    return int(lib().orc_num_threads())


def _depth_residual(rendered_depth, target_depth):
    """D_r - D of Eq. 16 / Eq. 26 where the sensor depth D is valid, 0 elsewhere.  Reading R25: the paper's
    frames are RGB-D sensor frames (L350) whose depth has holes encoded as 0 (or non-finite values); Eq. 16, 19 and 26 do not
    spell a mask out, and a hole is no measurement, so a pixel with D <= 0 or non-finite D carries no depth term (neither
    loss nor gradient); its colour term stays."""
    D = np.asarray(target_depth, dtype=np.float64)
    valid = np.isfinite(D) & (D > 0)
    return np.where(valid, rendered_depth - np.where(valid, D, 0.0), 0.0)


def tracking_loss(img, target_rgb, target_depth, camv, lambda_d, normal_sign=1.0):
    """Eq. 15-19 (L180-204) written out in numpy, fp64.  img: (8,H,W) rendered planes; returns
    (L_t, upstream (8,H,W)).  M_n = [sign * N_r . r > 0] (Eq. 17; R19: the harness scenes use outward
    normals so sign = -1 there), M_o = [O > 0.95] (Eq. 18); the masks carry no gradient."""
    img = np.asarray(img, dtype=np.float64)
    W, H = int(camv[0]), int(camv[1])
    fx, fy, cx, cy = camv[2:6]
    X, Y = np.meshgrid(np.arange(W) + 0.5, np.arange(H) + 0.5)
    rx, ry = (X - cx) / fx, (Y - cy) / fy   # un-normalised ray: only the sign of N.r is used
    nr = img[4] * rx + img[5] * ry + img[6]
    m = ((normal_sign * nr > 0) & (img[7] > float(np.float32(0.95)))).astype(np.float64)
    dI = img[0:3] - np.asarray(target_rgb, dtype=np.float64)
    dD = _depth_residual(img[3], target_depth)
    LI = np.abs(dI).sum(0)                   # Eq. 15: element-wise L1 over the colour channels
    LD = np.abs(dD)                          # Eq. 16
    L = (m * (LI + lambda_d * LD)).sum() / (W * H)     # Eq. 19
    up = np.zeros_like(img)
    up[0:3] = m * np.sign(dI) / (W * H)
    up[3] = m * lambda_d * np.sign(dD) / (W * H)
    return float(L), up


def normal_from_depth(depth, camv):
    """Eq. 23 (L226-228): N_D = (grad_x D x grad_y D) / |.|, "the cross product of neighbouring pixel differences in
    D" -- reading R23: the differences are those of the back-projected points
    P(x,y) = D(x,y) ((x+0.5-cx)/fx, (y+0.5-cy)/fy, 1), central: grad_x P = P(x+1,y) - P(x-1,y), grad_y P = P(x,y+1) -
    P(x,y-1).  Defined on interior pixels with a non-zero cross product; N_D = 0 elsewhere.  Returns (3,H,W) fp64."""
    D = np.asarray(depth, dtype=np.float64)
    W, H = int(camv[0]), int(camv[1])
    fx, fy, cx, cy = camv[2:6]
    X, Y = np.meshgrid(np.arange(W) + 0.5, np.arange(H) + 0.5)
    P = np.stack([D * (X - cx) / fx, D * (Y - cy) / fy, D], 0)
    N = np.zeros((3, H, W))
    a = P[:, 1:-1, 2:] - P[:, 1:-1, :-2]
    b = P[:, 2:, 1:-1] - P[:, :-2, 1:-1]
    c = np.cross(a, b, axis=0)
    nrm = np.sqrt((c * c).sum(0))
    ok = nrm > 0
    N[:, 1:-1, 1:-1] = np.where(ok, c / np.where(ok, nrm, 1.0), 0.0)
    return N


def mapping_loss(img, target_rgb, target_depth, camv, lambda_c, w_d, w_n, normal_sign=1.0):
    """Mapping loss of Eq. 24-26 (L232-248) WITHOUT the SSIM term (stated in DESIGN.md):
        L = 1/|Omega| sum_p [ lambda_c |I_r - I|_1 + w_d |D_r - D| + w_n (1 - sign N_{D_r} . N_r) ]
    with N_{D_r} = normal_from_depth(D_r) (Eq. 23, 25).  Returns (L, upstream (8,H,W)): dL/d(rgb, depth, normal, alpha)
    of the rendered planes, the depth gradient including the chain through N_{D_r}."""
    img = np.asarray(img, dtype=np.float64)
    W, H = int(camv[0]), int(camv[1])
    fx, fy, cx, cy = camv[2:6]
    HW = W * H
    dI = img[0:3] - np.asarray(target_rgb, dtype=np.float64)
    dD = _depth_residual(img[3], target_depth)
    ND = normal_from_depth(img[3], camv)
    Nr = img[4:7]
    Ln = 1.0 - normal_sign * (ND * Nr).sum(0)
    L = (lambda_c * np.abs(dI).sum(0) + w_d * np.abs(dD) + w_n * Ln).sum() / HW
    up = np.zeros_like(img)
    up[0:3] = lambda_c * np.sign(dI) / HW
    up[3] = w_d * np.sign(dD) / HW
    up[4:7] = -normal_sign * w_n * ND / HW
    # chain through N_D: f = N.m with N = c/|c|, c = a x b  =>  df/dc = (m - N (N.m))/|c|, df/da = b x df/dc,
    # df/db = df/dc x a; a, b are differences of P = D ray, so each interior pixel scatters to its four neighbours
    X, Y = np.meshgrid(np.arange(W) + 0.5, np.arange(H) + 0.5)
    ray = np.stack([(X - cx) / fx, (Y - cy) / fy, np.ones_like(X)], 0)
    P = img[3][None] * ray
    a = P[:, 1:-1, 2:] - P[:, 1:-1, :-2]
    b = P[:, 2:, 1:-1] - P[:, :-2, 1:-1]
    c = np.cross(a, b, axis=0)
    nrm = np.sqrt((c * c).sum(0))
    ok = nrm > 0
    inv = np.where(ok, 1.0 / np.where(ok, nrm, 1.0), 0.0)
    Nc = c * inv
    m = Nr[:, 1:-1, 1:-1]
    q = (m - Nc * (Nc * m).sum(0)) * inv
    coef = -normal_sign * w_n / HW
    dfa = np.cross(b, q, axis=0) * coef
    dfb = np.cross(q, a, axis=0) * coef
    gP = np.zeros((3, H, W))
    gP[:, 1:-1, 2:] += dfa
    gP[:, 1:-1, :-2] -= dfa
    gP[:, 2:, 1:-1] += dfb
    gP[:, :-2, 1:-1] -= dfb
    up[3] += (gP * ray).sum(0)
    return float(L), up


def quat_to_matrix(q):
    """R(q/|q|) for (n,4) quaternions (w,x,y,z), fp64 -- the unit-quaternion formula of Eq. 5-6's R."""
    q = np.asarray(q, dtype=np.float64)
    q = q / np.linalg.norm(q, axis=-1, keepdims=True)
    w, x, y, z = q[..., 0], q[..., 1], q[..., 2], q[..., 3]
    return np.stack([np.stack([1 - 2 * (y * y + z * z), 2 * (x * y - w * z), 2 * (x * z + w * y)], -1),
                     np.stack([2 * (x * y + w * z), 1 - 2 * (x * x + z * z), 2 * (y * z - w * x)], -1),
                     np.stack([2 * (x * z - w * y), 2 * (y * z + w * x), 1 - 2 * (x * x + y * y)], -1)], -2)


def map_correction(mean, quat, frame_id, T_orig, T_opt):
    """Map correction after pose-graph optimisation (Eq. 31-32): Delta T_i = T_i^o T_i^{-1} per keyframe;
    each splat moves with the increment of its closest observed keyframe f: mu' = Delta T_f mu, R' = Delta R_f R.
    T_orig, T_opt: (K,3,4) rigid transforms [R|t].  Returns (mu' (n,3), R' (n,3,3)) in fp64 -- the rotation as a MATRIX
    (a quaternion is unique only up to sign)."""
    To = np.asarray(T_orig, dtype=np.float64).reshape(-1, 3, 4)
    Tn = np.asarray(T_opt, dtype=np.float64).reshape(-1, 3, 4)
    K = To.shape[0]
    dT = np.zeros((K, 4, 4))
    for i in range(K):
        A = np.eye(4); A[:3] = To[i]
        B = np.eye(4); B[:3] = Tn[i]
        dT[i] = B @ np.linalg.inv(A)                 # Eq. 31
    f = np.asarray(frame_id).astype(np.int64)
    mu = np.asarray(mean, dtype=np.float64)
    mu2 = np.einsum("nij,nj->ni", dT[f, :3, :3], mu) + dT[f, :3, 3]      # Eq. 32
    R2 = np.einsum("nij,njk->nik", dT[f, :3, :3], quat_to_matrix(quat))
    return mu2, R2


def ssim_window(size=11, sigma=1.5):
    """The normalised Gaussian window of SSIM [87] (11 x 11, sigma 1.5), as a 1-D kernel; the 2-D window is its outer product."""
    x = np.arange(size, dtype=np.float64) - (size - 1) / 2.0
    g = np.exp(-x * x / (2.0 * sigma * sigma))
    return g / g.sum()


def ssim_loss(rgb_r, rgb_t, weight):
    """SSIM term of Eq. 24 (L236-238), reading R24: per channel the structural similarity index of [87]
    with the 11 x 11 Gaussian window (sigma 1.5), zero padding, C1 = 0.01^2, C2 = 0.03^2 (unit dynamic range);
    L_SSIM(p) = 1 - mean_c SSIM_c(p);  returns (weight/|Omega| sum_p L_SSIM(p), d/d rgb_r of that (3,H,W)), fp64."""
    from scipy.signal import convolve2d
    x = np.asarray(rgb_r, dtype=np.float64); y = np.asarray(rgb_t, dtype=np.float64)
    Cn, H, W = x.shape
    g = ssim_window()
    win = np.outer(g, g)
    conv = lambda a: convolve2d(a, win, mode="same", boundary="fill", fillvalue=0.0)
    C1, C2 = 0.01 ** 2, 0.03 ** 2
    L = 0.0
    grad = np.zeros_like(x)
    G = -weight / (Cn * H * W)          # dL/dSSIM_c(p)
    for c in range(Cn):
        mu1, mu2 = conv(x[c]), conv(y[c])
        e11, e22, e12 = conv(x[c] * x[c]), conv(y[c] * y[c]), conv(x[c] * y[c])
        s1, s2, s12 = e11 - mu1 * mu1, e22 - mu2 * mu2, e12 - mu1 * mu2
        a1, a2 = 2 * mu1 * mu2 + C1, 2 * s12 + C2
        b1, b2 = mu1 * mu1 + mu2 * mu2 + C1, s1 + s2 + C2
        S = a1 * a2 / (b1 * b2)
        L += weight * (1.0 - S).sum() / (Cn * H * W)
        dS_dmu1 = 2 * mu2 * (a2 - a1) / (b1 * b2) - S * (2 * mu1 / b1 - 2 * mu1 / b2)
        dS_de11 = -S / b2
        dS_de12 = 2 * a1 / (b1 * b2)
        grad[c] = conv(G * dS_dmu1) + 2 * x[c] * conv(G * dS_de11) + y[c] * conv(G * dS_de12)
    return float(L), grad
