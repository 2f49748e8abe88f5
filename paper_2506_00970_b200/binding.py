"""Thin ctypes binding over libsgs.so (include/sgs.h).  Argument marshalling only: every step of
the path runs in the CUDA kernels behind the C ABI.  torch is used for device memory (the ctx's
workspace comes from torch's caching allocator through the sgs_alloc_fn callbacks) and streams.
There is NO CPU fallback: a missing library or device raises."""
import atexit
import ctypes as C
import os
import weakref
import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libsgs.so")

SGS_OK, SGS_INVALID_ARGUMENT, SGS_OUT_OF_MEMORY, SGS_WORKSPACE_OVERFLOW, SGS_NO_FORWARD_STATE, SGS_CUDA_ERROR, SGS_LIMIT_EXCEEDED = range(7)
SGS_STATIC_MAX_FRAMES = 4096
SGS_FLAG_ASYNC = 1
SGS_FLAG_RADIX_BINNING = 2
SGS_FLAG_TRACK_REUSE = 4
SGS_FLAG_LAZY_GRADS = 8
SGS_FLAG_NORMALISED_DEPTH = 16
SGS_FLAG_GRAPH = 32
SGS_FLAG_TIGHT_BINNING = 64
SGS_FLAG_LOWPASS = 128

ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p, C.c_void_p)
FREE_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p, C.c_void_p)


class sgs_config(C.Structure):
    _fields_ = [("tile", C.c_int), ("cutoff", C.c_float), ("alpha_min", C.c_float), ("alpha_max", C.c_float),
                ("t_min", C.c_float), ("z_near", C.c_float), ("flags", C.c_int),
                ("alloc", ALLOC_FN), ("free", FREE_FN), ("user", C.c_void_p)]


class sgs_surfels(C.Structure):
    _fields_ = [("n", C.c_int64), ("mean", C.c_void_p), ("scale", C.c_void_p), ("quat", C.c_void_p),
                ("opacity", C.c_void_p), ("rgb", C.c_void_p), ("active", C.c_void_p)]


class sgs_camera(C.Structure):
    _fields_ = [("width", C.c_int), ("height", C.c_int), ("fx", C.c_float), ("fy", C.c_float),
                ("cx", C.c_float), ("cy", C.c_float), ("T_cw", C.c_float * 12)]


class sgs_images(C.Structure):
    _fields_ = [("rgb", C.c_void_p), ("depth", C.c_void_p), ("normal", C.c_void_p), ("alpha", C.c_void_p)]


class sgs_surfel_grads(C.Structure):
    _fields_ = [("mean", C.c_void_p), ("scale", C.c_void_p), ("quat", C.c_void_p), ("opacity", C.c_void_p),
                ("rgb", C.c_void_p)]


class sgs_stats(C.Structure):
    _fields_ = [("n_visible", C.c_int64), ("n_entries", C.c_int64), ("capacity", C.c_int64), ("overflow", C.c_int64),
                ("workspace_bytes", C.c_int64), ("kernel_launches", C.c_int64)]


EXPORTS = ["sgs_default_config", "sgs_create", "sgs_destroy", "sgs_render", "sgs_prepare", "sgs_backward", "sgs_wait_grads", "sgs_tracking_loss",
           "sgs_backward_tracking", "sgs_track_iter", "sgs_track_new_frame", "sgs_render_contrib", "sgs_render_median", "sgs_covisibility", "sgs_mapping_loss", "sgs_ssim_loss", "sgs_map_correction", "sgs_measure_fp32_peak", "sgs_get_binning", "sgs_get_stats", "sgs_upload_surfels", "sgs_render_host", "sgs_backward_host",
           "sgs_upload_target", "sgs_track_iter_host", "sgs_set_profiling", "sgs_get_profile", "sgs_status_string",
           "sgs_track_iter_dev", "sgs_probe_staging", "sgs_backward_accumulate", "sgs_zero_grads", "sgs_map_view_host", "sgs_fetch_grads_host", "sgs_sync_host", "sgs_fetch_grads_sparse_host", "sgs_map_correction_static"]

_lib = None
_LIVE = weakref.WeakSet()


@atexit.register
def _close_all():
    for r in list(_LIVE):
        r.close()


def load_library():
    """dlopen libsgs.so (built by build.py).  Fails loudly when it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise RuntimeError(f"{_LIB_PATH} is missing: run `python -m paper_2506_00970_b200.build` "
                               "(or __graft_entry__.build()); there is no CPU fallback")
        lib = C.CDLL(_LIB_PATH)
        for name in EXPORTS:
            getattr(lib, name)  # AttributeError if a declared symbol is not exported
        for name in EXPORTS:
            getattr(lib, name).restype = C.c_char_p if name == "sgs_status_string" else C.c_int
        _lib = lib
    return _lib


class SgsError(RuntimeError):
    def __init__(self, status, where):
        self.status = status
        super().__init__(f"{where}: {load_library().sgs_status_string(status).decode()} (status {status})")


def _check(status, where):
    if status != SGS_OK:
        raise SgsError(status, where)


def _ptr(t, dtype=torch.float32, device_type="cuda"):
    if t is None:
        return None
    if not isinstance(t, torch.Tensor) or t.dtype != dtype or not t.is_contiguous() or t.device.type != device_type:
        raise TypeError(f"expected a contiguous {dtype} {device_type} tensor")
    return C.c_void_p(t.data_ptr())


def make_camera(width, height, fx, fy, cx, cy, T_cw):
    cam = sgs_camera()
    cam.width, cam.height, cam.fx, cam.fy, cam.cx, cam.cy = int(width), int(height), fx, fy, cx, cy
    T = np.asarray(T_cw, dtype=np.float32)[:3].reshape(12)
    for i in range(12):
        cam.T_cw[i] = float(T[i])
    return cam


def _images(rgb=None, depth=None, normal=None, alpha=None, device_type="cuda"):
    im = sgs_images()
    im.rgb, im.depth = _ptr(rgb, device_type=device_type), _ptr(depth, device_type=device_type)
    im.normal, im.alpha = _ptr(normal, device_type=device_type), _ptr(alpha, device_type=device_type)
    return im


def _stream_ptr(stream):
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def measure_fp32_peak(stream=None):
    """sgs_measure_fp32_peak: measured FP32 FMA throughput of the current device in TFLOP/s."""
    if not torch.cuda.is_available():
        raise RuntimeError("paper_2506_00970_b200 needs a CUDA device; there is no CPU fallback")
    out = C.c_double(0.0)
    _check(load_library().sgs_measure_fp32_peak(C.byref(out), _stream_ptr(stream)), "sgs_measure_fp32_peak")
    return float(out.value)


def map_correction_static(mean, quat, frame_id, T_orig, T_opt, stream=None):
    """sgs_map_correction_static: sgs_map_correction (Eq. 31-32, in place) without a ctx and without any allocation; the
    keyframe increments sit in a static device array of SGS_STATIC_MAX_FRAMES entries (SgsError SGS_LIMIT_EXCEEDED beyond).
    Calls that overlap on the GPU race on that array."""
    if not torch.cuda.is_available():
        raise RuntimeError("paper_2506_00970_b200 needs a CUDA device; there is no CPU fallback")
    _check(load_library().sgs_map_correction_static(C.c_int64(mean.shape[0]), _ptr(mean), _ptr(quat), _ptr(frame_id, torch.int32),
                                                    C.c_int(T_orig.shape[0]), _ptr(T_orig), _ptr(T_opt), _stream_ptr(stream)),
           "sgs_map_correction_static")


class Renderer:
    """One sgs_ctx.  Method names follow the C calls (sgs_render -> render, ...)."""

    def __init__(self, tile=16, cutoff=3.0, alpha_min=1.0 / 255.0, alpha_max=0.99, t_min=1e-4, z_near=0.2,
                 async_mode=False, radix_binning=False, track_reuse=False, lazy_grads=False, normalised_depth=False, graph=False, tight_binning=False, lowpass=False, device="cuda:0", torch_allocator=True):
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2506_00970_b200 needs a CUDA device; there is no CPU fallback")
        self.lib = load_library()
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        torch.cuda.current_stream()  # make sure the primary context exists
        cfg = sgs_config()
        _check(self.lib.sgs_default_config(C.byref(cfg)), "sgs_default_config")
        cfg.tile, cfg.cutoff, cfg.alpha_min, cfg.alpha_max = tile, cutoff, alpha_min, alpha_max
        cfg.t_min, cfg.z_near = t_min, z_near
        cfg.flags = ((SGS_FLAG_ASYNC if async_mode else 0) | (SGS_FLAG_RADIX_BINNING if radix_binning else 0) |
                     (SGS_FLAG_TRACK_REUSE if track_reuse else 0) | (SGS_FLAG_LAZY_GRADS if lazy_grads else 0) |
                     (SGS_FLAG_NORMALISED_DEPTH if normalised_depth else 0) | (SGS_FLAG_GRAPH if graph else 0) |
                     (SGS_FLAG_TIGHT_BINNING if tight_binning else 0) | (SGS_FLAG_LOWPASS if lowpass else 0))
        if torch_allocator:
            dev_index = self.device.index or 0

            _t_alloc, _t_delete = torch.cuda.caching_allocator_alloc, torch.cuda.caching_allocator_delete

            def _alloc(nbytes, user, stream):
                try:
                    return _t_alloc(int(nbytes), dev_index, stream)
                except Exception:
                    return None

            def _free(ptr, user, stream):
                try:
                    _t_delete(ptr)
                except Exception:  # interpreter shutdown: the allocator is already gone
                    pass

            self._alloc_cb, self._free_cb = ALLOC_FN(_alloc), FREE_FN(_free)  # keep alive
            cfg.alloc, cfg.free = self._alloc_cb, self._free_cb
        self._cfg = cfg
        self._ctx = C.c_void_p()
        _check(self.lib.sgs_create(C.byref(self._ctx), C.byref(cfg)), "sgs_create")
        _LIVE.add(self)

    def close(self):
        if getattr(self, "_ctx", None) is not None and self._ctx:
            self.lib.sgs_destroy(self._ctx)
            self._ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- device path -------------------------------------------------------------------------
    @staticmethod
    def surfels(mean, scale, quat, opacity, rgb, active=None):
        s = sgs_surfels()
        s.n = mean.shape[0]
        s.mean, s.scale, s.quat, s.opacity, s.rgb = _ptr(mean), _ptr(scale), _ptr(quat), _ptr(opacity), _ptr(rgb)
        s.active = _ptr(active, torch.uint8)
        return s

    def render(self, surfels, cam, rgb=None, depth=None, normal=None, alpha=None, stream=None):
        """sgs_render.  `surfels` is a sgs_surfels (see Renderer.surfels); images are preallocated
        device tensors (any may be None)."""
        im = _images(rgb, depth, normal, alpha)
        _check(self.lib.sgs_render(self._ctx, C.byref(surfels), C.byref(cam), C.byref(im), _stream_ptr(stream)), "sgs_render")

    def wait_grads(self, stream=None):
        """sgs_wait_grads: with lazy_grads=True, orders `stream` behind the last backward()'s per-surfel kernel."""
        _check(self.lib.sgs_wait_grads(self._ctx, _stream_ptr(stream)), "sgs_wait_grads")

    def track_new_frame(self):
        """sgs_track_new_frame: with track_reuse=True, drops the survivor list kept across tracking iterations (call at
        every new frame / whenever the map arrays may have changed)."""
        _check(self.lib.sgs_track_new_frame(self._ctx), "sgs_track_new_frame")

    def prepare(self, surfels, cam, stream=None):
        """sgs_prepare: preprocess + tile binning only; the next render() of the same (surfels, cam) objects on this
        Renderer skips its binning and orders itself behind this call (the streams may differ)."""
        _check(self.lib.sgs_prepare(self._ctx, C.byref(surfels), C.byref(cam), _stream_ptr(stream)), "sgs_prepare")

    def render_median(self, surfels, cam, median, rgb=None, depth=None, normal=None, alpha=None, stream=None):
        """sgs_render_median: render + median depth image (R9m) into `median` (H x W floats, device)."""
        out = _images(rgb, depth, normal, alpha)
        _check(self.lib.sgs_render_median(self._ctx, C.byref(surfels), C.byref(cam), C.byref(out), _ptr(median),
                                          _stream_ptr(stream)), "sgs_render_median")

    def render_contrib(self, surfels, cam, contrib, rgb=None, depth=None, normal=None, alpha=None, stream=None):
        """sgs_render_contrib: render + per-splat contribution C_k^V (Eq. 20-21) into `contrib` (n floats, device)."""
        out = _images(rgb, depth, normal, alpha)
        _check(self.lib.sgs_render_contrib(self._ctx, C.byref(surfels), C.byref(cam), C.byref(out), _ptr(contrib),
                                           _stream_ptr(stream)), "sgs_render_contrib")

    def covisibility(self, contrib_a, contrib_b, result3, active=None, threshold=0.5, stream=None):
        """sgs_covisibility (Eq. 22): result3 <- (score, |intersection|, |union|)."""
        _check(self.lib.sgs_covisibility(self._ctx, _ptr(contrib_a), _ptr(contrib_b), C.c_int64(contrib_a.numel()),
                                         _ptr(active, torch.uint8), C.c_float(threshold), _ptr(result3),
                                         _stream_ptr(stream)), "sgs_covisibility")

    @staticmethod
    def _grads(grads, device_type="cuda"):
        g = sgs_surfel_grads()
        p = lambda t: _ptr(t, torch.float32, device_type)
        g.mean, g.scale, g.quat = p(grads.get("mean")), p(grads.get("scale")), p(grads.get("quat"))
        g.opacity, g.rgb = p(grads.get("opacity")), p(grads.get("rgb"))
        return g

    def backward(self, d_rgb=None, d_depth=None, d_normal=None, d_alpha=None, grads=None, d_pose6=None, stream=None,
                 accumulate=False):
        """sgs_backward.  grads: dict of preallocated device tensors mean/scale/quat/opacity/rgb, or None
        (pose-only).  d_pose6: device tensor of 6 floats or None.  accumulate=True: sgs_backward_accumulate (the surfel
        gradients are ADDED to `grads`, which the caller zeroes once per window: zero_grads)."""
        up = _images(d_rgb, d_depth, d_normal, d_alpha)
        g = self._grads(grads) if grads is not None else None
        fn, name = (self.lib.sgs_backward_accumulate, "sgs_backward_accumulate") if accumulate else (self.lib.sgs_backward, "sgs_backward")
        _check(fn(self._ctx, C.byref(up), C.byref(g) if g is not None else None, _ptr(d_pose6), _stream_ptr(stream)), name)

    def zero_grads(self, grads, stream=None):
        """sgs_zero_grads: the start of an accumulation window."""
        n = next(v for v in grads.values() if v is not None).shape[0]
        g = self._grads(grads)
        _check(self.lib.sgs_zero_grads(self._ctx, C.byref(g), C.c_int64(n), _stream_ptr(stream)), "sgs_zero_grads")

    def map_view_host(self, cam, target_rgb, target_depth, lambda_c, w_d, w_n, ssim_weight, normal_sign, loss=None, pose6=None,
                      stream=None):
        """sgs_map_view_host: one view of a mapping window on the resident map, HOST (ideally pinned) target frame in;
        loss (1 float) / pose6 (6 floats): HOST tensors filled by sync_host()."""
        self._win_keep = getattr(self, "_win_keep", [])
        self._win_keep.append((target_rgb, target_depth, loss, pose6))      # alive until sync_host
        _check(self.lib.sgs_map_view_host(self._ctx, C.byref(cam), _ptr(target_rgb, torch.float32, "cpu"),
                                          _ptr(target_depth, torch.float32, "cpu"), C.c_float(lambda_c), C.c_float(w_d),
                                          C.c_float(w_n), C.c_float(ssim_weight), C.c_float(normal_sign),
                                          _ptr(loss, torch.float32, "cpu"), _ptr(pose6, torch.float32, "cpu"),
                                          _stream_ptr(stream)), "sgs_map_view_host")

    def fetch_grads_host(self, grads, stream=None):
        """sgs_fetch_grads_host: ends the window; `grads` (HOST tensors) are complete after sync_host()."""
        self._win_keep = getattr(self, "_win_keep", [])
        self._win_keep.append(grads)
        g = self._grads(grads, "cpu")
        _check(self.lib.sgs_fetch_grads_host(self._ctx, C.byref(g), _stream_ptr(stream)), "sgs_fetch_grads_host")

    def fetch_grads_sparse_host(self, ids, rows, count, stream=None):
        """sgs_fetch_grads_sparse_host: ends the window; rows [0, count) of the PINNED host tensors in `rows` (dict like
        grads) hold the gradients of surfels ids[0..count) (int32, ascending); count: HOST int64 tensor of one element.
        All complete after sync_host()."""
        self._win_keep = getattr(self, "_win_keep", [])
        self._win_keep.append((ids, rows, count))
        g = self._grads(rows, "cpu")
        cap = min([ids.shape[0]] + [v.shape[0] for v in rows.values() if v is not None])
        _check(self.lib.sgs_fetch_grads_sparse_host(self._ctx, _ptr(ids, torch.int32, "cpu"), C.byref(g), C.c_int64(cap),
                                                    _ptr(count, torch.int64, "cpu"), _stream_ptr(stream)),
               "sgs_fetch_grads_sparse_host")

    def sync_host(self, stream=None):
        _check(self.lib.sgs_sync_host(self._ctx, _stream_ptr(stream)), "sgs_sync_host")
        self._win_keep = []

    def tracking_loss(self, cam, ren, target_rgb, target_depth, lambda_d, normal_sign, up, loss, stream=None):
        """sgs_tracking_loss.  ren/up: dicts with rgb, depth, normal, alpha device tensors."""
        r = _images(ren["rgb"], ren["depth"], ren["normal"], ren["alpha"])
        t = _images(target_rgb, target_depth)
        u = _images(up["rgb"], up["depth"], up["normal"], up["alpha"])
        _check(self.lib.sgs_tracking_loss(self._ctx, C.byref(cam), C.byref(r), C.byref(t), C.c_float(lambda_d),
                                          C.c_float(normal_sign), C.byref(u), _ptr(loss), _stream_ptr(stream)),
               "sgs_tracking_loss")

    def mapping_loss(self, cam, ren, target_rgb, target_depth, lambda_c, w_d, w_n, normal_sign, up, loss, stream=None):
        """sgs_mapping_loss (Eq. 24-26 without SSIM).  ren/up: dicts with rgb, depth, normal, alpha device tensors."""
        r = _images(ren["rgb"], ren["depth"], ren["normal"], ren["alpha"])
        t = _images(rgb=target_rgb, depth=target_depth)
        u = _images(up["rgb"], up["depth"], up["normal"], up["alpha"])
        _check(self.lib.sgs_mapping_loss(self._ctx, C.byref(cam), C.byref(r), C.byref(t), C.c_float(lambda_c), C.c_float(w_d),
                                         C.c_float(w_n), C.c_float(normal_sign), C.byref(u), _ptr(loss), _stream_ptr(stream)),
               "sgs_mapping_loss")

    def ssim_loss(self, rendered_rgb, target_rgb, weight, upstream_rgb, loss=None, stream=None):
        """sgs_ssim_loss (SSIM term of Eq. 24): ACCUMULATES into upstream_rgb and loss."""
        H, W = rendered_rgb.shape[-2], rendered_rgb.shape[-1]
        _check(self.lib.sgs_ssim_loss(self._ctx, C.c_int(W), C.c_int(H), _ptr(rendered_rgb), _ptr(target_rgb),
                                      C.c_float(weight), _ptr(upstream_rgb), _ptr(loss), _stream_ptr(stream)), "sgs_ssim_loss")

    def map_correction(self, mean, quat, frame_id, T_orig, T_opt, stream=None):
        """sgs_map_correction (Eq. 31-32), in place.  T_orig / T_opt: (n_frames, 12) CAMERA-TO-WORLD keyframe poses [R | t]
        (reading R29; pass the inverses of world-to-camera poses)."""
        """sgs_map_correction (Eq. 31-32), in place on mean / quat."""
        _check(self.lib.sgs_map_correction(self._ctx, C.c_int64(mean.shape[0]), _ptr(mean), _ptr(quat),
                                           _ptr(frame_id, torch.int32), C.c_int(T_orig.shape[0]), _ptr(T_orig), _ptr(T_opt),
                                           _stream_ptr(stream)), "sgs_map_correction")

    def backward_tracking(self, target_rgb, target_depth, lambda_d, normal_sign, d_pose6, loss=None, stream=None):
        """sgs_backward_tracking: pose-only backward with the Eq. 15-19 loss fused in."""
        t = _images(target_rgb, target_depth)
        _check(self.lib.sgs_backward_tracking(self._ctx, C.byref(t), C.c_float(lambda_d), C.c_float(normal_sign),
                                              _ptr(d_pose6), _ptr(loss), _stream_ptr(stream)), "sgs_backward_tracking")

    def track_iter(self, surfels, cam, target_rgb, target_depth, lambda_d, normal_sign, d_pose6, loss=None,
                   rgb=None, depth=None, normal=None, alpha=None, stream=None):
        """sgs_track_iter: preprocess + binning, then ONE kernel for render + Eq. 15-19 loss + pose-only backward."""
        t = _images(rgb=target_rgb, depth=target_depth)
        out = _images(rgb, depth, normal, alpha)
        _check(self.lib.sgs_track_iter(self._ctx, C.byref(surfels), C.byref(cam), C.byref(t), C.c_float(lambda_d),
                                       C.c_float(normal_sign), C.byref(out), _ptr(d_pose6), _ptr(loss),
                                       _stream_ptr(stream)), "sgs_track_iter")

    def track_iter_dev(self, surfels, cam, d_T_cw, target_rgb, target_depth, lambda_d, normal_sign, d_pose6, loss=None,
                       rgb=None, depth=None, normal=None, alpha=None, stream=None):
        """sgs_track_iter_dev: the pose is read from the DEVICE tensor d_T_cw (12 floats, row-major 3x4) when the kernels run."""
        t = _images(target_rgb, target_depth)
        out = _images(rgb, depth, normal, alpha)
        _check(self.lib.sgs_track_iter_dev(self._ctx, C.byref(surfels), C.byref(cam), _ptr(d_T_cw), C.byref(t), C.c_float(lambda_d),
                                           C.c_float(normal_sign), C.byref(out), _ptr(d_pose6), _ptr(loss), _stream_ptr(stream)),
               "sgs_track_iter_dev")

    def probe_staging(self, mode, reps=20, stream=None):
        """sgs_probe_staging: microseconds per launch of the staging alone over the last render's tile lists (mode 0: LDG
        gathers, mode 1: one cp.async.bulk per 128-byte record)."""
        us = C.c_double(0.0)
        _check(self.lib.sgs_probe_staging(self._ctx, C.c_int(mode), C.c_int(reps), C.byref(us), _stream_ptr(stream)), "sgs_probe_staging")
        return float(us.value)

    def get_binning(self, n, tiles):
        """sgs_get_binning -> numpy copies: keys (E,) u64, idx (E,) u32, ranges (tiles,2) u32, culled (n,) u8."""
        E = C.c_int64()
        keys, idx, rng, cul = C.c_void_p(), C.c_void_p(), C.c_void_p(), C.c_void_p()
        _check(self.lib.sgs_get_binning(self._ctx, C.byref(E), C.byref(keys), C.byref(idx), C.byref(rng), C.byref(cul)),
               "sgs_get_binning")
        e = int(E.value)

        def fetch(ptr, count, dtype):
            return _device_to_numpy(ptr.value, count, dtype)

        return dict(E=e, keys=fetch(keys, e, np.uint64), idx=fetch(idx, e, np.uint32),
                    ranges=fetch(rng, tiles * 2, np.uint32).reshape(tiles, 2), culled=fetch(cul, n, np.uint8))

    def stats(self):
        st = sgs_stats()
        _check(self.lib.sgs_get_stats(self._ctx, C.byref(st)), "sgs_get_stats")
        return {k: int(getattr(st, k)) for k, _ in sgs_stats._fields_}

    STAGES = ("preprocess", "sort", "forward", "loss", "backward", "track")

    def set_profiling(self, enabled):
        _check(self.lib.sgs_set_profiling(self._ctx, C.c_int(int(enabled))), "sgs_set_profiling")

    def get_profile(self, reset=True):
        """sgs_get_profile -> {stage: (total_ms, calls)}; waits for the device."""
        ms = (C.c_double * len(self.STAGES))()
        calls = (C.c_int64 * len(self.STAGES))()
        _check(self.lib.sgs_get_profile(self._ctx, ms, calls, C.c_int(int(reset))), "sgs_get_profile")
        return {k: (float(ms[i]), int(calls[i])) for i, k in enumerate(self.STAGES)}

    # ---- host path (end-to-end) --------------------------------------------------------------
    def upload_surfels(self, mean, scale, quat, opacity, rgb, active=None, stream=None):
        """sgs_upload_surfels: HOST (ideally pinned) tensors -> ctx-resident device map."""
        s = sgs_surfels()
        s.n = mean.shape[0]
        hp = lambda t, dt=torch.float32: _ptr(t, dt, "cpu")
        s.mean, s.scale, s.quat, s.opacity, s.rgb, s.active = hp(mean), hp(scale), hp(quat), hp(opacity), hp(rgb), hp(active, torch.uint8)
        _check(self.lib.sgs_upload_surfels(self._ctx, C.byref(s), _stream_ptr(stream)), "sgs_upload_surfels")

    def render_host(self, cam, rgb=None, depth=None, normal=None, alpha=None, stream=None):
        im = _images(rgb, depth, normal, alpha, device_type="cpu")
        _check(self.lib.sgs_render_host(self._ctx, C.byref(cam), C.byref(im), _stream_ptr(stream)), "sgs_render_host")

    def backward_host(self, d_rgb=None, d_depth=None, d_normal=None, d_alpha=None, grads=None, d_pose6=None, stream=None):
        up = _images(d_rgb, d_depth, d_normal, d_alpha, device_type="cpu")
        g = None
        if grads is not None:
            g = sgs_surfel_grads()
            hp = lambda t: _ptr(t, torch.float32, "cpu")
            g.mean, g.scale, g.quat, g.opacity, g.rgb = (hp(grads.get(k)) for k in ("mean", "scale", "quat", "opacity", "rgb"))
        _check(self.lib.sgs_backward_host(self._ctx, C.byref(up), C.byref(g) if g is not None else None,
                                          _ptr(d_pose6, torch.float32, "cpu"), _stream_ptr(stream)), "sgs_backward_host")

    def upload_target(self, cam, rgb, depth, stream=None):
        _check(self.lib.sgs_upload_target(self._ctx, C.byref(cam), _ptr(rgb, torch.float32, "cpu"),
                                          _ptr(depth, torch.float32, "cpu"), _stream_ptr(stream)), "sgs_upload_target")

    def track_iter_host(self, cam, lambda_d, normal_sign, stream=None):
        buf = getattr(self, "_h_track", None)
        if buf is None:  # one 7-float host buffer for the life of the Renderer: this call sits in a tracker's inner loop
            buf = self._h_track = (C.c_float * 7)()
            self._h_track_np = np.frombuffer(buf, dtype=np.float32)
        _check(self.lib.sgs_track_iter_host(self._ctx, C.byref(cam), C.c_float(lambda_d), C.c_float(normal_sign),
                                            buf, C.byref(buf, 4), _stream_ptr(stream)), "sgs_track_iter_host")
        return float(self._h_track_np[0]), self._h_track_np[1:].copy()


class _RawDeviceBytes:
    """Wraps a library-owned device pointer for torch through __cuda_array_interface__."""

    def __init__(self, ptr, nbytes):
        self.__cuda_array_interface__ = {"shape": (int(nbytes),), "typestr": "|u1", "data": (int(ptr), False), "version": 2}


def _device_to_numpy(dev_ptr, count, dtype):
    out = np.empty(count, dtype=dtype)
    if count:
        t = torch.as_tensor(_RawDeviceBytes(dev_ptr, out.nbytes), device="cuda")
        out.view(np.uint8)[:] = t.cpu().numpy()
    return out
