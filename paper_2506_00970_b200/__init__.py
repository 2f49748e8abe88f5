"""B200-native differentiable 2D-Gaussian (surfel) splatting renderer -- the hot path of
2DGS-SLAM (arxiv 2506.00970): hand-written CUDA for sm_100a behind the C ABI of include/sgs.h,
with this thin ctypes binding on top.  See DESIGN.md."""
from .binding import (Renderer, measure_fp32_peak, SgsError, make_camera, load_library, EXPORTS, sgs_camera, sgs_surfels, sgs_images,
                      sgs_surfel_grads, sgs_config, sgs_stats, SGS_OK, SGS_WORKSPACE_OVERFLOW, SGS_NO_FORWARD_STATE,
                      SGS_INVALID_ARGUMENT, SGS_FLAG_ASYNC, SGS_LIMIT_EXCEEDED, SGS_STATIC_MAX_FRAMES, map_correction_static)

__all__ = ["Renderer", "SgsError", "make_camera", "load_library", "EXPORTS"]
