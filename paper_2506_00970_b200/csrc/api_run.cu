// api_run.cu -- sgs_render / sgs_backward / sgs_tracking_loss / debug export (include/sgs.h).
#include <math.h>
#include <string.h>
#include "sgs_internal.h"

static inline bool radix_mode(const sgs_ctx* c) { return (c->cfg.flags & SGS_FLAG_RADIX_BINNING) != 0; }
// SGS_FLAG_GRAPH: no event is queried, waited for or shared with another stream and the ctx has no stream of its own, so a
// stream capture sees kernels and copies only; the counters still reach pinned memory, nobody polls them
static inline bool graph_mode(const sgs_ctx* c) { return (c->cfg.flags & SGS_FLAG_GRAPH) != 0; }

static int64_t grown_tile_cap(int64_t max_tile) { return max_tile + max_tile / 2 + 64; }

// async mode: examine the counters of the previous render (already copied to pinned memory)
static int check_pending(sgs_ctx* c, cudaStream_t s) {
    if (!c->pending_check || graph_mode(c)) return SGS_OK;
    if (c->pending_lazy) {
        // sgs_track_iter copies the counters after its fused kernel: waiting here would serialise host and device,
        // so an overflow of iteration i is reported by the first call that finds the copy complete
        const cudaError_t q = cudaEventQuery(c->counters_ready);
        if (q == cudaErrorNotReady) return SGS_OK;
        if (q != cudaSuccess) return SGS_CUDA_ERROR;
    } else if (cudaEventSynchronize(c->counters_ready) != cudaSuccess) return SGS_CUDA_ERROR;
    c->pending_check = false;
    c->pending_lazy = false;
    const int64_t E = (int64_t)c->counters_host->n_entries;
    c->last_entries = E;
    c->last_surv = (int64_t)c->counters_host->n_surv;
    c->last_vis = (int64_t)c->counters_host->n_visible;
    if (radix_mode(c)) {
        if (c->counters_host->overflow) {
            c->have_forward = c->have_binning = c->prepared = false;
            const int r = sgs_ensure_entries(c, E, s);
            return r != SGS_OK ? r : SGS_WORKSPACE_OVERFLOW;
        }
    } else if (c->counters_host->max_tile > (unsigned)c->tile_cap) {
        c->have_forward = c->have_binning = c->prepared = false;
        const int r = sgs_ensure_buckets(c, c->camd.tiles_x * c->camd.tiles_y, grown_tile_cap(c->counters_host->max_tile), s);
        return r != SGS_OK ? r : SGS_WORKSPACE_OVERFLOW;
    }
    return SGS_OK;
}

static int copy_counters(sgs_ctx* c, cudaStream_t s) {
    static_assert(sizeof(SgsCounters) % 4 == 0, "");
    c->launches += 1;   // (a one-warp kernel to mapped host memory, not a copy command: see k_publish_words)
    return sgs_launch_publish(c->counters_host_dev, c->counters, (int)(sizeof(SgsCounters) / 4), s) == cudaSuccess ? SGS_OK : SGS_CUDA_ERROR;
}

// binning through per-tile buckets + in-tile sort (default)
static int bin_buckets(sgs_ctx* c, const sgs_surfels* sf, bool async, bool want_order, cudaStream_t s) {
    const int tiles = c->camd.tiles_x * c->camd.tiles_y;
    if (c->copy_in_flight) {  // a copy of the LIVE counters (render path) may still run on the ctx's stream: normally long done
        if (cudaStreamWaitEvent(s, c->counters_ready, 0) != cudaSuccess) return SGS_CUDA_ERROR;
        c->copy_in_flight = false;
    }
    int r = sgs_ensure_buckets(c, tiles, c->tile_cap ? c->tile_cap : 2048, s);
    if (r != SGS_OK) return r;
    if (sgs_launch_preprocess_bucket(c, sf, s) != cudaSuccess) return SGS_CUDA_ERROR;
    const bool defer = async && c->defer_counters && c->tile_cap <= 2048;  // the fused kernel snapshots them
    c->defer_counters = defer;
    // async mode: the 32-byte copy runs on the ctx's own stream so that it is not a link of the caller's chain
    // (K-pre-B -> copy -> compositing); the next preprocess on this ctx waits for it before it clears the counters
    cudaStream_t cs = (async && c->aux_stream) ? c->aux_stream : s;
    c->stats_src = c->counters;
    if (!defer && !graph_mode(c)) {  // (capture mode: nobody polls; sgs_get_stats fetches them itself)
        if (cs != s && (cudaEventRecord(c->fork_ev, s) != cudaSuccess || cudaStreamWaitEvent(cs, c->fork_ev, 0) != cudaSuccess))
            return SGS_CUDA_ERROR;
        if ((r = copy_counters(c, cs)) != SGS_OK) return r;
    }
    if (!async) {
        if (cudaStreamSynchronize(s) != cudaSuccess) return SGS_CUDA_ERROR;
        if (c->counters_host->max_tile > (unsigned)c->tile_cap) {  // grow and emit again
            if ((r = sgs_ensure_buckets(c, tiles, grown_tile_cap(c->counters_host->max_tile), s)) != SGS_OK) return r;
            if (sgs_launch_preprocess_bucket(c, sf, s) != cudaSuccess) return SGS_CUDA_ERROR;
            if ((r = copy_counters(c, s)) != SGS_OK) return r;
            if (cudaStreamSynchronize(s) != cudaSuccess) return SGS_CUDA_ERROR;
        }
        c->last_entries = (int64_t)c->counters_host->n_entries;
        c->last_surv = (int64_t)c->counters_host->n_surv;
        c->last_vis = (int64_t)c->counters_host->n_visible;
    } else if (!defer && !graph_mode(c)) {
        cudaEventRecord(c->counters_ready, cs);
        c->copy_in_flight = cs != s;
        c->pending_check = true;
        c->pending_lazy = false;
    }
    c->fused_sort = c->tile_cap <= 2048;
    c->render_order_valid = false;
    if (want_order && sgs_launch_tile_order(c, s) != cudaSuccess) return SGS_CUDA_ERROR;
    if (c->fused_sort) {  // k_forward orders each bucket itself
        c->list_vals = reinterpret_cast<const uint32_t*>(c->bucket);
        c->list_stride = 2;
        return SGS_OK;
    }
    return sgs_launch_tilesort(c, s) == cudaSuccess ? SGS_OK : SGS_CUDA_ERROR;
}

// binning through the global LSD radix sort of (tile << 32 | depth) keys (SGS_FLAG_RADIX_BINNING)
static int bin_radix(sgs_ctx* c, const sgs_surfels* sf, bool async, cudaStream_t s) {
    int r;
    if (c->e_cap == 0) {
        int64_t guess = 2 * sf->n;
        if (guess < (1 << 20)) guess = 1 << 20;
        if ((r = sgs_ensure_entries(c, guess, s)) != SGS_OK) return r;
    }
    c->launch_entries = c->e_cap;
    if (async && c->last_entries > 0) {
        const int64_t hint = c->last_entries + c->last_entries / 4 + 4096;
        if (hint < c->launch_entries) c->launch_entries = hint;
    }
    if (sgs_launch_preprocess(c, sf, s) != cudaSuccess) return SGS_CUDA_ERROR;
    c->stats_src = c->counters;
    if (!graph_mode(c) && (r = copy_counters(c, s)) != SGS_OK) return r;
    if (!async) {
        if (cudaStreamSynchronize(s) != cudaSuccess) return SGS_CUDA_ERROR;
        const int64_t E = (int64_t)c->counters_host->n_entries;
        c->last_entries = E;
        if (E > c->e_cap) {  // grow and emit again
            if ((r = sgs_ensure_entries(c, E, s)) != SGS_OK) return r;
            c->launch_entries = c->e_cap;
            if (sgs_launch_preprocess(c, sf, s) != cudaSuccess) return SGS_CUDA_ERROR;
            if ((r = copy_counters(c, s)) != SGS_OK) return r;
            if (cudaStreamSynchronize(s) != cudaSuccess) return SGS_CUDA_ERROR;
        }
        c->launch_entries = E;  // exact grids
    } else if (!graph_mode(c)) {
        cudaEventRecord(c->counters_ready, s);
        c->pending_check = true;
        c->pending_lazy = false;
    }
    c->fused_sort = false;
    c->render_order_valid = false;
    return sgs_launch_sort_and_ranges(c, s) == cudaSuccess ? SGS_OK : SGS_CUDA_ERROR;
}

extern "C" {

// preprocess + tile binning of one view (shared by sgs_render and sgs_track_iter)
static int bin_view(sgs_ctx* c, const sgs_surfels* sf, const sgs_camera* cam, bool want_order, cudaStream_t s) {
    if (!c || !sf || !sgs_cam_valid(cam) || sf->n < 0 || sf->n >= (1ll << 24)) return SGS_INVALID_ARGUMENT;
    if (sf->n > 0 && (!sf->mean || !sf->scale || !sf->quat || !sf->opacity || !sf->rgb)) return SGS_INVALID_ARGUMENT;
    int r = check_pending(c, s);
    if (r != SGS_OK) return r;
    c->have_forward = false;
    c->have_binning = false;
    if (c->grads_on_aux) {  // SGS_FLAG_LAZY_GRADS: the last backward's per-surfel kernel still reads the lists this call rewrites
        if (c->work_recorded && cudaStreamWaitEvent(s, c->work_ev, 0) != cudaSuccess) return SGS_CUDA_ERROR;
        c->grads_on_aux = false;
    }
    if (!c->use_surv_cache) c->surv_valid = false;  // K-pre-A is about to overwrite the list
    sgs_fill_cam(cam, &c->camd);
    const int tiles = c->camd.tiles_x * c->camd.tiles_y;
    const int64_t pixels = (int64_t)cam->width * cam->height;
    if ((r = sgs_ensure_surfels(c, sf->n, s)) != SGS_OK) return r;
    if ((r = sgs_ensure_image(c, tiles, pixels, s)) != SGS_OK) return r;
    const bool async = (c->cfg.flags & (SGS_FLAG_ASYNC | SGS_FLAG_GRAPH)) != 0;
    c->last_surfels = *sf;
    c->last_cam = *cam;
    return radix_mode(c) ? bin_radix(c, sf, async, s) : bin_buckets(c, sf, async, want_order, s);
}

static void pick_planes(sgs_ctx* c, const sgs_images* out, int64_t pixels, bool scratch, float* planes[8]) {
    for (int i = 0; i < 8; ++i) planes[i] = scratch ? c->img_scratch + (size_t)i * pixels : nullptr;
    if (out) {
        if (out->rgb) for (int i = 0; i < 3; ++i) planes[i] = out->rgb + (size_t)i * pixels;
        if (out->depth) planes[3] = out->depth;
        if (out->normal) for (int i = 0; i < 3; ++i) planes[4 + i] = out->normal + (size_t)i * pixels;
        if (out->alpha) planes[7] = out->alpha;
    }
}

// cam = Exp(tau) o ref with |rho| and |theta| inside 80 % of the survivor list's margins (same image and intrinsics)
static bool pose_within_margin(const sgs_camera* ref, const sgs_camera* cam) {
    if (ref->width != cam->width || ref->height != cam->height || ref->fx != cam->fx || ref->fy != cam->fy ||
        ref->cx != cam->cx || ref->cy != cam->cy) return false;
    const float* A = cam->T_cw; const float* B = ref->T_cw;  // rows [R | t]
    double Rd[9], tr = 0.0;
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {  // R_d = R_cam R_ref^T
            double v = 0.0;
            for (int k = 0; k < 3; ++k) v += (double)A[4 * i + k] * (double)B[4 * j + k];
            Rd[3 * i + j] = v;
        }
    tr = Rd[0] + Rd[4] + Rd[8];
    double cosang = 0.5 * (tr - 1.0);
    if (!(cosang <= 1.0)) cosang = 1.0;
    if (!(cosang >= -1.0)) return false;
    double d2 = 0.0;
    for (int i = 0; i < 3; ++i) {  // t_d = t_cam - R_d t_ref
        const double v = (double)A[4 * i + 3] - (Rd[3 * i] * B[3] + Rd[3 * i + 1] * B[7] + Rd[3 * i + 2] * B[11]);
        d2 += v * v;
    }
    const double mt = 0.8 * SGS_REUSE_MARGIN_T, mr = 0.8 * SGS_REUSE_MARGIN_R;
    return d2 <= mt * mt && cosang >= cos(mr);
}

static bool same_view(const sgs_ctx* c, const sgs_surfels* sf, const sgs_camera* cam) {
    return sf && cam && memcmp(&c->last_surfels, sf, sizeof(*sf)) == 0 && memcmp(&c->last_cam, cam, sizeof(*cam)) == 0;
}

int sgs_prepare(sgs_ctx* c, const sgs_surfels* sf, const sgs_camera* cam, void* stream) {
    if (!c || graph_mode(c)) return SGS_INVALID_ARGUMENT;  // (two streams and an event between them: not for a capture)
    cudaStream_t s = (cudaStream_t)stream;
    c->prepared = false;
    // the binning buffers are still read by the ctx's last render / backward, possibly on another stream
    if (c->work_recorded && cudaStreamWaitEvent(s, c->work_ev, 0) != cudaSuccess) return SGS_CUDA_ERROR;
    c->narrow_prepare = 1;  // K-pre-B at one block per SM (measured: C4 1070 -> 1092 MP/s against the full grid)
    const int r = bin_view(c, sf, cam, true, s);
    c->narrow_prepare = 0;
    if (r != SGS_OK) return r;
    if (cudaEventRecord(c->prepared_ev, s) != cudaSuccess) return SGS_CUDA_ERROR;
    c->prepared = true;
    return SGS_OK;
}

int sgs_render(sgs_ctx* c, const sgs_surfels* sf, const sgs_camera* cam, const sgs_images* out, void* stream) {
    if (!c) return SGS_INVALID_ARGUMENT;
    cudaStream_t s = (cudaStream_t)stream;
    int r;
    if (c->prepared && same_view(c, sf, cam)) {  // binning already enqueued by sgs_prepare: order this stream behind it
        // async mode: its counters have usually arrived by now; an overflow is reported HERE (workspace grown, nothing
        // composited from truncated lists) and the caller renders again, which bins in line
        if ((r = check_pending(c, s)) != SGS_OK) return r;
        c->prepared = false;
        if (cudaStreamWaitEvent(s, c->prepared_ev, 0) != cudaSuccess) return SGS_CUDA_ERROR;
    } else {
        c->prepared = false;
        if ((r = bin_view(c, sf, cam, true, s)) != SGS_OK) return r;
    }
    const int64_t pixels = (int64_t)cam->width * cam->height;
    float* planes[8];
    pick_planes(c, out, pixels, true, planes);
    for (int i = 0; i < 8; ++i) c->last_img[i] = planes[i];
    if (sgs_launch_forward(c, planes, s) != cudaSuccess) return SGS_CUDA_ERROR;
    c->have_forward = true;
    c->have_binning = true;
    c->work_recorded = !graph_mode(c) && cudaEventRecord(c->work_ev, s) == cudaSuccess;
    return SGS_OK;
}

int sgs_render_median(sgs_ctx* c, const sgs_surfels* sf, const sgs_camera* cam, const sgs_images* out, float* median,
                      void* stream) {
    if (!c || !sf || !median || c->cfgd.lowpass) return SGS_INVALID_ARGUMENT;
    c->median_out = median;
    const int r = sgs_render(c, sf, cam, out, stream);
    c->median_out = nullptr;
    return r;
}

int sgs_render_contrib(sgs_ctx* c, const sgs_surfels* sf, const sgs_camera* cam, const sgs_images* out, float* contrib,
                       void* stream) {
    if (!c || !sf || !contrib || c->cfgd.lowpass) return SGS_INVALID_ARGUMENT;
    if (sf->n > 0 && cudaMemsetAsync(contrib, 0, sizeof(float) * (size_t)sf->n, (cudaStream_t)stream) != cudaSuccess)
        return SGS_CUDA_ERROR;
    c->contrib_out = contrib;
    const int r = sgs_render(c, sf, cam, out, stream);
    c->contrib_out = nullptr;
    return r;
}

int sgs_covisibility(sgs_ctx* c, const float* ca, const float* cb, int64_t n, const uint8_t* active, float threshold,
                     float* result3, void* stream) {
    if (!c || !ca || !cb || !result3 || n < 0) return SGS_INVALID_ARGUMENT;
    return sgs_launch_covisibility(c, ca, cb, n, active, threshold, result3, (cudaStream_t)stream) == cudaSuccess
               ? SGS_OK : SGS_CUDA_ERROR;
}

int sgs_track_iter(sgs_ctx* c, const sgs_surfels* sf, const sgs_camera* cam, const sgs_images* target, float lambda_d,
                   float normal_sign, const sgs_images* out, float* d_pose6, float* loss, void* stream) {
    if (!c || !target || !target->rgb || !target->depth || !d_pose6) return SGS_INVALID_ARGUMENT;
    cudaStream_t s = (cudaStream_t)stream;
    if (radix_mode(c) || c->cfgd.lowpass) {  // A/B binning path, SGS_FLAG_LOWPASS: the unfused sequence
        int r = sgs_render(c, sf, cam, out, stream);
        if (r != SGS_OK) return r;
        r = sgs_backward_tracking(c, target, lambda_d, normal_sign, d_pose6, loss, stream);
        c->have_forward = false;
        return r;
    }
    if ((c->cfg.flags & SGS_FLAG_TRACK_REUSE) && sf && sgs_cam_valid(cam)) {
        if (!c->surv_cnt && !(c->surv_cnt = (unsigned int*)sgs_ws_alloc(c, sizeof(unsigned int), s))) return SGS_OUT_OF_MEMORY;
        if (c->surv_in_cap < sf->n) {  // 52 B per splat of the map at most; every survivor list fits
            if (c->surv_in) sgs_ws_free(c, c->surv_in, s);
            c->surv_in_cap = 0; c->surv_valid = false;
            if (!(c->surv_in = sgs_ws_alloc(c, 52 * (size_t)sf->n + 64, s))) return SGS_OUT_OF_MEMORY;
            c->surv_in_cap = sf->n;
        }
        // (device-resident pose: the host cannot check the margin; K-pre-B does and the iteration turns NaN, see sgs_track_iter_dev)
        if (c->surv_valid && !(memcmp(&c->surv_sf, sf, sizeof(*sf)) == 0 && (c->pose_dev != nullptr || pose_within_margin(&c->surv_cam, cam))))
            c->surv_valid = false;  // another map, or the pose has left the list's margin: build it again, centred here
        c->use_surv_cache = true;
    }
    // capture mode with a kept list: the longest-first tile order is renewed by the first iteration of a frame only (it sits on
    // the iteration's chain there: no side stream); the order is a scheduling hint, results do not depend on it
    c->order_skip = graph_mode(c) && (c->cfg.flags & SGS_FLAG_TRACK_REUSE) && c->surv_valid;
    c->defer_counters = true;  // (bin_buckets clears it when it cannot honour it)
    c->track_binning = true;
    int r = bin_view(c, sf, cam, false, s);
    c->track_binning = false;
    c->use_surv_cache = false;
    const bool deferred = c->defer_counters;
    c->defer_counters = false;
    if (r != SGS_OK) return r;
    const int tiles = c->camd.tiles_x * c->camd.tiles_y;
    if ((r = sgs_ensure_partials(c, (int64_t)tiles + SGS_TRACK_HELPERS, s)) != SGS_OK) return r;  // K-track: one row per block, helpers included
    float* planes[8];
    pick_planes(c, out, (int64_t)cam->width * cam->height, false, planes);
    if (deferred && c->prev_copy_on_aux) {  // the slot this K-track overwrites was copied two iterations ago: done long since
        if (cudaStreamWaitEvent(s, c->counters_ready_prev, 0) != cudaSuccess) return SGS_CUDA_ERROR;
        c->prev_copy_on_aux = false;
    }
    if (sgs_launch_track(c, planes, target->rgb, target->depth, lambda_d, normal_sign, d_pose6, loss, deferred, s) != cudaSuccess)
        return SGS_CUDA_ERROR;
    if (deferred) {  // the counters of this iteration's preprocess, snapshotted by k_track's last block
        // ... copied on the ctx's own stream: a copy between K-track and the next iteration's K-pre-B is a link of the
        // iteration's dependency chain (measured on C2: 82.3 -> 72.2 us per iteration).  Two snapshot slots alternate, and
        // an iteration waits for the copy of the slot it is about to overwrite, which is one iteration old.
        c->stats_src = c->counters_snap + c->snap_slot;
        if (graph_mode(c)) { c->have_binning = true; return SGS_OK; }  // (one slot, one stream; no copy on the iteration's chain)
        cudaStream_t cs = c->aux_stream ? c->aux_stream : s;
        if (cs != s && (cudaEventRecord(c->fork_ev, s) != cudaSuccess || cudaStreamWaitEvent(cs, c->fork_ev, 0) != cudaSuccess))
            return SGS_CUDA_ERROR;
        if (cudaMemcpyAsync(c->counters_host, c->counters_snap + c->snap_slot, sizeof(SgsCounters), cudaMemcpyDeviceToHost, cs) != cudaSuccess)
            return SGS_CUDA_ERROR;
        const cudaEvent_t t = c->counters_ready_prev; c->counters_ready_prev = c->counters_ready; c->counters_ready = t;
        c->prev_copy_on_aux = c->snap_copy_on_aux;
        cudaEventRecord(c->counters_ready, cs);
        c->snap_copy_on_aux = cs != s;
        c->snap_slot ^= 1;
        c->pending_check = true;
        c->pending_lazy = true;
    }
    c->have_binning = true;
    return SGS_OK;
}

int sgs_track_iter_dev(sgs_ctx* c, const sgs_surfels* sf, const sgs_camera* cam, const float* d_T_cw, const sgs_images* target,
                       float lambda_d, float normal_sign, const sgs_images* out, float* d_pose6, float* loss, void* stream) {
    if (!c || !d_T_cw || radix_mode(c) || c->cfgd.lowpass) return SGS_INVALID_ARGUMENT;
    c->pose_dev = d_T_cw;
    const int r = sgs_track_iter(c, sf, cam, target, lambda_d, normal_sign, out, d_pose6, loss, stream);
    c->pose_dev = nullptr;
    return r;
}

int sgs_track_new_frame(sgs_ctx* c) {
    if (!c) return SGS_INVALID_ARGUMENT;
    c->surv_valid = false;
    return SGS_OK;
}

static int backward_impl(sgs_ctx* c, const sgs_images* upstream, const sgs_surfel_grads* dg, float* d_pose6, bool accumulate,
                         void* stream) {
    if (!c) return SGS_INVALID_ARGUMENT;
    cudaStream_t s = (cudaStream_t)stream;
    int r = check_pending(c, s);
    if (r != SGS_OK) return r;
    if (!c->have_forward) return SGS_NO_FORWARD_STATE;
    const int tiles = c->camd.tiles_x * c->camd.tiles_y;
    const int64_t pixels = (int64_t)c->camd.W * c->camd.H;
    int64_t blocks = (c->last_surfels.n + 255) / 256;
    if (blocks < tiles) blocks = tiles;
    if ((r = sgs_ensure_partials(c, blocks, s)) != SGS_OK) return r;
    const float* up[8] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    if (upstream) {
        if (upstream->rgb) for (int i = 0; i < 3; ++i) up[i] = upstream->rgb + (size_t)i * pixels;
        if (upstream->depth) up[3] = upstream->depth;
        if (upstream->normal) for (int i = 0; i < 3; ++i) up[4 + i] = upstream->normal + (size_t)i * pixels;
        if (upstream->alpha) up[7] = upstream->alpha;
    }
    c->grads_on_aux = false;
    if (sgs_launch_backward(c, up, dg, d_pose6, accumulate, s) != cudaSuccess) return SGS_CUDA_ERROR;
    c->work_recorded = !graph_mode(c) && cudaEventRecord(c->work_ev, c->grads_on_aux ? c->aux_stream : s) == cudaSuccess;
    return SGS_OK;
}

int sgs_backward(sgs_ctx* c, const sgs_images* upstream, const sgs_surfel_grads* dg, float* d_pose6, void* stream) {
    return backward_impl(c, upstream, dg, d_pose6, false, stream);
}

int sgs_backward_accumulate(sgs_ctx* c, const sgs_images* upstream, const sgs_surfel_grads* dg, float* d_pose6, void* stream) {
    if (!dg) return SGS_INVALID_ARGUMENT;
    return backward_impl(c, upstream, dg, d_pose6, true, stream);
}

int sgs_zero_grads(sgs_ctx* c, const sgs_surfel_grads* dg, int64_t n, void* stream) {
    if (!c || !dg || n < 0) return SGS_INVALID_ARGUMENT;
    cudaStream_t s = (cudaStream_t)stream;
    const size_t m = (size_t)n;
    bool ok = true;
    if (dg->mean) ok = ok && cudaMemsetAsync(dg->mean, 0, sizeof(float) * 3 * m, s) == cudaSuccess;
    if (dg->scale) ok = ok && cudaMemsetAsync(dg->scale, 0, sizeof(float) * 2 * m, s) == cudaSuccess;
    if (dg->quat) ok = ok && cudaMemsetAsync(dg->quat, 0, sizeof(float) * 4 * m, s) == cudaSuccess;
    if (dg->opacity) ok = ok && cudaMemsetAsync(dg->opacity, 0, sizeof(float) * m, s) == cudaSuccess;
    if (dg->rgb) ok = ok && cudaMemsetAsync(dg->rgb, 0, sizeof(float) * 3 * m, s) == cudaSuccess;
    return ok ? SGS_OK : SGS_CUDA_ERROR;
}

int sgs_wait_grads(sgs_ctx* c, void* stream) {
    if (!c) return SGS_INVALID_ARGUMENT;
    if (c->grads_on_aux && c->work_recorded && cudaStreamWaitEvent((cudaStream_t)stream, c->work_ev, 0) != cudaSuccess)
        return SGS_CUDA_ERROR;
    return SGS_OK;
}

int sgs_backward_tracking(sgs_ctx* c, const sgs_images* target, float lambda_d, float normal_sign, float* d_pose6,
                          float* loss, void* stream) {
    if (!c || !target || !target->rgb || !target->depth || !d_pose6) return SGS_INVALID_ARGUMENT;
    cudaStream_t s = (cudaStream_t)stream;
    int r = check_pending(c, s);
    if (r != SGS_OK) return r;
    if (!c->have_forward) return SGS_NO_FORWARD_STATE;
    if ((r = sgs_ensure_partials(c, c->camd.tiles_x * c->camd.tiles_y, s)) != SGS_OK) return r;
    if (sgs_launch_backward_tracking(c, target->rgb, target->depth, lambda_d, normal_sign, d_pose6, loss, s) != cudaSuccess)
        return SGS_CUDA_ERROR;
    return SGS_OK;
}

int sgs_tracking_loss(sgs_ctx* c, const sgs_camera* cam, const sgs_images* ren, const sgs_images* target, float lambda_d,
                      float normal_sign, const sgs_images* upstream, float* loss, void* stream) {
    if (!c || !sgs_cam_valid(cam) || !ren || !target || !upstream) return SGS_INVALID_ARGUMENT;
    if (!ren->rgb || !ren->depth || !ren->normal || !ren->alpha || !target->rgb || !target->depth)
        return SGS_INVALID_ARGUMENT;
    const int64_t pixels = (int64_t)cam->width * cam->height;
    const float* rp[8];
    float* upp[8];
    for (int i = 0; i < 3; ++i) {
        rp[i] = ren->rgb + (size_t)i * pixels;
        rp[4 + i] = ren->normal + (size_t)i * pixels;
        upp[i] = upstream->rgb ? upstream->rgb + (size_t)i * pixels : nullptr;
        upp[4 + i] = upstream->normal ? upstream->normal + (size_t)i * pixels : nullptr;
    }
    rp[3] = ren->depth; rp[7] = ren->alpha; upp[3] = upstream->depth; upp[7] = upstream->alpha;
    if (sgs_launch_tracking_loss(c, cam, rp, target->rgb, target->depth, lambda_d, normal_sign, upp, loss,
                                 (cudaStream_t)stream) != cudaSuccess)
        return SGS_CUDA_ERROR;
    return SGS_OK;
}

int sgs_mapping_loss(sgs_ctx* c, const sgs_camera* cam, const sgs_images* ren, const sgs_images* target, float lambda_c,
                     float w_d, float w_n, float normal_sign, const sgs_images* upstream, float* loss, void* stream) {
    if (!c || !sgs_cam_valid(cam) || !ren || !target || !upstream) return SGS_INVALID_ARGUMENT;
    if (!ren->rgb || !ren->depth || !ren->normal || !target->rgb || !target->depth) return SGS_INVALID_ARGUMENT;
    const int64_t pixels = (int64_t)cam->width * cam->height;
    const float* rp[8];
    float* upp[8];
    for (int i = 0; i < 3; ++i) {
        rp[i] = ren->rgb + (size_t)i * pixels;
        rp[4 + i] = ren->normal + (size_t)i * pixels;
        upp[i] = upstream->rgb ? upstream->rgb + (size_t)i * pixels : nullptr;
        upp[4 + i] = upstream->normal ? upstream->normal + (size_t)i * pixels : nullptr;
    }
    rp[3] = ren->depth; rp[7] = ren->alpha; upp[3] = upstream->depth; upp[7] = upstream->alpha;
    return sgs_launch_mapping_loss(c, cam, rp, target->rgb, target->depth, lambda_c, w_d, w_n, normal_sign, upp, loss,
                                   (cudaStream_t)stream) == cudaSuccess ? SGS_OK : SGS_CUDA_ERROR;
}

int sgs_ssim_loss(sgs_ctx* c, int width, int height, const float* rendered_rgb, const float* target_rgb, float weight,
                  float* upstream_rgb, float* loss, void* stream) {
    if (!c || width <= 0 || height <= 0 || !rendered_rgb || !target_rgb || !upstream_rgb) return SGS_INVALID_ARGUMENT;
    return sgs_launch_ssim_loss(c, width, height, rendered_rgb, target_rgb, weight, upstream_rgb, loss,
                                (cudaStream_t)stream) == cudaSuccess ? SGS_OK : SGS_CUDA_ERROR;
}

int sgs_map_correction(sgs_ctx* c, int64_t n, float* mean, float* quat, const int32_t* frame_id, int n_frames,
                       const float* T_orig, const float* T_opt, void* stream) {
    if (!c || n < 0 || n_frames < 0) return SGS_INVALID_ARGUMENT;
    if (n > 0 && (!mean || !quat || !frame_id || (n_frames > 0 && (!T_orig || !T_opt)))) return SGS_INVALID_ARGUMENT;
    if (reinterpret_cast<uintptr_t>(quat) & 15u) return SGS_INVALID_ARGUMENT;
    return sgs_launch_map_correction(c, n, mean, quat, frame_id, n_frames, T_orig, T_opt, (cudaStream_t)stream) == cudaSuccess
               ? SGS_OK : SGS_CUDA_ERROR;
}

int sgs_measure_fp32_peak(double* tflops, void* stream) {
    if (!tflops) return SGS_INVALID_ARGUMENT;
    return sgs_launch_fma_peak(tflops, (cudaStream_t)stream) == cudaSuccess ? SGS_OK : SGS_CUDA_ERROR;
}

int sgs_get_binning(sgs_ctx* c, int64_t* n_entries, const uint64_t** keys, const uint32_t** idx,
                    const uint32_t** tile_ranges, const uint8_t** culled) {
    if (!c) return SGS_INVALID_ARGUMENT;
    int r = check_pending(c, 0);
    if (r != SGS_OK) return r;
    if (!c->have_binning) return SGS_NO_FORWARD_STATE;
    if (cudaDeviceSynchronize() != cudaSuccess) return SGS_CUDA_ERROR;
    const int64_t E = (int64_t)c->counters_host->n_entries;
    if (n_entries) *n_entries = E;
    if (culled) *culled = c->culled;
    if (!radix_mode(c)) {
        const int tiles = c->camd.tiles_x * c->camd.tiles_y;
        if ((r = sgs_ensure_export(c, tiles, E, 0)) != SGS_OK) return r;
        if (sgs_launch_export_bucket(c, E, 0) != cudaSuccess || cudaDeviceSynchronize() != cudaSuccess) return SGS_CUDA_ERROR;
        if (keys) *keys = c->export_keys;
        if (idx) *idx = c->idx_export;
        if (tile_ranges) *tile_ranges = c->export_ranges;
        return SGS_OK;
    }
    if (sgs_launch_export_idx(c, 0) != cudaSuccess || cudaDeviceSynchronize() != cudaSuccess) return SGS_CUDA_ERROR;
    if (keys) *keys = c->keys[c->sorted_buf];
    if (idx) *idx = c->idx_export;
    if (tile_ranges) *tile_ranges = c->ranges;
    return SGS_OK;
}

int sgs_get_stats(sgs_ctx* c, sgs_stats* out) {
    if (!c || !out) return SGS_INVALID_ARGUMENT;
    if (graph_mode(c)) {
        if (cudaDeviceSynchronize() != cudaSuccess) return SGS_CUDA_ERROR;
        if (c->stats_src && cudaMemcpy(c->counters_host, c->stats_src, sizeof(SgsCounters), cudaMemcpyDeviceToHost) != cudaSuccess) return SGS_CUDA_ERROR;
    }
    else if (c->pending_check && cudaEventSynchronize(c->counters_ready) != cudaSuccess) return SGS_CUDA_ERROR;
    out->n_visible = c->counters_host->n_visible;
    out->n_entries = (int64_t)c->counters_host->n_entries;
    out->capacity = radix_mode(c) ? c->e_cap : c->tile_cap;
    out->overflow = radix_mode(c) ? c->counters_host->overflow : (c->counters_host->max_tile > (unsigned)c->tile_cap);
    out->workspace_bytes = c->bytes;
    out->kernel_launches = c->launches;
    return SGS_OK;
}

}  // extern "C"
