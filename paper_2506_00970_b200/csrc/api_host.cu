// api_host.cu -- HOST-buffer entry points of include/sgs.h (end-to-end path: copies in, runs the
// device path, copies out, waits).  No arithmetic here.
#include <string.h>
#include "sgs_internal.h"

template <typename T>
static bool grow(sgs_ctx* c, T*& p, int64_t& cap, int64_t need, cudaStream_t s) {
    if (need <= cap) return true;
    cudaStreamSynchronize(s);
    sgs_ws_free(c, p, s);
    p = (T*)sgs_ws_alloc(c, (size_t)need * sizeof(T), s);
    cap = p ? need : 0;
    return p != nullptr;
}

static int ensure_host_images(sgs_ctx* c, int64_t pixels, cudaStream_t s) {
    int64_t cap2 = c->host_img_cap;
    if (!grow(c, c->host_img_dev, c->host_img_cap, pixels * 8, s)) return SGS_OUT_OF_MEMORY;
    if (!grow(c, c->host_up_dev, cap2, pixels * 8, s)) return SGS_OUT_OF_MEMORY;
    return SGS_OK;
}

static void dev_images(float* base, int64_t pixels, sgs_images* im) {
    im->rgb = base; im->depth = base + 3 * pixels; im->normal = base + 4 * pixels; im->alpha = base + 7 * pixels;
}

// sgs_fetch_grads_sparse_host, second half: once the pack kernel of the last sparse fetch has run, the row count sits in
// mapped memory and the copy commands of exactly that many rows can be enqueued (on the ctx's copy stream, behind the pack).
// wait == false: only if the pack is already complete (called from the window calls that follow the fetch).
static int flush_sparse(sgs_ctx* c, bool wait) {
    if (!c->win_sp.pending) return SGS_OK;
    if (!wait) {
        const cudaError_t q = cudaEventQuery(c->win_packed);
        if (q == cudaErrorNotReady) return SGS_OK;
        if (q != cudaSuccess) return SGS_CUDA_ERROR;
    } else if (cudaEventSynchronize(c->win_packed) != cudaSuccess) return SGS_CUDA_ERROR;
    c->win_sp.pending = false;
    const int64_t n = c->win_sp.n;
    int64_t rows = (int64_t)c->win_counts[c->win_sp.ring];
    if (rows > c->win_sp.cap) rows = c->win_sp.cap;
    if (rows <= 0) return SGS_OK;
    const float* st = reinterpret_cast<const float*>(c->win_stage);
    cudaStream_t cs = c->copy_stream;
    const sgs_surfel_grads& h = c->win_sp.rows;
    const size_t r4 = sizeof(float) * (size_t)rows;
    bool ok = true;
    if (c->win_sp.ids) ok = ok && cudaMemcpyAsync(c->win_sp.ids, st, r4, cudaMemcpyDeviceToHost, cs) == cudaSuccess;
    if (h.mean) ok = ok && cudaMemcpyAsync(h.mean, st + n, 3 * r4, cudaMemcpyDeviceToHost, cs) == cudaSuccess;
    if (h.scale) ok = ok && cudaMemcpyAsync(h.scale, st + 4 * n, 2 * r4, cudaMemcpyDeviceToHost, cs) == cudaSuccess;
    if (h.quat) ok = ok && cudaMemcpyAsync(h.quat, st + 6 * n, 4 * r4, cudaMemcpyDeviceToHost, cs) == cudaSuccess;
    if (h.opacity) ok = ok && cudaMemcpyAsync(h.opacity, st + 10 * n, r4, cudaMemcpyDeviceToHost, cs) == cudaSuccess;
    if (h.rgb) ok = ok && cudaMemcpyAsync(h.rgb, st + 11 * n, 3 * r4, cudaMemcpyDeviceToHost, cs) == cudaSuccess;
    return ok ? SGS_OK : SGS_CUDA_ERROR;
}

extern "C" {

int sgs_upload_surfels(sgs_ctx* c, const sgs_surfels* h, void* stream) {
    if (!c || !h || h->n < 0 || (h->n > 0 && (!h->mean || !h->scale || !h->quat || !h->opacity || !h->rgb)))
        return SGS_INVALID_ARGUMENT;
    cudaStream_t s = (cudaStream_t)stream;
    const int64_t n = h->n;
    c->surv_valid = false;  // SGS_FLAG_TRACK_REUSE: the resident map is being rewritten
    if (n > c->resident_cap) {
        cudaStreamSynchronize(s);
        sgs_ws_free(c, c->resident_store, s);
        sgs_ws_free(c, c->resident_active, s);
        c->resident_store = (float*)sgs_ws_alloc(c, (size_t)n * 13 * sizeof(float), s);
        c->resident_active = (uint8_t*)sgs_ws_alloc(c, (size_t)n, s);
        if (!c->resident_store || !c->resident_active) { c->resident_cap = 0; return SGS_OUT_OF_MEMORY; }
        c->resident_cap = n;
    }
    float* b = c->resident_store;
    float* d_mean = b; float* d_scale = b + 3 * n; float* d_quat = b + 5 * n; float* d_op = b + 9 * n; float* d_rgb = b + 10 * n;
    bool ok = cudaMemcpyAsync(d_mean, h->mean, sizeof(float) * 3 * n, cudaMemcpyHostToDevice, s) == cudaSuccess &&
              cudaMemcpyAsync(d_scale, h->scale, sizeof(float) * 2 * n, cudaMemcpyHostToDevice, s) == cudaSuccess &&
              cudaMemcpyAsync(d_quat, h->quat, sizeof(float) * 4 * n, cudaMemcpyHostToDevice, s) == cudaSuccess &&
              cudaMemcpyAsync(d_op, h->opacity, sizeof(float) * n, cudaMemcpyHostToDevice, s) == cudaSuccess &&
              cudaMemcpyAsync(d_rgb, h->rgb, sizeof(float) * 3 * n, cudaMemcpyHostToDevice, s) == cudaSuccess;
    if (ok && h->active) ok = cudaMemcpyAsync(c->resident_active, h->active, (size_t)n, cudaMemcpyHostToDevice, s) == cudaSuccess;
    if (!ok) return SGS_CUDA_ERROR;
    c->resident.n = n; c->resident.mean = d_mean; c->resident.scale = d_scale; c->resident.quat = d_quat;
    c->resident.opacity = d_op; c->resident.rgb = d_rgb; c->resident.active = h->active ? c->resident_active : nullptr;
    return SGS_OK;
}

int sgs_render_host(sgs_ctx* c, const sgs_camera* cam, const sgs_images* ho, void* stream) {
    if (!c || !sgs_cam_valid(cam) || !ho) return SGS_INVALID_ARGUMENT;
    if (!c->resident.mean && c->resident.n != 0) return SGS_NO_FORWARD_STATE;
    cudaStream_t s = (cudaStream_t)stream;
    const int64_t px = (int64_t)cam->width * cam->height;
    int r = ensure_host_images(c, px, s);
    if (r != SGS_OK) return r;
    sgs_images d;
    dev_images(c->host_img_dev, px, &d);
    if ((r = sgs_render(c, &c->resident, cam, &d, stream)) != SGS_OK) return r;
    bool ok = true;
    if (ho->rgb) ok = ok && cudaMemcpyAsync(ho->rgb, d.rgb, sizeof(float) * 3 * px, cudaMemcpyDeviceToHost, s) == cudaSuccess;
    if (ho->depth) ok = ok && cudaMemcpyAsync(ho->depth, d.depth, sizeof(float) * px, cudaMemcpyDeviceToHost, s) == cudaSuccess;
    if (ho->normal) ok = ok && cudaMemcpyAsync(ho->normal, d.normal, sizeof(float) * 3 * px, cudaMemcpyDeviceToHost, s) == cudaSuccess;
    if (ho->alpha) ok = ok && cudaMemcpyAsync(ho->alpha, d.alpha, sizeof(float) * px, cudaMemcpyDeviceToHost, s) == cudaSuccess;
    if (!ok || cudaStreamSynchronize(s) != cudaSuccess) return SGS_CUDA_ERROR;
    return SGS_OK;
}

int sgs_backward_host(sgs_ctx* c, const sgs_images* hu, const sgs_surfel_grads* hg, float* h_pose6, void* stream) {
    if (!c || !hu) return SGS_INVALID_ARGUMENT;
    if (!c->have_forward) return SGS_NO_FORWARD_STATE;
    cudaStream_t s = (cudaStream_t)stream;
    const int64_t px = (int64_t)c->camd.W * c->camd.H, n = c->last_surfels.n;
    int r = ensure_host_images(c, px, s);
    if (r != SGS_OK) return r;
    sgs_images d;
    dev_images(c->host_up_dev, px, &d);
    sgs_images du = {nullptr, nullptr, nullptr, nullptr};
    bool ok = true;
    if (hu->rgb) { ok = ok && cudaMemcpyAsync(d.rgb, hu->rgb, sizeof(float) * 3 * px, cudaMemcpyHostToDevice, s) == cudaSuccess; du.rgb = d.rgb; }
    if (hu->depth) { ok = ok && cudaMemcpyAsync(d.depth, hu->depth, sizeof(float) * px, cudaMemcpyHostToDevice, s) == cudaSuccess; du.depth = d.depth; }
    if (hu->normal) { ok = ok && cudaMemcpyAsync(d.normal, hu->normal, sizeof(float) * 3 * px, cudaMemcpyHostToDevice, s) == cudaSuccess; du.normal = d.normal; }
    if (hu->alpha) { ok = ok && cudaMemcpyAsync(d.alpha, hu->alpha, sizeof(float) * px, cudaMemcpyHostToDevice, s) == cudaSuccess; du.alpha = d.alpha; }
    if (!ok) return SGS_CUDA_ERROR;
    sgs_surfel_grads dg;
    if (hg) {
        if (!grow(c, c->host_grads_dev, c->host_grads_cap, n * 13 + 16, s)) return SGS_OUT_OF_MEMORY;
        float* b = c->host_grads_dev;
        dg.mean = b; dg.scale = b + 3 * n; dg.quat = b + 5 * n; dg.opacity = b + 9 * n; dg.rgb = b + 10 * n;
    }
    if ((r = sgs_backward(c, &du, hg ? &dg : nullptr, h_pose6 ? c->pose6_dev : nullptr, stream)) != SGS_OK) return r;
    if ((r = sgs_wait_grads(c, stream)) != SGS_OK) return r;  // SGS_FLAG_LAZY_GRADS: the copies below need the last kernel
    if (hg) {
        if (hg->mean) ok = ok && cudaMemcpyAsync(hg->mean, dg.mean, sizeof(float) * 3 * n, cudaMemcpyDeviceToHost, s) == cudaSuccess;
        if (hg->scale) ok = ok && cudaMemcpyAsync(hg->scale, dg.scale, sizeof(float) * 2 * n, cudaMemcpyDeviceToHost, s) == cudaSuccess;
        if (hg->quat) ok = ok && cudaMemcpyAsync(hg->quat, dg.quat, sizeof(float) * 4 * n, cudaMemcpyDeviceToHost, s) == cudaSuccess;
        if (hg->opacity) ok = ok && cudaMemcpyAsync(hg->opacity, dg.opacity, sizeof(float) * n, cudaMemcpyDeviceToHost, s) == cudaSuccess;
        if (hg->rgb) ok = ok && cudaMemcpyAsync(hg->rgb, dg.rgb, sizeof(float) * 3 * n, cudaMemcpyDeviceToHost, s) == cudaSuccess;
    }
    if (h_pose6) ok = ok && cudaMemcpyAsync(c->pinned_small, c->pose6_dev, sizeof(float) * 6, cudaMemcpyDeviceToHost, s) == cudaSuccess;
    if (!ok || cudaStreamSynchronize(s) != cudaSuccess) return SGS_CUDA_ERROR;
    if (h_pose6) memcpy(h_pose6, c->pinned_small, sizeof(float) * 6);
    return SGS_OK;
}

int sgs_upload_target(sgs_ctx* c, const sgs_camera* cam, const float* h_rgb, const float* h_depth, void* stream) {
    if (!c || !sgs_cam_valid(cam) || !h_rgb || !h_depth) return SGS_INVALID_ARGUMENT;
    cudaStream_t s = (cudaStream_t)stream;
    const int64_t px = (int64_t)cam->width * cam->height;
    if (!grow(c, c->target_rgb, c->target_cap, px * 4, s)) return SGS_OUT_OF_MEMORY;
    c->target_depth = c->target_rgb + 3 * px;
    if (cudaMemcpyAsync(c->target_rgb, h_rgb, sizeof(float) * 3 * px, cudaMemcpyHostToDevice, s) != cudaSuccess ||
        cudaMemcpyAsync(c->target_depth, h_depth, sizeof(float) * px, cudaMemcpyHostToDevice, s) != cudaSuccess)
        return SGS_CUDA_ERROR;
    return SGS_OK;
}

int sgs_track_iter_host(sgs_ctx* c, const sgs_camera* cam, float lambda_d, float normal_sign, float* h_loss,
                        float* h_pose6, void* stream) {
    if (!c || !sgs_cam_valid(cam)) return SGS_INVALID_ARGUMENT;
    const int64_t px = (int64_t)cam->width * cam->height;
    if (!c->target_rgb || c->target_cap < px * 4 || (!c->resident.mean && c->resident.n != 0)) return SGS_NO_FORWARD_STATE;
    cudaStream_t s = (cudaStream_t)stream;
    int r = ensure_host_images(c, px, s);
    if (r != SGS_OK) return r;
    sgs_images ren, tgt = {c->target_rgb, c->target_depth, nullptr, nullptr};
    dev_images(c->host_img_dev, px, &ren);
    // Results through pinned host memory the kernel writes itself (6 + 1 floats, then a flag word the host polls): a
    // device-to-host copy and a stream synchronisation cost about 20 us of every iteration's turnaround.
    const unsigned int want = ++c->host_flag_val;
    *c->host_flag = want - 1u;
    c->host_flag_want = true;
    c->host_flag_armed = false;
    r = sgs_track_iter(c, &c->resident, cam, &tgt, lambda_d, normal_sign, &ren, c->pinned_small_dev + 1, c->pinned_small_dev, stream);
    c->host_flag_want = false;
    if (r != SGS_OK) return r;
    bool got = false;
    if (c->host_flag_armed) {
        volatile unsigned int* f = c->host_flag;
        for (unsigned long long spin = 0; !got; ++spin) {
            if (*f == want) { got = true; break; }
            if ((spin & 0xffffu) == 0xffffu) {  // every 65 k polls: has the stream finished (or failed) without the flag?
                const cudaError_t q = cudaStreamQuery(s);
                if (q == cudaSuccess) { got = (*f == want); break; }
                if (q != cudaErrorNotReady) return SGS_CUDA_ERROR;
            }
        }
    }
    if (!got && cudaStreamSynchronize(s) != cudaSuccess) return SGS_CUDA_ERROR;  // paths without the fused kernel (radix binning)
    if (h_loss) *h_loss = c->pinned_small[0];
    if (h_pose6) memcpy(h_pose6, c->pinned_small + 1, sizeof(float) * 6);
    return SGS_OK;
}


// ---- mapping window on the resident map (an iteration optimises over N_a + N_i views) ----
static int window_setup(sgs_ctx* c, int64_t n, cudaStream_t s) {
    if (!c->copy_stream) {
        if (cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking) != cudaSuccess ||
            cudaEventCreateWithFlags(&c->win_filled, cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&c->win_drained[0], cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&c->win_drained[1], cudaEventDisableTiming) != cudaSuccess ||
            cudaHostAlloc(&c->win_results, sizeof(float) * 8 * SGS_WIN_RING, cudaHostAllocMapped) != cudaSuccess ||
            cudaHostGetDevicePointer(&c->win_results_dev, c->win_results, 0) != cudaSuccess ||
            cudaHostAlloc(&c->win_counts, sizeof(uint32_t) * SGS_WIN_RING, cudaHostAllocMapped) != cudaSuccess ||
            cudaHostGetDevicePointer(&c->win_counts_dev, c->win_counts, 0) != cudaSuccess ||
            cudaEventCreateWithFlags(&c->win_packed, cudaEventDisableTiming) != cudaSuccess ||
            cudaStreamCreateWithFlags(&c->in_stream, cudaStreamNonBlocking) != cudaSuccess ||
            cudaEventCreateWithFlags(&c->win_tgt_ready[0], cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&c->win_tgt_ready[1], cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&c->win_tgt_free[0], cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&c->win_tgt_free[1], cudaEventDisableTiming) != cudaSuccess)
            return SGS_CUDA_ERROR;
    }
    for (int k = 0; k < 2; ++k) {
        if (c->win_cap[k] >= n * 13 + 16) continue;
        if (c->win_draining[k]) { cudaEventSynchronize(c->win_drained[k]); c->win_draining[k] = false; }
        if (!grow(c, c->win_grads[k], c->win_cap[k], n * 13 + 16, s)) return SGS_OUT_OF_MEMORY;
        if (cudaMemsetAsync(c->win_grads[k], 0, sizeof(float) * (size_t)(n * 13 + 16), s) != cudaSuccess) return SGS_CUDA_ERROR;
    }
    return SGS_OK;
}

static void window_grads(sgs_ctx* c, int slot, int64_t n, sgs_surfel_grads* dg) {
    float* b = c->win_grads[slot];
    dg->mean = b; dg->scale = b + 3 * n; dg->quat = b + 5 * n; dg->opacity = b + 9 * n; dg->rgb = b + 10 * n;
}

int sgs_map_view_host(sgs_ctx* c, const sgs_camera* cam, const float* h_rgb, const float* h_depth, float lambda_c, float w_d,
                      float w_n, float ssim_weight, float normal_sign, float* h_loss, float* h_pose6, void* stream) {
    if (!c || !sgs_cam_valid(cam) || !h_rgb || !h_depth) return SGS_INVALID_ARGUMENT;
    if (!c->resident.mean && c->resident.n != 0) return SGS_NO_FORWARD_STATE;
    if (c->win_n_pending >= SGS_WIN_RING) return SGS_INVALID_ARGUMENT;  // call sgs_sync_host first
    cudaStream_t s = (cudaStream_t)stream;
    const int64_t px = (int64_t)cam->width * cam->height, n = c->resident.n;
    int r = ensure_host_images(c, px, s);
    if (r != SGS_OK) return r;
    if ((r = window_setup(c, n, s)) != SGS_OK) return r;
    if ((r = flush_sparse(c, false)) != SGS_OK) return r;
    // keyframe: host -> one of two device buffers on the ctx's upload stream (runs under the previous view's kernels; the
    // buffer's previous user, two views ago, has recorded win_tgt_free behind its last reader)
    const int ts = c->win_tgt_slot;
    c->win_tgt_slot ^= 1;
    if (c->win_tgt_cap[ts] < px * 4) {
        if (c->win_tgt_used[ts]) { cudaEventSynchronize(c->win_tgt_free[ts]); c->win_tgt_used[ts] = false; }
        if (!grow(c, c->win_tgt[ts], c->win_tgt_cap[ts], px * 4, s)) return SGS_OUT_OF_MEMORY;
    }
    if (c->win_tgt_used[ts] && cudaStreamWaitEvent(c->in_stream, c->win_tgt_free[ts], 0) != cudaSuccess) return SGS_CUDA_ERROR;
    float* t_rgb = c->win_tgt[ts]; float* t_depth = t_rgb + 3 * px;
    if (cudaMemcpyAsync(t_rgb, h_rgb, sizeof(float) * 3 * px, cudaMemcpyHostToDevice, c->in_stream) != cudaSuccess ||
        cudaMemcpyAsync(t_depth, h_depth, sizeof(float) * px, cudaMemcpyHostToDevice, c->in_stream) != cudaSuccess ||
        cudaEventRecord(c->win_tgt_ready[ts], c->in_stream) != cudaSuccess)
        return SGS_CUDA_ERROR;
    const int slot = c->win_slot;
    if (c->win_draining[slot]) {  // the copy-out (and re-zeroing) of this accumulator, two windows ago, must be complete
        if (cudaStreamWaitEvent(s, c->win_drained[slot], 0) != cudaSuccess) return SGS_CUDA_ERROR;
        c->win_draining[slot] = false;
    }
    sgs_images ren, up, tgt = {t_rgb, t_depth, nullptr, nullptr};
    dev_images(c->host_img_dev, px, &ren);
    dev_images(c->host_up_dev, px, &up);
    if ((r = sgs_render(c, &c->resident, cam, &ren, stream)) != SGS_OK) return r;
    if (cudaStreamWaitEvent(s, c->win_tgt_ready[ts], 0) != cudaSuccess) return SGS_CUDA_ERROR;
    float* res = c->win_results_dev + 8 * c->win_n_pending;  // (mapped host memory; this view's loss and pose gradient land here)
    if (cudaMemsetAsync(c->loss_dev, 0, sizeof(float), s) != cudaSuccess) return SGS_CUDA_ERROR;
    if ((r = sgs_mapping_loss(c, cam, &ren, &tgt, lambda_c, w_d, w_n, normal_sign, &up, c->loss_dev, stream)) != SGS_OK) return r;
    if (ssim_weight != 0.f &&
        (r = sgs_ssim_loss(c, cam->width, cam->height, ren.rgb, tgt.rgb, ssim_weight, up.rgb, c->loss_dev, stream)) != SGS_OK)
        return r;
    sgs_surfel_grads dg;
    window_grads(c, slot, n, &dg);
    if (cudaEventRecord(c->win_tgt_free[ts], s) != cudaSuccess) return SGS_CUDA_ERROR;   // (the losses were its last readers)
    c->win_tgt_used[ts] = true;
    if ((r = sgs_backward_accumulate(c, &up, &dg, c->pose6_dev, stream)) != SGS_OK) return r;
    if ((r = sgs_wait_grads(c, stream)) != SGS_OK) return r;
    c->win_dirty = true;
    if (sgs_launch_publish(res, c->loss_dev, 7, s) != cudaSuccess) return SGS_CUDA_ERROR;
    c->launches += 1;
    c->win_pending[c->win_n_pending].loss = h_loss;
    c->win_pending[c->win_n_pending].pose6 = h_pose6;
    c->win_n_pending += 1;
    return flush_sparse(c, false);
}

int sgs_fetch_grads_host(sgs_ctx* c, const sgs_surfel_grads* hg, void* stream) {
    if (!c || !hg) return SGS_INVALID_ARGUMENT;
    if (!c->copy_stream || !c->win_grads[c->win_slot]) return SGS_NO_FORWARD_STATE;
    if (flush_sparse(c, true) != SGS_OK) return SGS_CUDA_ERROR;
    cudaStream_t s = (cudaStream_t)stream, cs = c->copy_stream;
    const int64_t n = c->resident.n;
    const int slot = c->win_slot;
    sgs_surfel_grads dg;
    window_grads(c, slot, n, &dg);
    bool ok = cudaEventRecord(c->win_filled, s) == cudaSuccess && cudaStreamWaitEvent(cs, c->win_filled, 0) == cudaSuccess;
    if (hg->mean) ok = ok && cudaMemcpyAsync(hg->mean, dg.mean, sizeof(float) * 3 * n, cudaMemcpyDeviceToHost, cs) == cudaSuccess;
    if (hg->scale) ok = ok && cudaMemcpyAsync(hg->scale, dg.scale, sizeof(float) * 2 * n, cudaMemcpyDeviceToHost, cs) == cudaSuccess;
    if (hg->quat) ok = ok && cudaMemcpyAsync(hg->quat, dg.quat, sizeof(float) * 4 * n, cudaMemcpyDeviceToHost, cs) == cudaSuccess;
    if (hg->opacity) ok = ok && cudaMemcpyAsync(hg->opacity, dg.opacity, sizeof(float) * n, cudaMemcpyDeviceToHost, cs) == cudaSuccess;
    if (hg->rgb) ok = ok && cudaMemcpyAsync(hg->rgb, dg.rgb, sizeof(float) * 3 * n, cudaMemcpyDeviceToHost, cs) == cudaSuccess;
    ok = ok && cudaMemsetAsync(c->win_grads[slot], 0, sizeof(float) * (size_t)(n * 13), cs) == cudaSuccess &&
         cudaEventRecord(c->win_drained[slot], cs) == cudaSuccess;
    if (!ok) return SGS_CUDA_ERROR;
    c->win_draining[slot] = true;
    c->win_slot ^= 1;
    c->win_dirty = false;
    return SGS_OK;
}

int sgs_fetch_grads_sparse_host(sgs_ctx* c, int32_t* h_ids, const sgs_surfel_grads* hg, int64_t cap, int64_t* h_count,
                                void* stream) {
    if (!c || !hg || cap < 0) return SGS_INVALID_ARGUMENT;
    if (!c->copy_stream || !c->win_grads[c->win_slot]) return SGS_NO_FORWARD_STATE;
    if (c->win_n_cnt_pending >= SGS_WIN_RING) return SGS_INVALID_ARGUMENT;  // call sgs_sync_host first
    cudaStream_t s = (cudaStream_t)stream, cs = c->copy_stream;
    const int64_t n = c->resident.n;
    const int slot = c->win_slot;
    int r = flush_sparse(c, true);   // the previous fetch's rows leave the staging buffer first (its pack ran a window ago)
    if (r != SGS_OK) return r;
    if (!grow(c, c->win_scratch, c->win_scratch_cap, sgs_window_scratch_words(n), cs) ||
        !grow(c, c->win_stage, c->win_stage_cap, sgs_window_stage_words(n), cs))
        return SGS_OUT_OF_MEMORY;
    const int k = c->win_n_cnt_pending;
    c->win_counts[k] = 0;
    bool ok = cudaEventRecord(c->win_filled, s) == cudaSuccess && cudaStreamWaitEvent(cs, c->win_filled, 0) == cudaSuccess &&
              sgs_launch_window_compact(c, c->win_grads[slot], n, c->win_scratch, c->win_stage, c->win_counts_dev + k, cs) == cudaSuccess &&
              cudaEventRecord(c->win_packed, cs) == cudaSuccess && cudaEventRecord(c->win_drained[slot], cs) == cudaSuccess;
    if (!ok) return SGS_CUDA_ERROR;
    c->win_sp.pending = true; c->win_sp.ring = k; c->win_sp.n = n; c->win_sp.cap = cap; c->win_sp.ids = h_ids; c->win_sp.rows = *hg;
    c->win_cnt_pending[k] = h_count;
    c->win_n_cnt_pending = k + 1;
    c->win_draining[slot] = true;
    c->win_slot ^= 1;
    c->win_dirty = false;
    return SGS_OK;
}

int sgs_sync_host(sgs_ctx* c, void* stream) {
    if (!c) return SGS_INVALID_ARGUMENT;
    if (flush_sparse(c, true) != SGS_OK) return SGS_CUDA_ERROR;
    if (cudaStreamSynchronize((cudaStream_t)stream) != cudaSuccess) return SGS_CUDA_ERROR;
    if (c->copy_stream && cudaStreamSynchronize(c->copy_stream) != cudaSuccess) return SGS_CUDA_ERROR;
    if (c->in_stream && cudaStreamSynchronize(c->in_stream) != cudaSuccess) return SGS_CUDA_ERROR;
    c->win_tgt_used[0] = c->win_tgt_used[1] = false;
    c->win_draining[0] = c->win_draining[1] = false;
    for (int k = 0; k < c->win_n_pending; ++k) {
        const float* res = c->win_results + 8 * k;
        if (c->win_pending[k].loss) *c->win_pending[k].loss = res[0];
        if (c->win_pending[k].pose6) memcpy(c->win_pending[k].pose6, res + 1, sizeof(float) * 6);
    }
    c->win_n_pending = 0;
    for (int k = 0; k < c->win_n_cnt_pending; ++k)
        if (c->win_cnt_pending[k]) *c->win_cnt_pending[k] = (int64_t)c->win_counts[k];
    c->win_n_cnt_pending = 0;
    return SGS_OK;
}

}  // extern "C"
