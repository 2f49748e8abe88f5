// api.cu -- the C ABI of include/sgs.h: ctx, workspace, and the launch sequences.
#include <math.h>
#include <new>
#include <stdlib.h>
#include <string.h>
#include "sgs_internal.h"

// A few words from device memory to MAPPED pinned host memory, written by a kernel.  Used instead of a device-to-host
// cudaMemcpyAsync for results the host polls or a stream's next kernel sits behind: a copy command queues on the copy
// engine BEHIND whatever bulk transfer is in flight (measured: with sgs_fetch_grads_host's 104 MB copy-out running, the 28-byte
// result copy of the next view -- and with it that view's kernels -- waited for it: 18.7 ms per C4 step instead of 12.9).
__global__ void k_publish_words(unsigned int* __restrict__ dst, const unsigned int* __restrict__ src, int n) {
    const int i = threadIdx.x;
    if (i < n) dst[i] = src[i];   // (visible to the host once the kernel has completed: every reader waits for that)
}
cudaError_t sgs_launch_publish(void* dst_mapped, const void* src, int words, cudaStream_t s) {
    k_publish_words<<<1, 32 * ((words + 31) / 32), 0, s>>>((unsigned int*)dst_mapped, (const unsigned int*)src, words);
    return cudaGetLastError();
}

void* sgs_ws_alloc(sgs_ctx* c, size_t bytes, cudaStream_t s) {
    if (bytes == 0) bytes = 16;
    void* p = nullptr;
    if (c->cfg.alloc) {
        p = c->cfg.alloc(bytes, c->cfg.user, (void*)s);
    } else if (cudaMalloc(&p, bytes) != cudaSuccess) {
        cudaGetLastError();
        p = nullptr;
    }
    if (p) c->bytes += (int64_t)bytes;
    return p;
}
void sgs_ws_free(sgs_ctx* c, void* p, cudaStream_t s) {
    if (!p) return;
    if (c->cfg.free) c->cfg.free(p, c->cfg.user, (void*)s);
    else if (!c->cfg.alloc) cudaFree(p);
}
template <typename T>
static bool ws_realloc(sgs_ctx* c, T*& p, size_t count, cudaStream_t s, bool zero = false) {
    sgs_ws_free(c, p, s);
    p = (T*)sgs_ws_alloc(c, count * sizeof(T), s);
    if (!p) return false;
    if (zero && cudaMemsetAsync(p, 0, count * sizeof(T), s) != cudaSuccess) return false;
    return true;
}

// per-surfel workspace
int sgs_ensure_surfels(sgs_ctx* c, int64_t n, cudaStream_t s) {
    if (n <= c->n_cap) return SGS_OK;
    cudaStreamSynchronize(s);
    const size_t m = (size_t)(n + n / 8 + 1024);
    const size_t blocks = (m + SGS_PRE_BLOCK - 1) / SGS_PRE_BLOCK + 1;
    bool ok = ws_realloc(c, c->scan_state, blocks, s) && ws_realloc(c, c->vis_to_surfel, m, s) && ws_realloc(c, c->vis_list, m, s) &&
              ws_realloc(c, c->culled, m, s) && ws_realloc(c, c->pay.store, m * 8, s) &&
              ws_realloc(c, c->acc, m * SGS_ACC_STRIDE, s, true);  // invariant: acc is all-zero between backward calls
    if (!ok) return SGS_OUT_OF_MEMORY;
    float4* st = c->pay.store;
    c->pay.g0.base = st; c->pay.g1.base = st + 1; c->pay.g2.base = st + 2; c->pay.g3.base = st + 3;
    c->pay.g4.base = st + 4; c->pay.g5.base = st + 5; c->pay.g6.base = st + 6; c->pay.g7.base = st + 7;
    c->n_cap = (int64_t)m;
    return SGS_OK;
}

int sgs_ensure_entries(sgs_ctx* c, int64_t e, cudaStream_t s) {
    if (e <= c->e_cap) return SGS_OK;
    cudaStreamSynchronize(s);
    const size_t m = (size_t)(e + e / 4 + 4096);
    const size_t st = (m + SGS_SORT_TILE - 1) / SGS_SORT_TILE + 1;
    bool ok = ws_realloc(c, c->keys[0], m, s) && ws_realloc(c, c->keys[1], m, s) && ws_realloc(c, c->vals[0], m, s) &&
              ws_realloc(c, c->vals[1], m, s) && ws_realloc(c, c->idx_export, m, s) &&
              ws_realloc(c, c->sort_state, st * 256 * 8, s);
    if (!ok) return SGS_OUT_OF_MEMORY;
    c->e_cap = (int64_t)m;
    c->sort_tiles_cap = (int64_t)st;
    return SGS_OK;
}

int sgs_ensure_image(sgs_ctx* c, int tiles, int64_t pixels, cudaStream_t s) {
    if (tiles > c->tiles_cap) {
        cudaStreamSynchronize(s);
        if (!ws_realloc(c, c->ranges, (size_t)tiles * 2, s)) return SGS_OUT_OF_MEMORY;
        c->tiles_cap = tiles;
    }
    if (pixels > c->pix_cap) {
        cudaStreamSynchronize(s);
        if (!(ws_realloc(c, c->T_final, (size_t)pixels, s) && ws_realloc(c, c->n_last, (size_t)pixels, s) &&
              ws_realloc(c, c->img_scratch, (size_t)pixels * 8, s)))
            return SGS_OUT_OF_MEMORY;
        if ((c->cfg.flags & SGS_FLAG_NORMALISED_DEPTH) && !ws_realloc(c, c->dn_state, (size_t)pixels, s)) return SGS_OUT_OF_MEMORY;
        c->pix_cap = pixels;
    }
    return SGS_OK;
}

int sgs_ensure_partials(sgs_ctx* c, int64_t blocks, cudaStream_t s) {
    static_assert(sizeof(float) == 4, "");
    if (blocks * 8 <= c->partial_cap) return SGS_OK;
    cudaStreamSynchronize(s);
    if (!ws_realloc(c, c->pose_partial, (size_t)blocks * 8 + 64, s)) return SGS_OUT_OF_MEMORY;
    c->partial_cap = blocks * 8 + 64;
    return SGS_OK;
}

int sgs_ensure_buckets(sgs_ctx* c, int tiles, int64_t tile_cap, cudaStream_t s) {
    int64_t cap = 256;
    while (cap < tile_cap) cap <<= 1;  // power of two (the bitonic network pads to it)
    if ((int64_t)tiles * cap >= (1ll << 32)) return SGS_OUT_OF_MEMORY;
    if (cap == c->tile_cap && (int64_t)tiles * cap <= c->bucket_cap && tiles <= c->cursor_cap) return SGS_OK;
    cudaStreamSynchronize(s);
    if (tiles > c->cursor_cap) {
        if (!(ws_realloc(c, c->cursor, (size_t)tiles + 64, s) && ws_realloc(c, c->tile_order, (size_t)tiles + 64, s) && ws_realloc(c, c->render_order, (size_t)tiles + 64, s) &&
              ws_realloc(c, c->tile_cost, (size_t)tiles + 64, s)))
            return SGS_OUT_OF_MEMORY;
        c->cursor_cap = tiles;
        c->cost_tiles = 0;
        c->prezero_tiles = 0;
    }
    if ((int64_t)tiles * cap > c->bucket_cap) {
        const size_t m = (size_t)tiles * (size_t)cap;
        if (!ws_realloc(c, c->bucket, m, s)) return SGS_OUT_OF_MEMORY;
        c->bucket_cap = (int64_t)m;
    }
    c->tile_cap = cap;
    return SGS_OK;
}

int sgs_ensure_export(sgs_ctx* c, int tiles, int64_t entries, cudaStream_t s) {
    if (entries + 2 * tiles <= c->export_cap) return SGS_OK;
    cudaStreamSynchronize(s);
    const size_t m = (size_t)entries + 1024;
    if (!(ws_realloc(c, c->export_keys, m, s) && ws_realloc(c, c->idx_export, m, s) &&
          ws_realloc(c, c->export_ranges, (size_t)tiles * 2 + 64, s)))
        return SGS_OUT_OF_MEMORY;
    c->export_cap = (int64_t)m + 2 * tiles;
    return SGS_OK;
}

void sgs_fill_cam(const sgs_camera* cam, SgsCamDev* d) {
    d->W = cam->width; d->H = cam->height;
    d->tiles_x = (cam->width + SGS_TILE - 1) / SGS_TILE;
    d->tiles_y = (cam->height + SGS_TILE - 1) / SGS_TILE;
    d->fx = cam->fx; d->fy = cam->fy; d->cx = cam->cx; d->cy = cam->cy;
    d->Kd[0] = cam->fx; d->Kd[1] = cam->fy; d->Kd[2] = cam->cx; d->Kd[3] = cam->cy;
    for (int i = 0; i < 3; ++i) {
        for (int j = 0; j < 3; ++j) { d->R[3 * i + j] = cam->T_cw[4 * i + j]; d->Rf[3 * i + j] = cam->T_cw[4 * i + j]; }
        d->t[i] = cam->T_cw[4 * i + 3]; d->tf[i] = cam->T_cw[4 * i + 3];
    }
    d->pc_cxr = cam->cx - (float)cam->width; d->pc_cyr = cam->cy - (float)cam->height;
    d->pc_n[0] = sqrtf(cam->fx * cam->fx + cam->cx * cam->cx) * 1.00001f;
    d->pc_n[1] = sqrtf(cam->fx * cam->fx + d->pc_cxr * d->pc_cxr) * 1.00001f;
    d->pc_n[2] = sqrtf(cam->fy * cam->fy + cam->cy * cam->cy) * 1.00001f;
    d->pc_n[3] = sqrtf(cam->fy * cam->fy + d->pc_cyr * d->pc_cyr) * 1.00001f;
    d->pc_tabs = fabsf(d->tf[0]) + fabsf(d->tf[1]) + fabsf(d->tf[2]) + 1.f;
    d->pm_t = 0.f; d->pm_r = 0.f;
}

bool sgs_cam_valid(const sgs_camera* cam) {
    if (!cam || cam->width <= 0 || cam->height <= 0 || cam->width > 16384 || cam->height > 16384) return false;
    if (!(cam->fx > 0.f) || !(cam->fy > 0.f) || !isfinite(cam->cx) || !isfinite(cam->cy)) return false;
    for (int i = 0; i < 12; ++i)
        if (!isfinite(cam->T_cw[i])) return false;
    return true;
}

SgsStage::SgsStage(sgs_ctx* c_, int stage, cudaStream_t s_) : c(c_), s(s_), slot(-1) {
    if (!c->prof_on) return;
    if (c->prof_n == c->prof_cap) {
        const int ncap = c->prof_cap ? c->prof_cap * 2 : 1024;
        cudaEvent_t* ev = (cudaEvent_t*)realloc(c->prof_ev, sizeof(cudaEvent_t) * 2 * (size_t)ncap);
        int* st = (int*)realloc(c->prof_stage, sizeof(int) * (size_t)ncap);
        if (ev) c->prof_ev = ev;
        if (st) c->prof_stage = st;
        if (!ev || !st) return;
        for (int i = 2 * c->prof_cap; i < 2 * ncap; ++i) cudaEventCreate(&c->prof_ev[i]);
        c->prof_cap = ncap;
    }
    slot = c->prof_n++;
    c->prof_stage[slot] = stage;
    cudaEventRecord(c->prof_ev[2 * slot], s);
}
SgsStage::~SgsStage() {
    if (slot >= 0) cudaEventRecord(c->prof_ev[2 * slot + 1], s);
}

extern "C" {

int sgs_default_config(sgs_config* cfg) {
    if (!cfg) return SGS_INVALID_ARGUMENT;
    memset(cfg, 0, sizeof(*cfg));
    cfg->tile = SGS_TILE; cfg->cutoff = 3.0f; cfg->alpha_min = 1.0f / 255.0f; cfg->alpha_max = 0.99f;
    cfg->t_min = 1e-4f; cfg->z_near = 0.2f; cfg->flags = 0;
    return SGS_OK;
}

int sgs_create(sgs_ctx** out, const sgs_config* cfg) {
    if (!out) return SGS_INVALID_ARGUMENT;
    *out = nullptr;
    sgs_config def;
    sgs_default_config(&def);
    if (!cfg) cfg = &def;
    if (cfg->tile != SGS_TILE || !(cfg->cutoff > 0.f) || !isfinite(cfg->cutoff) || !(cfg->alpha_min >= 0.f) ||
        !(cfg->alpha_max > 0.f) || !(cfg->alpha_max < 1.f) || !(cfg->t_min >= 0.f) || !(cfg->z_near > 0.f) ||
        ((cfg->alloc == nullptr) != (cfg->free == nullptr)) ||
        ((cfg->flags & SGS_FLAG_TIGHT_BINNING) && (cfg->flags & SGS_FLAG_RADIX_BINNING)) ||
        ((cfg->flags & SGS_FLAG_LOWPASS) && (cfg->flags & (SGS_FLAG_TIGHT_BINNING | SGS_FLAG_NORMALISED_DEPTH))))
        return SGS_INVALID_ARGUMENT;
    sgs_ctx* c = new (std::nothrow) sgs_ctx;
    if (!c) return SGS_OUT_OF_MEMORY;
    memset(c, 0, sizeof(*c));
    c->cfg = *cfg;
    c->cfgd.cutoff2 = cfg->cutoff * cfg->cutoff;
    c->cfgd.cutoff = sqrtf(c->cfgd.cutoff2);
    c->cfgd.alpha_min = cfg->alpha_min; c->cfgd.alpha_max = cfg->alpha_max;
    c->cfgd.t_min = cfg->t_min; c->cfgd.z_near = cfg->z_near;
    c->cfgd.cutoff2_d = (double)cfg->cutoff * (double)cfg->cutoff;
    c->cfgd.z_near_d = (double)cfg->z_near;
    c->cfgd.alpha_min_d = (double)cfg->alpha_min;
    c->cfgd.tight = (cfg->flags & SGS_FLAG_TIGHT_BINNING) ? 1 : 0;
    c->cfgd.lowpass = (cfg->flags & SGS_FLAG_LOWPASS) ? 1 : 0;
    int prio_lo = 0, prio_hi = 0;  // the ctx's own stream carries short latency-bound work: let it in first
    cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi);
    bool ok = cudaMalloc(&c->counters, sizeof(SgsCounters)) == cudaSuccess &&
              cudaMalloc(&c->counters_snap, 2 * sizeof(SgsCounters)) == cudaSuccess &&
              cudaEventCreateWithFlags(&c->counters_ready_prev, cudaEventDisableTiming) == cudaSuccess &&
              cudaHostAlloc(&c->counters_host, sizeof(SgsCounters), cudaHostAllocMapped) == cudaSuccess &&
              cudaHostGetDevicePointer(&c->counters_host_dev, c->counters_host, 0) == cudaSuccess &&
              cudaHostAlloc(&c->pinned_small, 8 * sizeof(float), cudaHostAllocMapped) == cudaSuccess &&
              cudaHostAlloc(&c->host_flag, sizeof(unsigned int), cudaHostAllocMapped) == cudaSuccess &&
              cudaMalloc(&c->split_state, sizeof(float) * 8 * SGS_BLOCK * SGS_TRACK_HELPERS) == cudaSuccess &&
              cudaMalloc(&c->split_flag, sizeof(unsigned int) * (SGS_TRACK_HELPERS + 1)) == cudaSuccess &&
              cudaMemset(c->split_flag, 0, sizeof(unsigned int) * (SGS_TRACK_HELPERS + 1)) == cudaSuccess &&
              cudaHostGetDevicePointer(&c->pinned_small_dev, c->pinned_small, 0) == cudaSuccess &&
              cudaHostGetDevicePointer(&c->host_flag_dev, c->host_flag, 0) == cudaSuccess &&
              cudaMalloc(&c->sort_hist, sizeof(uint32_t) * (8 * 256 + 8)) == cudaSuccess &&
              cudaMalloc(&c->surv_pose_dev, sizeof(float) * 12) == cudaSuccess &&
              cudaMalloc(&c->loss_dev, sizeof(float) * 8) == cudaSuccess &&
              cudaEventCreateWithFlags(&c->counters_ready, cudaEventDisableTiming) == cudaSuccess &&
              cudaEventCreateWithFlags(&c->prepared_ev, cudaEventDisableTiming) == cudaSuccess &&
              cudaEventCreateWithFlags(&c->work_ev, cudaEventDisableTiming) == cudaSuccess &&
              cudaEventCreateWithFlags(&c->fork_ev, cudaEventDisableTiming) == cudaSuccess &&
              cudaEventCreateWithFlags(&c->order_fork, cudaEventDisableTiming) == cudaSuccess &&
              cudaEventCreateWithFlags(&c->order_done, cudaEventDisableTiming) == cudaSuccess &&
              cudaEventCreateWithFlags(&c->join_ev, cudaEventDisableTiming) == cudaSuccess &&
              ((cfg->flags & SGS_FLAG_GRAPH) != 0 ||  // capture mode: everything stays on the caller's stream
               cudaStreamCreateWithPriority(&c->aux_stream, cudaStreamNonBlocking, prio_hi) == cudaSuccess);
    if (!ok) { cudaGetLastError(); sgs_destroy(c); return SGS_CUDA_ERROR; }
    c->pose6_dev = c->loss_dev + 1;
    if (const char* d = getenv("SGS_DEBUG_HELPER_DELAY_NS")) c->helper_delay_ns = (unsigned int)strtoul(d, nullptr, 10);
    cudaMemset(c->counters, 0, sizeof(SgsCounters));
    memset(c->counters_host, 0, sizeof(SgsCounters));
    *out = c;
    return SGS_OK;
}

int sgs_destroy(sgs_ctx* c) {
    if (!c) return SGS_OK;
    cudaDeviceSynchronize();
    cudaStream_t s = 0;
    void* ptrs[] = {c->scan_state, c->vis_to_surfel, c->vis_list, c->culled, c->pay.store, c->acc, c->keys[0], c->keys[1], c->vals[0], c->vals[1], c->idx_export,
                    c->sort_state, c->ranges, c->T_final, c->n_last, c->dn_state, c->img_scratch, c->pose_partial, c->resident_store,
                    c->resident_active, c->target_rgb, c->host_img_dev, c->host_up_dev, c->host_grads_dev,
                    c->win_grads[0], c->win_grads[1], c->win_tgt[0], c->win_tgt[1], c->win_scratch, c->win_stage, c->bucket, c->cursor, c->tile_order, c->render_order, c->tile_cost, c->pose_inc, c->ssim_maps, c->surv_cnt, c->surv_in, c->export_keys, c->export_ranges};
    for (void* p : ptrs) sgs_ws_free(c, p, s);
    if (c->counters) cudaFree(c->counters);
    if (c->counters_snap) cudaFree(c->counters_snap);
    if (c->counters_ready_prev) cudaEventDestroy(c->counters_ready_prev);
    if (c->counters_host) cudaFreeHost(c->counters_host);
    if (c->pinned_small) cudaFreeHost(c->pinned_small);
    if (c->host_flag) cudaFreeHost(c->host_flag);
    if (c->split_state) cudaFree(c->split_state);
    if (c->split_flag) cudaFree(c->split_flag);
    if (c->sort_hist) cudaFree(c->sort_hist);
    if (c->surv_pose_dev) cudaFree(c->surv_pose_dev);
    if (c->loss_dev) cudaFree(c->loss_dev);
    if (c->covis_cnt) cudaFree(c->covis_cnt);
    if (c->counters_ready) cudaEventDestroy(c->counters_ready);
    if (c->prepared_ev) cudaEventDestroy(c->prepared_ev);
    if (c->work_ev) cudaEventDestroy(c->work_ev);
    if (c->fork_ev) cudaEventDestroy(c->fork_ev);
    if (c->order_fork) cudaEventDestroy(c->order_fork);
    if (c->order_done) cudaEventDestroy(c->order_done);
    if (c->join_ev) cudaEventDestroy(c->join_ev);
    if (c->aux_stream) cudaStreamDestroy(c->aux_stream);
    if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
    if (c->in_stream) cudaStreamDestroy(c->in_stream);
    for (int k = 0; k < 2; ++k) {
        if (c->win_tgt_ready[k]) cudaEventDestroy(c->win_tgt_ready[k]);
        if (c->win_tgt_free[k]) cudaEventDestroy(c->win_tgt_free[k]);
    }
    if (c->win_filled) cudaEventDestroy(c->win_filled);
    if (c->win_drained[0]) cudaEventDestroy(c->win_drained[0]);
    if (c->win_drained[1]) cudaEventDestroy(c->win_drained[1]);
    if (c->win_results) cudaFreeHost(c->win_results);
    if (c->win_counts) cudaFreeHost(c->win_counts);
    if (c->win_packed) cudaEventDestroy(c->win_packed);
    for (int i = 0; i < 2 * c->prof_cap; ++i) cudaEventDestroy(c->prof_ev[i]);
    free(c->prof_ev); free(c->prof_stage);
    delete c;
    return SGS_OK;
}

int sgs_set_profiling(sgs_ctx* c, int enabled) {
    if (!c) return SGS_INVALID_ARGUMENT;
    c->prof_on = enabled ? 1 : 0;
    return SGS_OK;
}

int sgs_get_profile(sgs_ctx* c, double* ms, int64_t* calls, int reset) {
    if (!c) return SGS_INVALID_ARGUMENT;
    if (cudaDeviceSynchronize() != cudaSuccess) return SGS_CUDA_ERROR;
    for (int i = 0; i < SGS_STAGE_COUNT; ++i) { if (ms) ms[i] = 0.0; if (calls) calls[i] = 0; }
    for (int i = 0; i < c->prof_n; ++i) {
        float t = 0.f;
        if (cudaEventElapsedTime(&t, c->prof_ev[2 * i], c->prof_ev[2 * i + 1]) != cudaSuccess) { cudaGetLastError(); continue; }
        if (ms) ms[c->prof_stage[i]] += (double)t;
        if (calls) calls[c->prof_stage[i]] += 1;
    }
    if (reset) c->prof_n = 0;
    return SGS_OK;
}

const char* sgs_status_string(int status) {
    switch (status) {
        case SGS_OK: return "ok";
        case SGS_INVALID_ARGUMENT: return "invalid argument";
        case SGS_OUT_OF_MEMORY: return "out of memory";
        case SGS_WORKSPACE_OVERFLOW: return "workspace overflow: the previous render dropped tile entries; render again";
        case SGS_NO_FORWARD_STATE: return "no forward state: call sgs_render first";
        case SGS_CUDA_ERROR: return "CUDA error";
        case SGS_LIMIT_EXCEEDED: return "size beyond the static scratch limit (sgs_map_correction_static: n_frames > SGS_STATIC_MAX_FRAMES = 4096)";
        default: return "unknown status";
    }
}

}  // extern "C"
