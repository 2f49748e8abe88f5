// sgs_internal.h -- shared declarations of the CUDA path (ctx, workspace layout, launchers).
// Nothing here is used by the oracle.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/sgs.h"

#define SGS_TILE 16
#define SGS_BLOCK 256                // threads per compositing block = pixels per tile
#define SGS_SORT_ITEMS 8             // items per thread in the radix sort
#define SGS_SORT_TILE (256 * SGS_SORT_ITEMS)
#define SGS_PRE_BLOCK 256
#define SGS_ACC_STRIDE 16            // floats per visible surfel in the backward accumulator

// Per-visible-surfel payload, structure of float4 arrays indexed by the compact visible index v.
// Screen-centred adjugate form of the ray-splat intersection:
//   xt = x - x_c, yt = y - y_c  (x_c, y_c = projected centre, kept in fp64)
//   u = (xt P + yt Q) / den,  v = (xt R + yt S) / den,  den = D - xt E - yt F,  z = a u + b v + c
// Per-surfel payload written by the preprocess and gathered by the compositing kernels: ONE 128-byte record per surfel
// (eight 16-byte fields), so that a record is four whole 32-byte sectors.  As eight separate planes every field was
// half a sector: K-pre-B's stores cost a read-fill each (ncu, C5: 145 MB read for 17 MB of inputs) and the gathers
// fetched seven half-used sectors per entry.  g<k>[v] addresses field k of surfel v as before.
template <typename T>
struct PayField {
    float4* base;  // record 0's field
    __device__ __forceinline__ T& operator[](size_t v) const { return reinterpret_cast<T*>(base)[v * 8]; }
};
struct SgsPayload {
    PayField<float4> g0;   // P, Q, R, S
    PayField<float4> g1;   // D, E, F, opacity
    PayField<double2> g2;  // x_c, y_c
    PayField<float4> g3;   // a, b, c (= M20, M21, M22), rgb.r
    PayField<float4> g4;   // rgb.g, rgb.b, n_c.x, n_c.y
    PayField<float4> g5;   // n_c.z, a_u.x, a_u.y, a_u.z      (a_u = s_u t_uc, camera space)
    PayField<float4> g6;   // a_v.x, a_v.y, a_v.z, unused     (a_v = s_v t_vc)
    PayField<float4> g7;   // screen AABB of the cutoff ellipse: xmin, xmax, ymin, ymax (rounded outward)
    float4* store;         // n x 8 float4
};

struct SgsCamDev {
    int W, H, tiles_x, tiles_y;
    float fx, fy, cx, cy;
    double Kd[4];   // fx, fy, cx, cy widened
    double R[9];    // R_cw row-major
    double t[3];
    float Rf[9];
    float tf[3];
    // camera-only constants of the binary32 pre-cull (preprocess.cu precull_f32), filled on the host
    float pc_n[4];   // |(fx, cx)|, |(fx, cx - W)|, |(fy, cy)|, |(fy, cy - H)|, each rounded up by 1.00001
    float pc_cxr, pc_cyr, pc_tabs;  // cx - W, cy - H, |t|_1 + 1
    float pm_t, pm_r;  // pose margin of the pre-cull (metres, radians): 0 unless a survivor list is built for reuse
};

// SGS_FLAG_TRACK_REUSE: a survivor list stays valid for poses within this translation / rotation of the pose it was built for
constexpr float SGS_REUSE_MARGIN_T = 0.03f, SGS_REUSE_MARGIN_R = 0.02f;

constexpr int SGS_WIN_RING = 64;       // views whose (loss, pose gradient) may be in flight between two sgs_sync_host calls
constexpr int SGS_TRACK_HELPERS = 32;  // K-track: extra blocks that walk back the second half of the longest tile lists

struct SurvInputs { float4 *p0, *p1, *p2; float* p3; };  // (mean, opacity), quat, (scale, r, g), b

struct SgsCfgDev {
    float cutoff2, alpha_min, alpha_max, t_min, z_near;
    float cutoff;   // sqrt(cutoff2)
    double cutoff2_d, z_near_d;
    double alpha_min_d; int tight;   // SGS_FLAG_TIGHT_BINNING (R26, R27)
    int lowpass;                     // SGS_FLAG_LOWPASS (R28)
};

// Device-side counters of one render (also copied to pinned host memory).
struct SgsCounters {
    unsigned long long n_entries;   // E (may exceed capacity -> overflow)
    unsigned int n_visible;
    unsigned int overflow;
    unsigned int ticket_pre;        // dynamic block ids for the chained scan in K-pre
    unsigned int ticket_bwd;        // last-block-done ticket for the pose reduction
    unsigned int max_tile;          // bucket mode: largest per-tile entry count seen (> tile_cap => overflow)
    unsigned int n_surv;            // bucket mode: surfels that passed the cheap tests of K-pre-A (the list K-pre-B walks)
    unsigned int stale;             // sgs_track_iter_dev + SGS_FLAG_TRACK_REUSE: the device pose has left the kept survivor list's margin
    unsigned int pad_;
};

struct sgs_ctx {
    sgs_config cfg;
    SgsCfgDev cfgd;
    // sizes
    int64_t n_cap;        // surfel capacity of per-surfel workspace
    int64_t e_cap;        // entry capacity
    int64_t tiles_cap;
    int64_t pix_cap;
    int64_t bytes;
    // per-surfel
    unsigned long long* scan_state;  // chained-scan status words, one per K-pre block
    uint32_t* vis_to_surfel;         // n_cap: radix binning: compact visible index -> surfel; bucket binning: K-pre-A's survivor list
    uint32_t* vis_list;              // n_cap, bucket binning: the surfels that passed K-pre-B's exact culling (arrival order)
    int64_t last_vis;                // N_v of the last checked render (grid hint of the per-surfel backward), 0 = unknown
    uint8_t* culled;                 // n_cap
    SgsPayload pay;                  // n_cap each
    float* acc;                      // n_cap x 16 backward accumulators
    // per-entry (double buffered for the sort)
    uint64_t* keys[2];
    uint32_t* vals[2];
    uint32_t* idx_export;            // e_cap, original indices for sgs_get_binning
    uint32_t* sort_hist;             // passes x 256 global digit histograms
    uint32_t* sort_state;            // passes x sort_tiles x 256 look-back words
    uint32_t* sort_ticket;           // passes
    int64_t sort_tiles_cap;
    // bucket binning (default): tile t owns bucket[t * tile_cap .. ), filled through cursor[t]
    uint64_t* bucket;                // tiles x tile_cap keys: depth bits << 32 | surfel index
    uint32_t* cursor;                // tiles
    uint32_t* tile_order;            // tiles: tile ids by descending entry count (longest first), written by K-pre-B
    uint32_t* render_order;          // tiles: longest-first order of the last sgs_render's tiles (by entry count), or unused
    bool render_order_valid;
    float* ssim_maps; int64_t ssim_cap;  // 9 derivative planes of sgs_ssim_loss
    float* pose_inc; int inc_cap;    // per-keyframe increments of sgs_map_correction (16 floats each)
    unsigned int* covis_cnt;         // 4 counters of k_covisibility (cudaMalloc, lazily)
    float* median_out;               // sgs_render_median: median depth plane of the current forward, else nullptr
    float* contrib_out;              // sgs_render_contrib: per-splat contribution output of the current forward, or NULL
    int64_t cursor_cap;              // tiles the cursor / tile_order arrays hold
    int64_t tile_cap, bucket_cap;    // entries per tile; allocated keys
    uint64_t* export_keys;           // contiguous (tile << 32 | depth) list for sgs_get_binning
    uint32_t* export_ranges;
    int64_t export_cap;
    const uint32_t* list_vals; int list_stride;
    bool fused_sort;                 // bucket mode with tile_cap <= 2048: k_forward sorts its own bucket   // the sorted per-tile lists the compositing kernels walk
    // per-tile / per-pixel
    uint32_t* ranges;                // tiles x 2
    float* T_final;                  // pixels
    uint32_t* n_last;                // pixels: index (within the tile list) after the last composited entry
    float2* dn_state;                // pixels, SGS_FLAG_NORMALISED_DEPTH only: (D / O, 1 / O) of the last forward (0, 0 where O = 0)
    float* pose_partial;             // tiles x 8 (pose-only) or blocks x 8 (per-surfel)
    float* img_saved[8];             // planes the backward needs when the caller did not ask for them
    float* img_scratch;              // 8 planes, pix_cap each
    SgsCounters* counters;           // device
    SgsCounters* counters_host;      // pinned + mapped
    SgsCounters* counters_host_dev;  // its device address
    cudaEvent_t counters_ready;
    cudaStream_t aux_stream;           // sgs_backward: the gradient memsets run beside k_backward (fork / join by events)
    cudaEvent_t fork_ev, join_ev;
    cudaEvent_t prepared_ev, work_ev;   // sgs_prepare: binning enqueued / the ctx's last render or backward enqueued
    // SGS_FLAG_TRACK_REUSE: K-pre-A's survivor list (vis_to_surfel) outlives the iteration it was built in
    unsigned int* surv_cnt;            // device: its length
    void* surv_in; int64_t surv_in_cap; // the listed splats' parameters in list order (3 float4 planes + 1 float plane)
    bool surv_valid, use_surv_cache;   // list valid for (surv_sf, poses near surv_cam) / this preprocess launch uses it
    sgs_surfels surv_sf;
    sgs_camera surv_cam;
    float* surv_pose_dev;              // 12 floats: the DEVICE pose the kept list was built around (sgs_track_iter_dev)
    const float* pose_dev;             // non-NULL inside sgs_track_iter_dev: the preprocess kernels read T_cw from here
    bool track_binning;                // inside sgs_track_iter's fused path: K-pre-B need not build vis_list
    int narrow_prepare;                // > 0 inside sgs_prepare: K-pre-B blocks per SM
    bool grads_on_aux;                 // SGS_FLAG_LAZY_GRADS: the last sgs_backward left its final kernel on aux_stream
    bool copy_in_flight;               // counters_ready was recorded on aux_stream and nothing on the caller's stream waited for it yet
    bool prepared, work_recorded;      // binning of (last_surfels, last_cam) enqueued by sgs_prepare, not yet rendered
    // last forward
    bool have_forward;
    bool have_binning;               // sorted lists + ranges of the last render / track_iter are valid
    bool pending_check;              // async mode: counters_host not yet examined
    bool pending_lazy;               // ... and the copy was enqueued BEHIND the compositing kernel (sgs_track_iter): never wait for it
    sgs_surfels last_surfels;
    sgs_camera last_cam;
    SgsCamDev camd;
    const float* last_img[8];        // device planes of the last render: rgb(3), depth, normal(3), alpha
    int sorted_buf;                  // which of keys[]/vals[] holds the sorted list
    int64_t launch_entries;          // entries bound used for this render's launches
    // resident (host-path) state
    sgs_surfels resident;            // ctx-owned device copy
    int64_t resident_cap;
    float* resident_store;           // one allocation
    uint8_t* resident_active;
    float* target_rgb; float* target_depth; int64_t target_cap;
    float* host_img_dev;             // 8 planes staging for *_host
    float* host_up_dev;              // 8 planes staging
    float* host_grads_dev;           // n x 13 staging
    float* loss_dev; float* pose6_dev;
    float* pinned_small;             // 8 floats pinned
    // sgs_track_iter_host: K-track writes loss + pose gradient straight into pinned_small and then this flag word (pinned,
    // device-visible); the host polls it instead of a copy + stream synchronisation
    unsigned int* host_flag; unsigned int* host_flag_dev; float* pinned_small_dev;
    unsigned int host_flag_val; bool host_flag_want, host_flag_armed;
    // K-track helpers (track.cu): per helper 8 x 256 floats of per-pixel state and a flag word; split_flag[SGS_TRACK_HELPERS] is the
    // launch epoch the flag values are built from (device-side, so that graph replays stay distinct)
    float* split_state; unsigned int* split_flag; unsigned int helper_delay_ns;
    cudaEvent_t order_fork, order_done; bool order_pending;  // k_track_order on aux_stream
    bool order_skip;                 // SGS_FLAG_GRAPH + SGS_FLAG_TRACK_REUSE: the tile order is renewed once per frame only
    const SgsCounters* stats_src;    // SGS_FLAG_GRAPH: where the last binning's counters sit on the device (sgs_get_stats copies them)
    int64_t host_img_cap, host_grads_cap;
    // mapping window on the resident map (sgs_map_view_host / sgs_fetch_grads_host): two device accumulators of n x 13 floats
    // (one fills while the other drains to the host on copy_stream), and a pinned ring of per-view results
    float* win_grads[2]; int64_t win_cap[2]; int win_slot; bool win_dirty;
    cudaStream_t copy_stream; cudaEvent_t win_filled, win_drained[2]; bool win_draining[2];
    float* win_results; float* win_results_dev;   // pinned + mapped, SGS_WIN_RING x 8 floats: loss, pose6
    // keyframe uploads of sgs_map_view_host run on their own stream into one of two buffers, under the previous view's kernels
    cudaStream_t in_stream; float* win_tgt[2]; int64_t win_tgt_cap[2]; int win_tgt_slot;
    cudaEvent_t win_tgt_ready[2], win_tgt_free[2]; bool win_tgt_used[2];
    struct { float* loss; float* pose6; } win_pending[64]; int win_n_pending;
    // sgs_fetch_grads_sparse_host (window.cu): compaction scratch, row staging, a mapped ring of row counts; the copy-out of
    // the last fetch is enqueued by the first window call that finds its pack complete (win_sp: what it has to deliver)
    uint32_t* win_scratch; int64_t win_scratch_cap; uint32_t* win_stage; int64_t win_stage_cap;
    uint32_t* win_counts; uint32_t* win_counts_dev; cudaEvent_t win_packed;
    struct { bool pending; int ring; int64_t n, cap; int32_t* ids; sgs_surfel_grads rows; } win_sp;
    int64_t* win_cnt_pending[64]; int win_n_cnt_pending;
    int64_t partial_cap;             // floats in pose_partial
    int64_t launches;                // kernels launched by this ctx
    int prof_on; int prof_n, prof_cap; cudaEvent_t* prof_ev; int* prof_stage;  // event pairs: ev[2i], ev[2i+1]
    int64_t last_entries;            // E of the last checked render (async launch bound hint), 0 = unknown
    int64_t last_surv;               // K-pre-A survivors of the last checked render (K-pre-B grid hint), 0 = unknown
    uint32_t* tile_cost;             // tiles: cycles >> 8 each tile's k_track block took last time (scheduling feedback)
    int cost_tiles, cost_W, cost_H;  // camera the costs were measured for (0 = none)
    SgsCounters* counters_snap;      // device copies (two slots, alternating) of the counters taken by k_track's last block before it zeroes them
    int snap_slot;                   // slot the NEXT sgs_track_iter writes
    cudaEvent_t counters_ready_prev; // copy of the other slot (one iteration older) done; swapped with counters_ready
    bool prev_copy_on_aux, snap_copy_on_aux;
    bool defer_counters;             // sgs_track_iter (async): the counters reach the host after k_track, from the snapshot
    int prezero_tiles;               // k_track's last block left counters and cursor[0..prezero_tiles) zeroed for the next preprocess
};

// ---- launchers (each enqueues on `s`, returns the last CUDA error) ----
cudaError_t sgs_launch_preprocess(sgs_ctx* c, const sgs_surfels* sf, cudaStream_t s);
cudaError_t sgs_launch_sort_and_ranges(sgs_ctx* c, cudaStream_t s);
cudaError_t sgs_launch_forward(sgs_ctx* c, float* const planes[8], cudaStream_t s);
cudaError_t sgs_launch_backward(sgs_ctx* c, const float* const up[8], const sgs_surfel_grads* dg, float* d_pose6,
                                bool accumulate, cudaStream_t s);
cudaError_t sgs_launch_tracking_loss(sgs_ctx* c, const sgs_camera* cam, const float* const ren[8], const float* trgb,
                                     const float* tdepth, float lambda_d, float nsign, float* const up[8], float* loss,
                                     cudaStream_t s);
cudaError_t sgs_launch_mapping_loss(sgs_ctx* c, const sgs_camera* cam, const float* const ren[8], const float* trgb,
                                    const float* tdepth, float lambda_c, float w_d, float w_n, float nsign, float* const up[8],
                                    float* loss, cudaStream_t s);
cudaError_t sgs_launch_fma_peak(double* tflops, cudaStream_t s);
cudaError_t sgs_launch_ssim_loss(sgs_ctx* c, int W, int H, const float* rgb_r, const float* rgb_t, float weight, float* up_rgb,
                                 float* loss, cudaStream_t s);
cudaError_t sgs_launch_map_correction(sgs_ctx* c, int64_t n, float* mean, float* quat, const int* frame_id, int n_frames,
                                      const float* T_orig, const float* T_opt, cudaStream_t s);
cudaError_t sgs_launch_export_idx(sgs_ctx* c, cudaStream_t s);
cudaError_t sgs_launch_backward_tracking(sgs_ctx* c, const float* trgb, const float* tdepth, float lambda_d, float nsign,
                                         float* d_pose6, float* loss, cudaStream_t s);
cudaError_t sgs_launch_track(sgs_ctx* c, float* const planes[8], const float* trgb, const float* tdepth, float lambda_d,
                             float nsign, float* d_pose6, float* loss, bool after_preprocess, cudaStream_t s);
int sgs_sort_passes(int tiles);
cudaError_t sgs_launch_preprocess_bucket(sgs_ctx* c, const sgs_surfels* sf, cudaStream_t s);
cudaError_t sgs_launch_tilesort(sgs_ctx* c, cudaStream_t s);
cudaError_t sgs_launch_tile_order(sgs_ctx* c, cudaStream_t s);
cudaError_t sgs_launch_covisibility(sgs_ctx* c, const float* ca, const float* cb, int64_t n, const uint8_t* active, float thr,
                                    float* result3, cudaStream_t s);
cudaError_t sgs_launch_export_bucket(sgs_ctx* c, int64_t n_entries, cudaStream_t s);
int sgs_ensure_buckets(sgs_ctx* c, int tiles, int64_t tile_cap, cudaStream_t s);
int sgs_ensure_export(sgs_ctx* c, int tiles, int64_t entries, cudaStream_t s);

int64_t sgs_window_scratch_words(int64_t n);
int64_t sgs_window_stage_words(int64_t n);
cudaError_t sgs_launch_window_compact(sgs_ctx* c, float* acc, int64_t n, uint32_t* scratch, uint32_t* stage, uint32_t* count_mapped,
                                      cudaStream_t s);
cudaError_t sgs_launch_publish(void* dst_mapped, const void* src, int words, cudaStream_t s);  // <= 1024 words

// ---- workspace helpers (api.cu) ----
void* sgs_ws_alloc(sgs_ctx* c, size_t bytes, cudaStream_t s);
void sgs_ws_free(sgs_ctx* c, void* p, cudaStream_t s);
int sgs_ensure_surfels(sgs_ctx* c, int64_t n, cudaStream_t s);
int sgs_ensure_entries(sgs_ctx* c, int64_t e, cudaStream_t s);
int sgs_ensure_image(sgs_ctx* c, int tiles, int64_t pixels, cudaStream_t s);
int sgs_ensure_partials(sgs_ctx* c, int64_t blocks, cudaStream_t s);
void sgs_fill_cam(const sgs_camera* cam, SgsCamDev* d);
bool sgs_cam_valid(const sgs_camera* cam);

// profiling scope: records an event pair around a stage when ctx->prof_on
struct SgsStage {
    sgs_ctx* c; cudaStream_t s; int slot;
    SgsStage(sgs_ctx* c_, int stage, cudaStream_t s_);
    ~SgsStage();
};
