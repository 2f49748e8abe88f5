// track.cu -- K-track: ONE launch per tracking iteration after K-pre.
//
// A tracking iteration renders the active map (Eq. 8), evaluates the masked L1 colour + depth loss of
// Eq. 15-19 against the current frame, and back-propagates to the 6-DoF pose only (Eq. 11-13; the splats
// are frozen, L204).  The loss couples nothing across pixels, so the whole chain runs per tile inside one
// block:  in-tile sort -> forward compositing -> loss and upstream gradients in registers -> reverse
// traversal -> block reduction -> grid reduction.  Compared with k_forward + k_backward<pose-only> this
// removes a launch, the T_final / n_last / image round trip through L2, the backward's prologue loads and
// -- for tiles whose list fits one 256-entry batch (the common case in tracking) -- the second staging
// gather: the staged records of the forward walk are walked again in reverse.
// Arithmetic is pair.cuh's (identical decisions to k_forward / k_backward); the tracking loss has no
// normal / alpha gradient, so those terms of the general backward are dropped at compile time.
#include "pair.cuh"
#include "histsort.cuh"
#include "reduce.cuh"
#include "sgs_internal.h"

namespace {

struct TrackPlanes { float* p[8]; };

// Staging capacity: lists of up to TRK_CAP entries are walked from ONE staged batch (the fast path below).  384 keeps the
// kernel's static shared memory under 48 KB; C2's longest tile list (263) used to fall into the general path, and that
// one tile set the end of the whole launch.
constexpr int TRK_CAP = 384;
constexpr uint32_t TRK_PL = TRK_CAP * 16;  // bytes per staged plane
constexpr int TRK_ORDER_BINS = 2048;         // tile costs (cycles >> 8) are binned 0..2047
constexpr int TRK_K = 2;                     // entries per trip of the walks
// Lists of TRK_SPLIT_MIN+1 .. TRK_CAP entries are walked BACK by the two blocks of the tile's cluster at once: block 0 the front
// part [0, m), block 1 the back part [m, n) (m a multiple of 32, n - m <= TRK_CAP / 2).  One warp gets through a trip of two
// entries in ~340 cycles whatever else the SM does (profiles/r01_c2_track.md), so a long list is a long serial walk and
// the launch ended with a dozen of them; the forward walk stays with block 0 (bit-identical images), block 1 stages its
// part meanwhile, receives (g, T_final, last) per pixel through distributed shared memory and takes half of the way back.
constexpr uint32_t TRK_SPLIT_MIN = 160;

// One thread stages entry `v` of the tile: forward record (s0..s4; s4.w carries m.z) plus the backward's a_u, a_v and
// m = a_u x a_v: 7 planes of float4.
__device__ __forceinline__ unsigned stage_track(const SgsPayload& pay, uint32_t v, double px0, double py0, float tx0,
                                                float ty0, float4 (*sh)[TRK_CAP], int tid, const SgsCfgDev& cfg) {
    const float4 g0 = pay.g0[v], g1 = pay.g1[v], g3 = pay.g3[v], g4 = pay.g4[v], g5 = pay.g5[v], g6 = pay.g6[v];
    const float4 g7 = pay.g7[v];
    const double2 g2 = pay.g2[v];
    float4 s0, s1, s2;
    stage_entry(g0, g1, g2, g3, px0, py0, s0, s1, s2);
    // K-track's own plane layout: operands that meet in one packed (two binary32 lanes) instruction sit in aligned pairs --
    //   plane 0 (P, R, Q, S), plane 1 (U0, V0, E', F'): (un, vn) = (ly, ly) (Q, S) + ((lx, lx) (P, R) + (U0, V0))
    //   plane 3 (r, g, b, n.z), plane 4 (n.x, n.y, opacity, m.z): the forward's accumulations take (r, g), (b, n.z), (n.x, n.y)
    // Per lane the operations and their order are those of pair.cuh / k_forward: the results are bit-identical.
    sh[0][tid] = make_float4(s0.x, s1.x, s0.y, s1.y); sh[1][tid] = make_float4(s0.z, s1.z, s0.w, s1.w); sh[2][tid] = s2;
    sh[3][tid] = make_float4(g3.w, g4.x, g4.y, g5.x);
    const float aux = g5.y, auy = g5.z, auz = g5.w, avx = g6.x, avy = g6.y, avz = g6.z;
    sh[5][tid] = make_float4(aux, auy, auz, avx);
    sh[6][tid] = make_float4(avy, avz, auy * avz - auz * avy, auz * avx - aux * avz);
    sh[4][tid] = make_float4(g4.z, g4.w, g1.w, aux * avy - auy * avx);
    return refine_patch_mask(warp_patch_mask(g7, tx0, ty0), s0, s1, s2, g1.w, cfg.cutoff2, cfg.alpha_min);
}

// (u, v) and rho^2 of one pair (pair.cuh's sequence)
__device__ __forceinline__ float pair_rho2(const float4 s0, const float4 s1, const float4 s2, float lx, float ly, float& u,
                                           float& v) {
    // s0 = (P, R, Q, S), s1 = (U0, V0, E', F') (stage_track): un and vn in two packed FMAs
    const float2 uvn = __ffma2_rn(make_float2(ly, ly), make_float2(s0.z, s0.w),
                                  __ffma2_rn(make_float2(lx, lx), make_float2(s0.x, s0.y), make_float2(s1.x, s1.y)));
    const float dn = __fmaf_rn(ly, s1.w, __fmaf_rn(lx, s1.z, s2.x));
    const float inv = fast_rcp(dn);
    u = __fmul_rn(uvn.x, inv); v = __fmul_rn(uvn.y, inv);
    return __fmaf_rn(v, v, __fmul_rn(u, u));
}

// (out of line: inlined it cost the walks registers)
__device__ __noinline__ bool hist_sort_call(unsigned long long* g, uint32_t n, unsigned long long* sk, uint32_t* sw, uint32_t* s_misc, int tid) {
    return hist_sort_keys(g, n, sk, sw, s_misc, tid, g);
}

template <bool WRITE_IMAGES, bool NDEPTH>
__global__ void __launch_bounds__(SGS_BLOCK, 3)
k_track(uint32_t* tile_order, uint32_t* __restrict__ ranges, const uint32_t* cursor, unsigned long long* bucket, uint32_t tile_cap,
        int presorted, SgsPayload pay, int W, int H, int tiles_x, float fx, float fy, float cx, float cy, SgsCfgDev cfg,
        TrackPlanes out, const float* __restrict__ trgb, const float* __restrict__ tdepth, float lambda_d, float nsign,
        float* __restrict__ pose_partial, SgsCounters* __restrict__ counters, float* __restrict__ d_pose6,
        float* __restrict__ loss_out, uint32_t* __restrict__ tile_cost, uint32_t* cursor_rw, SgsCounters* __restrict__ counters_snap,
        unsigned int* host_flag, unsigned int flag_val, float* split_state, unsigned int* split_flag, unsigned int helper_delay_ns,
        int n_help) {
    const long long t_start = clock64();
    cudaTriggerProgrammaticLaunchCompletion();  // the next iteration's K-pre-B may be staged; it waits for this grid before it reads anything
    __shared__ float4 sh[7][TRK_CAP];
    __shared__ unsigned long long s_keys[TRK_CAP];
    __shared__ unsigned char sh_mask[TRK_CAP];
    __shared__ float s_red[8][7];
    __shared__ uint32_t s_wmax[8];
    const uint32_t sa = smem_addr(&sh[0][0]), sm_a = smem_addr(sh_mask);
    // blocks [0, n_help) are HELPERS of the n_help tiles predicted longest (tile_order[0 .. n_help)); block n_help + k owns tile_order[k]
    const bool helper = (int)blockIdx.x < n_help;
    const int slot = helper ? (int)blockIdx.x : (int)blockIdx.x - n_help;
    const int tile = (int)tile_order[slot];  // longest tiles first (order written by the previous launch)
    const int crank = helper ? 1 : 0;
    const bool has_helper = !helper && slot < n_help;
    const int tx = tile % tiles_x, ty = tile / tiles_x;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int lxi = (wid & 1) * 8 + (lane & 7), lyi = (wid >> 1) * 4 + (lane >> 3);
    const int px = tx * SGS_TILE + lxi, py = ty * SGS_TILE + lyi;
    const bool inside = px < W && py < H;
    const float lx = (float)lxi, ly = (float)lyi;
    const float tx0 = (float)(tx * SGS_TILE), ty0 = (float)(ty * SGS_TILE);
    const double px0 = (double)(tx * SGS_TILE) + 0.5, py0 = (double)(ty * SGS_TILE) + 0.5;
    const size_t pix = (size_t)py * W + px, HW = (size_t)W * H;

    // (the hand-over epoch of split tiles, see below: fetched here, with the frame's pixel, so that no later load depends on it)
    const unsigned int epoch_raw = n_help > 0 ? __ldcg(split_flag + SGS_TRACK_HELPERS) : 0u;
    // the current frame's pixel: issued first, consumed after the forward walk
    float tr = 0.f, tg = 0.f, tb = 0.f, td = 0.f;
    if (inside) { tr = __ldg(trgb + pix); tg = __ldg(trgb + HW + pix); tb = __ldg(trgb + 2 * HW + pix); td = __ldg(tdepth + pix); }

    // ---- forward walk over the staged batch [boff, boff + nb) (Eq. 8, as k_forward) ----
    float T = 1.f;
    float2 DO = make_float2(0.f, 0.f);   // (Dp, O): O + w * 1 is O + w exactly
#define Dp DO.x
#define O DO.y
    float2 C01 = make_float2(0.f, 0.f), C2N2 = make_float2(0.f, 0.f), N01 = make_float2(0.f, 0.f);   // (C0, C1), (C2, N2), (N0, N1)
#define C0 C01.x
#define C1 C01.y
#define C2 C2N2.x
#define N2 C2N2.y
#define N0 N01.x
#define N1 N01.y
    uint32_t last = 0;
    bool done = !inside;
    auto forward_walk = [&](const uint32_t boff, const uint32_t nb, const uint32_t j0 = 0u) {  // slots [j0, nb), j0 % 32 == 0
        for (uint32_t c0 = j0; c0 < nb; c0 += 32) {
            if (__all_sync(0xffffffffu, done)) break;  // per-warp early stop on saturation
            unsigned m = __ballot_sync(0xffffffffu, (lds_u8(sm_a + c0 + lane) >> wid) & 1u);
            while (m) {
                // TRK_K entries per trip, in three phases.  The time of a tile is the serial walk of its slowest
                // warp (profiles/r01_c2_track.md: a handful of 230-entry tiles set the whole kernel's duration at
                // ~180 cycles per entry), so everything that does not depend on the running transmittance --
                // loads, intersection, rho^2, z, G, alpha -- is evaluated for all TRK_K entries side by side
                // (phase 1), the T / stop recurrence is a few dependent instructions per entry (phase 2), and
                // the eight accumulations follow (phase 3).  Operations and their order per pixel are k_forward's.
                uint32_t ea[TRK_K], jl[TRK_K];
                float al[TRK_K], zz[TRK_K];
                bool anyv = false;
#pragma unroll
                for (int k = 0; k < TRK_K; ++k) {
                    const bool has = m != 0u;
                    const uint32_t j = has ? c0 + (uint32_t)__ffs(m) - 1u : c0;
                    m &= m - 1u;
                    jl[k] = boff + j + 1u;
                    ea[k] = sa + j * 16u;
                    const float4 s0 = lds128(ea[k]), s1 = lds128(ea[k] + TRK_PL), s2 = lds128(ea[k] + 2 * TRK_PL);
                    const float opac = lds32(ea[k] + 4 * TRK_PL + 8);
                    float u, v;
                    const float rho2 = pair_rho2(s0, s1, s2, lx, ly, u, v);
                    const float z = __fmaf_rn(s2.z, v, __fmaf_rn(s2.y, u, s2.w));
                    const float G = fast_ex2(__fmul_rn(rho2, -0.72134752044448170368f));
                    const float a = fminf(cfg.alpha_max, __fmul_rn(opac, G));
                    const bool valid = has && (rho2 <= cfg.cutoff2) && (z > cfg.z_near) && (a >= cfg.alpha_min);
                    al[k] = valid ? a : 0.f;  // alpha_min > 0 or not, a valid pair has a > 0 or contributes nothing
                    zz[k] = z;
                    anyv = anyv || valid;
                }
                if (!__any_sync(0xffffffffu, anyv && !done)) continue;
#pragma unroll
                for (int k = 0; k < TRK_K; ++k) {
                    const float a = al[k];
                    bool pass = !done && (a > 0.f);
                    const float Tn = __fmul_rn(T, 1.f - a);
                    const bool stop = pass && (Tn < cfg.t_min);  // R6: stop, this splat is not composited
                    done = done || stop;
                    pass = pass && !stop;
                    const float w = pass ? __fmul_rn(a, T) : 0.f;
                    T = pass ? Tn : T;
                    last = pass ? jl[k] : last;
                    const float4 s3 = lds128(ea[k] + 3 * TRK_PL), s4 = lds128(ea[k] + 4 * TRK_PL);
                    const float2 w2 = make_float2(w, w);
                    C01 = __ffma2_rn(w2, make_float2(s3.x, s3.y), C01);
                    C2N2 = __ffma2_rn(w2, make_float2(s3.z, s3.w), C2N2);
                    N01 = __ffma2_rn(w2, make_float2(s4.x, s4.y), N01);
                    DO = __ffma2_rn(w2, make_float2(zz[k], 1.f), DO);
                }
            }
        }
    };

    // ---- Eq. 15-19 in registers (same arithmetic as loss.cu): loss term and upstream gradients of rgb, depth ----
    const float rx = ((float)px + 0.5f - cx) / fx, ry = ((float)py + 0.5f - cy) / fy;  // pixel ray (rx, ry, 1)
    float g0 = 0.f, g1 = 0.f, g2 = 0.f, g3 = 0.f, my_loss = 0.f;
    // SGS_FLAG_NORMALISED_DEPTH: the depth image and the loss take D_n = D / O; its upstream g
    // becomes dL/dD = g / O (kept in g3) and dL/dO = -g3 D_n, which the walk back carries as g3 (z - zref), zref = D_n
    float zref = 0.f;
    auto finish_forward = [&]() {
        if (NDEPTH) {
            const float io = O > 0.f ? __frcp_rn(O) : 0.f;
            Dp = __fmul_rn(Dp, io);
            zref = Dp;
        }
        if (WRITE_IMAGES && inside) {
            if (out.p[0]) out.p[0][pix] = C0;
            if (out.p[1]) out.p[1][pix] = C1;
            if (out.p[2]) out.p[2][pix] = C2;
            if (out.p[3]) out.p[3][pix] = Dp;
            if (out.p[4]) out.p[4][pix] = N0;
            if (out.p[5]) out.p[5][pix] = N1;
            if (out.p[6]) out.p[6][pix] = N2;
            if (out.p[7]) out.p[7][pix] = O;
        }
        if (inside) {
            const float inv = 1.f / (float)HW;
            const float nr = N0 * rx + N1 * ry + N2;
            if ((nsign * nr > 0.f) && (O > 0.95f)) {  // M_n M_o (Eq. 17-18)
                float d = C0 - tr; my_loss += fabsf(d); g0 = d > 0.f ? inv : (d < 0.f ? -inv : 0.f);
                d = C1 - tg; my_loss += fabsf(d); g1 = d > 0.f ? inv : (d < 0.f ? -inv : 0.f);
                d = C2 - tb; my_loss += fabsf(d); g2 = d > 0.f ? inv : (d < 0.f ? -inv : 0.f);
                d = (td > 0.f && isfinite(td)) ? Dp - td : 0.f;  // R25: holes of the sensor depth carry no depth term
                my_loss += lambda_d * fabsf(d);
                g3 = d > 0.f ? lambda_d * inv : (d < 0.f ? -lambda_d * inv : 0.f);
                if (NDEPTH) g3 *= __frcp_rn(O);  // O > 0.95 here
            }
            my_loss *= inv;
        }
        if (!(g0 != 0.f || g1 != 0.f || g2 != 0.f || g3 != 0.f)) last = 0;  // every backward term carries a factor g
    };

    // ---- reverse walk over the staged batch (as k_backward<POSE_ONLY>, g_normal = g_alpha = 0) ----
    float T_after = 1.f, suffix = 0.f;
    float F2 = 0.f, Z2 = 0.f;
    float2 F01 = make_float2(0.f, 0.f), Z01 = make_float2(0.f, 0.f);
#define F0 F01.x
#define F1 F01.y
#define Z0 Z01.x
#define Z1 Z01.y
    auto backward_walk = [&](const uint32_t boff, const int jend) {  // entries [0, jend) of the staged batch, back to front
        for (int c0 = ((jend - 1) >> 5) << 5; c0 >= 0 && jend > 0; c0 -= 32) {
            unsigned m = __ballot_sync(0xffffffffu, (c0 + lane < jend) && ((lds_u8(sm_a + c0 + lane) >> wid) & 1u));
            while (m) {
                // TRK_K entries per trip, back to front, phases as in the forward walk: pair evaluation, 1/(1-a)
                // and g.v side by side; then the T_i / suffix recurrence (4 dependent instructions per entry);
                // then the geometric chain of each hit.
                uint32_t ea[TRK_K];
                PairResult r[TRK_K];
                float inv1ma[TRK_K], gv[TRK_K], opac[TRK_K], da[TRK_K], w[TRK_K];
                bool hit[TRK_K];
                bool anyh = false;
#pragma unroll
                for (int k = 0; k < TRK_K; ++k) {
                    const bool has = m != 0u;
                    const int hb = has ? 31 - __clz(m) : 0;
                    m &= ~(1u << hb);
                    const uint32_t j = (uint32_t)(c0 + hb);
                    ea[k] = sa + j * 16u;
                    const float4 s0 = lds128(ea[k]), s1 = lds128(ea[k] + TRK_PL), s2 = lds128(ea[k] + 2 * TRK_PL);
                    const float4 s3 = lds128(ea[k] + 3 * TRK_PL);
                    // branch-free pair evaluation (pair.cuh's sequence and decisions, no early exits) so that the four
                    // LDS -> FMA -> RCP -> EX2 chains of the trip are scheduled side by side
                    const float rho2 = pair_rho2(s0, s1, s2, lx, ly, r[k].u, r[k].v);
                    r[k].z = __fmaf_rn(s2.z, r[k].v, __fmaf_rn(s2.y, r[k].u, s2.w));
                    r[k].G = fast_ex2(__fmul_rn(rho2, -0.72134752044448170368f));
                    const float op = lds32(ea[k] + 4 * TRK_PL + 8);
                    r[k].a = fminf(cfg.alpha_max, __fmul_rn(op, r[k].G));
                    hit[k] = has && (boff + j) < last && (rho2 <= cfg.cutoff2) && (r[k].z > cfg.z_near) && (r[k].a >= cfg.alpha_min);
                    opac[k] = op;
                    inv1ma[k] = fast_rcp(1.f - r[k].a);
                    gv[k] = g0 * s3.x + g1 * s3.y + g2 * s3.z + g3 * (NDEPTH ? r[k].z - zref : r[k].z);
                    anyh = anyh || hit[k];
                }
                if (!__any_sync(0xffffffffu, anyh)) continue;
#pragma unroll
                for (int k = 0; k < TRK_K; ++k) {  // the recurrence: 4 dependent instructions per hit
                    const float Ti = T_after * inv1ma[k];  // transmittance in front of this splat
                    const float wk = r[k].a * Ti;
                    const float dak = Ti * gv[k] - suffix * inv1ma[k];
                    w[k] = hit[k] ? wk : 0.f;
                    da[k] = hit[k] ? dak : 0.f;
                    suffix = hit[k] ? fmaf(wk, gv[k], suffix) : suffix;
                    T_after = hit[k] ? Ti : T_after;
                }
#pragma unroll
                for (int k = 0; k < TRK_K; ++k) {  // the geometric chain, predicated per lane (no divergent branches)
                    const float4 s5 = lds128(ea[k] + 5 * TRK_PL), s6 = lds128(ea[k] + 6 * TRK_PL);
                    const float m2 = lds32(ea[k] + 4 * TRK_PL + 12);
                    const bool clamped = opac[k] * r[k].G > cfg.alpha_max;  // R5: true derivative, zero when clamped
                    const float dG = clamped ? 0.f : da[k] * opac[k];
                    const float gu = -r[k].u * r[k].G * dG, gvv = -r[k].v * r[k].G * dG, gz = g3 * w[k];
                    // f = [ r x (a_v gu - a_u gv) + m gz ] / (r . m)
                    const float q0 = s5.w * gu - s5.x * gvv, q1 = s6.x * gu - s5.y * gvv, q2 = s6.y * gu - s5.z * gvv;
                    const float m0 = s6.z, m1 = s6.w;
                    const float inv_rm = fast_rcp(rx * m0 + ry * m1 + m2);
                    const float f0 = hit[k] ? (ry * q2 - q1 + m0 * gz) * inv_rm : 0.f;
                    const float f1 = hit[k] ? (q0 - rx * q2 + m1 * gz) * inv_rm : 0.f;
                    const float f2 = hit[k] ? (rx * q1 - ry * q0 + m2 * gz) * inv_rm : 0.f;
                    const float zk = hit[k] ? r[k].z : 0.f;  // a rejected pair may carry inf / NaN
                    F01 = __fadd2_rn(F01, make_float2(f0, f1)); F2 += f2;
                    Z01 = __ffma2_rn(make_float2(zk, zk), make_float2(f0, f1), Z01); Z2 = fmaf(zk, f2, Z2);
                }
            }
        }
    };
    auto warp_max_last = [&]() {
        uint32_t wmax = last;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) wmax = max(wmax, __shfl_xor_sync(0xffffffffu, wmax, o));
        return wmax;
    };

    // ---- tile list: order the bucket by (depth bits, index) (tilesort.cu's contract) ----
    const uint32_t raw = cursor[tile];
    const uint32_t n = raw < tile_cap ? raw : tile_cap;
    const uint32_t start = tile * tile_cap;
    unsigned long long* g = bucket + (size_t)start;
    if (tid == 0) { ranges[2 * tile] = start; ranges[2 * tile + 1] = start + n; }

    // split tiles: both blocks of the cluster work; otherwise block 1 has nothing to do (it still writes a zero row of
    // partial sums and draws its ticket below, so that the grid reduction counts every block)
    const bool split = (helper || has_helper) && !presorted && n > TRK_SPLIT_MIN && n <= (uint32_t)TRK_CAP;
    const uint32_t msp = split ? (((n + 1u) / 2u + 31u) & ~31u) : n;  // block 0: [0, msp) on the way back, block 1: [msp, n)
    // per-pixel state the owner hands to its helper: 6 x 256 floats in global memory, published by the flag value
    // 4 * epoch + 2; the epoch is a device word (split_flag[SGS_TRACK_HELPERS]) that the launch's last block increments, so
    // a replayed CUDA graph -- whose kernel arguments are frozen -- never meets a flag value left by an earlier replay.
    // Owner and helper both rank the tile's RAW bucket by themselves, at the same time: the owner of a split tile therefore
    // does not write the sorted keys back in place (a helper scheduled late would rank a half-permuted bucket);
    // sgs_get_binning's export ranks short buckets itself (tilesort.cu, k_export_copy).
    float* st = split_state + (size_t)slot * (8 * SGS_BLOCK);  // g0..g3, T, last, zref (NDEPTH), one spare
    const unsigned int epoch4 = 4u * epoch_raw;
    volatile unsigned int* my_flag = reinterpret_cast<volatile unsigned int*>(split_flag + slot);
    if (crank == 1) {
        if (split) {
            if (helper_delay_ns) __nanosleep(helper_delay_ns);  // (test hook: SGS_DEBUG_HELPER_DELAY_NS, see sgs_create)
            for (uint32_t e = tid; e < (uint32_t)TRK_CAP; e += SGS_BLOCK) {
                s_keys[e] = e < n ? g[e] : ~0ull;   // the raw bucket: nobody writes it during this launch
                sh_mask[e] = 0;
            }
            __syncthreads();
            for (uint32_t e0 = 0; e0 < n; e0 += SGS_BLOCK) {
                if (e0 + (uint32_t)(wid * 32) < n) {
                    const uint32_t e = e0 + tid;
                    const bool mine = e < n;
                    const unsigned long long key = mine ? s_keys[e] : ~0ull;
                    uint32_t rank = 0;
                    for (uint32_t k = 0; k < n; ++k) rank += s_keys[k] < key ? 1u : 0u;
                    if (mine && rank >= msp)   // this block's part of the sorted list, at slot rank - msp
                        sh_mask[rank - msp] = (unsigned char)stage_track(pay, (uint32_t)key, px0, py0, tx0, ty0, sh, (int)(rank - msp), cfg);
                }
            }
            __syncthreads();
            if (tid == 0) {  // the owner has walked forward and stored these pixels' state
                while (*my_flag != epoch4 + 2u) __nanosleep(200);
                __threadfence();
            }
            __syncthreads();
            g0 = __ldcg(st + tid); g1 = __ldcg(st + SGS_BLOCK + tid); g2 = __ldcg(st + 2 * SGS_BLOCK + tid);
            g3 = __ldcg(st + 3 * SGS_BLOCK + tid); T_after = __ldcg(st + 4 * SGS_BLOCK + tid);
            last = __float_as_uint(__ldcg(st + 5 * SGS_BLOCK + tid));
            if (NDEPTH) zref = __ldcg(st + 6 * SGS_BLOCK + tid);
            const uint32_t wmax = warp_max_last();
            backward_walk(msp, (int)min(n - msp, wmax > msp ? wmax - msp : 0u));
        }
    } else if (!presorted && n <= TRK_CAP) {
        // ===== one batch (the common case in tracking): rank the keys by counting (they are unique), stage each
        // entry straight into the slot of its rank, walk forward, then walk the SAME staged records back.
        // No barrier between the two walks: a warp needs only its own pixels' state. =====
        for (uint32_t e = tid; e < (uint32_t)TRK_CAP; e += SGS_BLOCK) {
            s_keys[e] = e < n ? g[e] : ~0ull;
            sh_mask[e] = 0;
        }
        __syncthreads();
        for (uint32_t e0 = 0; e0 < n; e0 += SGS_BLOCK) {
            if (e0 + (uint32_t)(wid * 32) < n) {  // only warps that own keys walk the list
                const uint32_t e = e0 + tid;
                const bool mine = e < n;
                const unsigned long long key = mine ? s_keys[e] : ~0ull;
                uint32_t rank = 0;
                for (uint32_t k = 0; k < n; ++k) rank += s_keys[k] < key ? 1u : 0u;
                if (mine) {
                    if (!split) g[rank] = key;  // sorted list for sgs_get_binning (a split tile's bucket stays raw: its helper ranks it too)
                    sh_mask[rank] = (unsigned char)stage_track(pay, (uint32_t)key, px0, py0, tx0, ty0, sh, (int)rank, cfg);
                }
            }
        }
        __syncthreads();
        if (!split) {
            forward_walk(0u, n);
            finish_forward();
            T_after = T;
            backward_walk(0u, (int)min(n, warp_max_last()));
        } else {
            forward_walk(0u, msp);
            const float Tm = T, C0m = C0, C1m = C1, C2m = C2, Dpm = Dp;  // the pixel's state between the two parts
            const float Om = O;
            forward_walk(0u, n, msp);
            const float Draw = Dp;  // (finish_forward<NDEPTH> turns Dp into D / O)
            finish_forward();
            // hand (g, T_final, last) of this pixel to the helper
            st[tid] = g0; st[SGS_BLOCK + tid] = g1; st[2 * SGS_BLOCK + tid] = g2; st[3 * SGS_BLOCK + tid] = g3;
            st[4 * SGS_BLOCK + tid] = T; st[5 * SGS_BLOCK + tid] = __uint_as_float(last);
            if (NDEPTH) st[6 * SGS_BLOCK + tid] = zref;
            __threadfence();
            __syncthreads();
            if (tid == 0) *my_flag = epoch4 + 2u;
            // the way back over [0, msp): transmittance behind entry msp - 1 and the suffix sum of everything behind it,
            // sum_{j >= msp} w_j (g . v_j) = g . (V_final - V_msp) with V the running accumulators of Eq. 8
            T_after = Tm;
            suffix = g0 * (C0 - C0m) + g1 * (C1 - C1m) + g2 * (C2 - C2m) +
                     g3 * (NDEPTH ? (Draw - Dpm) - zref * (O - Om) : Draw - Dpm);
            backward_walk(0u, (int)min(msp, warp_max_last()));
        }
    } else {
        // ===== general path: 256-entry batches front to back, then back to front (restaging what was evicted) =====
        // Lists longer than the staging capacity (C5: a quarter of the tiles, 41 % of the entries): counting pass over the depth +
        // rank inside a depth bin (histsort.cuh, linear in n; scratch = the staging planes), keys back to the bucket; it declines
        // buckets whose depths crowd into one bin, which take the bitonic network.  (Lists of up to TRK_CAP keys keep the rank by
        // counting above: measured, the counting sort there gains nothing on C5 and costs C2 3 %.)
        static_assert(sizeof(float4) * 7 * TRK_CAP >= 2048 * 8 + HS_SCRATCH_WORDS * 4 && sizeof(s_red) >= 32 * 4, "");
        unsigned long long* hs_keys = reinterpret_cast<unsigned long long*>(&sh[0][0]);
        if (!presorted && n <= 2048u && hist_sort_call(g, n, hs_keys, reinterpret_cast<uint32_t*>(hs_keys + 2048), reinterpret_cast<uint32_t*>(&s_red[0][0]), tid)) {
        } else if (!presorted) {  // bitonic network in the staging memory, sorted keys back to the bucket
            unsigned long long* sk = reinterpret_cast<unsigned long long*>(&sh[0][0]);
            uint32_t npad = 512;
            while (npad < n) npad <<= 1;
            for (uint32_t i = tid; i < npad; i += SGS_BLOCK) sk[i] = i < n ? g[i] : ~0ull;
            __syncthreads();
            for (uint32_t k = 2; k <= npad; k <<= 1)
                for (uint32_t j = k >> 1; j > 0; j >>= 1) {
                    for (uint32_t t = tid; t < (npad >> 1); t += SGS_BLOCK) {
                        const uint32_t i = ((t & ~(j - 1)) << 1) | (t & (j - 1)), p = i | j;
                        const unsigned long long a = sk[i], b = sk[p];
                        if ((a > b) == ((i & k) == 0)) { sk[i] = b; sk[p] = a; }
                    }
                    __syncthreads();
                }
            for (uint32_t i = tid; i < n; i += SGS_BLOCK) g[i] = sk[i];
            __syncthreads();  // sorted bucket visible to the block; staging memory free
        }
        int staged_b = -1;  // batch currently held in shared memory
        for (uint32_t boff = 0; boff < n; boff += SGS_BLOCK) {
            if (__syncthreads_and(done)) break;
            const uint32_t nb = min((uint32_t)SGS_BLOCK, n - boff);
            unsigned mask = 0;
            // plain loads: the bucket may just have been rewritten by this block
            if ((uint32_t)tid < nb) mask = stage_track(pay, (uint32_t)g[boff + tid], px0, py0, tx0, ty0, sh, tid, cfg);
            sh_mask[tid] = (unsigned char)mask;
            staged_b = (int)(boff / SGS_BLOCK);
            __syncthreads();
            forward_walk(boff, nb);
        }
        finish_forward();
        T_after = T;
        const uint32_t wmax = warp_max_last();
        if (lane == 0) s_wmax[wid] = wmax;
        __syncthreads();  // also: every warp has left the forward walk
        uint32_t bmax = 0;
#pragma unroll
        for (int w2 = 0; w2 < 8; ++w2) bmax = max(bmax, s_wmax[w2]);
        const int n_batches = (int)((bmax + SGS_BLOCK - 1) / SGS_BLOCK);
        for (int b = n_batches - 1; b >= 0; --b) {
            const uint32_t boff = (uint32_t)b * SGS_BLOCK;
            const uint32_t nb = min((uint32_t)SGS_BLOCK, bmax - boff);
            if (b != staged_b) {  // block-uniform
                __syncthreads();  // previous batch fully consumed
                unsigned mask = 0;
                if ((uint32_t)tid < nb) mask = stage_track(pay, (uint32_t)g[boff + tid], px0, py0, tx0, ty0, sh, tid, cfg);
                sh_mask[tid] = (unsigned char)mask;
                staged_b = b;
                __syncthreads();
            }
            backward_walk(boff, (int)min(nb, wmax > boff ? wmax - boff : 0u));
        }
    }
    // Eq. 11-13 per pixel: rho += sum f; theta += r x sum(z f)   (g_N = 0 in tracking)
    float p6[7];
    p6[0] = F0; p6[1] = F1; p6[2] = F2;
    p6[3] = ry * Z2 - Z1; p6[4] = Z0 - rx * Z2; p6[5] = rx * Z1 - ry * Z0;
    p6[6] = my_loss;
#pragma unroll
    for (int c = 0; c < 7; ++c) {
        const float s = warp_sum(inside ? p6[c] : 0.f);
        if (lane == 0) s_red[wid][c] = s;
    }
    __syncthreads();
    if (tid < 7) {
        float s = 0.f;
#pragma unroll
        for (int w2 = 0; w2 < 8; ++w2) s += s_red[w2][tid];
        pose_partial[(size_t)blockIdx.x * 8 + tid] = s;
    }
    if (tid == 0 && crank == 0) tile_cost[tile] = (uint32_t)((clock64() - t_start) >> 8);  // feedback for the next iteration's order
    // A tile bucket that overflowed (entries dropped) or a kept survivor list the device-resident pose has left (splats
    // possibly missing) must not pass for a result: the iteration's loss and pose gradient are NaN.  Under SGS_FLAG_GRAPH and
    // with SGS_FLAG_ASYNC nothing else tells the caller in time (the host sees the counters one call later, or never).
    if (!finish_pose(pose_partial, gridDim.x, counters, d_pose6, loss_out, tile_cap)) return;
    if (host_flag) {  // sgs_track_iter_host: d_pose6 / loss_out are pinned HOST memory; publish them before the housekeeping below
        if (tid < 7) __threadfence_system();
        __syncthreads();
        if (tid == 0) *reinterpret_cast<volatile unsigned int*>(host_flag) = flag_val;
    }
    // ---- last block: housekeeping for the next iteration (the tile order is k_track_order's, off this stream) ----
    const int tiles = (int)gridDim.x - n_help;
    // ... and the next preprocess finds its counters and per-tile cursors already zeroed (every block of this launch
    // has read its cursor; the host copied the counters before this kernel started)
    for (int t = tid; t < tiles; t += SGS_BLOCK) cursor_rw[t] = 0u;
    if (tid == 0) {
        if (counters_snap) *counters_snap = *counters;  // what the host reads for overflow detection and hints
        counters->n_entries = 0ull; counters->n_visible = 0u; counters->overflow = 0u; counters->ticket_pre = 0u;
        counters->max_tile = 0u; counters->n_surv = 0u; counters->stale = 0u;
        if (n_help > 0) atomicAdd(split_flag + SGS_TRACK_HELPERS, 1u);  // next launch's epoch (every block of this one is past its hand-over); a RED: nothing waits for a load
    }
}

// Longest-first tile order for the NEXT iteration.  One block per tile, and tiles differ several-fold in work (C2: 20 k ..
// 100 k cycles), so a launch ends when its long tiles end: they have to start first.  Every block of K-track has stored
// the cycles it took (tile_cost); consecutive tracking iterations differ by a small pose step, so those costs predict
// the next iteration's.  Counting sort of the tiles by cost, descending, into tile_order.  Ties land in arbitrary order;
// the order steers scheduling, never a result.  Its own one-block kernel on the context's stream since the timeline of
// profiles/r01_c2_track.md: inside K-track's last block these 2.4 us sat between the last tile and the next K-pre-B.
__global__ void __launch_bounds__(SGS_BLOCK)
k_track_order(const uint32_t* __restrict__ tile_cost, uint32_t* __restrict__ tile_order, int tiles) {
    __shared__ unsigned int s_hist[TRK_ORDER_BINS];
    __shared__ uint32_t s_wmax[8];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    for (int b = tid; b < TRK_ORDER_BINS; b += SGS_BLOCK) s_hist[b] = 0;
    __syncthreads();
    constexpr int ORD_U = 8;  // one pass covers ORD_U * 256 = 2048 tiles with the keys kept in registers
    unsigned int kb[ORD_U];
    auto load_keys = [&](int t0) {
#pragma unroll
        for (int k = 0; k < ORD_U; ++k) {
            const int t = t0 + k * SGS_BLOCK;
            kb[k] = t < tiles ? min(__ldcg(tile_cost + t), (unsigned int)(TRK_ORDER_BINS - 1)) : 0xffffffffu;
        }
    };
    for (int t0 = tid; t0 < tiles; t0 += ORD_U * SGS_BLOCK) {
        load_keys(t0);
#pragma unroll
        for (int k = 0; k < ORD_U; ++k)
            if (kb[k] != 0xffffffffu) atomicAdd(&s_hist[kb[k]], 1u);
    }
    __syncthreads();
    // exclusive scan over the bins from the largest cost down: thread k owns a contiguous run of bins
    constexpr int PER = TRK_ORDER_BINS / SGS_BLOCK;
    unsigned int local = 0;
#pragma unroll
    for (int k = 0; k < PER; ++k) local += s_hist[TRK_ORDER_BINS - 1 - (tid * PER + k)];
    unsigned int incl = local;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
        const unsigned int t2 = __shfl_up_sync(0xffffffffu, incl, off);
        if (lane >= off) incl += t2;
    }
    if (lane == 31) s_wmax[wid] = incl;
    __syncthreads();
    unsigned int run = incl - local;
    for (int w2 = 0; w2 < wid; ++w2) run += s_wmax[w2];
#pragma unroll
    for (int k = 0; k < PER; ++k) {
        const int b = TRK_ORDER_BINS - 1 - (tid * PER + k);
        const unsigned int c2 = s_hist[b];
        s_hist[b] = run;  // first output slot of this bin
        run += c2;
    }
    __syncthreads();
    const bool one_pass = tiles <= ORD_U * SGS_BLOCK;
    for (int t0 = tid; t0 < tiles; t0 += ORD_U * SGS_BLOCK) {
        if (!one_pass) load_keys(t0);
#pragma unroll
        for (int k = 0; k < ORD_U; ++k)
            if (kb[k] != 0xffffffffu) tile_order[atomicAdd(&s_hist[kb[k]], 1u)] = (uint32_t)(t0 + k * SGS_BLOCK);
    }
}

__global__ void k_iota(uint32_t* __restrict__ p, int n) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) p[i] = (uint32_t)i;
}

#undef F0
#undef F1
#undef Z0
#undef Z1
#undef Dp
#undef O
#undef C0
#undef C1
#undef C2
#undef N0
#undef N1
#undef N2
}  // namespace

cudaError_t sgs_launch_track(sgs_ctx* c, float* const planes[8], const float* trgb, const float* tdepth, float lambda_d,
                             float nsign, float* d_pose6, float* loss, bool after_preprocess, cudaStream_t s) {
    const int tiles = c->camd.tiles_x * c->camd.tiles_y;
    const SgsCamDev& cam = c->camd;
    TrackPlanes out;
    bool any = false;
    for (int i = 0; i < 8; ++i) { out.p[i] = planes ? planes[i] : nullptr; any = any || out.p[i] != nullptr; }
    // the order written by the previous iteration's k_track_order (on the ctx's stream) must be complete
    if (c->order_pending) {
        if (cudaStreamWaitEvent(s, c->order_done, 0) != cudaSuccess) return cudaErrorUnknown;
        c->order_pending = false;
    }
    if (!(c->cost_tiles == tiles && c->cost_W == cam.W && c->cost_H == cam.H)) {  // no order yet for this camera
        k_iota<<<(tiles + 255) / 256, 256, 0, s>>>(c->tile_order, tiles);
        c->launches += 1;
    }
    SgsStage st(c, SGS_STAGE_TRACK, s);
    c->launches += 1;
    unsigned long long* bucket = reinterpret_cast<unsigned long long*>(c->bucket);
    const int presorted = c->fused_sort ? 0 : 1;
    // (A programmatic dependent launch of THIS kernel behind K-pre-B was measured twice: 3459 -> 2888 MP/s when K-pre-B
    // triggered at its start, and no change (4483 vs 4468) with the trigger behind K-pre-B's own wait and the target-pixel
    // loads in front of this kernel's wait; profiles/r01_c2_track.md.  The other edge, K-pre-B behind this kernel, pays.)
    const uint32_t tile_cap = (uint32_t)c->tile_cap;
    SgsCounters* snap = after_preprocess ? c->counters_snap + c->snap_slot : nullptr;
    unsigned int* hflag = c->host_flag_want ? c->host_flag_dev : nullptr;  // (sgs_track_iter_host)
    const bool ndepth = (c->cfg.flags & SGS_FLAG_NORMALISED_DEPTH) != 0;
    const int n_help = (c->split_state && tiles >= 4 * SGS_TRACK_HELPERS) ? SGS_TRACK_HELPERS : 0;
    c->host_flag_armed = hflag != nullptr;
#define SGS_TRK_ARGS c->tile_order, c->ranges, c->cursor, bucket, tile_cap, presorted, c->pay, cam.W, cam.H, cam.tiles_x, cam.fx, cam.fy, cam.cx, \
                     cam.cy, c->cfgd, out, trgb, tdepth, lambda_d, nsign, c->pose_partial, c->counters, d_pose6, loss, c->tile_cost, c->cursor,   \
                     snap, hflag, c->host_flag_val, c->split_state, c->split_flag, c->helper_delay_ns, n_help
    if (ndepth) {
        if (any) k_track<true, true><<<tiles + n_help, SGS_BLOCK, 0, s>>>(SGS_TRK_ARGS);
        else k_track<false, true><<<tiles + n_help, SGS_BLOCK, 0, s>>>(SGS_TRK_ARGS);
    } else {
        if (any) k_track<true, false><<<tiles + n_help, SGS_BLOCK, 0, s>>>(SGS_TRK_ARGS);
        else k_track<false, false><<<tiles + n_help, SGS_BLOCK, 0, s>>>(SGS_TRK_ARGS);
    }
#undef SGS_TRK_ARGS
    if (!c->order_skip) {   // next iteration's tile order from this launch's measured tile costs, beside the next K-pre-B
        cudaStream_t os = c->aux_stream ? c->aux_stream : s;
        if (os != s && (cudaEventRecord(c->order_fork, s) != cudaSuccess || cudaStreamWaitEvent(os, c->order_fork, 0) != cudaSuccess))
            return cudaErrorUnknown;
        c->launches += 1;
        k_track_order<<<1, SGS_BLOCK, 0, os>>>(c->tile_cost, c->tile_order, tiles);
        if (os != s) { if (cudaEventRecord(c->order_done, os) != cudaSuccess) return cudaErrorUnknown; c->order_pending = true; }
    }
    c->cost_tiles = tiles; c->cost_W = cam.W; c->cost_H = cam.H;
    c->prezero_tiles = tiles;
    return cudaGetLastError();
}
