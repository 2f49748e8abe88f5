// backward.cu -- K-bwd, K-sbwd and the pose reductions.
//
// K-bwd walks each tile's list in REVERSE from the last composited entry of each pixel, recomputes
// the pair with the forward's exact instruction sequence (pair.cuh), recovers T_i = T_{i+1}/(1-a_i)
// and keeps one scalar suffix  sum_{j>i} w_j (g.v_j)  so that
//     dL/da_i = T_i (g.v_i) - suffix / (1 - a_i)                       (derivative of Eq. 8).
// The geometric chain is taken in camera space as a "force" on the splat's plane:
// the constraint  mu_c + a_u u + a_v v = z r  (Eq. 1, 3-4; r = pixel ray, a_u = s_u t_uc) gives
//     f = [ r x (a_v g_u - a_u g_v) + (a_u x a_v) g_z ] / (r . (a_u x a_v))
//     dL/dmu_c = sum f,  dL/d(s_u t_uc) = sum u f,  dL/d(s_v t_vc) = sum v f
// which IS the matrix dL/dH_c of Eq. 9 (= W^T dL/dT) accumulated directly.
//   full mode     : 16 values per (warp, surfel) are summed over the warp through a shared-memory scratch (16 transposed
//                   STS per lane, 4 LDS.128 + packed adds over half a row, one shuffle joins the halves) and land as ONE
//                   64-byte red.global.add per warp into acc[surfel][16]; k_surfel_backward finishes per surfel.
//   pose-only mode: Eq. 11-13 applied per pixel: dL/drho = sum f, dL/dtheta = r x sum z f + N x g_N;
//                   no per-surfel traffic at all -- registers -> block -> grid reduction to 6 values.
#include "pair.cuh"
#include "sgs_internal.h"
#include "reduce.cuh"

namespace {

struct CPlanes { const float* p[8]; };

constexpr int BWD_K = 2;  // entries per trip of the reverse walk
#ifndef SGS_BWD_MIN_BLOCKS
#define SGS_BWD_MIN_BLOCKS 4
#endif

struct StagedBwd {
    float4 s0, s1, s2, s3, s4;  // as StagedFwd
    float4 s5;                  // a_u.xyz, a_v.x
    float4 s6;                  // a_v.yz, m.xy      (m = a_u x a_v); m.z rides in s4.w
};

// FUSED (pose-only only): `up` holds the RENDERED planes of the last forward and the upstream gradients of the
// tracking loss (Eq. 15-19, same arithmetic as loss.cu) are formed in registers -- no loss kernel, no
// upstream images through HBM; the loss itself rides in slot 6 of the pose partials.
struct FusedLoss { const float* trgb; const float* tdepth; float lambda_d, nsign; float* loss; };

template <bool POSE_ONLY, bool FUSED, bool NDEPTH, bool LOWPASS = false>
__global__ void __launch_bounds__(SGS_BLOCK, SGS_BWD_MIN_BLOCKS)
k_backward(const uint32_t* __restrict__ tile_order, const uint32_t* __restrict__ ranges, const uint32_t* __restrict__ vals, int vstride, SgsPayload pay, int W, int H,
           int tiles_x, float fx, float fy, float cx, float cy, SgsCfgDev cfg, CPlanes up,
           const float* __restrict__ T_final, const uint32_t* __restrict__ n_last, float* __restrict__ acc,
           float* __restrict__ pose_partial, SgsCounters* __restrict__ counters, float* __restrict__ d_pose6,
           FusedLoss fl, const float2* __restrict__ dn_state) {
    __shared__ StagedBwd sh[SGS_BLOCK];
    __shared__ unsigned char sh_mask[SGS_BLOCK];
    __shared__ uint32_t sh_v[SGS_BLOCK];  // surfel (accumulator) index of each staged entry
    // full mode: per-warp scratch of the 16-value reduction, [value][lane] with rows padded to 36 words
    __shared__ float red_s[POSE_ONLY ? 1 : 8 * 16 * 36];
    __shared__ float s_red[8][7];
    const int tile = tile_order ? (int)tile_order[blockIdx.x] : (int)blockIdx.x;  // longest tiles first
    const int tx = tile % tiles_x, ty = tile / tiles_x;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int lxi = (wid & 1) * 8 + (lane & 7), lyi = (wid >> 1) * 4 + (lane >> 3);
    const int px = tx * SGS_TILE + lxi, py = ty * SGS_TILE + lyi;
    const bool inside = px < W && py < H;
    const float lx = (float)lxi, ly = (float)lyi;
    const float2 lx2 = make_float2(lx, lx), ly2 = make_float2(ly, ly);
    const double px0 = (double)(tx * SGS_TILE) + 0.5, py0 = (double)(ty * SGS_TILE) + 0.5;
    const uint32_t start = ranges[2 * tile];

    float g[8];
    float T_after = 1.f;
    uint32_t last = 0;
    float my_loss = 0.f;
    const float rx = ((float)px + 0.5f - cx) / fx, ry = ((float)py + 0.5f - cy) / fy;  // pixel ray (rx, ry, 1)
#pragma unroll
    for (int c = 0; c < 8; ++c) g[c] = 0.f;
    if (inside) {
        const size_t pix = (size_t)py * W + px;
        if (FUSED) {
            const size_t HW = (size_t)W * H;
            const float inv = 1.f / (float)HW;
            const float nr = up.p[4][pix] * rx + up.p[5][pix] * ry + up.p[6][pix];
            if ((fl.nsign * nr > 0.f) && (up.p[7][pix] > 0.95f)) {   // M_n M_o (Eq. 17-18)
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    const float d = up.p[c][pix] - fl.trgb[c * HW + pix];
                    my_loss += fabsf(d);
                    g[c] = d > 0.f ? inv : (d < 0.f ? -inv : 0.f);
                }
                const float td = fl.tdepth[pix];
                const float d = (td > 0.f && isfinite(td)) ? up.p[3][pix] - td : 0.f;  // R25: holes carry no depth term
                my_loss += fl.lambda_d * fabsf(d);
                g[3] = d > 0.f ? fl.lambda_d * inv : (d < 0.f ? -fl.lambda_d * inv : 0.f);
            }
            my_loss *= inv;
        } else {
#pragma unroll
            for (int c = 0; c < 8; ++c) g[c] = up.p[c] ? up.p[c][pix] : 0.f;
        }
        if (NDEPTH) {  // SGS_FLAG_NORMALISED_DEPTH: g[3] is dL/dD_n; D_n = D / O  =>  dL/dD = g / O, dL/dO -= g D_n / O
            const float2 dn = dn_state[pix];
            g[3] *= dn.y;
            g[7] = __fmaf_rn(-g[3], dn.x, g[7]);
        }
        T_after = T_final[pix];
        last = n_last[pix];
        // every term of the backward carries a factor g: a pixel whose upstream gradient is exactly zero
        // (e.g. masked out by M_n M_o in tracking, Eq. 17-19) contributes exactly nothing -- skip its list
        bool nz = false;
#pragma unroll
        for (int c = 0; c < 8; ++c) nz = nz || (g[c] != 0.f);
        if (!nz) last = 0;
    }
    float suffix = 0.f;
    float F0 = 0.f, F1 = 0.f, F2 = 0.f, Z0 = 0.f, Z1 = 0.f, Z2 = 0.f, Nn0 = 0.f, Nn1 = 0.f, Nn2 = 0.f;
    float E0 = 0.f, E1 = 0.f, E2 = 0.f;  // R28, pose-only: sum of Z_c (d x f) over screen-term pairs, d = (ddx / fx, ddy / fy, 0)

    // block-wide maximum of `last` decides how many batches exist
    uint32_t wmax = last;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) wmax = max(wmax, __shfl_xor_sync(0xffffffffu, wmax, o));
    __shared__ uint32_t s_wmax[8];
    if (lane == 0) s_wmax[wid] = wmax;
    __syncthreads();
    uint32_t bmax = 0;
#pragma unroll
    for (int w2 = 0; w2 < 8; ++w2) bmax = max(bmax, s_wmax[w2]);

    const int n_batches = (int)((bmax + SGS_BLOCK - 1) / SGS_BLOCK);
    for (int b = n_batches - 1; b >= 0; --b) {
        const uint32_t boff = (uint32_t)b * SGS_BLOCK;
        const uint32_t nb = min((uint32_t)SGS_BLOCK, bmax - boff);
        __syncthreads();  // previous batch fully consumed
        unsigned pmask = 0;
        if ((uint32_t)tid < nb) {
            const uint32_t v = vals[(size_t)(start + boff + tid) * vstride];
            const float4 g0 = pay.g0[v], g1 = pay.g1[v], g3 = pay.g3[v], g4 = pay.g4[v], g5 = pay.g5[v], g6 = pay.g6[v];
            pmask = warp_patch_mask(pay.g7[v], (float)(tx * SGS_TILE), (float)(ty * SGS_TILE));
            const double2 g2 = pay.g2[v];
            StagedBwd st;
            float xy0[2];
            float4 t0, t1;
            stage_entry(g0, g1, g2, g3, px0, py0, t0, t1, st.s2, xy0);
            // (P, R, Q, S) and (U0, V0, E', F'): the operands of the packed (un, vn) in aligned pairs, as in K-track
            st.s0 = make_float4(t0.x, t1.x, t0.y, t1.y); st.s1 = make_float4(t0.z, t1.z, t0.w, t1.w);

            st.s3 = make_float4(g1.w, g3.w, g4.x, g4.y);
            st.s4 = make_float4(g4.z, g4.w, g5.x, 0.f);  // .w <- m.z below
            const float aux = g5.y, auy = g5.z, auz = g5.w, avx = g6.x, avy = g6.y, avz = g6.z;
            st.s5 = make_float4(aux, auy, auz, avx);
            st.s6 = make_float4(avy, avz, auy * avz - auz * avy, auz * avx - aux * avz);
            st.s4.w = aux * avy - auy * avx;
            // R28: the record has no spare slot and the kernel's static shared memory is at its 48 KB limit, so under the flag
            // the pixel-minus-centre offsets of the tile's first pixel take m.x, m.y's place and m = a_u x a_v is rebuilt per pair
            if (LOWPASS) { st.s6.z = xy0[0]; st.s6.w = xy0[1]; }
            sh_v[tid] = v;
            sh[tid] = st;
            if (!LOWPASS) pmask = refine_patch_mask(pmask, t0, t1, st.s2, g1.w, cfg.cutoff2, cfg.alpha_min);
        }
        sh_mask[tid] = (unsigned char)pmask;
        __syncthreads();
        // entries at or after the warp's largest `last` were composited by none of its pixels
        const int jend = (int)min(nb, wmax > boff ? wmax - boff : 0u);  // exclusive
        for (int c0 = ((jend - 1) >> 5) << 5; c0 >= 0 && jend > 0; c0 -= 32) {
          // this chunk's entries whose AABB reaches the warp's patch, walked from the back
          unsigned m = __ballot_sync(0xffffffffu, (c0 + lane < jend) && ((sh_mask[c0 + lane] >> wid) & 1u));
          while (m) {
            // BWD_K entries per trip, back to front, in phases (see track.cu): branch-free pair evaluation,
            // 1/(1-a) and g.v of all entries side by side; then the T_i / suffix recurrence (4 dependent
            // instructions per hit); then the geometric chain of each entry some lane hit.
            int jj[BWD_K];
            PairResult r[BWD_K];
            float inv1ma[BWD_K], gv[BWD_K], opac[BWD_K], da[BWD_K], w[BWD_K];
            float ddx[BWD_K], ddy[BWD_K], zc[BWD_K];   // R28 only
            bool hit[BWD_K], use2d[BWD_K];
#pragma unroll
            for (int k = 0; k < BWD_K; ++k) {
                const bool has = m != 0u;
                const int hb = has ? 31 - __clz(m) : 0;
                m &= ~(1u << hb);
                const int j = c0 + hb;
                jj[k] = j;
                const float4 s0 = sh[j].s0, s1 = sh[j].s1, s2 = sh[j].s2, s3 = sh[j].s3, s4 = sh[j].s4;
                const float2 uvn = __ffma2_rn(ly2, make_float2(s0.z, s0.w), __ffma2_rn(lx2, make_float2(s0.x, s0.y), make_float2(s1.x, s1.y)));
                const float dn = __fmaf_rn(ly, s1.w, __fmaf_rn(lx, s1.z, s2.x));
                const float inv = fast_rcp(dn);
                r[k].u = __fmul_rn(uvn.x, inv); r[k].v = __fmul_rn(uvn.y, inv);
                float rho2 = __fmaf_rn(r[k].v, r[k].v, __fmul_rn(r[k].u, r[k].u));
                r[k].z = __fmaf_rn(s2.z, r[k].v, __fmaf_rn(s2.y, r[k].u, s2.w));
                use2d[k] = false;
                if (LOWPASS) {   // R28, the forward's sequence: rho^2 = min(u^2 + v^2, 2 |x - x_c|^2), centre depth where the screen term wins
                    const float4 xy = sh[j].s6;
                    ddx[k] = __fadd_rn(lx, xy.z); ddy[k] = __fadd_rn(ly, xy.w); zc[k] = s2.w;
                    const float r2 = __fmul_rn(2.f, __fmaf_rn(ddy[k], ddy[k], __fmul_rn(ddx[k], ddx[k])));
                    use2d[k] = !(rho2 <= r2);
                    rho2 = use2d[k] ? r2 : rho2;
                    r[k].z = use2d[k] ? s2.w : r[k].z;
                }
                r[k].G = fast_ex2(__fmul_rn(rho2, -0.72134752044448170368f));
                r[k].a = fminf(cfg.alpha_max, __fmul_rn(s3.x, r[k].G));
                hit[k] = has && (boff + (uint32_t)j) < last && (rho2 <= cfg.cutoff2) && (r[k].z > cfg.z_near) &&
                         (r[k].a >= cfg.alpha_min);
                opac[k] = s3.x;
                inv1ma[k] = fast_rcp(1.f - r[k].a);
                gv[k] = g[0] * s3.y + g[1] * s3.z + g[2] * s3.w + g[3] * r[k].z + g[4] * s4.x + g[5] * s4.y + g[6] * s4.z + g[7];
            }
#pragma unroll
            for (int k = 0; k < BWD_K; ++k) {
                const float Ti = T_after * inv1ma[k];  // transmittance in front of this splat
                const float wk = r[k].a * Ti;
                const float dak = Ti * gv[k] - suffix * inv1ma[k];
                w[k] = hit[k] ? wk : 0.f;
                da[k] = hit[k] ? dak : 0.f;
                suffix = hit[k] ? fmaf(wk, gv[k], suffix) : suffix;
                T_after = hit[k] ? Ti : T_after;
            }
#pragma unroll
            for (int k = 0; k < BWD_K; ++k) {
                if (!__any_sync(0xffffffffu, hit[k])) continue;
                const int j = jj[k];
                const float4 s4 = sh[j].s4, s5 = sh[j].s5, s6 = sh[j].s6;
                const bool clamped = opac[k] * r[k].G > cfg.alpha_max;  // R5: true derivative, zero when clamped
                const float dG = clamped ? 0.f : da[k] * opac[k];
                const float gu = -r[k].u * r[k].G * dG, gvv = -r[k].v * r[k].G * dG, gz = g[3] * w[k];
                // f = [ r x (a_v gu - a_u gv) + m gz ] / (r . m)
                const float q0 = s5.w * gu - s5.x * gvv, q1 = s6.x * gu - s5.y * gvv, q2 = s6.y * gu - s5.z * gvv;
                const float m0 = LOWPASS ? s5.y * s6.y - s5.z * s6.x : s6.z, m1 = LOWPASS ? s5.z * s5.w - s5.x * s6.y : s6.w, m2 = s4.w;
                const float inv_rm = fast_rcp(rx * m0 + ry * m1 + m2);
                // a rejected pair may carry inf / NaN: its lanes contribute exact zeros
                float f0 = hit[k] ? (ry * q2 - q1 + m0 * gz) * inv_rm : 0.f;
                float f1 = hit[k] ? (q0 - rx * q2 + m1 * gz) * inv_rm : 0.f;
                float f2 = hit[k] ? (rx * q1 - ry * q0 + m2 * gz) * inv_rm : 0.f;
                float uk = hit[k] ? r[k].u : 0.f, vk = hit[k] ? r[k].v : 0.f;
                const float zk = hit[k] ? r[k].z : 0.f;
                if (LOWPASS) {
                    // R28, screen term: G = exp(-|x - x_c|^2) and z = Z_c depend on the centre only.  dL/dx_c = 2 ddx G dL/dG;
                    // x_c = fx X / Z + cx  =>  the force on mu_c is (gxc fx, gyc fy, -(gxc (x_c - cx) + gyc (y_c - cy))) / Z + (0, 0, gz),
                    // with x_c - cx = fx rx - ddx; the tangents get nothing (u f = v f = 0).
                    const float gxc = 2.f * ddx[k] * r[k].G * dG, gyc = 2.f * ddy[k] * r[k].G * dG, iz = fast_rcp(zc[k]);
                    const bool s2d = hit[k] && use2d[k];
                    f0 = s2d ? gxc * fx * iz : f0;
                    f1 = s2d ? gyc * fy * iz : f1;
                    f2 = s2d ? gz - (gxc * (fx * rx - ddx[k]) + gyc * (fy * ry - ddy[k])) * iz : f2;
                    uk = s2d ? 0.f : uk; vk = s2d ? 0.f : vk;
                    if (POSE_ONLY && s2d) {   // mu_c x f = Z_c (r - d) x f, d = (ddx / fx, ddy / fy, 0): the r part rides in Z0..Z2
                        const float dxr = zc[k] * ddx[k] / fx, dyr = zc[k] * ddy[k] / fy;
                        E0 = fmaf(dyr, f2, E0); E1 = fmaf(-dxr, f2, E1); E2 = fmaf(dxr, f1, fmaf(-dyr, f0, E2));
                    }
                }
                if (POSE_ONLY) {
                    F0 += f0; F1 += f1; F2 += f2;
                    Z0 = fmaf(zk, f0, Z0); Z1 = fmaf(zk, f1, Z1); Z2 = fmaf(zk, f2, Z2);
                    Nn0 = fmaf(w[k], s4.x, Nn0); Nn1 = fmaf(w[k], s4.y, Nn1); Nn2 = fmaf(w[k], s4.z, Nn2);
                } else {
                    float x[16];
                    x[0] = f0; x[1] = f1; x[2] = f2;
                    x[3] = uk * f0; x[4] = uk * f1; x[5] = uk * f2;
                    x[6] = vk * f0; x[7] = vk * f1; x[8] = vk * f2;
                    {   // six products w * g as three packed multiplies (g[4], g[5]), (g[6], g[0]), (g[1], g[2])
                        const float2 w2 = make_float2(w[k], w[k]);
                        const float2 a45 = __fmul2_rn(w2, make_float2(g[4], g[5])), a60 = __fmul2_rn(w2, make_float2(g[6], g[0])),
                                     a12 = __fmul2_rn(w2, make_float2(g[1], g[2]));
                        x[9] = a45.x; x[10] = a45.y; x[11] = a60.x; x[12] = a60.y; x[13] = a12.x; x[14] = a12.y;
                    }
                    x[15] = (clamped || !hit[k]) ? 0.f : da[k] * r[k].G;
                    // Sum of the 16 values over the warp through shared memory (ncu: the register butterfly -- 16 SHFL,
                    // 30 SEL, 16 FADD -- was 32 % of this kernel's instructions; removing it altogether saved 95 us per
                    // C3/C4 view): every lane stores its 16 values transposed (conflict-free), then lane l adds 16 of the
                    // 32 entries of row l & 15 (four LDS.128, conflict-free per quarter-warp thanks to the 36-word
                    // rows) and one shuffle joins the two halves; the shuffle is also the barrier before the next store.
                    float* rs = red_s + wid * (16 * 36);
#pragma unroll
                    for (int q = 0; q < 16; ++q) rs[q * 36 + lane] = x[q];
                    __syncwarp();
                    const float4* rp = reinterpret_cast<const float4*>(rs + (lane & 15) * 36 + (lane >> 4) * 16);
                    const float4 v0 = rp[0], v1 = rp[1], v2 = rp[2], v3 = rp[3];
                    // packed adds (FADD2: two binary32 sums per issue slot; the kernel is issue-bound): 7 + 1 instead of 15
                    const float2 h0 = __fadd2_rn(__fadd2_rn(make_float2(v0.x, v0.y), make_float2(v0.z, v0.w)),
                                                 __fadd2_rn(make_float2(v1.x, v1.y), make_float2(v1.z, v1.w)));
                    const float2 h1 = __fadd2_rn(__fadd2_rn(make_float2(v2.x, v2.y), make_float2(v2.z, v2.w)),
                                                 __fadd2_rn(make_float2(v3.x, v3.y), make_float2(v3.z, v3.w)));
                    const float2 hs = __fadd2_rn(h0, h1);
                    float red = hs.x + hs.y;
                    red += __shfl_xor_sync(0xffffffffu, red, 16);
                    if (lane < 16) atomicAdd(acc + (size_t)sh_v[j] * SGS_ACC_STRIDE + lane, red);
                }
            }
          }
        }
    }
    if (POSE_ONLY) {
        // Eq. 11-13 per pixel: rho += sum f; theta += X x f summed = r x sum(z f), plus t_nc x dL/dt_nc = N x g_N
        float p6[7];
        p6[6] = my_loss;
        p6[0] = F0; p6[1] = F1; p6[2] = F2;
        p6[3] = (ry * Z2 - Z1) + (Nn1 * g[6] - Nn2 * g[5]) - E0;
        p6[4] = (Z0 - rx * Z2) + (Nn2 * g[4] - Nn0 * g[6]) - E1;
        p6[5] = (rx * Z1 - ry * Z0) + (Nn0 * g[5] - Nn1 * g[4]) - E2;
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
            pose_partial[(size_t)tile * 8 + tid] = s;
        }
        finish_pose(pose_partial, gridDim.x, counters, d_pose6, FUSED ? fl.loss : nullptr);
    }
}


// K-sbwd: one thread per VISIBLE surfel.  Eq. 9-10 (with R11, R13): the accumulator already holds
// dL/dH_c = [dL/d(s_u t_uc), dL/d(s_v t_vc), dL/dmu_c] and dL/dt_nc; this applies the product rule
// to (s, t), rotates to world space, goes through R(q/|q|), and forms the surfel's share of the
// pose gradient (Eq. 11-13).  Leaves acc[v] zeroed for the next backward.
__global__ void __launch_bounds__(256)
k_surfel_backward(const SgsCounters* __restrict__ counters, const uint32_t* __restrict__ vis_to_surfel,
                  const uint8_t* __restrict__ culled,
                  float* __restrict__ acc, SgsPayload pay,
                  const float* __restrict__ quat, SgsCamDev cam, sgs_surfel_grads out,
                  float* __restrict__ pose_partial, SgsCounters* __restrict__ counters_rw,
                  float* __restrict__ d_pose6, int survivors, int accumulate) {
    __shared__ float s_red[8][6];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    // compacted mode: v < N_v, surfel = vis_to_surfel[v]; bucket mode (no compaction): v = surfel index
    // grid-stride over the surfels: a bounded grid keeps the per-block ticket of the pose reduction off the
    // critical path (one same-address atomic per block)
    float p6[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
    // list: the visible surfels, compact (radix binning: vis_to_surfel, acc indexed by the list position; bucket binning:
    // K-pre-B's vis_list, acc indexed by the surfel itself: `survivors` != 0).  Everything else -- inactive, culled --
    // keeps the zeros the launcher's memsets wrote.
    const unsigned int n_loop = counters->n_visible;
    for (unsigned int v = blockIdx.x * blockDim.x + tid; v < n_loop; v += gridDim.x * blockDim.x) {
    const uint32_t i = vis_to_surfel[v];
    {
        float a[16];
        float4* ap = reinterpret_cast<float4*>(acc + (size_t)(survivors ? i : v) * SGS_ACC_STRIDE);
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            const float4 t = ap[c];
            a[4 * c] = t.x; a[4 * c + 1] = t.y; a[4 * c + 2] = t.z; a[4 * c + 3] = t.w;
            ap[c] = make_float4(0.f, 0.f, 0.f, 0.f);
        }
        const float qw0 = quat[4 * i], qx0 = quat[4 * i + 1], qy0 = quat[4 * i + 2], qz0 = quat[4 * i + 3];
        const float qn = sqrtf(qw0 * qw0 + qx0 * qx0 + qy0 * qy0 + qz0 * qz0);
        const float qi = 1.f / qn;
        const float qw = qw0 * qi, qx = qx0 * qi, qy = qy0 * qi, qz = qz0 * qi;
        // The camera-space frame comes from the splat's payload record (contiguous, still in L2 from the compositing
        // kernels) instead of the map's mean / scale arrays (two or three more scattered DRAM sectors per splat; this
        // kernel moves 900 B of DRAM per visible splat at 5 % issue utilisation, profiles/r02_c4.md): a_u = s_u t_uc and
        // a_v = s_v t_vc give the scales as their lengths, n_c is t_nc, and mu_c = ((x_c - cx) / fx, (y_c - cy) / fy, 1) z_c.
        const size_t pv = survivors ? (size_t)i : (size_t)v;
        const float4 g3 = pay.g3[pv], g4 = pay.g4[pv], g5 = pay.g5[pv], g6 = pay.g6[pv];
        const double2 g2 = pay.g2[pv];
        const float au[3] = {g5.y, g5.z, g5.w}, av[3] = {g6.x, g6.y, g6.z};
        const float su = sqrtf(au[0] * au[0] + au[1] * au[1] + au[2] * au[2]), sv = sqrtf(av[0] * av[0] + av[1] * av[1] + av[2] * av[2]);
        const float isu = 1.f / su, isv = 1.f / sv;
        const float tuc[3] = {au[0] * isu, au[1] * isu, au[2] * isu}, tvc[3] = {av[0] * isv, av[1] * isv, av[2] * isv};
        const float tnc[3] = {g4.z, g4.w, g5.x};
        const float zc = g3.z;
        const float muc[3] = {(float)((g2.x - (double)cam.cx) / (double)cam.fx) * zc, (float)((g2.y - (double)cam.cy) / (double)cam.fy) * zc, zc};
        const float* dmu = a;        // dL/dmu_c
        const float* dau = a + 3;    // dL/d(s_u t_uc)
        const float* dav = a + 6;    // dL/d(s_v t_vc)
        const float* dtn = a + 9;    // dL/dt_nc
        float dtu[3], dtv[3];
#pragma unroll
        for (int r = 0; r < 3; ++r) { dtu[r] = su * dau[r]; dtv[r] = sv * dav[r]; }
        // sgs_backward_accumulate: this view's gradient is ADDED to what the window has so far (one thread per surfel and
        // kernel, kernels of a window in stream order: plain read-modify-write)
        auto put = [accumulate](float* p, float v) { *p = accumulate ? *p + v : v; };
        if (out.scale) {
            put(out.scale + 2 * i, tuc[0] * dau[0] + tuc[1] * dau[1] + tuc[2] * dau[2]);
            put(out.scale + 2 * i + 1, tvc[0] * dav[0] + tvc[1] * dav[1] + tvc[2] * dav[2]);
        }
        if (out.opacity) put(out.opacity + i, a[15]);
        if (out.rgb) { put(out.rgb + 3 * i, a[12]); put(out.rgb + 3 * i + 1, a[13]); put(out.rgb + 3 * i + 2, a[14]); }
        // pose share: rho += dmu; theta += mu_c x dmu + t_uc x dtu + t_vc x dtv + t_nc x dtn   (Eq. 13)
        p6[0] += dmu[0]; p6[1] += dmu[1]; p6[2] += dmu[2];
        p6[3] += (muc[1] * dmu[2] - muc[2] * dmu[1]) + (tuc[1] * dtu[2] - tuc[2] * dtu[1]) +
                (tvc[1] * dtv[2] - tvc[2] * dtv[1]) + (tnc[1] * dtn[2] - tnc[2] * dtn[1]);
        p6[4] += (muc[2] * dmu[0] - muc[0] * dmu[2]) + (tuc[2] * dtu[0] - tuc[0] * dtu[2]) +
                (tvc[2] * dtv[0] - tvc[0] * dtv[2]) + (tnc[2] * dtn[0] - tnc[0] * dtn[2]);
        p6[5] += (muc[0] * dmu[1] - muc[1] * dmu[0]) + (tuc[0] * dtu[1] - tuc[1] * dtu[0]) +
                (tvc[0] * dtv[1] - tvc[1] * dtv[0]) + (tnc[0] * dtn[1] - tnc[1] * dtn[0]);
        // world space: x_c = R_cw x_w  =>  dL/dx_w = R_cw^T dL/dx_c
        float G[3][3];  // dL/dR (world), columns t_u, t_v, t_n
#pragma unroll
        for (int r = 0; r < 3; ++r) {
            const float c0 = cam.Rf[r], c1 = cam.Rf[3 + r], c2 = cam.Rf[6 + r];
            if (out.mean) put(out.mean + 3 * i + r, c0 * dmu[0] + c1 * dmu[1] + c2 * dmu[2]);
            G[r][0] = c0 * dtu[0] + c1 * dtu[1] + c2 * dtu[2];
            G[r][1] = c0 * dtv[0] + c1 * dtv[1] + c2 * dtv[2];
            G[r][2] = c0 * dtn[0] + c1 * dtn[1] + c2 * dtn[2];
        }
        if (out.quat) {
            float dq[4];
            dq[0] = 2.f * (-qz * G[0][1] + qy * G[0][2] + qz * G[1][0] - qx * G[1][2] - qy * G[2][0] + qx * G[2][1]);
            dq[1] = 2.f * (qy * G[0][1] + qz * G[0][2] + qy * G[1][0] - 2.f * qx * G[1][1] - qw * G[1][2] + qz * G[2][0] +
                           qw * G[2][1] - 2.f * qx * G[2][2]);
            dq[2] = 2.f * (-2.f * qy * G[0][0] + qx * G[0][1] + qw * G[0][2] + qx * G[1][0] + qz * G[1][2] - qw * G[2][0] +
                           qz * G[2][1] - 2.f * qy * G[2][2]);
            dq[3] = 2.f * (-2.f * qz * G[0][0] - qw * G[0][1] + qx * G[0][2] + qw * G[1][0] - 2.f * qz * G[1][1] +
                           qy * G[1][2] + qx * G[2][0] + qy * G[2][1]);
            const float qd = qw * dq[0] + qx * dq[1] + qy * dq[2] + qz * dq[3];
            put(out.quat + 4 * i, (dq[0] - qw * qd) * qi);
            put(out.quat + 4 * i + 1, (dq[1] - qx * qd) * qi);
            put(out.quat + 4 * i + 2, (dq[2] - qy * qd) * qi);
            put(out.quat + 4 * i + 3, (dq[3] - qz * qd) * qi);
        }
    }
    }
    if (d_pose6 == nullptr) return;
#pragma unroll
    for (int c = 0; c < 6; ++c) {
        const float s = warp_sum(p6[c]);
        if (lane == 0) s_red[wid][c] = s;
    }
    __syncthreads();
    if (tid < 6) {
        float s = 0.f;
#pragma unroll
        for (int w2 = 0; w2 < 8; ++w2) s += s_red[w2][tid];
        pose_partial[(size_t)blockIdx.x * 8 + tid] = s;
    }
    finish_pose(pose_partial, gridDim.x, counters_rw, d_pose6);
}

}  // namespace

cudaError_t sgs_launch_backward(sgs_ctx* c, const float* const up[8], const sgs_surfel_grads* dg, float* d_pose6,
                                bool accumulate, cudaStream_t s) {
    SgsStage st(c, SGS_STAGE_BACKWARD, s);
    const int tiles = c->camd.tiles_x * c->camd.tiles_y;
    CPlanes u;
    for (int i = 0; i < 8; ++i) u.p[i] = up[i];
    const SgsCamDev& cam = c->camd;
    const float2* dn = (c->cfg.flags & SGS_FLAG_NORMALISED_DEPTH) ? c->dn_state : nullptr;
    if (dg == nullptr) {  // pose-only (tracking, L204)
        if (d_pose6 == nullptr) return cudaSuccess;
        c->launches += 1;
        if (c->cfgd.lowpass) k_backward<true, false, false, true><<<tiles, SGS_BLOCK, 0, s>>>(c->render_order_valid ? c->render_order : nullptr, c->ranges, c->list_vals, c->list_stride, c->pay, cam.W, cam.H, cam.tiles_x,
                                                     cam.fx, cam.fy, cam.cx, cam.cy, c->cfgd, u, c->T_final, c->n_last,
                                                     c->acc, c->pose_partial, c->counters, d_pose6, FusedLoss{}, dn);
        else if (dn) k_backward<true, false, true><<<tiles, SGS_BLOCK, 0, s>>>(c->render_order_valid ? c->render_order : nullptr, c->ranges, c->list_vals, c->list_stride, c->pay, cam.W, cam.H, cam.tiles_x,
                                                     cam.fx, cam.fy, cam.cx, cam.cy, c->cfgd, u, c->T_final, c->n_last,
                                                     c->acc, c->pose_partial, c->counters, d_pose6, FusedLoss{}, dn);
        else k_backward<true, false, false><<<tiles, SGS_BLOCK, 0, s>>>(c->render_order_valid ? c->render_order : nullptr, c->ranges, c->list_vals, c->list_stride, c->pay, cam.W, cam.H, cam.tiles_x,
                                                     cam.fx, cam.fy, cam.cx, cam.cy, c->cfgd, u, c->T_final, c->n_last,
                                                     c->acc, c->pose_partial, c->counters, d_pose6, FusedLoss{}, dn);
        return cudaGetLastError();
    }
    const int64_t n = c->last_surfels.n;
    cudaError_t e = cudaSuccess;
    // exact zeros for every surfel the per-surfel kernel does not visit (inactive, culled): 52 B per surfel of plain
    // HBM writes that nothing before k_surfel_backward depends on -- forked onto the ctx's own stream so that they run
    // beside the issue-bound k_backward, joined in front of k_surfel_backward
    // (sgs_backward_accumulate: nothing is zeroed -- surfels this view does not see keep what the window has so far)
    cudaStream_t ms = c->aux_stream ? c->aux_stream : s;
    const bool fill = !accumulate;
    if (ms != s && fill) {
        if ((e = cudaEventRecord(c->fork_ev, s)) != cudaSuccess) return e;
        if ((e = cudaStreamWaitEvent(ms, c->fork_ev, 0)) != cudaSuccess) return e;
    }
    if (fill)
    if (dg->mean && e == cudaSuccess) e = cudaMemsetAsync(dg->mean, 0, sizeof(float) * 3 * (size_t)n, ms);
    if (fill && dg->scale && e == cudaSuccess) e = cudaMemsetAsync(dg->scale, 0, sizeof(float) * 2 * (size_t)n, ms);
    if (fill && dg->quat && e == cudaSuccess) e = cudaMemsetAsync(dg->quat, 0, sizeof(float) * 4 * (size_t)n, ms);
    if (fill && dg->opacity && e == cudaSuccess) e = cudaMemsetAsync(dg->opacity, 0, sizeof(float) * (size_t)n, ms);
    if (fill && dg->rgb && e == cudaSuccess) e = cudaMemsetAsync(dg->rgb, 0, sizeof(float) * 3 * (size_t)n, ms);
    if (e != cudaSuccess) return e;
    if (ms != s && fill && (e = cudaEventRecord(c->join_ev, ms)) != cudaSuccess) return e;
    c->launches += 1;
    if (c->cfgd.lowpass) k_backward<false, false, false, true><<<tiles, SGS_BLOCK, 0, s>>>(c->render_order_valid ? c->render_order : nullptr, c->ranges, c->list_vals, c->list_stride, c->pay, cam.W, cam.H, cam.tiles_x,
                                                  cam.fx, cam.fy, cam.cx, cam.cy, c->cfgd, u, c->T_final, c->n_last,
                                                  c->acc, c->pose_partial, c->counters, nullptr, FusedLoss{}, dn);
    else if (dn) k_backward<false, false, true><<<tiles, SGS_BLOCK, 0, s>>>(c->render_order_valid ? c->render_order : nullptr, c->ranges, c->list_vals, c->list_stride, c->pay, cam.W, cam.H, cam.tiles_x,
                                                  cam.fx, cam.fy, cam.cx, cam.cy, c->cfgd, u, c->T_final, c->n_last,
                                                  c->acc, c->pose_partial, c->counters, nullptr, FusedLoss{}, dn);
    else k_backward<false, false, false><<<tiles, SGS_BLOCK, 0, s>>>(c->render_order_valid ? c->render_order : nullptr, c->ranges, c->list_vals, c->list_stride, c->pay, cam.W, cam.H, cam.tiles_x,
                                                  cam.fx, cam.fy, cam.cx, cam.cy, c->cfgd, u, c->T_final, c->n_last,
                                                  c->acc, c->pose_partial, c->counters, nullptr, FusedLoss{}, dn);
    // SGS_FLAG_LAZY_GRADS: the per-surfel kernel (latency-bound: 12 % issue utilisation) stays on the ctx's stream, behind
    // k_backward by an event, and the caller's stream does NOT wait for it: sgs_wait_grads does (the next view's kernels
    // run meanwhile).  Otherwise the caller's stream joins here.
    const bool lazy = (c->cfg.flags & SGS_FLAG_LAZY_GRADS) != 0 && ms != s;
    cudaStream_t ks = lazy ? ms : s;
    if (lazy) {
        if ((e = cudaEventRecord(c->fork_ev, s)) != cudaSuccess) return e;       // k_backward enqueued
        if ((e = cudaStreamWaitEvent(ms, c->fork_ev, 0)) != cudaSuccess) return e;
    } else if (ms != s && fill && (e = cudaStreamWaitEvent(s, c->join_ev, 0)) != cudaSuccess) return e;
    // one thread per listed surfel; the list length is only known on the device: grid-stride from a hinted grid
    const bool bucket_mode = c->list_stride == 2;
    int64_t want = n;
    if (c->last_vis > 0 && c->last_vis + c->last_vis / 4 < want) want = c->last_vis + c->last_vis / 4;
    int blocks = (int)((want + 255) / 256);
    if (blocks > 148 * 8) blocks = 148 * 8;
    if (n == 0) return d_pose6 ? cudaMemsetAsync(d_pose6, 0, sizeof(float) * 6, ks) : cudaSuccess;
    if (blocks < 1) blocks = 1;
    c->launches += 1;
    c->grads_on_aux = lazy;
    k_surfel_backward<<<blocks, 256, 0, ks>>>(c->counters, bucket_mode ? c->vis_list : c->vis_to_surfel, c->culled, c->acc, c->pay,
                                             c->last_surfels.quat, cam, *dg, c->pose_partial,
                                             c->counters, d_pose6, bucket_mode ? 1 : 0, accumulate ? 1 : 0);
    return cudaGetLastError();
}

// Tracking iteration backward with the Eq. 15-19 loss fused in (pose-only): see FusedLoss.
cudaError_t sgs_launch_backward_tracking(sgs_ctx* c, const float* trgb, const float* tdepth, float lambda_d, float nsign,
                                         float* d_pose6, float* loss, cudaStream_t s) {
    SgsStage st(c, SGS_STAGE_BACKWARD, s);
    const int tiles = c->camd.tiles_x * c->camd.tiles_y;
    CPlanes u;
    for (int i = 0; i < 8; ++i) u.p[i] = c->last_img[i];
    const SgsCamDev& cam = c->camd;
    const float2* dn = (c->cfg.flags & SGS_FLAG_NORMALISED_DEPTH) ? c->dn_state : nullptr;
    FusedLoss fl{trgb, tdepth, lambda_d, nsign, loss};
    c->launches += 1;
    if (c->cfgd.lowpass) k_backward<true, true, false, true><<<tiles, SGS_BLOCK, 0, s>>>(c->render_order_valid ? c->render_order : nullptr, c->ranges, c->list_vals, c->list_stride, c->pay, cam.W, cam.H,
                                                       cam.tiles_x, cam.fx, cam.fy, cam.cx, cam.cy, c->cfgd, u, c->T_final,
                                                       c->n_last, c->acc, c->pose_partial, c->counters, d_pose6, fl, dn);
    else if (dn) k_backward<true, true, true><<<tiles, SGS_BLOCK, 0, s>>>(c->render_order_valid ? c->render_order : nullptr, c->ranges, c->list_vals, c->list_stride, c->pay, cam.W, cam.H,
                                                       cam.tiles_x, cam.fx, cam.fy, cam.cx, cam.cy, c->cfgd, u, c->T_final,
                                                       c->n_last, c->acc, c->pose_partial, c->counters, d_pose6, fl, dn);
    else k_backward<true, true, false><<<tiles, SGS_BLOCK, 0, s>>>(c->render_order_valid ? c->render_order : nullptr, c->ranges, c->list_vals, c->list_stride, c->pay, cam.W, cam.H,
                                                       cam.tiles_x, cam.fx, cam.fy, cam.cx, cam.cy, c->cfgd, u, c->T_final,
                                                       c->n_last, c->acc, c->pose_partial, c->counters, d_pose6, fl, dn);
    return cudaGetLastError();
}
