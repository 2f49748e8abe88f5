// preprocess.cu -- K-pre: one thread per surfel (SURVEY §8(a) step 1 + the emit half of step 2).
//
// Builds the ray-splat homography M = K [s_u t_uc, s_v t_vc, mu_c] (Eq. 5-7), culls,
// derives the screen AABB of the cutoff ellipse and the tile rectangle, and -- fused in the same
// kernel through a single-pass chained scan (decoupled look-back over dynamically numbered blocks)
// -- compacts the visible surfels and emits their 64-bit (tile id << 32 | depth bits) keys in
// surfel-major, tile row-major order.
//
// THIS FILE IS COMPILED WITH -fmad=false.  Everything that takes a binning decision (cull flag,
// depth bits, tile rectangle) is evaluated in IEEE-754 binary64 in the operation order DESIGN.md §3
// (O2) fixes, so that the list is bit-identical to the CPU oracle's.  B200 has full-rate-enough
// FP64 for this: the kernel is HBM-bound (52 B in, ~130 B out per visible surfel).
#include "sgs_internal.h"

namespace {

constexpr unsigned long long FLAG_AGG = 1ull << 62;
constexpr unsigned long long FLAG_INC = 2ull << 62;
constexpr unsigned long long FLAG_MASK = 3ull << 62;
constexpr int VIS_SHIFT = 38;  // value = vis (24 bits) << 38 | entries (38 bits)

__device__ __forceinline__ unsigned long long warp_incl_scan(unsigned long long v, int lane) {
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        unsigned long long t = __shfl_up_sync(0xffffffffu, v, o);
        if (lane >= o) v += t;
    }
    return v;
}

// R26 (oracle: two_ln_upper): an upper bound of 2 ln r, r >= 1, from +, -, x, / alone in the oracle's operation order
__device__ __forceinline__ double two_ln_upper(double r) {
    double m = r, e = 0.0;
    while (m >= 2.0) { m = m * 0.5; e = e + 1.0; }
    const double t = (m - 1.0) / (m + 1.0), t2 = t * t;
    double p = 1.0 / 25.0;
    p = p * t2 + 1.0 / 23.0; p = p * t2 + 1.0 / 21.0; p = p * t2 + 1.0 / 19.0; p = p * t2 + 1.0 / 17.0;
    p = p * t2 + 1.0 / 15.0; p = p * t2 + 1.0 / 13.0; p = p * t2 + 1.0 / 11.0; p = p * t2 + 1.0 / 9.0;
    p = p * t2 + 1.0 / 7.0; p = p * t2 + 1.0 / 5.0; p = p * t2 + 1.0 / 3.0; p = p * t2 + 1.0;
    const double ln_m = 2.0 * (t * p);
    const double ln_r = e * 0.69314718055994540 + ln_m;
    return (2.0 * ln_r) * (1.0 + 1e-9) + 1e-9;
}

// R27: the support ellipse as a screen conic relative to (cx, cy); ok = well-conditioned ellipse (else: list every tile)
struct Conic { double cx, cy, A, B, C, D, E, F; int ok; };

__device__ __forceinline__ double conic_q(const Conic& k, double x, double y) {
    return ((((k.A * x) * x + (2.0 * k.B) * (x * y)) + (k.C * y) * y) + ((2.0 * k.D) * x + (2.0 * k.E) * y)) + k.F;
}
__device__ __forceinline__ double clampd(double v, double lo, double hi) { return v < lo ? lo : (v > hi ? hi : v); }
// the oracle's tile_listed(), same binary64 sequence
__device__ __forceinline__ bool tile_listed(const Conic& k, int tx, int ty, int W, int H) {
    if (!k.ok) return true;
    const double ts = (double)SGS_TILE;
    double x1 = ts * tx + (ts - 0.5), y1 = ts * ty + (ts - 0.5);
    if (x1 > W - 0.5) x1 = W - 0.5;
    if (y1 > H - 0.5) y1 = H - 0.5;
    const double x0 = (ts * tx + 0.5) - k.cx, y0 = (ts * ty + 0.5) - k.cy;
    x1 = x1 - k.cx; y1 = y1 - k.cy;
    const double det = k.A * k.C - k.B * k.B;
    const double xc = (k.B * k.E - k.C * k.D) / det, yc = (k.B * k.D - k.A * k.E) / det;
    double qm = conic_q(k, clampd(xc, x0, x1), clampd(yc, y0, y1));
    double v;
    v = conic_q(k, x0, clampd(-(k.B * x0 + k.E) / k.C, y0, y1)); if (v < qm) qm = v;
    v = conic_q(k, x1, clampd(-(k.B * x1 + k.E) / k.C, y0, y1)); if (v < qm) qm = v;
    v = conic_q(k, clampd(-(k.B * y0 + k.D) / k.A, x0, x1), y0); if (v < qm) qm = v;
    v = conic_q(k, clampd(-(k.B * y1 + k.D) / k.A, x0, x1), y1); if (v < qm) qm = v;
    double R = fabs(x0);
    if (fabs(x1) > R) R = fabs(x1);
    if (fabs(y0) > R) R = fabs(y0);
    if (fabs(y1) > R) R = fabs(y1);
    const double tol = 1e-9 * ((fabs(k.F) + (2.0 * (fabs(k.D) + fabs(k.E))) * R) + ((k.A + k.C) + 2.0 * fabs(k.B)) * (R * R));
    return qm <= tol;
}

struct PreOut {
    bool vis;
    uint32_t depth_bits;
    int tx0, ty0, tx1, ty1;
    // payload
    float P, Q, R, S, D, E, F;
    double xc, yc;
    float a, b, c;
    float n[3], au[3], av[3];
    float bb[4];
};

__device__ __forceinline__ void preprocess_one(const float* __restrict__ mean, const float* __restrict__ scale,
                                               const float* __restrict__ quat, const SgsCamDev& cam,
                                               const SgsCfgDev& cfg, PreOut& o, const float opacity = 1.f, Conic* conic = nullptr) {
    o.vis = false;
    const double w = quat[0], x = quat[1], y = quat[2], z = quat[3];
    const double qn = sqrt(((w * w + x * x) + y * y) + z * z);
    if (!(qn > 0.0) || !isfinite(qn)) return;
    const double qw = w / qn, qx = x / qn, qy = y / qn, qz = z / qn;
    double Rw[9];
    Rw[0] = 1.0 - 2.0 * (qy * qy + qz * qz); Rw[1] = 2.0 * (qx * qy - qw * qz); Rw[2] = 2.0 * (qx * qz + qw * qy);
    Rw[3] = 2.0 * (qx * qy + qw * qz); Rw[4] = 1.0 - 2.0 * (qx * qx + qz * qz); Rw[5] = 2.0 * (qy * qz - qw * qx);
    Rw[6] = 2.0 * (qx * qz - qw * qy); Rw[7] = 2.0 * (qy * qz + qw * qx); Rw[8] = 1.0 - 2.0 * (qx * qx + qy * qy);
    const double m0 = mean[0], m1 = mean[1], m2 = mean[2];
    double tuc[3], tvc[3], tnc[3], muc[3];
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        const double r0 = cam.R[3 * i], r1 = cam.R[3 * i + 1], r2 = cam.R[3 * i + 2];
        tuc[i] = (r0 * Rw[0] + r1 * Rw[3]) + r2 * Rw[6];
        tvc[i] = (r0 * Rw[1] + r1 * Rw[4]) + r2 * Rw[7];
        tnc[i] = (r0 * Rw[2] + r1 * Rw[5]) + r2 * Rw[8];
        muc[i] = ((r0 * m0 + r1 * m1) + r2 * m2) + cam.t[i];
    }
    const double su = scale[0], sv = scale[1];
    const double A0[3] = {su * tuc[0], sv * tvc[0], muc[0]};
    const double A1[3] = {su * tuc[1], sv * tvc[1], muc[1]};
    const double A2[3] = {su * tuc[2], sv * tvc[2], muc[2]};
    double M[9];
#pragma unroll
    for (int j = 0; j < 3; ++j) {
        M[j] = cam.Kd[0] * A0[j] + cam.Kd[2] * A2[j];
        M[3 + j] = cam.Kd[1] * A1[j] + cam.Kd[3] * A2[j];
        M[6 + j] = A2[j];
    }
    o.depth_bits = __float_as_uint((float)muc[2]);
    if (!(muc[2] > cfg.z_near_d)) return;
    double c2 = cfg.cutoff2_d;
    if (conic != nullptr && cfg.alpha_min_d > 0.0) {   // SGS_FLAG_TIGHT_BINNING, R26: the splat's own support
        const double r = (double)opacity / cfg.alpha_min_d;
        if (!(r >= 1.0)) return;
        const double c2o = two_ln_upper(r);
        if (c2o < c2) c2 = c2o;
    }
    const double den = c2 * (M[6] * M[6] + M[7] * M[7]) - M[8] * M[8];
    if (!(den < 0.0)) return;
    const double ctrx = (c2 * (M[0] * M[6] + M[1] * M[7]) - M[2] * M[8]) / den;
    const double ctry = (c2 * (M[3] * M[6] + M[4] * M[7]) - M[5] * M[8]) / den;
    const double hx = sqrt(ctrx * ctrx - (c2 * (M[0] * M[0] + M[1] * M[1]) - M[2] * M[2]) / den);
    const double hy = sqrt(ctry * ctry - (c2 * (M[3] * M[3] + M[4] * M[4]) - M[5] * M[5]) / den);
    double xmin = ctrx - hx, xmax = ctrx + hx, ymin = ctry - hy, ymax = ctry + hy;
    if (cfg.lowpass) {   // R28: footprint = cutoff ellipse united with the filter's disc (the oracle's sequence, prep_surfel)
        const double xcf = M[2] / M[8], ycf = M[5] / M[8], rf = (double)cfg.cutoff * 0.70710678118654757;
        if (!(isfinite(xmin) && isfinite(xmax))) { xmin = xcf; xmax = xcf; }
        if (!(isfinite(ymin) && isfinite(ymax))) { ymin = ycf; ymax = ycf; }
        if (xcf - rf < xmin) xmin = xcf - rf;
        if (xcf + rf > xmax) xmax = xcf + rf;
        if (ycf - rf < ymin) ymin = ycf - rf;
        if (ycf + rf > ymax) ymax = ycf + rf;
    }
    if (!(isfinite(xmin) && isfinite(xmax) && isfinite(ymin) && isfinite(ymax))) return;
    if (!(xmax > 0.0 && xmin < (double)cam.W && ymax > 0.0 && ymin < (double)cam.H)) return;
    const double ts = (double)SGS_TILE;
    double fx0 = floor(xmin / ts), fx1 = floor(xmax / ts), fy0 = floor(ymin / ts), fy1 = floor(ymax / ts);
    if (fx0 < 0.0) fx0 = 0.0;
    if (fy0 < 0.0) fy0 = 0.0;
    if (fx1 > (double)(cam.tiles_x - 1)) fx1 = (double)(cam.tiles_x - 1);
    if (fy1 > (double)(cam.tiles_y - 1)) fy1 = (double)(cam.tiles_y - 1);
    o.tx0 = (int)fx0; o.tx1 = (int)fx1; o.ty0 = (int)fy0; o.ty1 = (int)fy1;
    o.vis = true;
    if (conic != nullptr) {   // R27: the footprint as a conic (the oracle's sequence, prep_surfel)
        const double C0[3] = {M[1] * M[5] - M[2] * M[4], M[2] * M[3] - M[0] * M[5], M[0] * M[4] - M[1] * M[3]};
        const double Cx[3] = {M[4] * M[8] - M[5] * M[7], M[5] * M[6] - M[3] * M[8], M[3] * M[7] - M[4] * M[6]};
        const double Cy[3] = {M[7] * M[2] - M[8] * M[1], M[8] * M[0] - M[6] * M[2], M[6] * M[1] - M[7] * M[0]};
        const double a1 = Cx[0], a2 = Cy[0], a3 = (Cx[0] * ctrx + Cy[0] * ctry) + C0[0];
        const double b1 = Cx[1], b2 = Cy[1], b3 = (Cx[1] * ctrx + Cy[1] * ctry) + C0[1];
        const double c1 = Cx[2], c2_ = Cy[2], c3 = (Cx[2] * ctrx + Cy[2] * ctry) + C0[2];
        conic->cx = ctrx; conic->cy = ctry;
        conic->A = (a1 * a1 + b1 * b1) - c2 * (c1 * c1);
        conic->B = (a1 * a2 + b1 * b2) - c2 * (c1 * c2_);
        conic->C = (a2 * a2 + b2 * b2) - c2 * (c2_ * c2_);
        conic->D = (a1 * a3 + b1 * b3) - c2 * (c1 * c3);
        conic->E = (a2 * a3 + b2 * b3) - c2 * (c2_ * c3);
        conic->F = (a3 * a3 + b3 * b3) - c2 * (c3 * c3);
        const double det = conic->A * conic->C - conic->B * conic->B;
        conic->ok = (conic->A > 0.0 && conic->C > 0.0 && det > 1e-12 * (conic->A * conic->C)) ? 1 : 0;
    }
    o.bb[0] = __double2float_rd(xmin); o.bb[1] = __double2float_ru(xmax);
    o.bb[2] = __double2float_rd(ymin); o.bb[3] = __double2float_ru(ymax);
    // ---- payload (no decision depends on it; rounded to fp32 at the end) ----
    const double xc = M[2] / M[8], yc = M[5] / M[8];
    const double B00 = M[0] - xc * M[6], B01 = M[1] - xc * M[7];
    const double B10 = M[3] - yc * M[6], B11 = M[4] - yc * M[7];
    const double a = M[6], b = M[7], c = M[8];
    o.P = (float)(c * B11); o.Q = (float)(-(c * B01)); o.R = (float)(-(c * B10)); o.S = (float)(c * B00);
    o.D = (float)(B00 * B11 - B01 * B10);
    o.E = (float)(a * B11 - b * B10);
    o.F = (float)(b * B00 - a * B01);
    o.xc = xc; o.yc = yc;
    o.a = (float)a; o.b = (float)b; o.c = (float)c;
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        o.n[i] = (float)tnc[i];
        o.au[i] = (float)(su * tuc[i]);
        o.av[i] = (float)(sv * tvc[i]);
    }
}

// Conservative binary32 pre-cull.  Returns true only when the strict binary64 path above is CERTAIN to
// cull the surfel, so the cull flags stay bit-identical to the oracle's while ~80-90 % of a room-scale
// map never touches the FP64 pipe.  The surfel's cutoff disk lies inside the sphere of radius
// r = cutoff * max(s_u, s_v) around mu_c.  (i) mu_c.z + d < z_near  =>  mu_c.z <= z_near (culled).
// (ii) sphere entirely beyond a frustum side plane (through the eye and an image border): every disk
// point in front of the camera projects off that border, so either the disk crosses the camera plane
// (den >= 0, culled) or its AABB misses the screen (culled).  d = 1e-5 (|mu|_1 + |t|_1 + 1) metres
// covers the binary32 rounding of mu_c (~20x its bound) and dwarfs the oracle's own 1e-10 px.
__device__ __forceinline__ bool precull_f32(const float* __restrict__ mean, const float* __restrict__ scale,
                                            const SgsCamDev& cam, const SgsCfgDev& cfg) {
    const float m0 = mean[0], m1 = mean[1], m2 = mean[2];
    const float X = cam.Rf[0] * m0 + cam.Rf[1] * m1 + cam.Rf[2] * m2 + cam.tf[0];
    const float Y = cam.Rf[3] * m0 + cam.Rf[4] * m1 + cam.Rf[5] * m2 + cam.tf[1];
    const float Z = cam.Rf[6] * m0 + cam.Rf[7] * m1 + cam.Rf[8] * m2 + cam.tf[2];
    // pm_t, pm_r > 0 (survivor list kept for later poses T' = Exp(tau) T with |rho| <= pm_t, |theta| <= pm_r): the
    // camera-space centre moves by at most pm_r |X_c| + pm_t, and every test below is linear in it with a unit normal
    const float d = 1e-5f * (fabsf(m0) + fabsf(m1) + fabsf(m2) + cam.pc_tabs) + cam.pm_t +
                    cam.pm_r * (fabsf(X) + fabsf(Y) + fabsf(Z));
    if (Z + d < cfg.z_near) return true;
    float r = cfg.cutoff * fmaxf(fabsf(scale[0]), fabsf(scale[1])) * 1.00001f + d;
    // SGS_FLAG_LOWPASS (R28): the footprint also holds the disc of cutoff / sqrt 2 pixels around the projected centre, i.e.
    // that many pixels times Z / f sideways at the centre's depth (every side-plane normal below is at least f long)
    if (cfg.lowpass) r += cfg.cutoff * 0.70711f * (fmaxf(Z, 0.f) + d) / fminf(cam.fx, cam.fy) * 1.0001f;
    // left: fx X + cx Z < 0 ; right: fx X + (cx - W) Z > 0 ; top / bottom alike.  Normals un-normalised:
    // compare against r * |normal| (|normal| rounded up on the host, cam.pc_n, and r rounded up above).
    if (cam.fx * X + cam.cx * Z < -r * cam.pc_n[0]) return true;
    if (cam.fx * X + cam.pc_cxr * Z > r * cam.pc_n[1]) return true;
    if (cam.fy * Y + cam.cy * Z < -r * cam.pc_n[2]) return true;
    if (cam.fy * Y + cam.pc_cyr * Z > r * cam.pc_n[3]) return true;
    return false;
}

__global__ void __launch_bounds__(SGS_PRE_BLOCK)
k_preprocess(int64_t n, const float* __restrict__ mean, const float* __restrict__ scale,
             const float* __restrict__ quat, const float* __restrict__ opacity, const float* __restrict__ rgb,
             const uint8_t* __restrict__ active, SgsCamDev cam, SgsCfgDev cfg, SgsPayload pay,
             uint32_t* __restrict__ vis_to_surfel, uint8_t* __restrict__ culled,
             unsigned long long* __restrict__ scan_state, SgsCounters* __restrict__ counters,
             uint64_t* __restrict__ keys, uint32_t* __restrict__ vals, unsigned long long e_cap) {
    __shared__ unsigned int s_bid;
    __shared__ unsigned long long s_warp[SGS_PRE_BLOCK / 32];
    __shared__ unsigned long long s_prefix;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    if (tid == 0) s_bid = atomicAdd(&counters->ticket_pre, 1u);  // dynamic id: predecessors are running or done
    __syncthreads();
    const unsigned int bid = s_bid;
    const int64_t i = (int64_t)bid * SGS_PRE_BLOCK + tid;

    PreOut o;
    o.vis = false;
    if (i < n && (active == nullptr || active[i] != 0) && !precull_f32(mean + 3 * i, scale + 2 * i, cam, cfg))
        preprocess_one(mean + 3 * i, scale + 2 * i, quat + 4 * i, cam, cfg, o);
    unsigned int cnt = 0;
    if (o.vis) cnt = (unsigned int)((o.tx1 - o.tx0 + 1) * (o.ty1 - o.ty0 + 1));
    if (i < n) culled[i] = o.vis ? 0 : 1;

    // block-exclusive scan of (visible, entries) packed in one 64-bit word
    const unsigned long long mine = ((unsigned long long)(o.vis ? 1 : 0) << VIS_SHIFT) | cnt;
    const unsigned long long incl = warp_incl_scan(mine, lane);
    if (lane == 31) s_warp[wid] = incl;
    __syncthreads();
    if (wid == 0) {
        unsigned long long wv = lane < SGS_PRE_BLOCK / 32 ? s_warp[lane] : 0ull;
        const unsigned long long wi = warp_incl_scan(wv, lane);
        if (lane < SGS_PRE_BLOCK / 32) s_warp[lane] = wi - wv;  // exclusive warp offsets
        const unsigned long long block_total = __shfl_sync(0xffffffffu, wi, SGS_PRE_BLOCK / 32 - 1);
        // chained scan: publish the aggregate, look back over predecessors 32 at a time
        unsigned long long prefix = 0;
        if (bid == 0) {
            if (lane == 0) atomicExch(&scan_state[0], FLAG_INC | block_total);
        } else {
            if (lane == 0) atomicExch(&scan_state[bid], FLAG_AGG | block_total);
            int64_t look = (int64_t)bid - 1;
            while (true) {
                const int64_t j = look - lane;
                unsigned long long st = FLAG_INC;  // lanes before block 0 read as "inclusive 0"
                if (j >= 0) {
                    do { st = *((volatile unsigned long long*)&scan_state[j]); } while ((st & FLAG_MASK) == 0);
                }
                const unsigned int inc_mask = __ballot_sync(0xffffffffu, (st & FLAG_MASK) == FLAG_INC);
                const int first_inc = inc_mask ? __ffs(inc_mask) - 1 : 32;
                unsigned long long v = (lane <= first_inc) ? (st & ~FLAG_MASK) : 0ull;
#pragma unroll
                for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
                prefix += v;
                if (inc_mask) break;
                look -= 32;
            }
            if (lane == 0) atomicExch(&scan_state[bid], FLAG_INC | (prefix + block_total));
        }
        if (lane == 0) {
            s_prefix = prefix;
            if (bid == gridDim.x - 1) {  // totals: E, N_v, overflow
                const unsigned long long tot = prefix + block_total;
                const unsigned long long E = tot & ((1ull << VIS_SHIFT) - 1);
                counters->n_entries = E;
                counters->n_visible = (unsigned int)(tot >> VIS_SHIFT);
                counters->overflow = E > e_cap ? 1u : 0u;
            }
        }
    }
    __syncthreads();
    if (!o.vis) return;
    const unsigned long long excl = s_prefix + s_warp[wid] + (incl - mine);
    const uint32_t v = (uint32_t)(excl >> VIS_SHIFT);
    unsigned long long pos = excl & ((1ull << VIS_SHIFT) - 1);

    vis_to_surfel[v] = (uint32_t)i;
    pay.g0[v] = make_float4(o.P, o.Q, o.R, o.S);
    pay.g1[v] = make_float4(o.D, o.E, o.F, opacity[i]);
    pay.g2[v] = make_double2(o.xc, o.yc);
    pay.g3[v] = make_float4(o.a, o.b, o.c, rgb[3 * i]);
    pay.g4[v] = make_float4(rgb[3 * i + 1], rgb[3 * i + 2], o.n[0], o.n[1]);
    pay.g5[v] = make_float4(o.n[2], o.au[0], o.au[1], o.au[2]);
    pay.g6[v] = make_float4(o.av[0], o.av[1], o.av[2], 0.f);
    pay.g7[v] = make_float4(o.bb[0], o.bb[1], o.bb[2], o.bb[3]);

    // emit keys: tile row-major within the surfel (R2: key = tile id << 32 | depth bits)
    for (int ty = o.ty0; ty <= o.ty1; ++ty)
        for (int tx = o.tx0; tx <= o.tx1; ++tx) {
            if (pos < e_cap) {
                keys[pos] = ((unsigned long long)(uint32_t)(ty * cam.tiles_x + tx) << 32) | o.depth_bits;
                vals[pos] = v;
            }
            ++pos;
        }
}

// Bucket variant (default path): no scan at all.  Tile t owns a fixed-capacity bucket; a visible surfel
// appends (depth bits << 32 | surfel index) to every tile of its rectangle through an atomic cursor.
// Arrival order is irrelevant: the in-tile sort orders each bucket by the full 64-bit key, which is unique
// inside a tile, so the result is the stable (tile, depth, index) order of the contract.  The payload
// is indexed by the surfel index itself (no compaction of the payload in HBM).
//
// Two kernels (ncu, profiles/r01_*: with one thread per surfel doing everything, 73 % of the warps of a
// 20 %-active map dragged all 32 lanes through the ~700-instruction binary64 path for one or two
// survivors, the kernel sat at 3 blocks/SM on its 78 registers and 42 % of the stall samples were
// dependent global loads):
//   K-pre-A  light (few registers, full occupancy, 4 surfels per thread with all loads in flight together):
//            active flag + binary32 pre-cull; writes culled = 1 for the rejected, compacts the survivors of
//            the block in shared memory and appends them to a global list with ONE atomic per block.
//   K-pre-B  dense: one thread per survivor runs the binary64 sequence, writes the payload, and the
//            block's tile entries are spread over its threads (one (surfel, tile) pair each).
// sgs_track_iter_dev: the pose T_cw (row-major 3x4) lives in DEVICE memory -- a tracker's own update kernel writes it between
// the iterations of one stream or CUDA graph -- and replaces the pose fields of the camera struct the host filled.
__device__ __forceinline__ void load_pose(SgsCamDev& cam, const float* __restrict__ T) {
    float ta = 1.f;
#pragma unroll
    for (int i = 0; i < 3; ++i) {
#pragma unroll
        for (int j = 0; j < 3; ++j) { const float v = __ldg(T + 4 * i + j); cam.R[3 * i + j] = (double)v; cam.Rf[3 * i + j] = v; }
        const float t = __ldg(T + 4 * i + 3);
        cam.t[i] = (double)t; cam.tf[i] = t; ta += fabsf(t);
    }
    cam.pc_tabs = ta;
}

// is `cur` = Exp(tau) o `ref` with |rho|, |theta| inside 80 % of the survivor list's margins?  (api_run.cu: pose_within_margin)
__device__ __forceinline__ bool pose_inside_margin(const float* __restrict__ ref, const float* __restrict__ cur) {
    double Rd[9];
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
            double v = 0.0;
            for (int k = 0; k < 3; ++k) v += (double)cur[4 * i + k] * (double)ref[4 * j + k];
            Rd[3 * i + j] = v;
        }
    double cosang = 0.5 * (Rd[0] + Rd[4] + Rd[8] - 1.0);
    if (!(cosang <= 1.0)) cosang = 1.0;
    if (!(cosang >= -1.0)) return false;
    double d2 = 0.0;
    for (int i = 0; i < 3; ++i) {
        const double v = (double)cur[4 * i + 3] - (Rd[3 * i] * ref[3] + Rd[3 * i + 1] * ref[7] + Rd[3 * i + 2] * ref[11]);
        d2 += v * v;
    }
    const double mt = 0.8 * SGS_REUSE_MARGIN_T, mr = 0.8 * SGS_REUSE_MARGIN_R;
    return d2 <= mt * mt && cosang >= 1.0 - 0.5 * mr * mr;   // (cos mr >= 1 - mr^2 / 2: slightly stricter, no transcendental)
}

template <int SGS_PREA_ITEMS, bool DEVPOSE>
__global__ void __launch_bounds__(SGS_PRE_BLOCK)
k_pre_select(int64_t n, const float* __restrict__ mean, const float* __restrict__ scale,
             const uint8_t* __restrict__ active, SgsCamDev cam_in, SgsCfgDev cfg, uint8_t* __restrict__ culled,
             unsigned int* __restrict__ n_surv, uint32_t* __restrict__ surv_list, const float* __restrict__ pose_dev,
             float* __restrict__ surv_pose) {
    constexpr int SGS_PREA_SPAN = SGS_PREA_ITEMS * SGS_PRE_BLOCK;
    cudaTriggerProgrammaticLaunchCompletion();  // K-pre-B may be staged now; it waits for this grid before reading
    SgsCamDev camL;
    if (DEVPOSE) {
        camL = cam_in;
        load_pose(camL, pose_dev);
        if (surv_pose != nullptr && blockIdx.x == 0 && threadIdx.x < 12) surv_pose[threadIdx.x] = __ldg(pose_dev + threadIdx.x);
    }
    const SgsCamDev& cam = DEVPOSE ? camL : cam_in;
    __shared__ unsigned short s_list[SGS_PREA_SPAN];
    __shared__ unsigned int s_n, s_base;
    const int tid = threadIdx.x, lane = tid & 31;
    const int64_t base = (int64_t)blockIdx.x * SGS_PREA_SPAN;
    if (tid == 0) s_n = 0;
    __syncthreads();
    // all loads of the thread's items are issued before the first use
    bool act[SGS_PREA_ITEMS];
    float m[SGS_PREA_ITEMS][3], sc[SGS_PREA_ITEMS][2];
#pragma unroll
    for (int it = 0; it < SGS_PREA_ITEMS; ++it) {
        const int64_t i = base + it * SGS_PRE_BLOCK + tid;
        act[it] = i < n && (active == nullptr || active[i] != 0);
    }
#pragma unroll
    for (int it = 0; it < SGS_PREA_ITEMS; ++it) {
        const int64_t i = base + it * SGS_PRE_BLOCK + tid;
        m[it][0] = m[it][1] = m[it][2] = 0.f; sc[it][0] = sc[it][1] = 0.f;
        if (act[it]) {
            m[it][0] = mean[3 * i]; m[it][1] = mean[3 * i + 1]; m[it][2] = mean[3 * i + 2];
            sc[it][0] = scale[2 * i]; sc[it][1] = scale[2 * i + 1];
        }
    }
#pragma unroll
    for (int it = 0; it < SGS_PREA_ITEMS; ++it) {
        const int local = it * SGS_PRE_BLOCK + tid;
        const int64_t i = base + local;
        const bool surv = act[it] && !precull_f32(m[it], sc[it], cam, cfg);
        if (i < n && !surv) culled[i] = 1;
        const unsigned int bal = __ballot_sync(0xffffffffu, surv);
        unsigned int wbase = 0;
        if (lane == 0 && bal) wbase = atomicAdd(&s_n, (unsigned int)__popc(bal));
        wbase = __shfl_sync(0xffffffffu, wbase, 0);
        if (surv) s_list[wbase + __popc(bal & ((1u << lane) - 1u))] = (unsigned short)local;
    }
    __syncthreads();
    const unsigned int ns = s_n;
    if (ns == 0) return;
    if (tid == 0) s_base = atomicAdd(n_surv, ns);
    __syncthreads();
    const unsigned int gb = s_base;
    for (unsigned int k = tid; k < ns; k += SGS_PRE_BLOCK) surv_list[gb + k] = (uint32_t)(base + s_list[k]);
}

// SGS_FLAG_TRACK_REUSE: one copy of the listed splats' parameters in list order (52 B each, 7.8 MB for 150 k survivors:
// resident in L2 across the iterations of a frame), so that K-pre-B reads coalesced lines instead of gathering 12-16 B
// pieces of a map that does not fit the L2 (ncu, C5: 43 % of its stall samples were those gathers, L2 hit rate 7 %).
__global__ void __launch_bounds__(256)
k_surv_gather(const uint32_t* __restrict__ surv_list, const unsigned int* __restrict__ n_surv_in,
              const float* __restrict__ mean, const float* __restrict__ scale, const float* __restrict__ quat,
              const float* __restrict__ opacity, const float* __restrict__ rgb, float4* __restrict__ p0,
              float4* __restrict__ p1, float4* __restrict__ p2, float* __restrict__ p3) {
    const unsigned int n = *n_surv_in;
    for (unsigned int j = blockIdx.x * blockDim.x + threadIdx.x; j < n; j += gridDim.x * blockDim.x) {
        const size_t i = surv_list[j];
        p0[j] = make_float4(mean[3 * i], mean[3 * i + 1], mean[3 * i + 2], opacity[i]);
        p1[j] = make_float4(quat[4 * i], quat[4 * i + 1], quat[4 * i + 2], quat[4 * i + 3]);
        p2[j] = make_float4(scale[2 * i], scale[2 * i + 1], rgb[3 * i], rgb[3 * i + 1]);
        p3[j] = rgb[3 * i + 2];
    }
}

constexpr int SGS_PREB_BLOCK = 128, SGS_PREB_LOG2 = 7, PREB_EMIT = 4;  // K-pre-B block: small, so that few survivors still spread over the SMs

template <bool TIGHT, bool DEVPOSE>
__global__ void __launch_bounds__(SGS_PREB_BLOCK)
k_pre_project(const float* __restrict__ mean, const float* __restrict__ scale, const float* __restrict__ quat,
              const float* __restrict__ opacity, const float* __restrict__ rgb, SgsCamDev cam_in, SgsCfgDev cfg,
              SgsPayload pay, uint8_t* __restrict__ culled, SgsCounters* __restrict__ counters,
              const uint32_t* surv_list, const unsigned int* n_surv_in,  // written by the PREVIOUS grid: no __restrict__,
              // or the compiler may hoist their loads above the conditional grid-dependency wait (it did: stale counts)
              uint32_t* __restrict__ cursor, uint64_t* __restrict__ bucket, uint32_t tile_cap, SurvInputs cin, int early,
              uint32_t* __restrict__ vis_list, const float* __restrict__ pose_dev, const float* surv_pose) {
    SgsCamDev camL;
    if (DEVPOSE) { camL = cam_in; load_pose(camL, pose_dev); }
    const SgsCamDev& cam = DEVPOSE ? camL : cam_in;
    __shared__ unsigned int s_off[SGS_PREB_BLOCK + 1];
    __shared__ unsigned long long s_key[SGS_PREB_BLOCK];
    __shared__ unsigned int s_rect[SGS_PREB_BLOCK];   // tile index of the rectangle's first tile
    __shared__ unsigned int s_w[SGS_PREB_BLOCK];      // rectangle width in tiles
    __shared__ unsigned int s_wsum[SGS_PREB_BLOCK / 32];
    __shared__ Conic s_conic[TIGHT ? SGS_PREB_BLOCK : 1];   // SGS_FLAG_TIGHT_BINNING: each survivor's support conic (R27)
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    // early (list and inputs kept from an earlier iteration, this grid staged programmatically behind K-track): nothing
    // the first round reads is written by the previous kernel, so its loads and the projection run before the wait and
    // only the stores (records K-track still gathers, cursors it zeroes at its end) stay behind it
    bool must_wait = early != 0;
    if (!must_wait) cudaGridDependencySynchronize();   // K-pre-A complete: survivor list and count are final
    const unsigned int n_surv = *(const volatile unsigned int*)n_surv_in;   // written by K-pre-A (previous launch on the stream, or an earlier iteration)
    for (unsigned int r0 = blockIdx.x * SGS_PREB_BLOCK; r0 < n_surv; r0 += gridDim.x * SGS_PREB_BLOCK) {
        const bool have = r0 + tid < n_surv;
        const int64_t i = have ? (int64_t)__ldcg(surv_list + r0 + tid) : 0;
        PreOut o;
        o.vis = false;
        o.depth_bits = 0;
        float in_m[3] = {0.f, 0.f, 0.f}, in_s[2] = {0.f, 0.f}, in_q[4] = {0.f, 0.f, 0.f, 0.f}, in_o = 0.f, in_c[3] = {0.f, 0.f, 0.f};
        if (have) {
            if (cin.p0) {  // SGS_FLAG_TRACK_REUSE: the survivors' parameters, copied in list order when the list was built
                const float4 a = cin.p0[r0 + tid], q = cin.p1[r0 + tid], c2 = cin.p2[r0 + tid];
                in_m[0] = a.x; in_m[1] = a.y; in_m[2] = a.z; in_o = a.w;
                in_q[0] = q.x; in_q[1] = q.y; in_q[2] = q.z; in_q[3] = q.w;
                in_s[0] = c2.x; in_s[1] = c2.y; in_c[0] = c2.z; in_c[1] = c2.w; in_c[2] = cin.p3[r0 + tid];
            } else {
                in_m[0] = mean[3 * i]; in_m[1] = mean[3 * i + 1]; in_m[2] = mean[3 * i + 2];
                in_s[0] = scale[2 * i]; in_s[1] = scale[2 * i + 1];
                in_q[0] = quat[4 * i]; in_q[1] = quat[4 * i + 1]; in_q[2] = quat[4 * i + 2]; in_q[3] = quat[4 * i + 3];
                if (TIGHT) in_o = opacity[i];
            }
            Conic kq;
            kq.ok = 0;
            preprocess_one(in_m, in_s, in_q, cam, cfg, o, in_o, TIGHT ? &kq : nullptr);
            if (TIGHT) s_conic[tid] = kq;
        }
        if (must_wait) { cudaGridDependencySynchronize(); must_wait = false; }
        if (n_surv_in != &counters->n_surv && r0 == 0 && tid == 0) counters->n_surv = n_surv;  // for the host's grid hint
        // a kept survivor list covers poses near the one it was built around; the host cannot see a device-resident pose,
        // so the check is made here and K-track turns the iteration's results into NaN when it fails
        if (DEVPOSE && surv_pose != nullptr && r0 == 0 && tid == 0 && !pose_inside_margin(surv_pose, pose_dev)) counters->stale = 1u;
        if (have) culled[i] = o.vis ? 0 : 1;
        const unsigned int cnt = o.vis ? (unsigned int)((o.tx1 - o.tx0 + 1) * (o.ty1 - o.ty0 + 1)) : 0u;
        // totals: one atomic per warp
        const unsigned int vis_mask = __ballot_sync(0xffffffffu, o.vis);
        unsigned int wcnt = cnt;
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) wcnt += __shfl_xor_sync(0xffffffffu, wcnt, off);
        unsigned int vbase = 0;
        if (lane == 0 && vis_mask) {
            if (vis_list != nullptr) vbase = atomicAdd(&counters->n_visible, (unsigned int)__popc(vis_mask));
            else atomicAdd(&counters->n_visible, (unsigned int)__popc(vis_mask));   // (no return value: a RED, nothing waits)
            if (!TIGHT) atomicAdd(&counters->n_entries, (unsigned long long)wcnt);   // (TIGHT: counted at emission, below)
        }
        // (vis_list == nullptr inside sgs_track_iter: no per-surfel backward follows, and waiting for the atomic's return value
        // is a dependent L2 round trip per round of a kernel that sits on the tracking iteration's chain)
        if (vis_list != nullptr) vbase = __shfl_sync(0xffffffffu, vbase, 0);
        if (o.vis) {
            // the visible surfels, compact (arrival order): what the per-surfel backward walks -- K-pre-A's survivor list
            // is several times longer (C4: every splat the frustum test cannot exclude) and costs it a sector per entry
            if (vis_list != nullptr) vis_list[vbase + __popc(vis_mask & ((1u << lane) - 1u))] = (uint32_t)i;
            if (!cin.p0) { if (!TIGHT) in_o = opacity[i]; in_c[0] = rgb[3 * i]; in_c[1] = rgb[3 * i + 1]; in_c[2] = rgb[3 * i + 2]; }
            pay.g0[i] = make_float4(o.P, o.Q, o.R, o.S);
            pay.g1[i] = make_float4(o.D, o.E, o.F, in_o);
            pay.g2[i] = make_double2(o.xc, o.yc);
            pay.g3[i] = make_float4(o.a, o.b, o.c, in_c[0]);
            pay.g4[i] = make_float4(in_c[1], in_c[2], o.n[0], o.n[1]);
            pay.g5[i] = make_float4(o.n[2], o.au[0], o.au[1], o.au[2]);
            pay.g6[i] = make_float4(o.av[0], o.av[1], o.av[2], 0.f);
            pay.g7[i] = make_float4(o.bb[0], o.bb[1], o.bb[2], o.bb[3]);
        }
        // Cooperative emission: the round's entries (sum of tile counts) are spread over the block's threads,
        // one (surfel, tile) pair each, so the cursor atomics are all in flight together instead of one
        // thread walking its rectangle serially (a surfel covering hundreds of tiles costs no more than
        // hundreds of small ones).
        unsigned int incl = cnt;
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            const unsigned int t2 = __shfl_up_sync(0xffffffffu, incl, off);
            if (lane >= off) incl += t2;
        }
        if (lane == 31) s_wsum[wid] = incl;
        s_key[tid] = ((unsigned long long)o.depth_bits << 32) | (unsigned long long)(uint32_t)i;
        s_rect[tid] = o.vis ? (unsigned int)(o.ty0 * cam.tiles_x + o.tx0) : 0u;
        s_w[tid] = o.vis ? (unsigned int)(o.tx1 - o.tx0 + 1) : 1u;
        __syncthreads();
        unsigned int wbase = 0, total = 0;
#pragma unroll
        for (int w2 = 0; w2 < SGS_PREB_BLOCK / 32; ++w2) {
            const unsigned int x = s_wsum[w2];
            wbase += (w2 < wid) ? x : 0u;
            total += x;
        }
        s_off[tid] = wbase + incl - cnt;  // exclusive
        if (tid == 0) s_off[SGS_PREB_BLOCK] = total;
        __syncthreads();
        unsigned int n_listed = 0;
        for (unsigned int e0 = tid; e0 < total; e0 += PREB_EMIT * SGS_PREB_BLOCK) {
            // PREB_EMIT entries per trip so that their cursor atomics are all in flight before the first dependent store
            uint32_t t[PREB_EMIT];
            unsigned long long key[PREB_EMIT];
            bool ok[PREB_EMIT];
#pragma unroll
            for (int k = 0; k < PREB_EMIT; ++k) {
                const unsigned int e = e0 + k * SGS_PREB_BLOCK;
                ok[k] = e < total;
                // owner = last thread whose exclusive offset is <= e (and whose count is non-zero by construction)
                int lo = 0, hi = SGS_PREB_BLOCK;  // invariant: s_off[lo] <= e < s_off[hi]
#pragma unroll
                for (int it = 0; it < SGS_PREB_LOG2; ++it) {
                    const int mid = (lo + hi) >> 1;
                    if (s_off[mid] <= e) lo = mid; else hi = mid;
                }
                const unsigned int local = e - s_off[lo], w = s_w[lo];
                t[k] = s_rect[lo] + (local / w) * (unsigned int)cam.tiles_x + (local % w);
                key[k] = s_key[lo];
                if (TIGHT && ok[k]) {   // R27: only tiles the support ellipse reaches are listed
                    ok[k] = tile_listed(s_conic[lo], (int)(t[k] % (unsigned int)cam.tiles_x), (int)(t[k] / (unsigned int)cam.tiles_x), cam.W, cam.H);
                    n_listed += ok[k] ? 1u : 0u;
                }
            }
            uint32_t pos[PREB_EMIT];
#pragma unroll
            for (int k = 0; k < PREB_EMIT; ++k)
                pos[k] = ok[k] ? atomicAdd(&cursor[t[k]], 1u) : 0u;
#pragma unroll
            for (int k = 0; k < PREB_EMIT; ++k)
                if (ok[k]) {
                    if (pos[k] < tile_cap) bucket[(size_t)t[k] * tile_cap + pos[k]] = key[k];
                    else atomicMax(&counters->max_tile, pos[k] + 1u);
                }
        }
        if (TIGHT) {
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) n_listed += __shfl_xor_sync(0xffffffffu, n_listed, off);
            if (lane == 0 && n_listed) atomicAdd(&counters->n_entries, (unsigned long long)n_listed);
        }
        __syncthreads();  // the round's shared arrays are free again
    }
}

}  // namespace

cudaError_t sgs_launch_preprocess(sgs_ctx* c, const sgs_surfels* sf, cudaStream_t s) {
    const int64_t n = sf->n;
    const int blocks = (int)((n + SGS_PRE_BLOCK - 1) / SGS_PRE_BLOCK);
    cudaError_t e = cudaMemsetAsync(c->counters, 0, sizeof(SgsCounters), s);
    if (e != cudaSuccess) return e;
    if (blocks == 0) return cudaSuccess;
    e = cudaMemsetAsync(c->scan_state, 0, sizeof(unsigned long long) * (size_t)blocks, s);
    if (e != cudaSuccess) return e;
    SgsStage st(c, SGS_STAGE_PREPROCESS, s);
    c->launches += 1;
    k_preprocess<<<blocks, SGS_PRE_BLOCK, 0, s>>>(n, sf->mean, sf->scale, sf->quat, sf->opacity, sf->rgb, sf->active,
                                                  c->camd, c->cfgd, c->pay, c->vis_to_surfel, c->culled, c->scan_state,
                                                  c->counters, c->keys[0], c->vals[0], (unsigned long long)c->e_cap);
    return cudaGetLastError();
}

cudaError_t sgs_launch_preprocess_bucket(sgs_ctx* c, const sgs_surfels* sf, cudaStream_t s) {
    const int64_t n = sf->n;
    const int tiles = c->camd.tiles_x * c->camd.tiles_y;
    cudaError_t e = cudaSuccess;
    const bool prezeroed = c->prezero_tiles >= tiles;
    if (!prezeroed) {  // else: the previous sgs_track_iter's kernel already zeroed both (two stream ops saved)
        e = cudaMemsetAsync(c->counters, 0, sizeof(SgsCounters), s);
        if (e != cudaSuccess) return e;
        e = cudaMemsetAsync(c->cursor, 0, sizeof(uint32_t) * (size_t)tiles, s);
        if (e != cudaSuccess) return e;
    }
    c->prezero_tiles = 0;
    SgsStage st(c, SGS_STAGE_PREPROCESS, s);
    // K-pre-A: 4 surfels per thread once that still gives every SM several blocks (large maps), else 1
    const bool wide = (n + 1023) / 1024 >= 4 * 148;
    const int span = wide ? 1024 : 256;
    const int blocks_a = (int)((n + span - 1) / span);
    // SGS_FLAG_TRACK_REUSE: the list built (with pose margins) by an earlier iteration still covers this pose
    const bool cached = c->use_surv_cache && c->surv_valid;
    unsigned int* n_surv = c->use_surv_cache ? c->surv_cnt : &c->counters->n_surv;
    const bool run_a = blocks_a > 0 && !cached;
    c->launches += run_a ? 2 : 1;
    SgsCamDev cam_a = c->camd;
    if (run_a && c->use_surv_cache) {  // this list has to cover the poses of the coming iterations too
        if ((e = cudaMemsetAsync(c->surv_cnt, 0, sizeof(unsigned int), s)) != cudaSuccess) return e;
        cam_a.pm_t = SGS_REUSE_MARGIN_T; cam_a.pm_r = SGS_REUSE_MARGIN_R;
        c->surv_valid = true; c->surv_sf = *sf; c->surv_cam = c->last_cam;
    }
    const float* pd = c->pose_dev;
    float* sp_w = (pd && c->use_surv_cache) ? c->surv_pose_dev : nullptr;          // K-pre-A records the pose the list is built around
    const float* sp_r = (pd && cached) ? c->surv_pose_dev : nullptr;                // K-pre-B checks a kept list against it
    if (run_a) {
#define SGS_PREA_ARGS n, sf->mean, sf->scale, sf->active, cam_a, c->cfgd, c->culled, n_surv, c->vis_to_surfel, pd, sp_w
        if (wide) { if (pd) k_pre_select<4, true><<<blocks_a, SGS_PRE_BLOCK, 0, s>>>(SGS_PREA_ARGS); else k_pre_select<4, false><<<blocks_a, SGS_PRE_BLOCK, 0, s>>>(SGS_PREA_ARGS); }
        else { if (pd) k_pre_select<1, true><<<blocks_a, SGS_PRE_BLOCK, 0, s>>>(SGS_PREA_ARGS); else k_pre_select<1, false><<<blocks_a, SGS_PRE_BLOCK, 0, s>>>(SGS_PREA_ARGS); }
#undef SGS_PREA_ARGS
    }
    SurvInputs cin = {nullptr, nullptr, nullptr, nullptr};
    if (c->use_surv_cache && c->surv_in) {
        cin.p0 = reinterpret_cast<float4*>(c->surv_in);
        cin.p1 = cin.p0 + c->surv_in_cap; cin.p2 = cin.p1 + c->surv_in_cap;
        cin.p3 = reinterpret_cast<float*>(cin.p2 + c->surv_in_cap);
        if (run_a) {
            c->launches += 1;
            k_surv_gather<<<148 * 4, 256, 0, s>>>(c->vis_to_surfel, n_surv, sf->mean, sf->scale, sf->quat, sf->opacity, sf->rgb,
                                                 cin.p0, cin.p1, cin.p2, cin.p3);
        }
    }
    // K-pre-B walks the survivor list with a grid-stride loop: the count is only known on the device
    // (the grid follows the last known survivor count)
    int64_t blocks_b = (n + SGS_PREB_BLOCK - 1) / SGS_PREB_BLOCK;
    if (c->last_surv > 0) {
        const int64_t hint = (c->last_surv + c->last_surv / 4 + SGS_PREB_BLOCK - 1) / SGS_PREB_BLOCK;
        if (hint < blocks_b) blocks_b = hint;
    }
    if (blocks_b > 148 * 8) blocks_b = 148 * 8;
    // sgs_prepare: the binning runs under another view's compositing kernels and has a whole view's time to finish;
    // a narrow grid (one block per SM) keeps it from displacing their blocks (each of these holds 13.8 k registers)
    if (c->narrow_prepare && blocks_b > 148 * c->narrow_prepare) blocks_b = 148 * c->narrow_prepare;
    if (blocks_b < 1) blocks_b = 1;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)blocks_b); cfg.blockDim = dim3(SGS_PREB_BLOCK); cfg.dynamicSmemBytes = 0; cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    // programmatic dependent launch behind K-pre-A, or (list reused, previous launch on the stream = K-track) behind K-track
    cfg.numAttrs = ((run_a && !cin.p0) || (cached && prezeroed)) ? 1 : 0;
    auto kern = c->cfgd.tight ? (pd ? k_pre_project<true, true> : k_pre_project<true, false>)
                              : (pd ? k_pre_project<false, true> : k_pre_project<false, false>);
    const cudaError_t le = cudaLaunchKernelEx(&cfg, kern, sf->mean, sf->scale, sf->quat, sf->opacity, sf->rgb, c->camd,
                                              c->cfgd, c->pay, c->culled, c->counters, (const uint32_t*)c->vis_to_surfel,
                                              (const unsigned int*)n_surv, c->cursor, c->bucket, (uint32_t)c->tile_cap, cin,
                                              (cached && prezeroed && cin.p0) ? 1 : 0, c->track_binning ? nullptr : c->vis_list, pd, sp_r);
    if (le != cudaSuccess) return le;
    return cudaGetLastError();
}
