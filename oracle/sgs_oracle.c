/*
 * sgs_oracle.c -- CPU ORACLE for the 2D-Gaussian (surfel) splatting renderer of 2DGS-SLAM
 * (arxiv 2506.00970).  TEST INFRASTRUCTURE ONLY: nothing but tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call this file.
 * It shares no code with the CUDA path under paper_2506_00970_b200/.
 *
 * Plain, slow, fp64, one pixel at a time over all surfels in depth order, in the paper's
 * notation (citations are PAPER.md line numbers; "R<n>" are the readings listed in DESIGN.md §3):
 *   Eq. 1-2  (L83-93)   surfel frame  P(u,v) = mu + s_u t_u u + s_v t_v v
 *   Eq. 3-7  (L95-110)  homography    M = K [s_u t_uc, s_v t_vc, mu_c]   (3x3 reduction of  W T_cw H, R14)
 *   L112                ray-splat intersection (u,v,1) ~ (M0 - x M2) x (M1 - y M2)           (R1)
 *   Eq. 8    (L114-120) depth-ordered alpha blending of colour, depth, normal, opacity
 *   Eq. 9-13 (L130-152) gradient to H_c, R_c and the SE(3) pose (left perturbation)
 *
 * Pins (tests/test_oracle_pins.py): P1 closed-form footprint, P2 ray-plane depth, P3 hand-computed
 * stacks, P4 invariants, P5 channel consistency, P6 truncation limit, P7 binning conservativeness,
 * P8 central finite differences of every gradient incl. pose, P9 rigid-motion identity, P10
 * symmetries.  Parity UNPINNED: absolute image values on the paper's datasets (not available).
 *
 * Build: gcc -O2 -fopenmp -ffp-contract=off -fPIC -shared (oracle/__init__.py: build()).
 * -ffp-contract=off matters: the binning stage (orc_preprocess) is the bit-exact contract with
 * the GPU and must evaluate the documented IEEE-754 binary64 operation sequence without FMA.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int W, H;
    double fx, fy, cx, cy;
    double R[9], t[3]; /* T_cw = [R | t], row-major */
} Cam;

typedef struct {
    int tile;
    double cutoff, alpha_min, alpha_max, t_min, z_near;
    int tight; /* binning variant of readings R26 + R27: opacity-aware cutoff and tile-exact culling */
    int lowpass; /* compositing variant of reading R28: screen-space low-pass filter */
} Cfg;

/* Per-surfel derived quantities (all fp64). */
typedef struct {
    int culled;          /* 1 = inactive, behind / across the camera plane, off-screen or non-finite */
    uint32_t depth_bits; /* bit pattern of (float)mu_c.z */
    int rect[4];         /* tile rect tx0, ty0, tx1, ty1 (inclusive) */
    double aabb[4];      /* xmin, xmax, ymin, ymax of the cutoff ellipse on screen (pixels) */
    double qn;           /* |q| */
    double qh[4];        /* q / |q| */
    double Rw[9];        /* R(qh), columns t_u, t_v, t_n (world) */
    double tuc[3], tvc[3], tnc[3], muc[3];
    double M[9];         /* rows M0, M1, M2 of K [s_u t_uc, s_v t_vc, mu_c] */
    /* tight binning only: c2k = the splat's own cutoff^2 (R26); the footprint rho^2 <= c2k as the screen conic
     * q(x', y') = A x'^2 + 2 B x' y' + C y'^2 + 2 D x' + 2 E y' + F <= 0 in coordinates relative to (q_cx, q_cy) (R27) */
    double c2k, q_cx, q_cy, qA, qB, qC, qD, qE, qF;
    int q_ok;            /* the conic is a well-conditioned ellipse: the per-tile test applies (else every tile of the rect is listed) */
} Prep;

static void load_cam(const double* c, Cam* cam) {
    cam->W = (int)c[0]; cam->H = (int)c[1];
    cam->fx = c[2]; cam->fy = c[3]; cam->cx = c[4]; cam->cy = c[5];
    for (int i = 0; i < 3; ++i) {
        for (int j = 0; j < 3; ++j) cam->R[3 * i + j] = c[6 + 4 * i + j];
        cam->t[i] = c[6 + 4 * i + 3];
    }
}
static void load_cfg(const double* c, Cfg* cfg) {
    cfg->tile = (int)c[0]; cfg->cutoff = c[1]; cfg->alpha_min = c[2];
    cfg->alpha_max = c[3]; cfg->t_min = c[4]; cfg->z_near = c[5];
    cfg->tight = c[6] != 0.0;
    cfg->lowpass = c[7] != 0.0;
}

/* R26: an UPPER bound of 2 ln r (r >= 1) from +, -, x, / alone, so that the CUDA preprocess can evaluate the identical
 * binary64 sequence (no transcendental in the binning path):  r = m 2^e with m in [1, 2) by exact halvings;
 * ln m = 2 atanh(t), t = (m - 1) / (m + 1) <= 1/3, by 13 terms of the odd series in Horner form (truncation < 2e-13);
 * the result is inflated by 1e-9 relative + 1e-9 absolute, far above the series' and the roundings' error.  An upper bound
 * keeps the variant conservative: a pair with o G >= alpha_min always has rho^2 <= 2 ln(o / alpha_min) <= two_ln_upper(). */
static double two_ln_upper(double r) {
    double m = r, e = 0.0;
    while (m >= 2.0) { m = m * 0.5; e = e + 1.0; }
    const double t = (m - 1.0) / (m + 1.0), t2 = t * t;
    double p = 1.0 / 25.0;
    p = p * t2 + 1.0 / 23.0; p = p * t2 + 1.0 / 21.0; p = p * t2 + 1.0 / 19.0; p = p * t2 + 1.0 / 17.0;
    p = p * t2 + 1.0 / 15.0; p = p * t2 + 1.0 / 13.0; p = p * t2 + 1.0 / 11.0; p = p * t2 + 1.0 / 9.0;
    p = p * t2 + 1.0 / 7.0; p = p * t2 + 1.0 / 5.0; p = p * t2 + 1.0 / 3.0; p = p * t2 + 1.0;
    const double ln_m = 2.0 * (t * p);
    const double ln_r = e * 0.69314718055994540 + ln_m;   /* (0.6931471805599454 > ln 2 = 0.693147180559945309...) */
    return (2.0 * ln_r) * (1.0 + 1e-9) + 1e-9;
}
double orc_two_ln_upper(double r) { return two_ln_upper(r); }

static uint32_t f32_bits(float f) { uint32_t u; memcpy(&u, &f, 4); return u; }

/*
 * O2: the binning reference.  STRICT operation order -- the GPU preprocess kernel
 * evaluates exactly this binary64 sequence (no FMA, IEEE sqrt and division, no transcendental).
 *   q_hat = q / sqrt(((w*w + x*x) + y*y) + z*z)
 *   R(q_hat) by the unit-quaternion formula, (w,x,y,z) order
 *   t_uc = R_cw t_u, t_vc = R_cw t_v, t_nc = R_cw t_n, mu_c = R_cw mu + t_cw      (Eq. 5-6)
 *   M = K [s_u t_uc, s_v t_vc, mu_c]                                               (Eq. 7)
 *   cull iff inactive, mu_c.z <= z_near, den = c^2 (M20^2 + M21^2) - M22^2 >= 0,
 *            non-finite, or the AABB misses [0,W] x [0,H]
 *   AABB of u^2+v^2 = c^2 under the homography (closed form from Eq. 4):
 *     ctr_x = (c^2 (M00 M20 + M01 M21) - M02 M22) / den
 *     half_x = sqrt(ctr_x^2 - (c^2 (M00^2 + M01^2) - M02^2) / den),  same for y with M1
 *   tile rect = floor(min/tile) .. floor(max/tile), clamped to the tile grid
 */
static inline double dot3r(const double* r, const double* v) { return (r[0] * v[0] + r[1] * v[1]) + r[2] * v[2]; }

static void prep_surfel(const float* mean, const float* scale, const float* quat, float opacity, int is_active,
                        const Cam* cam, const Cfg* cfg, Prep* p) {
    memset(p, 0, sizeof(*p));
    p->culled = 1;
    if (!is_active) return;
    const double w = quat[0], x = quat[1], y = quat[2], z = quat[3];
    const double qn = sqrt(((w * w + x * x) + y * y) + z * z);
    p->qn = qn;
    if (!(qn > 0.0) || !isfinite(qn)) return;
    const double qw = w / qn, qx = x / qn, qy = y / qn, qz = z / qn;
    p->qh[0] = qw; p->qh[1] = qx; p->qh[2] = qy; p->qh[3] = qz;
    double* R = p->Rw;
    R[0] = 1.0 - 2.0 * (qy * qy + qz * qz); R[1] = 2.0 * (qx * qy - qw * qz); R[2] = 2.0 * (qx * qz + qw * qy);
    R[3] = 2.0 * (qx * qy + qw * qz); R[4] = 1.0 - 2.0 * (qx * qx + qz * qz); R[5] = 2.0 * (qy * qz - qw * qx);
    R[6] = 2.0 * (qx * qz - qw * qy); R[7] = 2.0 * (qy * qz + qw * qx); R[8] = 1.0 - 2.0 * (qx * qx + qy * qy);
    const double tu[3] = {R[0], R[3], R[6]}, tv[3] = {R[1], R[4], R[7]}, tn[3] = {R[2], R[5], R[8]};
    const double mu[3] = {mean[0], mean[1], mean[2]};
    for (int i = 0; i < 3; ++i) {
        p->tuc[i] = dot3r(cam->R + 3 * i, tu);
        p->tvc[i] = dot3r(cam->R + 3 * i, tv);
        p->tnc[i] = dot3r(cam->R + 3 * i, tn);
        p->muc[i] = dot3r(cam->R + 3 * i, mu) + cam->t[i];
    }
    const double su = scale[0], sv = scale[1];
    const double A0[3] = {su * p->tuc[0], sv * p->tvc[0], p->muc[0]};
    const double A1[3] = {su * p->tuc[1], sv * p->tvc[1], p->muc[1]};
    const double A2[3] = {su * p->tuc[2], sv * p->tvc[2], p->muc[2]};
    double* M = p->M;
    for (int j = 0; j < 3; ++j) {
        M[j] = cam->fx * A0[j] + cam->cx * A2[j];
        M[3 + j] = cam->fy * A1[j] + cam->cy * A2[j];
        M[6 + j] = A2[j];
    }
    p->depth_bits = f32_bits((float)p->muc[2]);
    if (!(p->muc[2] > cfg->z_near)) return;
    const int tiles_x = (cam->W + cfg->tile - 1) / cfg->tile, tiles_y = (cam->H + cfg->tile - 1) / cfg->tile;
    if (isinf(cfg->cutoff)) { /* oracle-only smooth mode (plain Eq. 8, used for finite differences): no footprint */
        p->aabb[0] = p->aabb[2] = -INFINITY; p->aabb[1] = p->aabb[3] = INFINITY;
        p->rect[0] = 0; p->rect[1] = 0; p->rect[2] = tiles_x - 1; p->rect[3] = tiles_y - 1;
        p->culled = 0;
        return;
    }
    double c2 = cfg->cutoff * cfg->cutoff;
    if (cfg->tight && cfg->alpha_min > 0.0) {
        /* R26: the splat's own support.  a = min(alpha_max, o G) >= alpha_min  <=>  o exp(-rho^2 / 2) >= alpha_min  <=>
         * rho^2 <= 2 ln(o / alpha_min); a splat with o < alpha_min contributes nowhere and is culled. */
        const double r = (double)opacity / cfg->alpha_min;
        if (!(r >= 1.0)) return;
        const double c2o = two_ln_upper(r);
        if (c2o < c2) c2 = c2o;
    }
    p->c2k = c2;
    const double den = c2 * (M[6] * M[6] + M[7] * M[7]) - M[8] * M[8];
    if (!(den < 0.0)) return;
    const double ctrx = (c2 * (M[0] * M[6] + M[1] * M[7]) - M[2] * M[8]) / den;
    const double ctry = (c2 * (M[3] * M[6] + M[4] * M[7]) - M[5] * M[8]) / den;
    const double hx = sqrt(ctrx * ctrx - (c2 * (M[0] * M[0] + M[1] * M[1]) - M[2] * M[2]) / den);
    const double hy = sqrt(ctry * ctry - (c2 * (M[3] * M[3] + M[4] * M[4]) - M[5] * M[5]) / den);
    double xmin = ctrx - hx, xmax = ctrx + hx, ymin = ctry - hy, ymax = ctry + hy;
    if (cfg->lowpass) {
        /* R28: the screen-space Gaussian of the filter reaches rho_2d^2 = 2 |x - x_c|^2 <= c^2, a disc of radius c / sqrt 2
         * around the projected centre; the footprint is the union.  A splat so close to edge-on that its own ellipse is not
         * representable (non-finite half axes) is kept through the disc. */
        const double xc = M[2] / M[8], yc = M[5] / M[8], rf = cfg->cutoff * 0.70710678118654757;
        if (!(isfinite(xmin) && isfinite(xmax))) { xmin = xc; xmax = xc; }
        if (!(isfinite(ymin) && isfinite(ymax))) { ymin = yc; ymax = yc; }
        if (xc - rf < xmin) xmin = xc - rf;
        if (xc + rf > xmax) xmax = xc + rf;
        if (yc - rf < ymin) ymin = yc - rf;
        if (yc + rf > ymax) ymax = yc + rf;
    }
    p->aabb[0] = xmin; p->aabb[1] = xmax; p->aabb[2] = ymin; p->aabb[3] = ymax;
    if (!(isfinite(xmin) && isfinite(xmax) && isfinite(ymin) && isfinite(ymax))) return;
    if (!(xmax > 0.0 && xmin < (double)cam->W && ymax > 0.0 && ymin < (double)cam->H)) return;
    const double ts = (double)cfg->tile;
    /* floor and clamp in double (exact: tile is a power of two or small integer), then cast */
    double fx0 = floor(xmin / ts), fx1 = floor(xmax / ts), fy0 = floor(ymin / ts), fy1 = floor(ymax / ts);
    if (fx0 < 0.0) fx0 = 0.0;
    if (fy0 < 0.0) fy0 = 0.0;
    if (fx1 > (double)(tiles_x - 1)) fx1 = (double)(tiles_x - 1);
    if (fy1 > (double)(tiles_y - 1)) fy1 = (double)(tiles_y - 1);
    const int tx0 = (int)fx0, tx1 = (int)fx1, ty0 = (int)fy0, ty1 = (int)fy1;
    p->rect[0] = tx0; p->rect[1] = ty0; p->rect[2] = tx1; p->rect[3] = ty1;
    p->culled = 0;
    if (cfg->tight) {
        /* R27: the footprint as a conic.  k = (M0 - x M2) x (M1 - y M2) = C0 + x Cx + y Cy with C0 = M0 x M1, Cx = M1 x M2,
         * Cy = M2 x M0, so k_x = a.p, k_y = b.p, k_z = c.p for p = (x, y, 1) and rho^2 <= c2k  <=>
         * (a.p)^2 + (b.p)^2 - c2k (c.p)^2 <= 0.  Coordinates are taken relative to the AABB's centre (ctr_x, ctr_y). */
        const double C0[3] = {M[1] * M[5] - M[2] * M[4], M[2] * M[3] - M[0] * M[5], M[0] * M[4] - M[1] * M[3]};
        const double Cx[3] = {M[4] * M[8] - M[5] * M[7], M[5] * M[6] - M[3] * M[8], M[3] * M[7] - M[4] * M[6]};
        const double Cy[3] = {M[7] * M[2] - M[8] * M[1], M[8] * M[0] - M[6] * M[2], M[6] * M[1] - M[7] * M[0]};
        const double a1 = Cx[0], a2 = Cy[0], a3 = (Cx[0] * ctrx + Cy[0] * ctry) + C0[0];
        const double b1 = Cx[1], b2 = Cy[1], b3 = (Cx[1] * ctrx + Cy[1] * ctry) + C0[1];
        const double c1 = Cx[2], c2_ = Cy[2], c3 = (Cx[2] * ctrx + Cy[2] * ctry) + C0[2];
        p->q_cx = ctrx; p->q_cy = ctry;
        p->qA = (a1 * a1 + b1 * b1) - c2 * (c1 * c1);
        p->qB = (a1 * a2 + b1 * b2) - c2 * (c1 * c2_);
        p->qC = (a2 * a2 + b2 * b2) - c2 * (c2_ * c2_);
        p->qD = (a1 * a3 + b1 * b3) - c2 * (c1 * c3);
        p->qE = (a2 * a3 + b2 * b3) - c2 * (c2_ * c3);
        p->qF = (a3 * a3 + b3 * b3) - c2 * (c3 * c3);
        const double det = p->qA * p->qC - p->qB * p->qB;
        p->q_ok = p->qA > 0.0 && p->qC > 0.0 && det > 1e-12 * (p->qA * p->qC);
    }
}

/* R27: is tile (tx, ty) of the surfel's rectangle LISTED?  Always in the default binning.  Tight binning: iff the
 * ellipse q <= 0 meets the rectangle spanned by the tile's pixel centres (clipped to the image).  q is convex, so its
 * minimum over the rectangle is attained at the ellipse centre clamped into the rectangle or on one of the four edges
 * (each a 1-D convex quadratic, minimised and clamped); listed iff that minimum is <= tol, tol = 1e-9 of the largest
 * magnitude q's terms reach on the rectangle (conservative against the binary64 rounding of the coefficients). */
static inline double conic_q(const Prep* p, double x, double y) {
    return ((((p->qA * x) * x + (2.0 * p->qB) * (x * y)) + (p->qC * y) * y) + ((2.0 * p->qD) * x + (2.0 * p->qE) * y)) + p->qF;
}
static inline double clampd(double v, double lo, double hi) { return v < lo ? lo : (v > hi ? hi : v); }
static int tile_listed(const Prep* p, int tx, int ty, const Cam* cam, const Cfg* cfg) {
    if (!cfg->tight || !p->q_ok) return 1;
    const double ts = (double)cfg->tile;
    double x1 = ts * tx + (ts - 0.5), y1 = ts * ty + (ts - 0.5);
    if (x1 > cam->W - 0.5) x1 = cam->W - 0.5;
    if (y1 > cam->H - 0.5) y1 = cam->H - 0.5;
    const double x0 = (ts * tx + 0.5) - p->q_cx, y0 = (ts * ty + 0.5) - p->q_cy;
    x1 = x1 - p->q_cx; y1 = y1 - p->q_cy;
    const double det = p->qA * p->qC - p->qB * p->qB;
    const double xc = (p->qB * p->qE - p->qC * p->qD) / det, yc = (p->qB * p->qD - p->qA * p->qE) / det;
    double qm = conic_q(p, clampd(xc, x0, x1), clampd(yc, y0, y1));
    double v;
    v = conic_q(p, x0, clampd(-(p->qB * x0 + p->qE) / p->qC, y0, y1)); if (v < qm) qm = v;
    v = conic_q(p, x1, clampd(-(p->qB * x1 + p->qE) / p->qC, y0, y1)); if (v < qm) qm = v;
    v = conic_q(p, clampd(-(p->qB * y0 + p->qD) / p->qA, x0, x1), y0); if (v < qm) qm = v;
    v = conic_q(p, clampd(-(p->qB * y1 + p->qD) / p->qA, x0, x1), y1); if (v < qm) qm = v;
    double R = fabs(x0);
    if (fabs(x1) > R) R = fabs(x1);
    if (fabs(y0) > R) R = fabs(y0);
    if (fabs(y1) > R) R = fabs(y1);
    const double tol = 1e-9 * ((fabs(p->qF) + (2.0 * (fabs(p->qD) + fabs(p->qE))) * R) + ((p->qA + p->qC) + 2.0 * fabs(p->qB)) * (R * R));
    return qm <= tol;
}

static Prep* prep_all(int64_t n, const float* mean, const float* scale, const float* quat, const float* opacity,
                      const uint8_t* active, const Cam* cam, const Cfg* cfg) {
    Prep* P = (Prep*)malloc(sizeof(Prep) * (size_t)(n > 0 ? n : 1));
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i)
        prep_surfel(mean + 3 * i, scale + 2 * i, quat + 4 * i, opacity ? opacity[i] : 1.f, active ? active[i] != 0 : 1, cam, cfg, P + i);
    return P;
}

/* ---- public: stage O2, per-surfel part.  Returns E = sum of tile counts. ---- */
int64_t orc_preprocess(int64_t n, const float* mean, const float* scale, const float* quat, const float* opacity,
                       const uint8_t* active, const double* camv, const double* cfgv,
                       uint8_t* culled, uint32_t* depth_bits, int32_t* rect, uint32_t* count,
                       double* M_out, double* aabb_out) {
    Cam cam; Cfg cfg; load_cam(camv, &cam); load_cfg(cfgv, &cfg);
    Prep* P = prep_all(n, mean, scale, quat, opacity, active, &cam, &cfg);
    int64_t E = 0;
    for (int64_t i = 0; i < n; ++i) {
        const Prep* p = P + i;
        culled[i] = (uint8_t)p->culled;
        depth_bits[i] = p->culled ? 0u : p->depth_bits;
        uint32_t c = 0;
        for (int j = 0; j < 4; ++j) rect[4 * i + j] = p->culled ? 0 : p->rect[j];
        if (!p->culled)
            for (int ty = p->rect[1]; ty <= p->rect[3]; ++ty)
                for (int tx = p->rect[0]; tx <= p->rect[2]; ++tx) c += (uint32_t)tile_listed(p, tx, ty, &cam, &cfg);
        count[i] = c;
        E += c;
        if (M_out) memcpy(M_out + 9 * i, p->M, sizeof(double) * 9);
        if (aabb_out) memcpy(aabb_out + 4 * i, p->aabb, sizeof(double) * 4);
    }
    free(P);
    return E;
}

typedef struct { uint64_t key; uint32_t idx; } Entry;
static int cmp_entry(const void* a, const void* b) {
    const Entry* x = (const Entry*)a; const Entry* y = (const Entry*)b;
    if (x->key != y->key) return x->key < y->key ? -1 : 1;
    if (x->idx != y->idx) return x->idx < y->idx ? -1 : 1; /* stable sort of a surfel-major emission */
    return 0;
}

/* ---- public: stage O2, list part.  key = tile_id << 32 | depth bits (R2); entries emitted
 * surfel-major, tiles row-major; stable sort => ties ordered by surfel index; ranges[t] = [start,end). */
void orc_bin(int64_t n, const float* mean, const float* scale, const float* quat, const float* opacity,
             const uint8_t* active, const double* camv, const double* cfgv, int64_t E, uint64_t* keys, uint32_t* idx,
             uint32_t* ranges) {
    Cam cam; Cfg cfg; load_cam(camv, &cam); load_cfg(cfgv, &cfg);
    Prep* P = prep_all(n, mean, scale, quat, opacity, active, &cam, &cfg);
    const int tiles_x = (cam.W + cfg.tile - 1) / cfg.tile, tiles_y = (cam.H + cfg.tile - 1) / cfg.tile;
    Entry* e = (Entry*)malloc(sizeof(Entry) * (size_t)(E > 0 ? E : 1));
    int64_t m = 0;
    for (int64_t i = 0; i < n; ++i) {
        const Prep* p = P + i;
        if (p->culled) continue;
        for (int ty = p->rect[1]; ty <= p->rect[3]; ++ty)
            for (int tx = p->rect[0]; tx <= p->rect[2]; ++tx) {
                if (!tile_listed(p, tx, ty, &cam, &cfg)) continue;
                e[m].key = ((uint64_t)(uint32_t)(ty * tiles_x + tx) << 32) | p->depth_bits;
                e[m].idx = (uint32_t)i;
                ++m;
            }
    }
    free(P);
    qsort(e, (size_t)m, sizeof(Entry), cmp_entry);
    const int tiles = tiles_x * tiles_y;
    for (int t = 0; t < tiles; ++t) { ranges[2 * t] = 0; ranges[2 * t + 1] = 0; }
    for (int64_t i = 0; i < m; ++i) {
        keys[i] = e[i].key; idx[i] = e[i].idx;
        const uint32_t t = (uint32_t)(e[i].key >> 32);
        if (i == 0 || (uint32_t)(e[i - 1].key >> 32) != t) ranges[2 * t] = (uint32_t)i;
        if (i == m - 1 || (uint32_t)(e[i + 1].key >> 32) != t) ranges[2 * t + 1] = (uint32_t)(i + 1);
    }
    free(e);
}

/* ---- global compositing order (R2): depth bits of the centre, ties by surfel index ---- */
typedef struct { uint32_t d; uint32_t i; } OrdKey;
static int cmp_ord(const void* a, const void* b) {
    const OrdKey* x = (const OrdKey*)a; const OrdKey* y = (const OrdKey*)b;
    if (x->d != y->d) return x->d < y->d ? -1 : 1;
    return x->i < y->i ? -1 : (x->i > y->i ? 1 : 0);
}
static uint32_t* global_order(int64_t n, const Prep* P, int64_t* n_vis) {
    OrdKey* k = (OrdKey*)malloc(sizeof(OrdKey) * (size_t)(n > 0 ? n : 1));
    int64_t m = 0;
    for (int64_t i = 0; i < n; ++i)
        if (!P[i].culled) { k[m].d = P[i].depth_bits; k[m].i = (uint32_t)i; ++m; }
    qsort(k, (size_t)m, sizeof(OrdKey), cmp_ord);
    uint32_t* ord = (uint32_t*)malloc(sizeof(uint32_t) * (size_t)(m > 0 ? m : 1));
    for (int64_t i = 0; i < m; ++i) ord[i] = k[i].i;
    free(k);
    *n_vis = m;
    return ord;
}

/*
 * Candidate lists for the "skipping" mode (O4): bucket b (B x B pixels) lists, in global order,
 * every surfel whose fp64 AABB PADDED BY 1 PIXEL touches the bucket.  A pixel outside the padded
 * AABB has rho^2 > c^2 by a margin no rounding can close, so skipping it cannot change the result.
 * Bit 31 of an entry marks "also inside the UNPADDED tile rect of stage O2" (used only to count
 * Q_t, the pairs a tile-list traversal tests).  B equals the tile size so the flag is meaningful.
 */
typedef struct { int bx, by, B; int64_t* start; uint32_t* list; } Buckets;
static void build_buckets(const Prep* P, const uint32_t* ord, int64_t n_vis, const Cam* cam, const Cfg* cfg, int B, Buckets* bk) {
    bk->B = B; bk->bx = (cam->W + B - 1) / B; bk->by = (cam->H + B - 1) / B;
    const int nb = bk->bx * bk->by;
    bk->start = (int64_t*)calloc((size_t)nb + 1, sizeof(int64_t));
    for (int pass = 0; pass < 2; ++pass) {
        int64_t* fill = NULL;
        if (pass == 1) {
            int64_t acc = 0;
            for (int b = 0; b < nb; ++b) { int64_t c = bk->start[b]; bk->start[b] = acc; acc += c; }
            bk->start[nb] = acc;
            bk->list = (uint32_t*)malloc(sizeof(uint32_t) * (size_t)(acc > 0 ? acc : 1));
            fill = (int64_t*)malloc(sizeof(int64_t) * (size_t)nb);
            memcpy(fill, bk->start, sizeof(int64_t) * (size_t)nb);
        }
        for (int64_t j = 0; j < n_vis; ++j) {
            const Prep* p = P + ord[j];
            double x0 = floor((p->aabb[0] - 1.0) / B), x1 = floor((p->aabb[1] + 1.0) / B);
            double y0 = floor((p->aabb[2] - 1.0) / B), y1 = floor((p->aabb[3] + 1.0) / B);
            if (x0 < 0) x0 = 0;
            if (y0 < 0) y0 = 0;
            if (x1 > bk->bx - 1) x1 = bk->bx - 1;
            if (y1 > bk->by - 1) y1 = bk->by - 1;
            for (int by = (int)y0; by <= (int)y1; ++by)
                for (int bx = (int)x0; bx <= (int)x1; ++bx) {
                    const int b = by * bk->bx + bx;
                    if (pass == 0) { bk->start[b]++; continue; }
                    const int inside = bx >= p->rect[0] && bx <= p->rect[2] && by >= p->rect[1] && by <= p->rect[3] &&
                                       tile_listed(p, bx, by, cam, cfg);
                    bk->list[fill[b]++] = (uint32_t)j | (inside ? 0x80000000u : 0u); /* j = rank in ord */
                }
        }
        if (fill) free(fill);
    }
}
static void free_buckets(Buckets* bk) { free(bk->start); free(bk->list); }

/* ---------------------------------------------------------------------------------------------
 * O3 + O4: one (pixel, surfel) pair.  Ray-splat intersection derived from Eq. 4 (R1):
 *   h_u = M0 - x M2,  h_v = M1 - y M2,  k = h_u x h_v,  (u,v) = k_xy / k_z,  z = M2 . (u,v,1)
 * then Eq. 8 with the truncation conventions R3-R7:
 *   skip if k_z == 0 or non-finite; skip if rho^2 > c^2; skip if z <= z_near;
 *   G = exp(-rho^2/2); a = min(alpha_max, o G); skip if a < alpha_min;
 *   T' = T (1 - a); if T' < t_min: STOP the pixel, this surfel is not composited.
 * Returns 0 = skipped, 1 = composited, 2 = stop.  *frag is OR-ed with 1 when any decision taken
 * had relative margin < 1e-4.
 * ------------------------------------------------------------------------------------------- */
typedef struct {
    double hu[3], hv[3], k[3], u, v, z, G, a;
    int clamped;
    int use2d;      /* R28: the screen-space term of the low-pass filter gave rho^2 (and the depth is the centre's) */
    double dx, dy;  /* R28: pixel minus projected centre */
} Pair;

#define FRAG_EPS 1e-4
#define KAPPA_MAX 32.0
static inline int eval_pair(const Prep* p, double opac, double x, double y, double T, const Cfg* cfg,
                            Pair* r, int* frag, int* covers) {
    const double* M = p->M;
    for (int j = 0; j < 3; ++j) { r->hu[j] = M[j] - x * M[6 + j]; r->hv[j] = M[3 + j] - y * M[6 + j]; }
    r->k[0] = r->hu[1] * r->hv[2] - r->hu[2] * r->hv[1];
    r->k[1] = r->hu[2] * r->hv[0] - r->hu[0] * r->hv[2];
    r->k[2] = r->hu[0] * r->hv[1] - r->hu[1] * r->hv[0];
    *covers = 0;
    r->use2d = 0;
    double rho2;
    if (cfg->lowpass) {
        /* R28: rho^2 = min(u^2 + v^2, 2 |x - x_c|^2), x_c = (M02, M12) / M22 the projected centre; the screen term also
         * stands in where the intersection is undefined.  Where it wins the pair's depth is the centre depth M22. */
        r->dx = x - M[2] / M[8]; r->dy = y - M[5] / M[8];
        const double rho2_2d = 2.0 * (r->dx * r->dx + r->dy * r->dy);
        double rho2_3d = INFINITY;
        r->u = 0.0; r->v = 0.0;
        if (r->k[2] != 0.0) {
            r->u = r->k[0] / r->k[2]; r->v = r->k[1] / r->k[2];
            rho2_3d = r->u * r->u + r->v * r->v;
            if (!isfinite(rho2_3d)) rho2_3d = INFINITY;
        }
        if (isfinite(rho2_3d) && fabs(rho2_3d - rho2_2d) < FRAG_EPS * rho2_2d) *frag |= 1;   /* which term wins decides depth and gradient */
        r->use2d = !(rho2_3d <= rho2_2d);
        rho2 = r->use2d ? rho2_2d : rho2_3d;
    } else {
        if (r->k[2] == 0.0) return 0;
        r->u = r->k[0] / r->k[2];
        r->v = r->k[1] / r->k[2];
        rho2 = r->u * r->u + r->v * r->v;
        if (!isfinite(rho2)) return 0;
    }
    const double c2 = cfg->cutoff * cfg->cutoff;
    if (isfinite(c2) && fabs(rho2 - c2) < FRAG_EPS * c2) *frag |= 1;
    if (rho2 > c2) return 0;
    r->z = r->use2d ? M[8] : M[6] * r->u + M[7] * r->v + M[8];
    if (cfg->z_near > 0.0 && fabs(r->z - cfg->z_near) < FRAG_EPS * cfg->z_near) *frag |= 1;
    if (!(r->z > cfg->z_near)) return 0;
    *covers = 1;
    r->G = exp(-0.5 * rho2);
    const double og = opac * r->G;
    if (fabs(og - cfg->alpha_max) < FRAG_EPS * cfg->alpha_max) *frag |= 2; /* matters to gradients only */
    r->clamped = og > cfg->alpha_max;
    r->a = r->clamped ? cfg->alpha_max : og;
    if (cfg->alpha_min > 0.0 && fabs(r->a - cfg->alpha_min) < FRAG_EPS * cfg->alpha_min) *frag |= 1;
    if (r->a < cfg->alpha_min) return 0;
    const double Tn = T * (1.0 - r->a);
    if (cfg->t_min > 0.0 && fabs(Tn - cfg->t_min) < FRAG_EPS * cfg->t_min) *frag |= 1;
    if (Tn < cfg->t_min) return 2;
    /* Ill-conditioned intersection: kappa = |h_u||h_v| / |k_z| (uv parts) is ~ 1/cos(tilt) of the
     * splat against the ray.  Beyond KAPPA_MAX the fp32 rounding of the INPUTS already moves (u,v)
     * by more than the image tolerance allows (delta G / G ~ rho^2 kappa 2e-7), so no binary32
     * renderer can be held to 1e-4 there: flag bit 2 (value 4) of the fragile mask. */
    if (!r->use2d) {
        const double nu = r->hu[0] * r->hu[0] + r->hu[1] * r->hu[1], nv = r->hv[0] * r->hv[0] + r->hv[1] * r->hv[1];
        if (sqrt(nu * nv) > KAPPA_MAX * fabs(r->k[2])) *frag |= 4;
    }
    return 1;
}

typedef struct {
    int64_t n;
    const float *opacity, *rgb;
    Cam cam; Cfg cfg;
    Prep* P;
    uint32_t* ord; int64_t n_vis;
    Buckets bk; int brute;
} Ctx;

static void ctx_init(Ctx* c, int64_t n, const float* mean, const float* scale, const float* quat,
                     const float* opacity, const float* rgb, const uint8_t* active,
                     const double* camv, const double* cfgv, int brute) {
    load_cam(camv, &c->cam); load_cfg(cfgv, &c->cfg);
    c->n = n; c->opacity = opacity; c->rgb = rgb; c->brute = brute;
    c->P = prep_all(n, mean, scale, quat, opacity, active, &c->cam, &c->cfg);
    c->ord = global_order(n, c->P, &c->n_vis);
    build_buckets(c->P, c->ord, c->n_vis, &c->cam, &c->cfg, c->cfg.tile, &c->bk);
}
static void ctx_free(Ctx* c) { free(c->P); free(c->ord); free_buckets(&c->bk); }

/* candidate iteration for pixel (i,j): brute = every visible surfel in global order;
 * skipping = the pixel's bucket list, further filtered by the padded AABB. */
static inline int64_t cand_count(const Ctx* c, int i, int j, const uint32_t** lst) {
    if (c->brute) { *lst = NULL; return c->n_vis; }
    const int b = (j / c->bk.B) * c->bk.bx + (i / c->bk.B);
    *lst = c->bk.list + c->bk.start[b];
    return c->bk.start[b + 1] - c->bk.start[b];
}

/* ---- public: forward (O4).  img = 8 planes H*W: r,g,b, depth, nx,ny,nz, alpha (un-normalised
 * blends, R9/R10; background 0, R17).  counters: [0]=Q_t tile-list pairs tested up to and incl.
 * the stopping entry, [1]=Q_c composited pairs, [2]=covering pairs (rho^2<=c^2, z>z_near) over
 * ALL surfels ignoring termination (depth complexity), [3]=n_vis, [4]=fragile pixels,
 * [5]=Q_tb tile-list pairs up to and incl. each pixel's LAST COMPOSITED entry (what a reverse traversal revisits). */
static inline void atomic_add_fwd(double* p, double v) {
#pragma omp atomic
    *p += v;
}

/* contrib (nullable, n doubles, zero-initialised by the caller): the contribution of splat k to the view,
 * C_k^V = sum over pixels of its blending coefficient w_k(p) = a_k T_k (Eq. 20-21). */
void orc_render_ex2(int64_t n, const float* mean, const float* scale, const float* quat, const float* opacity, const float* rgb,
                    const uint8_t* active, const double* camv, const double* cfgv, int brute, double* img, double* T_final,
                    int32_t* n_comp, uint8_t* fragile, int64_t* counters, int32_t* qtb_pix, double* contrib, double* median,
                    uint8_t* median_fragile);

void orc_render_ex(int64_t n, const float* mean, const float* scale, const float* quat,
                   const float* opacity, const float* rgb, const uint8_t* active,
                   const double* camv, const double* cfgv, int brute,
                   double* img, double* T_final, int32_t* n_comp, uint8_t* fragile, int64_t* counters,
                   int32_t* qtb_pix /* nullable: per-pixel Q_tb */, double* contrib) {
    orc_render_ex2(n, mean, scale, quat, opacity, rgb, active, camv, cfgv, brute, img, T_final, n_comp, fragile, counters, qtb_pix,
                   contrib, NULL, NULL);
}

/* + median depth (DESIGN R9m; a variant of the depth image of L118-120): along the pixel's ray
 * the blending weights w_i of Eq. 8 and the remaining transmittance T_final form a distribution over the
 * intersection depths z_i (and "nothing hit"); its median is the z_i of the composited splat at which the
 * transmittance first falls to T_{i+1} = prod_{j<=i}(1 - a_j) <= 1/2.  0 where T_final > 1/2.  median_fragile: some
 * composited splat left T within 1e-4 of 1/2 (the GPU's fp32 may pick the neighbouring splat there). */
void orc_render_ex2(int64_t n, const float* mean, const float* scale, const float* quat,
                    const float* opacity, const float* rgb, const uint8_t* active,
                    const double* camv, const double* cfgv, int brute,
                    double* img, double* T_final, int32_t* n_comp, uint8_t* fragile, int64_t* counters,
                    int32_t* qtb_pix, double* contrib, double* median, uint8_t* median_fragile) {
    Ctx c; ctx_init(&c, n, mean, scale, quat, opacity, rgb, active, camv, cfgv, brute);
    const int W = c.cam.W, H = c.cam.H; const int64_t HW = (int64_t)W * H;
    int64_t Qt = 0, Qc = 0, Qcover = 0, nfrag = 0, Qtb = 0;
    const int count_all = counters != NULL; /* the covering count needs the traversal past termination */
#pragma omp parallel for schedule(dynamic, 1) reduction(+ : Qt, Qc, Qcover, nfrag, Qtb)
    for (int j = 0; j < H; ++j) {
        for (int i = 0; i < W; ++i) {
            const double x = i + 0.5, y = j + 0.5; /* pixel centres at half integers (R17) */
            const uint32_t* lst; const int64_t m = cand_count(&c, i, j, &lst);
            double acc[8] = {0, 0, 0, 0, 0, 0, 0, 0}, T = 1.0;
            int frag = 0, stopped = 0, nc = 0, medfrag = 0;
            double med = 0.0;
            int64_t qt_pix = 0, qt_last = 0;
            for (int64_t e = 0; e < m; ++e) {
                const uint32_t raw = lst ? lst[e] : (uint32_t)e;
                const uint32_t k = c.ord[raw & 0x7fffffffu];
                const Prep* p = c.P + k;
                if (lst) {
                    if (x < p->aabb[0] - 1.0 || x > p->aabb[1] + 1.0 || y < p->aabb[2] - 1.0 || y > p->aabb[3] + 1.0) {
                        if ((raw >> 31) && !stopped) ++qt_pix;
                        continue;
                    }
                }
                Pair r; int covers, f = 0;
                const int st = eval_pair(p, opacity[k], x, y, T, &c.cfg, &r, &f, &covers);
                Qcover += covers;
                if (stopped) continue; /* past termination: only the covering count continues */
                if (!lst || (raw >> 31)) ++qt_pix;
                frag |= f;
                if (st == 2) { stopped = 1; if (!count_all) break; continue; }
                if (st == 0) continue;
                const double w = r.a * T;
                acc[0] += w * rgb[3 * k]; acc[1] += w * rgb[3 * k + 1]; acc[2] += w * rgb[3 * k + 2];
                acc[3] += w * r.z;
                acc[4] += w * p->tnc[0]; acc[5] += w * p->tnc[1]; acc[6] += w * p->tnc[2];
                acc[7] += w;
                if (contrib) atomic_add_fwd(contrib + k, w); /* Eq. 21 */
                if (T > 0.5 && T * (1.0 - r.a) <= 0.5) med = r.z; /* the one splat that takes T across 1/2 */
                if (fabs(T * (1.0 - r.a) - 0.5) < 1e-4) medfrag = 1;
                T *= (1.0 - r.a);
                ++nc; ++Qc;
                qt_last = qt_pix;
            }
            const int64_t pix = (int64_t)j * W + i;
            for (int ch = 0; ch < 8; ++ch) img[ch * HW + pix] = acc[ch];
            if (T_final) T_final[pix] = T;
            if (n_comp) n_comp[pix] = nc;
            if (qtb_pix) qtb_pix[pix] = (int32_t)qt_last;
            if (fragile) fragile[pix] = (uint8_t)frag;
            if (median) median[pix] = med;
            if (median_fragile) median_fragile[pix] = (uint8_t)medfrag;
            nfrag += (frag & 5) != 0;
            Qt += qt_pix; Qtb += qt_last;
        }
    }
    if (counters) { counters[0] = Qt; counters[1] = Qc; counters[2] = Qcover; counters[3] = c.n_vis; counters[4] = nfrag; counters[5] = Qtb; }
    ctx_free(&c);
}

void orc_render(int64_t n, const float* mean, const float* scale, const float* quat,
                const float* opacity, const float* rgb, const uint8_t* active,
                const double* camv, const double* cfgv, int brute,
                double* img, double* T_final, int32_t* n_comp, uint8_t* fragile, int64_t* counters,
                int32_t* qtb_pix) {
    orc_render_ex(n, mean, scale, quat, opacity, rgb, active, camv, cfgv, brute, img, T_final, n_comp, fragile, counters,
                  qtb_pix, NULL);
}

/* ---------------------------------------------------------------------------------------------
 * O5-O7: analytic backward.
 * Per pixel, over its composited list i = 0..m-1 (front to back) with w_i = a_i T_i and
 * v_i = (rgb_k, z_i, t_nc_k, 1) (Eq. 8 and L118-120), g = upstream gradient of the 8 planes:
 *   dL/dv_i   = g w_i                          -> rgb_k, t_nc_k, z_i
 *   dL/da_i   = T_i (g.v_i) - (sum_{j>i} w_j (g.v_j)) / (1 - a_i)
 *   a = min(alpha_max, o G): zero derivative when clamped (R5), else da/do = G, da/dG = o
 *   dG/du = -u G, dG/dv = -v G;  z = M20 u + M21 v + M22
 *   dL/dk = (dL/du, dL/dv, -(u dL/du + v dL/dv)) / k_z
 *   dL/dh_u = h_v x dL/dk,  dL/dh_v = dL/dk x h_u
 *   dL/dM0 += dL/dh_u, dL/dM1 += dL/dh_v, dL/dM2 -= x dL/dh_u + y dL/dh_v      (this is dL/dT of L130)
 * Per surfel (O6, Eq. 9-10 with R11, R13, R14):
 *   G = K^T dL/dM = [dL/d(s_u t_uc), dL/d(s_v t_vc), dL/dmu_c]
 *   dL/dt_uc = s_u G[:,0], dL/ds_u = t_uc . G[:,0] (same for v); dL/dt_nc from the normal planes
 *   world: dL/dmu = R_cw^T dL/dmu_c, dL/dR = R_cw^T [dL/dt_uc, dL/dt_vc, dL/dt_nc];
 *   then the Jacobian of R(q/|q|).
 * Pose (O7, Eq. 11-13, left perturbation Exp(tau) o T_cw, tau = (rho, theta), R12, R15):
 *   dL/drho = sum_k dL/dmu_c;  dL/dtheta = sum_k [mu_c x dL/dmu_c + sum_i R_c[:,i] x dL/dR_c[:,i]]
 * ------------------------------------------------------------------------------------------- */
typedef struct { uint32_t k; Pair r; double T; } Hit;

static inline void atomic_add(double* p, double v) {
#pragma omp atomic
    *p += v;
}
static inline void cross3(const double* a, const double* b, double* o) {
    o[0] = a[1] * b[2] - a[2] * b[1]; o[1] = a[2] * b[0] - a[0] * b[2]; o[2] = a[0] * b[1] - a[1] * b[0];
}

void orc_backward(int64_t n, const float* mean, const float* scale, const float* quat,
                  const float* opacity, const float* rgb, const uint8_t* active,
                  const double* camv, const double* cfgv, int brute, const double* up /* 8*H*W */,
                  double* d_mean, double* d_scale, double* d_quat, double* d_opacity, double* d_rgb,
                  double* d_pose /* 6 */, double* dM_out /* n*9, nullable */, double* dnc_out /* n*3, nullable */,
                  uint8_t* surfel_fragile /* n, nullable */) {
    Ctx c; ctx_init(&c, n, mean, scale, quat, opacity, rgb, active, camv, cfgv, brute);
    const int W = c.cam.W, H = c.cam.H; const int64_t HW = (int64_t)W * H;
    const size_t nn = (size_t)(n > 0 ? n : 1);
    double* dM = (double*)calloc(nn * 9, sizeof(double));
    double* dnc = (double*)calloc(nn * 3, sizeof(double));
    memset(d_mean, 0, sizeof(double) * 3 * (size_t)n); memset(d_scale, 0, sizeof(double) * 2 * (size_t)n);
    memset(d_quat, 0, sizeof(double) * 4 * (size_t)n); memset(d_opacity, 0, sizeof(double) * (size_t)n);
    memset(d_rgb, 0, sizeof(double) * 3 * (size_t)n);
    if (surfel_fragile) memset(surfel_fragile, 0, (size_t)n);
#pragma omp parallel
    {
        size_t cap = 256; Hit* hits = (Hit*)malloc(sizeof(Hit) * cap);
#pragma omp for schedule(dynamic, 1)
        for (int j = 0; j < H; ++j) {
            for (int i = 0; i < W; ++i) {
                const double x = i + 0.5, y = j + 0.5;
                const int64_t pix = (int64_t)j * W + i;
                double g[8];
                for (int ch = 0; ch < 8; ++ch) g[ch] = up[ch * HW + pix];
                const uint32_t* lst; const int64_t m = cand_count(&c, i, j, &lst);
                /* forward replay, storing the composited list */
                size_t nh = 0; double T = 1.0;
                for (int64_t e = 0; e < m; ++e) {
                    const uint32_t raw = lst ? lst[e] : (uint32_t)e;
                    const uint32_t k = c.ord[raw & 0x7fffffffu];
                    const Prep* p = c.P + k;
                    if (lst && (x < p->aabb[0] - 1.0 || x > p->aabb[1] + 1.0 || y < p->aabb[2] - 1.0 || y > p->aabb[3] + 1.0))
                        continue;
                    Pair r; int covers, f = 0;
                    const int st = eval_pair(p, opacity[k], x, y, T, &c.cfg, &r, &f, &covers);
                    if (f && surfel_fragile) surfel_fragile[k] = 1; /* benign race: any writer stores 1 */
                    if (st == 2) break;
                    if (st == 0) continue;
                    if (nh == cap) { cap *= 2; hits = (Hit*)realloc(hits, sizeof(Hit) * cap); }
                    hits[nh].k = k; hits[nh].r = r; hits[nh].T = T; ++nh;
                    T *= (1.0 - r.a);
                }
                /* reverse sweep */
                double suffix = 0.0; /* sum_{j>i} w_j (g . v_j) */
                for (size_t q = nh; q-- > 0;) {
                    const Hit* h = hits + q; const uint32_t k = h->k; const Prep* p = c.P + k; const Pair* r = &h->r;
                    const double w = r->a * h->T;
                    const double gv = g[0] * rgb[3 * k] + g[1] * rgb[3 * k + 1] + g[2] * rgb[3 * k + 2] + g[3] * r->z +
                                      g[4] * p->tnc[0] + g[5] * p->tnc[1] + g[6] * p->tnc[2] + g[7];
                    for (int ch = 0; ch < 3; ++ch) {
                        atomic_add(d_rgb + 3 * k + ch, g[ch] * w);
                        atomic_add(dnc + 3 * k + ch, g[4 + ch] * w);
                    }
                    const double dz = g[3] * w;
                    const double da = h->T * gv - suffix / (1.0 - r->a);
                    suffix += w * gv;
                    double dG = 0.0;
                    if (!r->clamped) { atomic_add(d_opacity + k, da * r->G); dG = da * opacity[k]; }
                    if (r->use2d) {
                        /* R28, screen term: G = exp(-|x - x_c|^2), z = M22;  x_c = M02 / M22, y_c = M12 / M22:
                         * dG/dx_c = 2 dx G, dG/dy_c = 2 dy G;  dx_c/dM02 = 1 / M22, dx_c/dM22 = -x_c / M22 (same for y) */
                        const double gxc = 2.0 * r->dx * r->G * dG, gyc = 2.0 * r->dy * r->G * dG, m22 = p->M[8];
                        atomic_add(dM + 9 * k + 2, gxc / m22);
                        atomic_add(dM + 9 * k + 5, gyc / m22);
                        atomic_add(dM + 9 * k + 8, dz - (gxc * (p->M[2] / m22) + gyc * (p->M[5] / m22)) / m22);
                        continue;
                    }
                    const double du = -r->u * r->G * dG + dz * p->M[6];
                    const double dv = -r->v * r->G * dG + dz * p->M[7];
                    const double dk[3] = {du / r->k[2], dv / r->k[2], -(r->u * du + r->v * dv) / r->k[2]};
                    double dhu[3], dhv[3];
                    cross3(r->hv, dk, dhu);
                    cross3(dk, r->hu, dhv);
                    const double uv1[3] = {r->u, r->v, 1.0};
                    for (int t = 0; t < 3; ++t) {
                        atomic_add(dM + 9 * k + t, dhu[t]);
                        atomic_add(dM + 9 * k + 3 + t, dhv[t]);
                        atomic_add(dM + 9 * k + 6 + t, dz * uv1[t] - x * dhu[t] - y * dhv[t]);
                    }
                }
            }
        }
        free(hits);
    }
    /* O6 + O7 */
    double pose[6] = {0, 0, 0, 0, 0, 0};
    const double* Rc = c.cam.R;
    for (int64_t k = 0; k < n; ++k) {
        const Prep* p = c.P + k;
        if (p->culled) continue;
        const double* m = dM + 9 * k;
        const double su = scale[2 * k], sv = scale[2 * k + 1];
        double Gc[3][3]; /* Gc[row][col] = dL/dA, A = [s_u t_uc, s_v t_vc, mu_c]  (Eq. 9, K^T dL/dM) */
        for (int col = 0; col < 3; ++col) {
            Gc[0][col] = c.cam.fx * m[col];
            Gc[1][col] = c.cam.fy * m[3 + col];
            Gc[2][col] = c.cam.cx * m[col] + c.cam.cy * m[3 + col] + m[6 + col];
        }
        double dtuc[3], dtvc[3], dtnc[3], dmuc[3];
        double dsu = 0, dsv = 0;
        for (int r = 0; r < 3; ++r) {
            dtuc[r] = su * Gc[r][0]; dtvc[r] = sv * Gc[r][1]; dmuc[r] = Gc[r][2]; dtnc[r] = dnc[3 * k + r];
            dsu += p->tuc[r] * Gc[r][0]; dsv += p->tvc[r] * Gc[r][1];
        }
        d_scale[2 * k] = dsu; d_scale[2 * k + 1] = dsv;
        /* pose, Eq. 11-13 */
        double t0[3], t1[3], t2[3], t3[3];
        cross3(p->muc, dmuc, t0); cross3(p->tuc, dtuc, t1); cross3(p->tvc, dtvc, t2); cross3(p->tnc, dtnc, t3);
        for (int r = 0; r < 3; ++r) { pose[r] += dmuc[r]; pose[3 + r] += t0[r] + t1[r] + t2[r] + t3[r]; }
        /* to world: x_c = R_cw x_w  =>  dL/dx_w = R_cw^T dL/dx_c */
        double GR[3][3]; /* dL/dR (world), columns t_u, t_v, t_n */
        for (int r = 0; r < 3; ++r) {
            d_mean[3 * k + r] = Rc[0 + r] * dmuc[0] + Rc[3 + r] * dmuc[1] + Rc[6 + r] * dmuc[2];
            GR[r][0] = Rc[0 + r] * dtuc[0] + Rc[3 + r] * dtuc[1] + Rc[6 + r] * dtuc[2];
            GR[r][1] = Rc[0 + r] * dtvc[0] + Rc[3 + r] * dtvc[1] + Rc[6 + r] * dtvc[2];
            GR[r][2] = Rc[0 + r] * dtnc[0] + Rc[3 + r] * dtnc[1] + Rc[6 + r] * dtnc[2];
        }
        const double qw = p->qh[0], qx = p->qh[1], qy = p->qh[2], qz = p->qh[3];
        double dq[4];
        dq[0] = 2.0 * (-qz * GR[0][1] + qy * GR[0][2] + qz * GR[1][0] - qx * GR[1][2] - qy * GR[2][0] + qx * GR[2][1]);
        dq[1] = 2.0 * (qy * GR[0][1] + qz * GR[0][2] + qy * GR[1][0] - 2.0 * qx * GR[1][1] - qw * GR[1][2] + qz * GR[2][0] + qw * GR[2][1] - 2.0 * qx * GR[2][2]);
        dq[2] = 2.0 * (-2.0 * qy * GR[0][0] + qx * GR[0][1] + qw * GR[0][2] + qx * GR[1][0] + qz * GR[1][2] - qw * GR[2][0] + qz * GR[2][1] - 2.0 * qy * GR[2][2]);
        dq[3] = 2.0 * (-2.0 * qz * GR[0][0] - qw * GR[0][1] + qx * GR[0][2] + qw * GR[1][0] - 2.0 * qz * GR[1][1] + qy * GR[1][2] + qx * GR[2][0] + qy * GR[2][1]);
        const double qd = qw * dq[0] + qx * dq[1] + qy * dq[2] + qz * dq[3];
        for (int r = 0; r < 4; ++r) d_quat[4 * k + r] = (dq[r] - p->qh[r] * qd) / p->qn; /* through q/|q| */
    }
    for (int r = 0; r < 6; ++r) d_pose[r] = pose[r];
    if (dM_out) memcpy(dM_out, dM, sizeof(double) * 9 * (size_t)n);
    if (dnc_out) memcpy(dnc_out, dnc, sizeof(double) * 3 * (size_t)n);
    free(dM); free(dnc);
    ctx_free(&c);
}

/* ---------------------------------------------------------------------------------------------
 * Comparison support (DESIGN.md §6 "fragile pixels"): NOT part of the rendered function or its gradient.
 *
 * A binary32 renderer and this binary64 oracle may take a DIFFERENT discrete decision (rho^2 <= c^2, z > z_near,
 * a >= alpha_min, o G > alpha_max, T (1 - a) < t_min) at a pixel where the oracle's margin is below FRAG_EPS, and cannot
 * agree to the image tolerance on a pair whose intersection is ill-conditioned (kappa > KAPPA_MAX).  Such pixels are
 * compared against a bound DERIVED here instead of a flat allowance:
 *
 *  orc_pixel_bounds: per pixel, for the forward images,
 *    flip_w  = sum over the pixel's fragile decisions of the blending weight at stake, a T of the pair (+ T' behind a
 *              fragile stop): flipping one decision moves a blended value by at most 2 vmax flip_w
 *              (|dV/da_i| <= 2 T_i vmax by Eq. 8, and the pair's own term is a T v);
 *    kerr    = sum over composited pairs of w rho^2 kappa: first-order sensitivity of the blend to the relative rounding
 *              eps of the intersection's inputs, delta G / G = rho^2 kappa eps  =>  |delta V| <= 2 vmax eps kerr;
 *    kerr_z  = sum over composited pairs of w kappa (|M20 u| + |M21 v|): the same for the depth value z itself;
 *    zmax    = largest intersection depth among the pixel's composited or fragile pairs (vmax of the depth channel).
 *
 *  orc_exposure: per surfel and parameter, the summed |contribution| of the "exposed" pixels (fragile ones, plus a mask
 *    the caller passes) to the gradient, evaluated on the oracle's own composited list AND on the list with every fragile
 *    decision of that pixel inverted; likewise for the pose 6-vector.  A renderer that decides differently at those pixels
 *    differs from the oracle's gradient by at most a small multiple of this sum.  With signed_all != 0 it instead
 *    accumulates the SIGNED contributions of the oracle's own list over ALL pixels, i.e. recomputes orc_backward pair by
 *    pair through surfel_chain() -- the self-check that pins this function to orc_backward (tests/test_oracle_pins.py).
 * ------------------------------------------------------------------------------------------- */
static inline double pair_kappa(const Pair* r) {
    const double nu = r->hu[0] * r->hu[0] + r->hu[1] * r->hu[1], nv = r->hv[0] * r->hv[0] + r->hv[1] * r->hv[1];
    return sqrt(nu * nv) / fabs(r->k[2]);
}
/* fields eval_pair() leaves unset when it rejects a pair early (u, v are set whenever k_z != 0) */
/* the pair's rho^2 (R28: of the term r->use2d names) */
static inline double pair_rho2(const Cfg* cfg, const Pair* r) {
    return (cfg->lowpass && r->use2d) ? 2.0 * (r->dx * r->dx + r->dy * r->dy) : r->u * r->u + r->v * r->v;
}
/* does eval_pair() define the pair's geometry at all? (default: the intersection must exist; R28: the screen term always does) */
static inline int pair_defined(const Cfg* cfg, const Pair* r) {
    if (cfg->lowpass) return 1;
    return r->k[2] != 0.0 && isfinite(r->u * r->u + r->v * r->v);
}
static inline void pair_complete(const Prep* p, double opac, const Cfg* cfg, Pair* r) {
    const double rho2 = pair_rho2(cfg, r);
    r->z = (cfg->lowpass && r->use2d) ? p->M[8] : p->M[6] * r->u + p->M[7] * r->v + p->M[8];
    r->G = exp(-0.5 * rho2);
    const double og = opac * r->G;
    r->clamped = og > cfg->alpha_max;
    r->a = r->clamped ? cfg->alpha_max : og;
}

void orc_pixel_bounds(int64_t n, const float* mean, const float* scale, const float* quat, const float* opacity,
                      const float* rgb, const uint8_t* active, const double* camv, const double* cfgv,
                      double* flip_w, double* kerr, double* kerr_z, double* zmax) {
    Ctx c; ctx_init(&c, n, mean, scale, quat, opacity, rgb, active, camv, cfgv, 0);
    const int W = c.cam.W, H = c.cam.H;
#pragma omp parallel for schedule(dynamic, 1)
    for (int j = 0; j < H; ++j) {
        for (int i = 0; i < W; ++i) {
            const double x = i + 0.5, y = j + 0.5;
            const uint32_t* lst; const int64_t m = cand_count(&c, i, j, &lst);
            double T = 1.0, fw = 0.0, ke = 0.0, kz = 0.0, zm = 0.0;
            for (int64_t e = 0; e < m; ++e) {
                const uint32_t k = c.ord[lst[e] & 0x7fffffffu];
                const Prep* p = c.P + k;
                if (x < p->aabb[0] - 1.0 || x > p->aabb[1] + 1.0 || y < p->aabb[2] - 1.0 || y > p->aabb[3] + 1.0) continue;
                Pair r; int covers, f = 0;
                const int st = eval_pair(p, opacity[k], x, y, T, &c.cfg, &r, &f, &covers);
                if ((f & 1) && pair_defined(&c.cfg, &r)) {
                    if (st != 1) pair_complete(p, opacity[k], &c.cfg, &r);
                    fw += r.a * T + (st == 2 ? T * (1.0 - r.a) : 0.0);
                    if (fabs(r.z) > zm) zm = fabs(r.z);
                }
                if (st == 2) break;
                if (st == 0) continue;
                const double w = r.a * T, kap = r.use2d ? 0.0 : pair_kappa(&r);   /* (R28 screen term: no intersection, no kappa) */
                ke += w * (r.u * r.u + r.v * r.v) * kap;
                kz += w * kap * (fabs(p->M[6] * r.u) + fabs(p->M[7] * r.v));
                if (fabs(r.z) > zm) zm = fabs(r.z);
                T *= (1.0 - r.a);
            }
            const int64_t pix = (int64_t)j * W + i;
            flip_w[pix] = fw; kerr[pix] = ke; kerr_z[pix] = kz; zmax[pix] = zm;
        }
    }
    ctx_free(&c);
}

/* O6 + O7 for ONE set of per-surfel accumulators (dL/dM 9, dL/dt_nc 3): out13 = d mean (3), d scale (2), d quat (4),
 * [9..12 left to the caller: opacity, rgb], pose6 = this surfel's share of (dL/drho, dL/dtheta).  Same formulas as the loop
 * at the end of orc_backward (Eq. 9-13, R11-R15), written once more so that orc_backward stays one readable function. */
static void surfel_chain(const Ctx* c, int64_t k, const float* scale, const double* m, const double* dnc, double* out13,
                         double* pose6) {
    const Prep* p = c->P + k;
    const double* Rc = c->cam.R;
    const double su = scale[2 * k], sv = scale[2 * k + 1];
    double Gc[3][3];
    for (int col = 0; col < 3; ++col) {
        Gc[0][col] = c->cam.fx * m[col];
        Gc[1][col] = c->cam.fy * m[3 + col];
        Gc[2][col] = c->cam.cx * m[col] + c->cam.cy * m[3 + col] + m[6 + col];
    }
    double dtuc[3], dtvc[3], dtnc[3], dmuc[3], dsu = 0, dsv = 0;
    for (int r = 0; r < 3; ++r) {
        dtuc[r] = su * Gc[r][0]; dtvc[r] = sv * Gc[r][1]; dmuc[r] = Gc[r][2]; dtnc[r] = dnc[r];
        dsu += p->tuc[r] * Gc[r][0]; dsv += p->tvc[r] * Gc[r][1];
    }
    out13[3] = dsu; out13[4] = dsv;
    double t0[3], t1[3], t2[3], t3[3];
    cross3(p->muc, dmuc, t0); cross3(p->tuc, dtuc, t1); cross3(p->tvc, dtvc, t2); cross3(p->tnc, dtnc, t3);
    for (int r = 0; r < 3; ++r) { pose6[r] = dmuc[r]; pose6[3 + r] = t0[r] + t1[r] + t2[r] + t3[r]; }
    double GR[3][3];
    for (int r = 0; r < 3; ++r) {
        out13[r] = Rc[0 + r] * dmuc[0] + Rc[3 + r] * dmuc[1] + Rc[6 + r] * dmuc[2];
        GR[r][0] = Rc[0 + r] * dtuc[0] + Rc[3 + r] * dtuc[1] + Rc[6 + r] * dtuc[2];
        GR[r][1] = Rc[0 + r] * dtvc[0] + Rc[3 + r] * dtvc[1] + Rc[6 + r] * dtvc[2];
        GR[r][2] = Rc[0 + r] * dtnc[0] + Rc[3 + r] * dtnc[1] + Rc[6 + r] * dtnc[2];
    }
    const double qw = p->qh[0], qx = p->qh[1], qy = p->qh[2], qz = p->qh[3];
    double dq[4];
    dq[0] = 2.0 * (-qz * GR[0][1] + qy * GR[0][2] + qz * GR[1][0] - qx * GR[1][2] - qy * GR[2][0] + qx * GR[2][1]);
    dq[1] = 2.0 * (qy * GR[0][1] + qz * GR[0][2] + qy * GR[1][0] - 2.0 * qx * GR[1][1] - qw * GR[1][2] + qz * GR[2][0] + qw * GR[2][1] - 2.0 * qx * GR[2][2]);
    dq[2] = 2.0 * (-2.0 * qy * GR[0][0] + qx * GR[0][1] + qw * GR[0][2] + qx * GR[1][0] + qz * GR[1][2] - qw * GR[2][0] + qz * GR[2][1] - 2.0 * qy * GR[2][2]);
    dq[3] = 2.0 * (-2.0 * qz * GR[0][0] - qw * GR[0][1] + qx * GR[0][2] + qw * GR[1][0] - 2.0 * qz * GR[1][1] + qy * GR[1][2] + qx * GR[2][0] + qy * GR[2][1]);
    const double qd = qw * dq[0] + qx * dq[1] + qy * dq[2] + qz * dq[3];
    for (int r = 0; r < 4; ++r) out13[5 + r] = (dq[r] - p->qh[r] * qd) / p->qn;
}

typedef struct { uint32_t k; Pair r; double T; int clamped; int64_t e; /* position in the pixel's candidate list */ } XHit;

/* Reverse sweep of O5 over one pixel's list; every pair's contribution goes through surfel_chain() on its own and is
 * added, times `sign`, to row e of `loc` (19 values: 13 parameters + 6 pose); |contribution| to `absl` if non-NULL. */
static void exposure_sweep(const Ctx* c, const float* scale, const float* opacity, const float* rgb, const XHit* hits,
                           size_t nh, const double* g, double x, double y, double sign, double* loc, double* absl) {
    double suffix = 0.0;
    for (size_t q = nh; q-- > 0;) {
        const XHit* h = hits + q; const uint32_t k = h->k; const Prep* p = c->P + k; const Pair* r = &h->r;
        const double w = r->a * h->T;
        const double gv = g[0] * rgb[3 * k] + g[1] * rgb[3 * k + 1] + g[2] * rgb[3 * k + 2] + g[3] * r->z +
                          g[4] * p->tnc[0] + g[5] * p->tnc[1] + g[6] * p->tnc[2] + g[7];
        const double dz = g[3] * w;
        const double da = h->T * gv - suffix / (1.0 - r->a);
        suffix += w * gv;
        double out[19], lm[9], lnc[3], dG = 0.0;
        out[9] = 0.0;
        if (!h->clamped) { out[9] = da * r->G; dG = da * opacity[k]; }
        for (int ch = 0; ch < 3; ++ch) { out[10 + ch] = g[ch] * w; lnc[ch] = g[4 + ch] * w; }
        if (r->use2d) {   /* R28, screen term (as in orc_backward) */
            const double gxc = 2.0 * r->dx * r->G * dG, gyc = 2.0 * r->dy * r->G * dG, m22 = p->M[8];
            for (int t = 0; t < 9; ++t) lm[t] = 0.0;
            lm[2] = gxc / m22; lm[5] = gyc / m22;
            lm[8] = dz - (gxc * (p->M[2] / m22) + gyc * (p->M[5] / m22)) / m22;
        } else {
        const double du = -r->u * r->G * dG + dz * p->M[6];
        const double dv = -r->v * r->G * dG + dz * p->M[7];
        const double dk[3] = {du / r->k[2], dv / r->k[2], -(r->u * du + r->v * dv) / r->k[2]};
        double dhu[3], dhv[3];
        cross3(r->hv, dk, dhu);
        cross3(dk, r->hu, dhv);
        const double uv1[3] = {r->u, r->v, 1.0};
        for (int t = 0; t < 3; ++t) { lm[t] = dhu[t]; lm[3 + t] = dhv[t]; lm[6 + t] = dz * uv1[t] - x * dhu[t] - y * dhv[t]; }
        }
        surfel_chain(c, k, scale, lm, lnc, out, out + 13);
        for (int t = 0; t < 19; ++t) {
            loc[19 * h->e + t] += sign * out[t];
            if (absl) absl[19 * h->e + t] += fabs(out[t]);
        }
    }
}

/*
 * expo[k][t], pose_expo[t]: what a renderer that decides differently at the EXPOSED pixels can add to / remove from
 * gradient element t of surfel k (pose: of the 6-vector).  Summed over the exposed pixels p:
 *     | c2(p,k) - c1(p,k) |                the pixel's contribution on the list with its fragile decisions inverted (c2)
 *                                          minus the contribution on the oracle's own list (c1): the effect of the flip
 *   + phi_p | c1(p,k) |                    phi_p = min(1, C eps sum_{i composited, kappa_i > KAPPA_MAX} kappa_i (1 + rho_i^2)):
 *                                          first-order effect of the binary32 rounding of an ill-conditioned
 *                                          intersection's inputs (C eps = round_eps, passed in)
 *   + | c1(p,k) |  where extra_mask[p]     the caller's pixels: the whole term may appear or vanish (a loss mask)
 * (pose: the same with the pixel's pairs summed before the | |).
 */
void orc_exposure(int64_t n, const float* mean, const float* scale, const float* quat, const float* opacity,
                  const float* rgb, const uint8_t* active, const double* camv, const double* cfgv,
                  const double* up /* 8*H*W */, const uint8_t* extra_mask /* H*W, nullable */, int signed_all, double round_eps,
                  double* expo /* n*13, zeroed here */, double* pose_expo /* 6 */, uint8_t* pix_exposed /* H*W, nullable */) {
    Ctx c; ctx_init(&c, n, mean, scale, quat, opacity, rgb, active, camv, cfgv, 0);
    const int W = c.cam.W, H = c.cam.H; const int64_t HW = (int64_t)W * H;
    const Cfg* cfg = &c.cfg;
    memset(expo, 0, sizeof(double) * 13 * (size_t)(n > 0 ? n : 0));
    for (int t = 0; t < 6; ++t) pose_expo[t] = 0.0;
#pragma omp parallel
    {
        size_t cap = 256, lcap = 256;
        XHit* l1 = (XHit*)malloc(sizeof(XHit) * cap); XHit* l2 = (XHit*)malloc(sizeof(XHit) * cap);
        double* loc = (double*)malloc(sizeof(double) * 19 * lcap); double* absl = (double*)malloc(sizeof(double) * 19 * lcap);
#pragma omp for schedule(dynamic, 1)
        for (int j = 0; j < H; ++j) {
            for (int i = 0; i < W; ++i) {
                const double x = i + 0.5, y = j + 0.5;
                const int64_t pix = (int64_t)j * W + i;
                double g[8];
                for (int ch = 0; ch < 8; ++ch) g[ch] = up[ch * HW + pix];
                const uint32_t* lst; const int64_t m = cand_count(&c, i, j, &lst);
                /* the oracle's own list (as orc_backward's replay), the pixel's fragile bits, and phi */
                size_t n1 = 0; double T = 1.0, ksum = 0.0; int frag = 0;
                for (int64_t e = 0; e < m; ++e) {
                    const uint32_t k = c.ord[lst[e] & 0x7fffffffu];
                    const Prep* p = c.P + k;
                    if (x < p->aabb[0] - 1.0 || x > p->aabb[1] + 1.0 || y < p->aabb[2] - 1.0 || y > p->aabb[3] + 1.0) continue;
                    Pair r; int covers, f = 0;
                    const int st = eval_pair(p, opacity[k], x, y, T, cfg, &r, &f, &covers);
                    frag |= f;
                    if (st == 2) break;
                    if (st == 0) continue;
                    if (f & 4) ksum += pair_kappa(&r) * (1.0 + r.u * r.u + r.v * r.v);
                    if (n1 == cap) { cap *= 2; l1 = (XHit*)realloc(l1, sizeof(XHit) * cap); l2 = (XHit*)realloc(l2, sizeof(XHit) * cap); }
                    l1[n1].k = k; l1[n1].r = r; l1[n1].T = T; l1[n1].clamped = r.clamped; l1[n1].e = e; ++n1;
                    T *= (1.0 - r.a);
                }
                const int extra = extra_mask && extra_mask[pix];
                const int exposed = frag != 0 || extra;
                if (pix_exposed) pix_exposed[pix] = (uint8_t)exposed;
                if (!exposed && !signed_all) continue;
                if ((size_t)m > lcap) {
                    lcap = (size_t)m * 2;
                    loc = (double*)realloc(loc, sizeof(double) * 19 * lcap); absl = (double*)realloc(absl, sizeof(double) * 19 * lcap);
                }
                memset(loc, 0, sizeof(double) * 19 * (size_t)m); memset(absl, 0, sizeof(double) * 19 * (size_t)m);
                if (signed_all) {   /* self-check mode: orc_backward recomputed pair by pair */
                    exposure_sweep(&c, scale, opacity, rgb, l1, n1, g, x, y, 1.0, loc, NULL);
                    for (size_t q = 0; q < n1; ++q) {
                        for (int t = 0; t < 13; ++t) atomic_add(expo + 13 * (size_t)l1[q].k + t, loc[19 * l1[q].e + t]);
                        for (int t = 0; t < 6; ++t) atomic_add(pose_expo + t, loc[19 * l1[q].e + 13 + t]);
                    }
                    continue;
                }
                exposure_sweep(&c, scale, opacity, rgb, l1, n1, g, x, y, -1.0, loc, absl);
                /* the list with every fragile decision of this pixel inverted */
                size_t n2 = 0; T = 1.0;
                for (int64_t e = 0; e < m; ++e) {
                    const uint32_t k = c.ord[lst[e] & 0x7fffffffu];
                    const Prep* p = c.P + k;
                    if (x < p->aabb[0] - 1.0 || x > p->aabb[1] + 1.0 || y < p->aabb[2] - 1.0 || y > p->aabb[3] + 1.0) continue;
                    Pair r; int covers, f = 0;
                    (void)eval_pair(p, opacity[k], x, y, T, cfg, &r, &f, &covers);   /* fills h_u, h_v, k, u, v */
                    if (!pair_defined(cfg, &r)) continue;
                    if (cfg->lowpass && r.k[2] != 0.0) {   /* R28: which term wins is a decision too */
                        const double r3 = r.u * r.u + r.v * r.v, r2 = 2.0 * (r.dx * r.dx + r.dy * r.dy);
                        if (isfinite(r3) && fabs(r3 - r2) < FRAG_EPS * r2) r.use2d = !r.use2d;
                    }
                    const double rho2 = pair_rho2(cfg, &r);
                    pair_complete(p, opacity[k], cfg, &r);
                    const double c2 = cfg->cutoff * cfg->cutoff, og = opacity[k] * r.G;
                    int in = (rho2 <= c2) ^ (isfinite(c2) && fabs(rho2 - c2) < FRAG_EPS * c2);
                    in = in && ((r.z > cfg->z_near) ^ (cfg->z_near > 0.0 && fabs(r.z - cfg->z_near) < FRAG_EPS * cfg->z_near));
                    in = in && ((r.a >= cfg->alpha_min) ^ (cfg->alpha_min > 0.0 && fabs(r.a - cfg->alpha_min) < FRAG_EPS * cfg->alpha_min));
                    if (!in) continue;
                    const double Tn = T * (1.0 - r.a);
                    const int stop = (Tn < cfg->t_min) ^ (cfg->t_min > 0.0 && fabs(Tn - cfg->t_min) < FRAG_EPS * cfg->t_min);
                    if (stop) break;
                    if (n2 == cap) { cap *= 2; l1 = (XHit*)realloc(l1, sizeof(XHit) * cap); l2 = (XHit*)realloc(l2, sizeof(XHit) * cap); }
                    l2[n2].k = k; l2[n2].r = r; l2[n2].T = T; l2[n2].e = e;
                    l2[n2].clamped = r.clamped ^ (fabs(og - cfg->alpha_max) < FRAG_EPS * cfg->alpha_max);
                    ++n2;
                    T = Tn;
                }
                exposure_sweep(&c, scale, opacity, rgb, l2, n2, g, x, y, 1.0, loc, NULL);
                double phi = round_eps * ksum + (extra ? 1.0 : 0.0);
                if (phi > 1.0) phi = 1.0;
                double pd[6] = {0, 0, 0, 0, 0, 0}, pa[6] = {0, 0, 0, 0, 0, 0}, p1[6] = {0, 0, 0, 0, 0, 0};
                for (int64_t e = 0; e < m; ++e) {   /* rows touched by either list */
                    const double* le = loc + 19 * e; const double* ae = absl + 19 * e;
                    int any = 0;
                    for (int t = 0; t < 19 && !any; ++t) any = le[t] != 0.0 || ae[t] != 0.0;
                    if (!any) continue;
                    const uint32_t k = c.ord[lst[e] & 0x7fffffffu];
                    for (int t = 0; t < 13; ++t) atomic_add(expo + 13 * (size_t)k + t, fabs(le[t]) + phi * ae[t]);
                    for (int t = 0; t < 6; ++t) { pd[t] += le[13 + t]; pa[t] += ae[13 + t]; }
                }
                /* the oracle's own signed pose contribution of this pixel (for a mask that may flip) */
                if (extra) {
                    memset(loc, 0, sizeof(double) * 19 * (size_t)m);
                    exposure_sweep(&c, scale, opacity, rgb, l1, n1, g, x, y, 1.0, loc, NULL);
                    for (size_t q = 0; q < n1; ++q) for (int t = 0; t < 6; ++t) p1[t] += loc[19 * l1[q].e + 13 + t];
                }
                const double phk = round_eps * ksum > 1.0 ? 1.0 : round_eps * ksum;
                for (int t = 0; t < 6; ++t) atomic_add(pose_expo + t, fabs(pd[t]) + phk * pa[t] + fabs(p1[t]));
            }
        }
        free(l1); free(l2); free(loc); free(absl);
    }
    ctx_free(&c);
}

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
