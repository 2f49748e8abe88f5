// pair.cuh -- one (pixel, surfel) pair, shared by the forward and backward compositing kernels so
// that both take bit-identical decisions (explicit _rn intrinsics pin the instruction sequence).
//
// Ray-splat intersection (Eq. 4) in the screen-centred adjugate form:
// with the tile-relative staged coefficients
//   un = U0 + lx P + ly Q,  vn = V0 + lx R + ly S,  dn = D0 + lx E' + ly F'
//   (u, v) = (un, vn) / dn,   z = a u + b v + c
// which is algebraically (u,v,1) ~ (M0 - x M2) x (M1 - y M2) with the pixel-independent factors of
// the cross product hoisted per surfel and the pixel coordinate taken relative to the surfel's
// projected centre, the well-conditioned choice in fp32.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

// Staged per-(tile, entry) record in shared memory: 5 x float4, read as warp-wide broadcasts.
struct StagedFwd {
    float4 s0;  // P, Q, U0, E'
    float4 s1;  // R, S, V0, F'
    float4 s2;  // D0, a, b, c
    float4 s3;  // opacity, r, g, b
    float4 s4;  // nx, ny, nz, unused
};

// Shared-memory access by 32-bit shared-window address (computed once per kernel): keeps the
// address arithmetic of the inner loops to one multiply-add.
__device__ __forceinline__ uint32_t smem_addr(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ float4 lds128(uint32_t addr) {
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ float lds32(uint32_t addr) {
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ uint32_t lds_u8(uint32_t addr) {
    uint32_t v;
    asm volatile("ld.shared.u8 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
    return v;
}

struct PairResult {
    float u, v, z, G, a;
};

__device__ __forceinline__ float fast_rcp(float x) {
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ float fast_ex2(float x) {
    float r;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

// Returns true when the pair passes the geometric tests (rho^2 <= c^2, finite, z > z_near) and
// a >= alpha_min.  The saturation stop is the caller's (it needs T).
__device__ __forceinline__ bool eval_pair(const float4 s0, const float4 s1, const float4 s2, const float opacity,
                                          const float lx, const float ly, const float cutoff2, const float alpha_min,
                                          const float alpha_max, const float z_near, PairResult& r) {
    const float un = __fmaf_rn(ly, s0.y, __fmaf_rn(lx, s0.x, s0.z));
    const float vn = __fmaf_rn(ly, s1.y, __fmaf_rn(lx, s1.x, s1.z));
    const float dn = __fmaf_rn(ly, s1.w, __fmaf_rn(lx, s0.w, s2.x));
    const float inv = fast_rcp(dn);
    r.u = __fmul_rn(un, inv);
    r.v = __fmul_rn(vn, inv);
    const float rho2 = __fmaf_rn(r.v, r.v, __fmul_rn(r.u, r.u));
    if (!(rho2 <= cutoff2)) return false;  // also rejects NaN/inf (dn == 0)
    r.z = __fmaf_rn(s2.z, r.v, __fmaf_rn(s2.y, r.u, s2.w));
    if (!(r.z > z_near)) return false;
    r.G = fast_ex2(__fmul_rn(rho2, -0.72134752044448170368f));  // exp(-rho2/2) = 2^(-rho2 / (2 ln 2))
    r.a = fminf(alpha_max, __fmul_rn(opacity, r.G));
    return r.a >= alpha_min;
}

// 8-bit mask of the warps (8x4 pixel patches, warp w at x0 = (w&1)*8, y0 = (w>>1)*4 inside the tile)
// whose pixel CENTRES the surfel's screen AABB can reach.  Pixels outside the AABB have rho^2 > c^2,
// so a warp whose bit is clear would reject the entry at every lane: it skips it without testing.
__device__ __forceinline__ unsigned warp_patch_mask(const float4 bb, const float tile_x0, const float tile_y0) {
    unsigned m = 0;
#pragma unroll
    for (int w = 0; w < 8; ++w) {
        const float xl = tile_x0 + (float)((w & 1) * 8) + 0.5f, yl = tile_y0 + (float)((w >> 1) * 4) + 0.5f;
        const bool hit = bb.y >= xl && bb.x <= xl + 7.f && bb.w >= yl && bb.z <= yl + 3.f;
        m |= hit ? (1u << w) : 0u;
    }
    return m;
}

// Second, exact stage of the warp-patch mask.  With the staged rows a = (P, Q, U0), b = (R, S, V0), c = (E', F', D0)
// and p = (lx, ly, 1), rho^2 = ((a.p)^2 + (b.p)^2) / (c.p)^2, so rho^2 <= k2 is the conic
//   q(x, y) = (a.p)^2 + (b.p)^2 - k2 (c.p)^2 = A x^2 + 2 B x y + C y^2 + 2 D x + 2 E y + F <= 0.
// k2 = min(cutoff^2, 2 ln(opacity / alpha_min)) also folds the alpha >= alpha_min test in (eval_pair).  Where q is
// convex (the splat's footprint is an ellipse) its minimum over a patch's rectangle of pixel centres, grown by a
// quarter pixel against rounding, is attained at the centre clamped onto the rectangle along one axis and
// minimised along the other; a patch whose minimum is positive holds no pixel that eval_pair() accepts and loses its
// bit.  Non-convex or badly conditioned conics (horizon through the tile, edge-on splats) keep the AABB answer.
// Measured need: in C3 two of three (warp, entry) trips that passed the AABB mask found no lane that hits.
__device__ __forceinline__ unsigned refine_patch_mask(const unsigned m, const float4 s0, const float4 s1, const float4 s2,
                                                      const float opacity, const float cutoff2, const float alpha_min) {
    const float ratio = opacity / alpha_min;
    if (!(ratio >= 1.f)) return 0u;  // alpha < alpha_min everywhere (also NaN opacity)
    const float k2 = fminf(cutoff2, fmaf(2.002f, __logf(ratio), 1e-3f));
    const float a1 = s0.x, a2 = s0.y, a3 = s0.z, b1 = s1.x, b2 = s1.y, b3 = s1.z, c1 = s0.w, c2 = s1.w, c3 = s2.x;
    const float kc1 = k2 * c1, kc2 = k2 * c2, kc3 = k2 * c3;
    const float A = fmaf(a1, a1, fmaf(b1, b1, -kc1 * c1)), B = fmaf(a1, a2, fmaf(b1, b2, -kc1 * c2));
    const float C = fmaf(a2, a2, fmaf(b2, b2, -kc2 * c2)), D = fmaf(a1, a3, fmaf(b1, b3, -kc1 * c3));
    const float E = fmaf(a2, a3, fmaf(b2, b3, -kc2 * c3)), F = fmaf(a3, a3, fmaf(b3, b3, -kc3 * c3));
    const float det = fmaf(A, C, -B * B);
    if (!(A > 0.f && C > 0.f && det > 1e-4f * A * C)) return m;
    const float idet = 1.f / det, nia = -1.f / A, nic = -1.f / C;
    const float xc = (B * E - C * D) * idet, yc = (B * D - A * E) * idet;
    const float B2 = B + B, D2 = D + D, E2 = E + E;
    // rounding allowance: 32 ulp of the largest term q can hold inside the tile (|x|, |y| <= 16)
    const float tol = 4e-6f * (fabsf(F) + 32.f * (fabsf(D) + fabsf(E)) + 256.f * (A + C + fabsf(B2)));
    unsigned out = 0;
#pragma unroll
    for (int w = 0; w < 8; ++w) {
        const float x0 = (float)((w & 1) * 8) - 0.25f, x1 = x0 + 7.5f, y0 = (float)((w >> 1) * 4) - 0.25f, y1 = y0 + 3.5f;
        const float X = fminf(fmaxf(xc, x0), x1), Y = fminf(fmaxf(yc, y0), y1);
        const float ys = fminf(fmaxf(fmaf(B, X, E) * nic, y0), y1);   // argmin over y of q(X, y), clamped
        const float xs = fminf(fmaxf(fmaf(B, Y, D) * nia, x0), x1);   // argmin over x of q(x, Y), clamped
        const float q1 = fmaf(X, fmaf(A, X, fmaf(B2, ys, D2)), fmaf(ys, fmaf(C, ys, E2), F));
        const float q2 = fmaf(xs, fmaf(A, xs, fmaf(B2, Y, D2)), fmaf(Y, fmaf(C, Y, E2), F));
        out |= (fminf(q1, q2) <= tol) ? (1u << w) : 0u;
    }
    return m & out;
}

// Builds the staged record of entry `v` for the tile whose first pixel centre is (px0, py0).
__device__ __forceinline__ void stage_entry(const float4 g0, const float4 g1, const double2 g2, const float4 g3,
                                            const double px0, const double py0, float4& s0, float4& s1, float4& s2,
                                            float* xy0 = nullptr) {
    const float X0 = (float)(px0 - g2.x), Y0 = (float)(py0 - g2.y);  // xt, yt of the tile's first pixel
    if (xy0) { xy0[0] = X0; xy0[1] = Y0; }   // (SGS_FLAG_LOWPASS: pixel - projected centre = (lx + X0, ly + Y0))
    const float P = g0.x, Q = g0.y, R = g0.z, S = g0.w, D = g1.x, E = g1.y, F = g1.z;
    s0 = make_float4(P, Q, __fmaf_rn(Y0, Q, __fmul_rn(X0, P)), -E);
    s1 = make_float4(R, S, __fmaf_rn(Y0, S, __fmul_rn(X0, R)), -F);
    s2 = make_float4(__fmaf_rn(-Y0, F, __fmaf_rn(-X0, E, D)), g3.x, g3.y, g3.z);
}
