// ssim.cu -- the SSIM term of the mapping loss (Eq. 24; reading R24 in
// DESIGN.md): per channel the structural similarity index of [87] with the 11 x 11 Gaussian window (sigma 1.5),
// zero padding, C1 = 0.01^2, C2 = 0.03^2;  L = weight / (3 |Omega|) sum_c sum_p (1 - SSIM_c(p)).
//
// Two kernels of the same shape.  A block of 64 threads owns a strip 64 pixels wide and `rows` pixels tall of one
// channel and marches down it one input row at a time: the row (64 + 10 halo pixels, zero outside the image) is
// staged in shared memory by `cp.async`, three rows ahead; every thread takes the 11
// taps ACROSS for its column from shared memory, and the 11 taps DOWN never leave registers: each finished row is
// scattered with the window's weights into the 11 pending output rows' accumulators (a ring indexed statically by
// unrolling the march 11-fold), and the row that has just received its last tap is emitted.
//   k_ssim_forward : window sums of x, y, x^2, y^2, xy -> SSIM -> loss; writes the three derivative maps
//                    G dS/dmu1, G dS/de11, G dS/de12  (G = dL/dSSIM = -weight / (3 |Omega|))
//   k_ssim_backward: the same window over the three maps;  dL/dx = conv(m0) + 2 x conv(m1) + y conv(m2)  is ADDED to
//                    the caller's upstream colour gradient (the window is symmetric: correlation = convolution).
// The first version (16 x 16 output tiles, 26 x 26 inputs, both passes through shared memory) spent 99 shared-memory
// accesses per output pixel and channel and ran 52 + 46 us at 1200 x 680; this one spends 12, and its arithmetic is
// packed two binary32 lanes per instruction (FFMA2 / FMUL2 / FADD2: same flops per clock, half the issue slots).
#include "sgs_internal.h"

namespace {

constexpr int SB_W = 64, SS_R = 5, SS_TAPS = 2 * SS_R + 1, SB_IN = SB_W + 2 * SS_R, SB_ST = 4;  // 4 staged rows in flight
__constant__ float c_win[SS_TAPS];

// 4-byte asynchronous global -> shared copy; `valid == false` writes a zero (the zero padding) without touching src
__device__ __forceinline__ void cp_async4(void* dst, const float* src, bool valid) {
    const uint32_t d = (uint32_t)__cvta_generic_to_shared(dst);
    const int sz = valid ? 4 : 0;
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4, %2;" ::"r"(d), "l"(src), "r"(sz) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait2() { asm volatile("cp.async.wait_group 2;" ::: "memory"); }

__global__ void __launch_bounds__(SB_W)
k_ssim_forward(const float* __restrict__ xr, const float* __restrict__ yt, int W, int H, int rows, float G, float lscale,
               float* __restrict__ maps /* 3 channels x 3 maps x HW */, float* __restrict__ slots /* 64 partial sums */) {
    __shared__ float2 sxy[SB_ST][SB_IN + 2];  // (x, y) interleaved: one LDS.64 per tap feeds the packed FMAs
    __shared__ float s_part[SB_W / 32];
    const int c = blockIdx.z, tx = threadIdx.x;
    const size_t HW = (size_t)W * H;
    const float* x = xr + (size_t)c * HW;
    const float* y = yt + (size_t)c * HW;
    float* m = maps + (size_t)c * 3 * HW;
    const int px = blockIdx.x * SB_W + tx, yb = blockIdx.y * rows, gx0 = blockIdx.x * SB_W - SS_R;
    const int nrow = min(rows, H - yb), nin = nrow + 2 * SS_R;
    const int gxa = gx0 + tx, gxb = gx0 + SB_W + tx;               // this thread's one or two columns of a staged row
    const bool ina = gxa >= 0 && gxa < W, inb = gxb < W;
    // running source pointers of this thread's column(s): one row further per issue_row() call
    int gy_n = yb - SS_R;
    const float* xa = x + (ptrdiff_t)gy_n * W + gxa;
    const float* ya = y + (ptrdiff_t)gy_n * W + gxa;
    auto issue_row = [&](int j) {  // input row j of the strip -> stage j % 4
        if (j < nin) {
            const bool rin = (unsigned)gy_n < (unsigned)H;
            float2* d = sxy[j & (SB_ST - 1)];
            cp_async4(&d[tx].x, (rin && ina) ? xa : x, rin && ina);
            cp_async4(&d[tx].y, (rin && ina) ? ya : y, rin && ina);
            if (tx < 2 * SS_R) {
                cp_async4(&d[SB_W + tx].x, (rin && inb) ? xa + SB_W : x, rin && inb);
                cp_async4(&d[SB_W + tx].y, (rin && inb) ? ya + SB_W : y, rin && inb);
            }
        }
        cp_async_commit();
        ++gy_n; xa += W; ya += W;
    };
    issue_row(0); issue_row(1); issue_row(2);
    float2 w2[SS_TAPS];
#pragma unroll
    for (int t = 0; t < SS_TAPS; ++t) w2[t] = make_float2(c_win[t], c_win[t]);
    float2 A01[SS_TAPS], A23[SS_TAPS];
    float A4[SS_TAPS];
#pragma unroll
    for (int k = 0; k < SS_TAPS; ++k) { A01[k] = make_float2(0.f, 0.f); A23[k] = make_float2(0.f, 0.f); A4[k] = 0.f; }
    float lsum = 0.f;
    for (int j0 = 0; j0 < nin; j0 += SS_TAPS) {
#pragma unroll
        for (int s = 0; s < SS_TAPS; ++s) {
            const int j = j0 + s;
            if (j < nin) {  // block-uniform
                cp_async_wait2();   // row j has landed (rows j+1, j+2 may still be in flight)
                __syncthreads();    // ... for every thread; and stage (j+3) % 4, read at step j-1, is free again
                issue_row(j + 3);
                const int gy = yb - SS_R + j;
                if (gy >= 0 && gy < H) {  // rows outside the image are zero padding: nothing to add
                    const float2* row = sxy[j & (SB_ST - 1)] + tx;
                    float2 h01 = make_float2(0.f, 0.f), h23 = make_float2(0.f, 0.f);
                    float h4 = 0.f;
#pragma unroll
                    for (int t = 0; t < SS_TAPS; ++t) {  // 11 taps across: sums of x, y | x^2, y^2 | xy
                        const float2 ab = row[t];
                        const float2 wab = __fmul2_rn(w2[t], ab);
                        h01 = __fadd2_rn(h01, wab);
                        h23 = __ffma2_rn(wab, ab, h23);
                        h4 = fmaf(wab.x, ab.y, h4);
                    }
#pragma unroll
                    for (int t = 1; t < SS_TAPS; ++t) {  // 11 taps down: this row is tap t of output row j - t
                        const int k = (s - t + SS_TAPS) % SS_TAPS;
                        A01[k] = __ffma2_rn(w2[t], h01, A01[k]);
                        A23[k] = __ffma2_rn(w2[t], h23, A23[k]);
                        A4[k] = fmaf(w2[t].x, h4, A4[k]);
                    }
                    // tap 0 opens output row j in the slot that row j - 11 left at the previous step
                    A01[s] = __fmul2_rn(w2[0], h01); A23[s] = __fmul2_rn(w2[0], h23); A4[s] = w2[0].x * h4;
                } else {
                    A01[s] = make_float2(0.f, 0.f); A23[s] = make_float2(0.f, 0.f); A4[s] = 0.f;
                }
                {   // output row j - 10 has all its taps
                    const int k = (s + 1) % SS_TAPS, o = j - 2 * SS_R;
                    if (o >= 0 && px < W) {
                        const float mu1 = A01[k].x, mu2 = A01[k].y, e11 = A23[k].x, e22 = A23[k].y, e12 = A4[k];
                        const float C1 = 1e-4f, C2 = 9e-4f;
                        const float s1 = e11 - mu1 * mu1, s2 = e22 - mu2 * mu2, s12 = e12 - mu1 * mu2;
                        const float a1 = 2.f * mu1 * mu2 + C1, a2 = 2.f * s12 + C2, b1 = mu1 * mu1 + mu2 * mu2 + C1, b2 = s1 + s2 + C2;
                        const float ib = 1.f / (b1 * b2);  // b1, b2 > 0; 1/b1 = b2 ib and 1/b2 = b1 ib below
                        const float S = a1 * a2 * ib;
                        lsum += 1.f - S;
                        float* mo = m + (size_t)(yb + o) * W + px;
                        mo[0] = G * (2.f * ib * (mu2 * (a2 - a1) - S * mu1 * (b2 - b1)));  // G dS/dmu1
                        mo[HW] = -G * S * b1 * ib;                                           // G dS/de11 = -G S / b2
                        mo[2 * HW] = G * (2.f * a1 * ib);                                    // G dS/de12
                    }
                }
            }
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) lsum += __shfl_xor_sync(0xffffffffu, lsum, o);
    if ((tx & 31) == 0) s_part[tx >> 5] = lsum;
    __syncthreads();
    if (tx == 0) {  // 64 slots instead of one address: a thousand blocks would serialise on a single atomic
        float t = 0.f;
#pragma unroll
        for (int w = 0; w < SB_W / 32; ++w) t += s_part[w];
        atomicAdd(slots + ((blockIdx.x + 7 * blockIdx.y + 13 * blockIdx.z) & 63), t * lscale);
    }
}

__global__ void __launch_bounds__(SB_W)
k_ssim_backward(const float* __restrict__ xr, const float* __restrict__ yt, int W, int H, int rows,
                const float* __restrict__ maps, float* __restrict__ up_rgb, float* __restrict__ slots, float* __restrict__ loss) {
    __shared__ float2 s01[SB_ST][SB_IN + 2];  // maps 0 and 1 interleaved
    __shared__ float s2[SB_ST][SB_IN + 2];
    const int c = blockIdx.z, tx = threadIdx.x;
    if (blockIdx.x == 0 && blockIdx.y == 0 && blockIdx.z == 0 && tx < 32) {  // the forward's loss: 64 slots -> *loss, slots re-zeroed
        float t = slots[tx] + slots[tx + 32];
        slots[tx] = 0.f; slots[tx + 32] = 0.f;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
        if (tx == 0 && loss) atomicAdd(loss, t);
    }
    const size_t HW = (size_t)W * H;
    const float* m = maps + (size_t)c * 3 * HW;
    const int px = blockIdx.x * SB_W + tx, yb = blockIdx.y * rows, gx0 = blockIdx.x * SB_W - SS_R;
    const int nrow = min(rows, H - yb), nin = nrow + 2 * SS_R;
    const int gxa = gx0 + tx, gxb = gx0 + SB_W + tx;
    const bool ina = gxa >= 0 && gxa < W, inb = gxb < W;
    int gy_n = yb - SS_R;
    const float* ma = m + (ptrdiff_t)gy_n * W + gxa;
    auto issue_row = [&](int j) {
        if (j < nin) {
            const bool rin = (unsigned)gy_n < (unsigned)H;
            const int st = j & (SB_ST - 1);
            const float* pa = (rin && ina) ? ma : m;
            cp_async4(&s01[st][tx].x, pa, rin && ina);
            cp_async4(&s01[st][tx].y, pa + HW, rin && ina);
            cp_async4(&s2[st][tx], pa + 2 * HW, rin && ina);
            if (tx < 2 * SS_R) {
                const float* pb = (rin && inb) ? ma + SB_W : m;
                cp_async4(&s01[st][SB_W + tx].x, pb, rin && inb);
                cp_async4(&s01[st][SB_W + tx].y, pb + HW, rin && inb);
                cp_async4(&s2[st][SB_W + tx], pb + 2 * HW, rin && inb);
            }
        }
        cp_async_commit();
        ++gy_n; ma += W;
    };
    issue_row(0); issue_row(1); issue_row(2);
    float2 w2[SS_TAPS];
#pragma unroll
    for (int t = 0; t < SS_TAPS; ++t) w2[t] = make_float2(c_win[t], c_win[t]);
    float2 A01[SS_TAPS];
    float A2[SS_TAPS];
#pragma unroll
    for (int k = 0; k < SS_TAPS; ++k) { A01[k] = make_float2(0.f, 0.f); A2[k] = 0.f; }
    for (int j0 = 0; j0 < nin; j0 += SS_TAPS) {
#pragma unroll
        for (int s = 0; s < SS_TAPS; ++s) {
            const int j = j0 + s;
            if (j < nin) {
                cp_async_wait2();
                __syncthreads();
                issue_row(j + 3);
                // the output row that completes at this step: its pixel values are needed for the final combination
                const int k = (s + 1) % SS_TAPS, o = j - 2 * SS_R;
                const bool emit = o >= 0 && px < W;
                const size_t pix = emit ? (size_t)c * HW + (size_t)(yb + o) * W + px : 0;
                float xv = 0.f, yv = 0.f, uv = 0.f;
                if (emit) { xv = xr[pix]; yv = yt[pix]; uv = up_rgb[pix]; }
                const int gy = yb - SS_R + j;
                if (gy >= 0 && gy < H) {
                    const int st = j & (SB_ST - 1);
                    const float2* r01 = s01[st] + tx;
                    const float* r2 = s2[st] + tx;
                    float2 h01 = make_float2(0.f, 0.f);
                    float h2 = 0.f;
#pragma unroll
                    for (int t = 0; t < SS_TAPS; ++t) {
                        h01 = __ffma2_rn(w2[t], r01[t], h01);
                        h2 = fmaf(w2[t].x, r2[t], h2);
                    }
#pragma unroll
                    for (int t = 1; t < SS_TAPS; ++t) {
                        const int kk = (s - t + SS_TAPS) % SS_TAPS;
                        A01[kk] = __ffma2_rn(w2[t], h01, A01[kk]);
                        A2[kk] = fmaf(w2[t].x, h2, A2[kk]);
                    }
                    A01[s] = __fmul2_rn(w2[0], h01); A2[s] = w2[0].x * h2;  // tap 0 opens output row j in the freed slot
                } else {
                    A01[s] = make_float2(0.f, 0.f); A2[s] = 0.f;
                }
                if (emit) up_rgb[pix] = uv + (A01[k].x + 2.f * xv * A01[k].y + yv * A2[k]);
            }
        }
    }
}

}  // namespace

cudaError_t sgs_launch_ssim_loss(sgs_ctx* c, int W, int H, const float* rgb_r, const float* rgb_t, float weight,
                                 float* up_rgb, float* loss, cudaStream_t s) {
    static bool win_set = false;
    if (!win_set) {  // normalised Gaussian, sigma 1.5, evaluated in double and rounded once (as the oracle's)
        double g[2 * SS_R + 1], sum = 0.0;
        for (int t = 0; t <= 2 * SS_R; ++t) { const double d = t - SS_R; g[t] = exp(-d * d / (2.0 * 1.5 * 1.5)); sum += g[t]; }
        float gf[SS_TAPS];
        for (int t = 0; t <= 2 * SS_R; ++t) gf[t] = (float)(g[t] / sum);
        const cudaError_t e = cudaMemcpyToSymbol(c_win, gf, sizeof(gf));
        if (e != cudaSuccess) return e;
        win_set = true;
    }
    const int64_t HW = (int64_t)W * H;
    if (HW * 9 > c->ssim_cap) {  // 9 derivative planes + 64 loss slots (kept zero between calls)
        if (c->ssim_maps) sgs_ws_free(c, c->ssim_maps, s);
        c->ssim_maps = (float*)sgs_ws_alloc(c, sizeof(float) * (9 * (size_t)HW + 64), s);
        if (!c->ssim_maps) { c->ssim_cap = 0; return cudaErrorMemoryAllocation; }
        c->ssim_cap = HW * 9;
        const cudaError_t e = cudaMemsetAsync(c->ssim_maps + 9 * (size_t)HW, 0, 64 * sizeof(float), s);
        if (e != cudaSuccess) return e;
    }
    float* slots = c->ssim_maps + c->ssim_cap;
    SgsStage st(c, SGS_STAGE_LOSS, s);
    c->launches += 2;
    // strip height: 10 halo rows are re-convolved per strip, so tall strips waste less, but the grid should still
    // hold a few blocks per SM (2 warps each)
    int rows = 68;
    while (rows > 17 && (int64_t)((W + SB_W - 1) / SB_W) * ((H + rows - 1) / rows) * 3 < 148 * 6) rows = (rows + 1) / 2;
    const dim3 grid((W + SB_W - 1) / SB_W, (H + rows - 1) / rows, 3);
    const float inv = 1.f / (3.f * (float)HW);
    k_ssim_forward<<<grid, SB_W, 0, s>>>(rgb_r, rgb_t, W, H, rows, -weight * inv, weight * inv, c->ssim_maps, slots);
    k_ssim_backward<<<grid, SB_W, 0, s>>>(rgb_r, rgb_t, W, H, rows, c->ssim_maps, up_rgb, slots, loss);
    return cudaGetLastError();
}
