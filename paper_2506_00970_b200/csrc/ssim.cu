// ssim.cu -- the SSIM term of the mapping loss (Eq. 24; reading R24 in
// DESIGN.md): per channel the structural similarity index of [87] with the 11 x 11 Gaussian window (sigma 1.5),
// zero padding, C1 = 0.01^2, C2 = 0.03^2;  L = weight / (3 |Omega|) sum_c sum_p (1 - SSIM_c(p)).
//
// Two kernels, one block per 16 x 16 output tile and channel, the 26 x 26 input tile (halo 5) staged in shared memory
// and convolved separably there (11 taps across, then 11 taps down), so every input pixel crosses HBM once:
//   k_ssim_forward : window sums of x, y, x^2, y^2, xy -> SSIM -> loss; writes the three derivative maps
//                    G dS/dmu1, G dS/de11, G dS/de12  (G = dL/dSSIM = -weight / (3 |Omega|))
//   k_ssim_backward: the same window over the three maps;  dL/dx = conv(m0) + 2 x conv(m1) + y conv(m2)  is ADDED to
//                    the caller's upstream colour gradient (the window is symmetric: correlation = convolution).
#include "sgs_internal.h"

namespace {

constexpr int SS_T = 16, SS_R = 5, SS_IN = SS_T + 2 * SS_R;  // 16 x 16 outputs, 26 x 26 inputs
// Row strides chosen against bank conflicts: a warp works on two consecutive tile rows x 16 columns, so a stride of
// 16 (mod 32) words puts its 32 accesses on 32 banks (ncu before: half of all shared-memory wavefronts were conflicts).
constexpr int SS_IS = 48, SS_HS = 16;
__constant__ float c_win[2 * SS_R + 1];

__global__ void __launch_bounds__(SS_T * SS_T)
k_ssim_forward(const float* __restrict__ xr, const float* __restrict__ yt, int W, int H, float G, float lscale,
               float* __restrict__ maps /* 3 channels x 3 maps x HW */, float* __restrict__ slots /* 64 partial sums */) {
    __shared__ float sx[SS_IN][SS_IS], sy[SS_IN][SS_IS];
    __shared__ float hs[5][SS_IN][SS_HS];
    __shared__ float s_part[8];
    const int c = blockIdx.z, tid = threadIdx.x;
    const size_t HW = (size_t)W * H;
    const float* x = xr + (size_t)c * HW;
    const float* y = yt + (size_t)c * HW;
    const int x0 = blockIdx.x * SS_T - SS_R, y0 = blockIdx.y * SS_T - SS_R;
    {   // 26 x 26 inputs by 16 x 16 threads: up to four (row, column) positions each, no division
        const int tx = tid & 15, tyy = tid >> 4;
#pragma unroll
        for (int j = 0; j < 2; ++j)
#pragma unroll
            for (int i = 0; i < 2; ++i) {
                const int r = tyy + 16 * j, q = tx + 16 * i;
                if (r < SS_IN && q < SS_IN) {
                    const int gx = x0 + q, gy = y0 + r;
                    const bool in = gx >= 0 && gx < W && gy >= 0 && gy < H;
                    sx[r][q] = in ? x[(size_t)gy * W + gx] : 0.f;
                    sy[r][q] = in ? y[(size_t)gy * W + gx] : 0.f;
                }
            }
    }
    __syncthreads();
    for (int k = tid; k < SS_IN * SS_T; k += SS_T * SS_T) {  // 11 taps across
        const int r = k / SS_T, q = k % SS_T;
        float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f, a4 = 0.f;
#pragma unroll
        for (int t = 0; t <= 2 * SS_R; ++t) {
            const float w = c_win[t], a = sx[r][q + t], b = sy[r][q + t];
            a0 = fmaf(w, a, a0); a1 = fmaf(w, b, a1); a2 = fmaf(w * a, a, a2); a3 = fmaf(w * b, b, a3); a4 = fmaf(w * a, b, a4);
        }
        hs[0][r][q] = a0; hs[1][r][q] = a1; hs[2][r][q] = a2; hs[3][r][q] = a3; hs[4][r][q] = a4;
    }
    __syncthreads();
    const int lx = tid % SS_T, ly = tid / SS_T, px = blockIdx.x * SS_T + lx, py = blockIdx.y * SS_T + ly;
    float one_minus = 0.f;
    if (px < W && py < H) {
        float mu1 = 0.f, mu2 = 0.f, e11 = 0.f, e22 = 0.f, e12 = 0.f;
#pragma unroll
        for (int t = 0; t <= 2 * SS_R; ++t) {  // 11 taps down
            const float w = c_win[t];
            mu1 = fmaf(w, hs[0][ly + t][lx], mu1); mu2 = fmaf(w, hs[1][ly + t][lx], mu2);
            e11 = fmaf(w, hs[2][ly + t][lx], e11); e22 = fmaf(w, hs[3][ly + t][lx], e22); e12 = fmaf(w, hs[4][ly + t][lx], e12);
        }
        const float C1 = 1e-4f, C2 = 9e-4f;
        const float s1 = e11 - mu1 * mu1, s2 = e22 - mu2 * mu2, s12 = e12 - mu1 * mu2;
        const float a1 = 2.f * mu1 * mu2 + C1, a2 = 2.f * s12 + C2, b1 = mu1 * mu1 + mu2 * mu2 + C1, b2 = s1 + s2 + C2;
        const float ib = 1.f / (b1 * b2);
        const float S = a1 * a2 * ib;
        one_minus = 1.f - S;
        const size_t pix = (size_t)py * W + px;
        float* m = maps + (size_t)c * 3 * HW;
        m[pix] = G * (2.f * mu2 * (a2 - a1) * ib - S * (2.f * mu1 / b1 - 2.f * mu1 / b2));  // G dS/dmu1
        m[HW + pix] = G * (-S / b2);                                                          // G dS/de11
        m[2 * HW + pix] = G * (2.f * a1 * ib);                                                // G dS/de12
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) one_minus += __shfl_xor_sync(0xffffffffu, one_minus, o);
    if ((tid & 31) == 0) s_part[tid >> 5] = one_minus;
    __syncthreads();
    if (tid == 0) {  // 64 slots instead of one address: ~10 k blocks would serialise on a single atomic
        float t = 0.f;
        for (int w = 0; w < 8; ++w) t += s_part[w];
        atomicAdd(slots + ((blockIdx.x + 7 * blockIdx.y + 13 * blockIdx.z) & 63), t * lscale);
    }
}

__global__ void __launch_bounds__(SS_T * SS_T)
k_ssim_backward(const float* __restrict__ xr, const float* __restrict__ yt, int W, int H, const float* __restrict__ maps,
                float* __restrict__ up_rgb, float* __restrict__ slots, float* __restrict__ loss) {
    __shared__ float sm[3][SS_IN][SS_IS];
    __shared__ float hs[3][SS_IN][SS_HS];
    const int c = blockIdx.z, tid = threadIdx.x;
    if (blockIdx.x == 0 && blockIdx.y == 0 && blockIdx.z == 0 && tid < 32) {  // the forward's loss: 64 slots -> *loss, slots re-zeroed
        float t = slots[tid] + slots[tid + 32];
        slots[tid] = 0.f; slots[tid + 32] = 0.f;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
        if (tid == 0 && loss) atomicAdd(loss, t);
    }
    const size_t HW = (size_t)W * H;
    const float* m = maps + (size_t)c * 3 * HW;
    const int x0 = blockIdx.x * SS_T - SS_R, y0 = blockIdx.y * SS_T - SS_R;
    {
        const int tx = tid & 15, tyy = tid >> 4;
#pragma unroll
        for (int j = 0; j < 2; ++j)
#pragma unroll
            for (int i = 0; i < 2; ++i) {
                const int r = tyy + 16 * j, q = tx + 16 * i;
                if (r < SS_IN && q < SS_IN) {
                    const int gx = x0 + q, gy = y0 + r;
                    const bool in = gx >= 0 && gx < W && gy >= 0 && gy < H;
                    const size_t p = (size_t)gy * W + gx;
                    sm[0][r][q] = in ? m[p] : 0.f; sm[1][r][q] = in ? m[HW + p] : 0.f; sm[2][r][q] = in ? m[2 * HW + p] : 0.f;
                }
            }
    }
    __syncthreads();
    for (int k = tid; k < SS_IN * SS_T; k += SS_T * SS_T) {
        const int r = k / SS_T, q = k % SS_T;
        float a0 = 0.f, a1 = 0.f, a2 = 0.f;
#pragma unroll
        for (int t = 0; t <= 2 * SS_R; ++t) {
            const float w = c_win[t];
            a0 = fmaf(w, sm[0][r][q + t], a0); a1 = fmaf(w, sm[1][r][q + t], a1); a2 = fmaf(w, sm[2][r][q + t], a2);
        }
        hs[0][r][q] = a0; hs[1][r][q] = a1; hs[2][r][q] = a2;
    }
    __syncthreads();
    const int lx = tid % SS_T, ly = tid / SS_T, px = blockIdx.x * SS_T + lx, py = blockIdx.y * SS_T + ly;
    if (px < W && py < H) {
        float c0 = 0.f, c1 = 0.f, c2 = 0.f;
#pragma unroll
        for (int t = 0; t <= 2 * SS_R; ++t) {
            const float w = c_win[t];
            c0 = fmaf(w, hs[0][ly + t][lx], c0); c1 = fmaf(w, hs[1][ly + t][lx], c1); c2 = fmaf(w, hs[2][ly + t][lx], c2);
        }
        const size_t pix = (size_t)py * W + px;
        const float xv = xr[(size_t)c * HW + pix], yv = yt[(size_t)c * HW + pix];
        up_rgb[(size_t)c * HW + pix] += c0 + 2.f * xv * c1 + yv * c2;
    }
}

}  // namespace

cudaError_t sgs_launch_ssim_loss(sgs_ctx* c, int W, int H, const float* rgb_r, const float* rgb_t, float weight,
                                 float* up_rgb, float* loss, cudaStream_t s) {
    static bool win_set = false;
    if (!win_set) {  // normalised Gaussian, sigma 1.5, evaluated in double and rounded once (as the oracle's)
        double g[2 * SS_R + 1], sum = 0.0;
        for (int t = 0; t <= 2 * SS_R; ++t) { const double d = t - SS_R; g[t] = exp(-d * d / (2.0 * 1.5 * 1.5)); sum += g[t]; }
        float gf[2 * SS_R + 1];
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
    const dim3 grid((W + SS_T - 1) / SS_T, (H + SS_T - 1) / SS_T, 3);
    const float inv = 1.f / (3.f * (float)HW);
    k_ssim_forward<<<grid, SS_T * SS_T, 0, s>>>(rgb_r, rgb_t, W, H, -weight * inv, weight * inv, c->ssim_maps, slots);
    k_ssim_backward<<<grid, SS_T * SS_T, 0, s>>>(rgb_r, rgb_t, W, H, c->ssim_maps, up_rgb, slots, loss);
    return cudaGetLastError();
}
