// loss.cu -- tracking loss of PAPER.md Eq. 15-19 (L180-204): the harness around the renderer that
// turns a rendered frame and a target RGB-D frame into the upstream image gradients of the
// pose-only backward.  Element-wise, HBM-bound (reads 8+4 planes, writes 8 planes).
//   L_I = |I_r - I|_1 (Eq. 15), L_D = |D_r - D| (Eq. 16), M_n = [sign * N_r . r > 0] (Eq. 17, R19),
//   M_o = [O > 0.95] (Eq. 18), L_t = mean(M_n M_o (L_I + lambda_d L_D)) (Eq. 19).
#include "sgs_internal.h"

namespace {

struct LP { const float* ren[8]; float* up[8]; };

__global__ void __launch_bounds__(256)
k_tracking_loss(LP p, const float* __restrict__ trgb, const float* __restrict__ tdepth, int W, int H, float fx,
                float fy, float cx, float cy, float lambda_d, float nsign, float* __restrict__ loss) {
    __shared__ float s_part[8];
    const int64_t HW = (int64_t)W * H;
    const float inv = 1.f / (float)HW;
    float acc = 0.f;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < HW; i += (int64_t)gridDim.x * blockDim.x) {
        const int px = (int)(i % W), py = (int)(i / W);
        const float rx = ((float)px + 0.5f - cx) / fx, ry = ((float)py + 0.5f - cy) / fy;
        const float nr = p.ren[4][i] * rx + p.ren[5][i] * ry + p.ren[6][i];
        const bool m = (nsign * nr > 0.f) && (p.ren[7][i] > 0.95f);
        float g[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
        if (m) {
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const float d = p.ren[c][i] - trgb[c * HW + i];
                acc += fabsf(d);
                g[c] = d > 0.f ? inv : (d < 0.f ? -inv : 0.f);
            }
            const float d = p.ren[3][i] - tdepth[i];
            acc += lambda_d * fabsf(d);
            g[3] = d > 0.f ? lambda_d * inv : (d < 0.f ? -lambda_d * inv : 0.f);
        }
#pragma unroll
        for (int c = 0; c < 8; ++c)
            if (p.up[c]) p.up[c][i] = g[c];
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) s_part[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        float s = 0.f;
        for (int w = 0; w < 8; ++w) s += s_part[w];
        if (loss) atomicAdd(loss, s * inv);
    }
}

// Covisibility of two views (Eq. 22): counts of the intersection and the union of the visible
// sets G_V = {k active : C_k^V > threshold}; the last block forms the score.  Integer counts: exact.
__global__ void __launch_bounds__(256)
k_covisibility(const float* __restrict__ ca, const float* __restrict__ cb, long long n, const uint8_t* __restrict__ active,
               float thr, unsigned int* __restrict__ cnt /* inter, union, ticket */, float* __restrict__ result3) {
    unsigned int inter = 0, uni = 0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const bool act = active == nullptr || active[i] != 0;
        const bool a = act && ca[i] > thr, b = act && cb[i] > thr;
        inter += (a && b) ? 1u : 0u;
        uni += (a || b) ? 1u : 0u;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        inter += __shfl_xor_sync(0xffffffffu, inter, o);
        uni += __shfl_xor_sync(0xffffffffu, uni, o);
    }
    __shared__ bool s_last;
    if ((threadIdx.x & 31) == 0) {
        if (inter) atomicAdd(&cnt[0], inter);
        if (uni) atomicAdd(&cnt[1], uni);
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        s_last = atomicAdd(&cnt[2], 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (s_last && threadIdx.x == 0) {
        __threadfence();
        const unsigned int it = atomicAdd(&cnt[0], 0u), un = atomicAdd(&cnt[1], 0u);
        result3[0] = un ? (float)it / (float)un : 0.f;
        result3[1] = (float)it;
        result3[2] = (float)un;
        cnt[0] = 0; cnt[1] = 0; cnt[2] = 0;  // self-cleaning
    }
}

}  // namespace

cudaError_t sgs_launch_covisibility(sgs_ctx* c, const float* ca, const float* cb, int64_t n, const uint8_t* active, float thr,
                                    float* result3, cudaStream_t s) {
    if (!c->covis_cnt) {
        if (cudaMalloc(&c->covis_cnt, 4 * sizeof(unsigned int)) != cudaSuccess) return cudaErrorMemoryAllocation;
        cudaMemset(c->covis_cnt, 0, 4 * sizeof(unsigned int));
    }
    int blocks = (int)((n + 255) / 256);
    if (blocks > 148 * 8) blocks = 148 * 8;
    if (blocks < 1) blocks = 1;
    c->launches += 1;
    k_covisibility<<<blocks, 256, 0, s>>>(ca, cb, (long long)n, active, thr, c->covis_cnt, result3);
    return cudaGetLastError();
}

cudaError_t sgs_launch_tracking_loss(sgs_ctx* c, const sgs_camera* cam, const float* const ren[8], const float* trgb,
                                     const float* tdepth, float lambda_d, float nsign, float* const up[8], float* loss,
                                     cudaStream_t s) {
    SgsStage st(c, SGS_STAGE_LOSS, s);
    c->launches += 1;
    LP p;
    for (int i = 0; i < 8; ++i) { p.ren[i] = ren[i]; p.up[i] = up[i]; }
    const int64_t HW = (int64_t)cam->width * cam->height;
    int blocks = (int)((HW + 255) / 256);
    if (blocks > 148 * 8) blocks = 148 * 8;
    cudaError_t e = cudaSuccess;
    if (loss) e = cudaMemsetAsync(loss, 0, sizeof(float), s);
    if (e != cudaSuccess) return e;
    k_tracking_loss<<<blocks, 256, 0, s>>>(p, trgb, tdepth, cam->width, cam->height, cam->fx, cam->fy, cam->cx, cam->cy,
                                           lambda_d, nsign, loss);
    return cudaGetLastError();
}
