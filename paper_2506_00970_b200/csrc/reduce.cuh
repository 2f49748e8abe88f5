// reduce.cuh -- warp / block / grid reductions shared by the backward kernels (backward.cu, track.cu):
// PAPER.md Eq. 11-13 sum per-pixel (or per-surfel) contributions into one 6-vector dL/dtau; this is the
// "block-then-grid" reduction of SURVEY 8(a) step 5.  Nothing here is used by the oracle.
#pragma once
#include "sgs_internal.h"

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Grid reduction: every block has written 6 partial sums at partial[block*8 ..]; the block that
// draws the last ticket adds them all in fp64 and writes the pose gradient (block-then-grid).
// Returns (to every thread of the block) whether this block was the last one.
__device__ __forceinline__ bool finish_pose(const float* __restrict__ partial, unsigned int n_blocks,
                                            SgsCounters* __restrict__ counters, float* __restrict__ d_pose6,
                                            float* __restrict__ loss_out = nullptr, unsigned int check_tile_cap = 0u) {
    __shared__ bool s_is_last;
    __shared__ double s_sum[8][7];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    __syncthreads();
    if (tid == 0) {
        __threadfence();
        const unsigned int t = atomicAdd(&counters->ticket_bwd, 1u);
        s_is_last = (t == n_blocks - 1);
    }
    __syncthreads();
    if (!s_is_last) return false;
    __threadfence();
    // (K-track's validity check, see below: the two counters are fetched here so that their latency hides under the partial sums)
    unsigned int chk_max = 0u, chk_stale = 0u;
    if (check_tile_cap != 0u) {
        chk_max = *reinterpret_cast<volatile unsigned int*>(&counters->max_tile);
        chk_stale = *reinterpret_cast<volatile unsigned int*>(&counters->stale);
    }
    double a[7] = {0, 0, 0, 0, 0, 0, 0};
    for (unsigned int b = tid; b < n_blocks; b += blockDim.x) {
        const float4 lo = __ldcg(reinterpret_cast<const float4*>(partial + (size_t)b * 8));
        const float4 hi = __ldcg(reinterpret_cast<const float4*>(partial + (size_t)b * 8 + 4));
        a[0] += lo.x; a[1] += lo.y; a[2] += lo.z; a[3] += lo.w; a[4] += hi.x; a[5] += hi.y; a[6] += hi.z;
    }
#pragma unroll
    for (int c = 0; c < 7; ++c) {
        double v = a[c];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) s_sum[wid][c] = v;
    }
    __syncthreads();
    if (tid < 7) {
        double v = 0;
        for (int w2 = 0; w2 < (int)(blockDim.x >> 5); ++w2) v += s_sum[w2][tid];
        // check_tile_cap != 0 (K-track): a tile bucket that overflowed (entries dropped) or a kept survivor list the
        // device-resident pose has left (splats possibly missing) must not pass for a result -- NaN, not a plausible number.
        // Only this, the last, block looks (the counters are final since the preprocess ended).
        if (check_tile_cap != 0u && (chk_max > check_tile_cap || chk_stale != 0u)) v = (double)__int_as_float(0x7fc00000);
        if (tid < 6) d_pose6[tid] = (float)v;
        else if (loss_out) *loss_out = (float)v;
    }
    if (tid == 0) counters->ticket_bwd = 0;  // self-cleaning: backward may run again on the same render
    return true;
}

