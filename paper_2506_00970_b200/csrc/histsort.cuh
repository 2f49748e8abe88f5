// histsort.cuh -- in-tile sort of a bucket's 64-bit keys (depth bits << 32 | surfel index, unique inside a tile) for
// buckets of more than 128 keys: one counting pass over the DEPTH, then a rank inside each depth bin.
//   1. block minimum / maximum of the keys' depth words;  bin = (depth - min) >> s  with the smallest s that leaves
//      at most HS_BINS bins: bins are monotone in the key, so the order ACROSS bins is final
//   2. histogram in shared memory (one atomic per key), exclusive scan over the bins (1024: the sort's scratch is the
//      20 KB of the staging planes: 2048 keys + 1024 counters)
//   3. keys scattered into shared memory, grouped by bin (a second atomic per key hands out the slots)
//   4. every key is ranked among the keys of its own bin (a few to a few dozen) and written to its final place
// Linear in n where the bitonic network (regsort.cuh) is n log^2 n: ncu on C4 (profiles/r02_final.md) has the network at
// 21 % of k_forward's instructions and 30 % of its stall samples, the 512 < n <= 2048 shared-memory network alone at 9 %.
// A bucket whose keys crowd into one bin (more than HS_MAX_BIN of them: near-equal depths against a wide depth range)
// would turn step 4 quadratic: the function then leaves the bucket untouched and returns false (the caller's network
// sorts it).  The contract is the sorted list (tilesort.cu), not the algorithm.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

constexpr int HS_BINS = 1024, HS_MAX_BIN = 96;
constexpr int HS_SCRATCH_WORDS = HS_BINS;   // histogram, then the bins' end cursors (+ 32 words of reduction scratch, passed apart)

// g: the bucket (n keys, 128 < n <= 2048), sk: shared memory for n keys, sw: HS_SCRATCH_WORDS words and s_misc: 32 words of
// shared memory.
// All 256 threads must call; ends with the sorted keys written and a __syncthreads().
// out0 / out1: where the sorted keys go (out1 may be null; either may be g itself: g is read for the last time before the
// barrier in front of step 4).
__device__ __forceinline__ bool hist_sort_keys(const unsigned long long* g, const uint32_t n, unsigned long long* sk, uint32_t* sw,
                                               uint32_t* s_misc, const int tid, unsigned long long* out0,
                                               unsigned long long* out1 = nullptr) {
    uint32_t* s_cnt = sw;                 // [HS_BINS] histogram, then scatter cursors = end of each bin
    const int lane = tid & 31, wid = tid >> 5;
    // 1. depth range
    uint32_t dmin = 0xffffffffu, dmax = 0u;
    for (uint32_t e = tid; e < n; e += 256) {
        const uint32_t d = (uint32_t)(g[e] >> 32);
        dmin = min(dmin, d); dmax = max(dmax, d);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        dmin = min(dmin, __shfl_xor_sync(0xffffffffu, dmin, o));
        dmax = max(dmax, __shfl_xor_sync(0xffffffffu, dmax, o));
    }
    if (lane == 0) { s_misc[wid] = dmin; s_misc[8 + wid] = dmax; }
    for (int b = tid; b < HS_BINS; b += 256) s_cnt[b] = 0u;
    __syncthreads();
#pragma unroll
    for (int w = 0; w < 8; ++w) { dmin = min(dmin, s_misc[w]); dmax = max(dmax, s_misc[8 + w]); }
    const uint32_t range = dmax - dmin;
    const int bits = 32 - __clz(range | 1u);                    // range < 2^bits
    const int sh = bits > 10 ? bits - 10 : 0;                   // (range >> sh) < 1024
    // 2. histogram
    for (uint32_t e = tid; e < n; e += 256) atomicAdd(&s_cnt[((uint32_t)(g[e] >> 32) - dmin) >> sh], 1u);
    __syncthreads();
    // exclusive scan over the bins (four per thread) and the largest bin
    const uint4 c = *reinterpret_cast<const uint4*>(s_cnt + 4 * tid);
    uint32_t incl = c.x + c.y + c.z + c.w, big = max(max(c.x, c.y), max(c.z, c.w));
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t y = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += y;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) big = max(big, __shfl_xor_sync(0xffffffffu, big, o));
    if (lane == 31) s_misc[16 + wid] = incl;
    if (lane == 0) s_misc[24 + wid] = big;
    __syncthreads();
    uint32_t before = 0;
#pragma unroll
    for (int w = 0; w < 8; ++w) { before += (w < wid) ? s_misc[16 + w] : 0u; big = max(big, s_misc[24 + w]); }
    if (big > (uint32_t)HS_MAX_BIN) { __syncthreads(); return false; }   // (block-uniform)
    const uint32_t ex = before + incl - (c.x + c.y + c.z + c.w);
    *reinterpret_cast<uint4*>(s_cnt + 4 * tid) = make_uint4(ex, ex + c.x, ex + c.x + c.y, ex + c.x + c.y + c.z);   // cursors of the scatter
    __syncthreads();
    // 3. scatter, grouped by bin
    for (uint32_t e = tid; e < n; e += 256) {
        const unsigned long long key = g[e];
        sk[atomicAdd(&s_cnt[((uint32_t)(key >> 32) - dmin) >> sh], 1u)] = key;
    }
    __syncthreads();   // every read of g is done, the bins are complete (s_cnt[b] = end of bin b)
    // 4. rank inside the bin, final place
    for (uint32_t p = tid; p < n; p += 256) {
        const unsigned long long key = sk[p];
        const uint32_t b = ((uint32_t)(key >> 32) - dmin) >> sh;
        const uint32_t lo = b ? s_cnt[b - 1] : 0u, hi = s_cnt[b];   // (a bin's end cursor is the next bin's start)
        uint32_t rank = lo;
        for (uint32_t k = lo; k < hi; ++k) rank += sk[k] < key ? 1u : 0u;
        out0[rank] = key;
        if (out1) out1[rank] = key;
    }
    __syncthreads();
    return true;
}
