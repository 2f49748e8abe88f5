// regsort.cuh -- in-tile sort of a bucket's 64-bit keys (depth bits << 32 | surfel index, unique inside a tile) held in
// REGISTERS: a bitonic network over 256 * R elements, element e = tid + 256 r in register r of thread tid.  Strides below
// 32 are warp shuffles, strides of 256 and more are compare-exchanges between a thread's own registers, and only the strides
// 32, 64, 128 go through shared memory (two barriers each): 6 of the 36 stages for 256 keys, 9 of 45 for 512.
// Why (ncu, profiles/r02_c4.md): the sort fused into k_forward was 20 % of its instructions and 25 % of its stall samples on C4:
// the rank-by-counting path (n <= 256) costs n x 10 instructions per thread (2450 at n = 245) and the shared-memory network
// (n > 256) a barrier per stage (45 at 512 keys, 18 % of the kernel's samples).  This network is ~350 / ~700 instructions per
// thread for 256 / 512 keys.  The contract is the sorted list (tilesort.cu), not the algorithm.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

// sorts ascending; npad = power of two >= number of real keys (slots beyond hold ~0ull), 32 <= npad <= 256 * R, block-uniform.
// sk: shared scratch of 256 * R keys.  All 256 threads must call.
template <int R>
__device__ __forceinline__ void block_sort_keys(unsigned long long (&key)[R], unsigned long long* sk, const int tid, const uint32_t npad) {
#pragma unroll
    for (int k = 2; k <= 256 * R; k <<= 1) {
        if ((uint32_t)k > npad) break;   // (block-uniform: slots at and beyond npad already hold the maximum)
#pragma unroll
        for (int j = k >> 1; j > 0; j >>= 1) {
            if (j >= 256) {
                constexpr int dummy = 0; (void)dummy;
                const int dr = j >> 8;
#pragma unroll
                for (int r = 0; r < R; ++r)
                    if ((r & dr) == 0) {
                        const bool asc = (((tid + 256 * r) & k) == 0);
                        const unsigned long long a = key[r], b = key[r | dr];
                        const bool sw = (a > b) == asc;
                        key[r] = sw ? b : a; key[r | dr] = sw ? a : b;
                    }
            } else if (j >= 32) {
                __syncthreads();
#pragma unroll
                for (int r = 0; r < R; ++r) sk[tid + 256 * r] = key[r];
                __syncthreads();
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const int e = tid + 256 * r;
                    const unsigned long long o = sk[e ^ j];
                    const bool keep_min = (((e & j) == 0) == ((e & k) == 0));
                    key[r] = keep_min ? (o < key[r] ? o : key[r]) : (o > key[r] ? o : key[r]);
                }
            } else {
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const int e = tid + 256 * r;
                    const unsigned long long o = __shfl_xor_sync(0xffffffffu, key[r], j);
                    const bool keep_min = (((e & j) == 0) == ((e & k) == 0));
                    key[r] = keep_min ? (o < key[r] ? o : key[r]) : (o > key[r] ? o : key[r]);
                }
            }
        }
    }
}
