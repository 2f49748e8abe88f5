// tilesort.cu -- tile binning, second half, default path (hard part H7: "the
// contract is the resulting list, not the sorting algorithm").
//
// The binning is a most-significant-digit-first radix sort of the 64-bit (tile id | depth bits) keys
// whose first digit IS the tile id: k_preprocess_bucket has already distributed the entries to their
// tile's bucket (a counting pass with an atomic cursor per tile), so what remains is to order each
// bucket by (depth bits, surfel index).  One block per tile does that entirely in shared memory with
// a bitonic network over the unique keys  depth_bits << 32 | index  -- entries move through HBM once
// instead of once per 8-bit digit, and there is no chained look-back (the global LSD radix sort of
// sort.cu spent 10 us per pass on it at E = 83 k; ncu, profiles/r01_*).  Buckets too large for shared
// memory are sorted in place in global memory by the same network.
// The per-tile ranges fall out of the cursors; the sorted list the forward/backward kernels walk is
// the low 32 bits of each key.
#include "sgs_internal.h"

namespace {

template <typename P>
__device__ __forceinline__ void bitonic_sort(P keys, uint32_t npad) {
    for (uint32_t k = 2; k <= npad; k <<= 1) {
        for (uint32_t j = k >> 1; j > 0; j >>= 1) {
            for (uint32_t t = threadIdx.x; t < (npad >> 1); t += blockDim.x) {
                const uint32_t i = ((t & ~(j - 1)) << 1) | (t & (j - 1));
                const uint32_t p = i | j;
                const unsigned long long a = keys[i], b = keys[p];
                const bool up = (i & k) == 0;
                if ((a > b) == up) { keys[i] = b; keys[p] = a; }
            }
            __syncthreads();
        }
    }
}

__global__ void __launch_bounds__(256)
k_tilesort(uint64_t* __restrict__ bucket, const uint32_t* __restrict__ cursor, uint32_t tile_cap,
           uint32_t smem_keys, uint32_t* __restrict__ ranges, SgsCounters* __restrict__ counters) {
    extern __shared__ unsigned long long sk[];
    const uint32_t t = blockIdx.x;
    const uint32_t raw = cursor[t];
    const uint32_t n = raw < tile_cap ? raw : tile_cap;
    unsigned long long* g = reinterpret_cast<unsigned long long*>(bucket) + (size_t)t * tile_cap;
    if (threadIdx.x == 0) {
        ranges[2 * t] = t * tile_cap;  // index into the bucket array; host guarantees tiles * tile_cap < 2^32
        ranges[2 * t + 1] = t * tile_cap + n;
        if (raw > tile_cap) counters->overflow = 1u;
    }
    if (n < 2) return;
    uint32_t npad = 2;
    while (npad < n) npad <<= 1;
    if (n <= 256 && n <= smem_keys) {
        // short bucket (the common case in tracking: ~70 entries): rank by counting.  Keys are unique, so
        // rank = #{keys smaller}; one key per thread, n broadcast reads, two barriers instead of ~30.
        const bool mine = threadIdx.x < n;
        const unsigned long long key = mine ? g[threadIdx.x] : ~0ull;
        if (mine) sk[threadIdx.x] = key;
        __syncthreads();
        uint32_t rank = 0;
        for (uint32_t k = 0; k < n; ++k) rank += sk[k] < key ? 1u : 0u;
        if (mine) g[rank] = key;
    } else if (npad <= smem_keys) {
        for (uint32_t i = threadIdx.x; i < npad; i += blockDim.x) sk[i] = i < n ? g[i] : ~0ull;
        __syncthreads();
        bitonic_sort(sk, npad);
        for (uint32_t i = threadIdx.x; i < n; i += blockDim.x) g[i] = sk[i];
    } else {
        // rare: in place in global memory; npad <= tile_cap because tile_cap is a power of two
        for (uint32_t i = n + threadIdx.x; i < npad; i += blockDim.x) g[i] = ~0ull;
        __syncthreads();
        bitonic_sort(g, npad);
    }
}

// Longest-first tile order for the compositing kernels of sgs_render / sgs_backward (one block per tile; ncu,
// profiles/r01_c3_c4_c5.md: SMs were active 80 % of k_forward's and k_backward's duration because the long tiles
// started late).  One block: counting sort of the tiles by entry count, descending.  Ties land in arbitrary
// order; the order steers scheduling only, never a result.
constexpr int ORDER_BINS = 2048, ORDER_THREADS = 1024;
__global__ void __launch_bounds__(ORDER_THREADS)
k_tile_order(const uint32_t* __restrict__ cursor, int tiles, uint32_t* __restrict__ order) {
    __shared__ unsigned int s_hist[ORDER_BINS];
    __shared__ unsigned int s_wsum[ORDER_THREADS / 32];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    for (int b = tid; b < ORDER_BINS; b += ORDER_THREADS) s_hist[b] = 0;
    __syncthreads();
    constexpr int U = 4;  // keys of one pass (U * 1024 = 4096 tiles) stay in registers for the scatter
    unsigned int kb[U];
    auto load_keys = [&](int t0) {
#pragma unroll
        for (int k = 0; k < U; ++k) {
            const int t = t0 + k * ORDER_THREADS;
            kb[k] = t < tiles ? min(cursor[t], (unsigned int)(ORDER_BINS - 1)) : 0xffffffffu;
        }
    };
    for (int t0 = tid; t0 < tiles; t0 += U * ORDER_THREADS) {
        load_keys(t0);
#pragma unroll
        for (int k = 0; k < U; ++k)
            if (kb[k] != 0xffffffffu) atomicAdd(&s_hist[kb[k]], 1u);
    }
    __syncthreads();
    constexpr int PER = ORDER_BINS / ORDER_THREADS;
    unsigned int local = 0;
#pragma unroll
    for (int k = 0; k < PER; ++k) local += s_hist[ORDER_BINS - 1 - (tid * PER + k)];
    unsigned int incl = local;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
        const unsigned int t2 = __shfl_up_sync(0xffffffffu, incl, off);
        if (lane >= off) incl += t2;
    }
    if (lane == 31) s_wsum[wid] = incl;
    __syncthreads();
    unsigned int run = incl - local;
    for (int w2 = 0; w2 < wid; ++w2) run += s_wsum[w2];
#pragma unroll
    for (int k = 0; k < PER; ++k) {
        const int b = ORDER_BINS - 1 - (tid * PER + k);
        const unsigned int c2 = s_hist[b];
        s_hist[b] = run;
        run += c2;
    }
    __syncthreads();
    const bool one_pass = tiles <= U * ORDER_THREADS;
    for (int t0 = tid; t0 < tiles; t0 += U * ORDER_THREADS) {
        if (!one_pass) load_keys(t0);
#pragma unroll
        for (int k = 0; k < U; ++k)
            if (kb[k] != 0xffffffffu) order[atomicAdd(&s_hist[kb[k]], 1u)] = (uint32_t)(t0 + k * ORDER_THREADS);
    }
}

// ---- debug export for sgs_get_binning: contiguous (tile << 32 | depth) keys, indices and ranges ----
__global__ void k_export_scan(const uint32_t* __restrict__ ranges, int tiles, uint32_t* __restrict__ xr) {
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        uint32_t acc = 0;
        for (int t = 0; t < tiles; ++t) {
            const uint32_t n = ranges[2 * t + 1] - ranges[2 * t];
            xr[2 * t] = n ? acc : 0u;
            xr[2 * t + 1] = n ? acc + n : 0u;
            acc += n;
        }
    }
}
__global__ void k_export_copy(const uint64_t* __restrict__ bucket, const uint32_t* __restrict__ ranges,
                              const uint32_t* __restrict__ xr, uint64_t* __restrict__ keys, uint32_t* __restrict__ idx) {
    const uint32_t t = blockIdx.x;
    const uint32_t s = ranges[2 * t], n = ranges[2 * t + 1] - s, d = xr[2 * t];
    // Buckets of up to 384 entries are ranked here (keys are unique): K-track leaves the bucket of a tile it splits
    // between an owner and a helper block unsorted in memory (both rank the raw bucket concurrently, track.cu).  Longer
    // buckets were sorted in place by whichever kernel walked them.
    const bool rank_here = n <= 384u;
    for (uint32_t i = threadIdx.x; i < n; i += blockDim.x) {
        const uint64_t k = bucket[s + i];
        uint32_t pos = i;
        if (rank_here) {
            pos = 0;
            for (uint32_t j = 0; j < n; ++j) pos += bucket[s + j] < k ? 1u : 0u;
        }
        keys[d + pos] = ((uint64_t)t << 32) | (k >> 32);
        idx[d + pos] = (uint32_t)k;
    }
}

}  // namespace

cudaError_t sgs_launch_tilesort(sgs_ctx* c, cudaStream_t s) {
    const int tiles = c->camd.tiles_x * c->camd.tiles_y;
    uint32_t smem_keys = (uint32_t)c->tile_cap;
    const uint32_t max_keys = (200u << 10) / 8u;  // 200 KB of dynamic shared memory
    if (smem_keys > max_keys) {
        smem_keys = 1;
        while (smem_keys * 2 <= max_keys) smem_keys <<= 1;
    }
    static bool attr_set = false;
    if (!attr_set) {
        cudaFuncSetAttribute(k_tilesort, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(max_keys * 8));
        attr_set = true;
    }
    SgsStage st(c, SGS_STAGE_SORT, s);
    c->launches += 1;
    k_tilesort<<<tiles, 256, smem_keys * 8, s>>>(c->bucket, c->cursor, (uint32_t)c->tile_cap, smem_keys, c->ranges,
                                                c->counters);
    c->list_vals = reinterpret_cast<const uint32_t*>(c->bucket);
    c->list_stride = 2;
    return cudaGetLastError();
}

cudaError_t sgs_launch_tile_order(sgs_ctx* c, cudaStream_t s) {
    const int tiles = c->camd.tiles_x * c->camd.tiles_y;
    SgsStage st(c, SGS_STAGE_SORT, s);
    c->launches += 1;
    k_tile_order<<<1, ORDER_THREADS, 0, s>>>(c->cursor, tiles, c->render_order);
    c->render_order_valid = true;
    return cudaGetLastError();
}

cudaError_t sgs_launch_export_bucket(sgs_ctx* c, int64_t n_entries, cudaStream_t s) {
    (void)n_entries;
    const int tiles = c->camd.tiles_x * c->camd.tiles_y;
    c->launches += 2;
    k_export_scan<<<1, 32, 0, s>>>(c->ranges, tiles, c->export_ranges);
    k_export_copy<<<tiles, 256, 0, s>>>(c->bucket, c->ranges, c->export_ranges, c->export_keys, c->idx_export);
    return cudaGetLastError();
}
