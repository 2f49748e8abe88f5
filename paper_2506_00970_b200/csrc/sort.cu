// sort.cu -- tile binning, second half: a least-significant-digit radix sort
// of the 64-bit (tile id << 32 | depth bits) keys with their 32-bit values, written for this
// project, plus the per-tile [start, end) ranges.
//
// One histogram kernel counts every digit of every pass in a single read of the keys; each pass
// is then ONE kernel ("one sweep"): a block takes a tile of 2048 keys (dynamic tile id), ranks them
// stably inside the block with warp match-any multisplit, resolves its global digit offsets with a
// decoupled look-back over the preceding tiles (thread d owns digit d), and scatters.  Only the live
// key bits are sorted: 32 depth bits + ceil(log2(tiles)) tile bits.  The number of entries E lives
// in device memory (no host round trip): blocks past ceil(E / 2048) exit at once.
#include "sgs_internal.h"

namespace {

constexpr int RADIX_BITS = 8;
constexpr int RADIX = 1 << RADIX_BITS;
constexpr int MAX_PASSES = 8;
constexpr uint32_t ST_AGG = 1u << 30;
constexpr uint32_t ST_INC = 2u << 30;
constexpr uint32_t ST_MASK = 3u << 30;

__device__ __forceinline__ uint32_t digit_of(uint64_t key, int pass) {
    return (uint32_t)(key >> (pass * RADIX_BITS)) & (RADIX - 1);
}

// All passes' digit histograms in one read of the keys.
__global__ void __launch_bounds__(256)
k_histogram(const uint64_t* __restrict__ keys, const SgsCounters* __restrict__ counters, unsigned long long e_cap,
            int passes, uint32_t* __restrict__ hist /* passes x 256 */) {
    __shared__ uint32_t sh[MAX_PASSES * RADIX];
    for (int i = threadIdx.x; i < passes * RADIX; i += blockDim.x) sh[i] = 0;
    __syncthreads();
    unsigned long long E = counters->n_entries;
    if (E > e_cap) E = e_cap;
    const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
    for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < E; i += stride) {
        const uint64_t k = keys[i];
        for (int p = 0; p < passes; ++p) atomicAdd(&sh[p * RADIX + digit_of(k, p)], 1u);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < passes * RADIX; i += blockDim.x)
        if (sh[i]) atomicAdd(&hist[i], sh[i]);
}

// One pass.  256 threads, 8 items per thread.  Item order inside a tile is (warp, iteration, lane)
// so that "position in the tile" == "position in the input"; ranks are assigned in that order,
// which makes the pass stable.
__global__ void __launch_bounds__(256)
k_onesweep(const uint64_t* __restrict__ keys_in, const uint32_t* __restrict__ vals_in,
           uint64_t* __restrict__ keys_out, uint32_t* __restrict__ vals_out,
           const SgsCounters* __restrict__ counters, unsigned long long e_cap, int pass,
           const uint32_t* __restrict__ hist /* this pass: 256 */, uint32_t* __restrict__ state /* tiles x 256 */,
           uint32_t* __restrict__ ticket) {
    __shared__ uint32_t s_tile;
    __shared__ uint32_t s_cnt[8][RADIX];   // per-warp digit counters, then per-warp exclusive bases
    __shared__ uint32_t s_base[RADIX];     // global base of this tile's digit d
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    unsigned long long E = counters->n_entries;
    if (E > e_cap) E = e_cap;
    const uint32_t n_tiles = (uint32_t)((E + SGS_SORT_TILE - 1) / SGS_SORT_TILE);
    if (tid == 0) s_tile = atomicAdd(ticket, 1u);
    for (int i = tid; i < 8 * RADIX; i += 256) (&s_cnt[0][0])[i] = 0;
    __syncthreads();
    const uint32_t tile = s_tile;
    if (tile >= n_tiles) return;
    const unsigned long long tile_base = (unsigned long long)tile * SGS_SORT_TILE + (unsigned long long)wid * (32 * SGS_SORT_ITEMS);

    uint64_t k[SGS_SORT_ITEMS];
    uint32_t v[SGS_SORT_ITEMS];
    uint32_t rank[SGS_SORT_ITEMS];
    const uint32_t lanemask_lt = (1u << lane) - 1u;
#pragma unroll
    for (int j = 0; j < SGS_SORT_ITEMS; ++j) {
        const unsigned long long idx = tile_base + (unsigned long long)j * 32 + lane;
        const bool valid = idx < E;
        k[j] = valid ? keys_in[idx] : ~0ull;
        v[j] = valid ? vals_in[idx] : 0u;
    }
#pragma unroll
    for (int j = 0; j < SGS_SORT_ITEMS; ++j) {
        const unsigned long long idx = tile_base + (unsigned long long)j * 32 + lane;
        const bool valid = idx < E;
        // invalid lanes take digit 256 (their own group) so they never perturb real counters
        const uint32_t d = valid ? digit_of(k[j], pass) : RADIX;
        const uint32_t peers = __match_any_sync(0xffffffffu, d);
        uint32_t base = 0;
        if (valid) base = s_cnt[wid][d];
        __syncwarp();
        if (valid && (peers & lanemask_lt) == 0) s_cnt[wid][d] = base + __popc(peers);
        __syncwarp();
        rank[j] = base + __popc(peers & lanemask_lt);
    }
    __syncthreads();
    // thread d: exclusive scan of digit d over the 8 warps, tile total, look-back
    {
        const int d = tid;
        uint32_t run = 0;
#pragma unroll
        for (int w = 0; w < 8; ++w) { const uint32_t c = s_cnt[w][d]; s_cnt[w][d] = run; run += c; }
        const uint32_t total = run;
        uint32_t* st = state + (size_t)tile * RADIX + d;
        uint32_t prefix = 0;
        if (tile == 0) {
            atomicExch(st, ST_INC | total);
        } else {
            atomicExch(st, ST_AGG | total);
            // Look back LB predecessors at a time: the loads are independent (one L2 round trip per
            // batch instead of one per predecessor); a word that is not published yet is re-read.
            constexpr int LB = 16;
            bool found = false;
            for (int64_t t = (int64_t)tile - 1; !found; t -= LB) {
                uint32_t sv[LB];
#pragma unroll
                for (int k = 0; k < LB; ++k)
                    sv[k] = (t - k >= 0) ? *((volatile uint32_t*)(state + (size_t)(t - k) * RADIX + d)) : (2u << 30);
#pragma unroll
                for (int k = 0; k < LB; ++k) {
                    if (!found) {
                        uint32_t x = sv[k];
                        while ((x & ST_MASK) == 0) x = *((volatile uint32_t*)(state + (size_t)(t - k) * RADIX + d));
                        prefix += x & ~ST_MASK;
                        found = (x & ST_MASK) == ST_INC;
                    }
                }
            }
            atomicExch(st, ST_INC | (prefix + total));
        }
        // global digit base = exclusive scan of the histogram: warp shuffles + one smem hop
        __shared__ uint32_t s_wsum[8];
        const uint32_t h = hist[d];
        uint32_t incl = h;
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            const uint32_t t2 = __shfl_up_sync(0xffffffffu, incl, off);
            if (lane >= off) incl += t2;
        }
        if (lane == 31) s_wsum[wid] = incl;
        __syncthreads();
        uint32_t wbase = 0;
#pragma unroll
        for (int w = 0; w < 8; ++w) wbase += (w < wid) ? s_wsum[w] : 0u;
        s_base[d] = wbase + incl - h + prefix;
    }
    __syncthreads();
#pragma unroll
    for (int j = 0; j < SGS_SORT_ITEMS; ++j) {
        const unsigned long long idx = tile_base + (unsigned long long)j * 32 + lane;
        if (idx < E) {
            const uint32_t d = digit_of(k[j], pass);
            const uint32_t pos = s_base[d] + s_cnt[wid][d] + rank[j];
            keys_out[pos] = k[j];
            vals_out[pos] = v[j];
        }
    }
}

// ranges[t] = [first, last+1) of tile t in the sorted list; tiles without entries get (0,0)
__global__ void k_ranges(const uint64_t* __restrict__ keys, const SgsCounters* __restrict__ counters,
                         unsigned long long e_cap, uint32_t* __restrict__ ranges) {
    unsigned long long E = counters->n_entries;
    if (E > e_cap) E = e_cap;
    const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
    for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < E; i += stride) {
        const uint32_t t = (uint32_t)(keys[i] >> 32);
        if (i == 0 || (uint32_t)(keys[i - 1] >> 32) != t) ranges[2 * t] = (uint32_t)i;
        if (i == E - 1 || (uint32_t)(keys[i + 1] >> 32) != t) ranges[2 * t + 1] = (uint32_t)(i + 1);
    }
}

__global__ void k_export_idx(const uint32_t* __restrict__ vals, const uint32_t* __restrict__ vis_to_surfel,
                             const SgsCounters* __restrict__ counters, unsigned long long e_cap,
                             uint32_t* __restrict__ out) {
    unsigned long long E = counters->n_entries;
    if (E > e_cap) E = e_cap;
    const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
    for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < E; i += stride)
        out[i] = vis_to_surfel[vals[i]];
}

}  // namespace

int sgs_sort_passes(int tiles) {
    int tile_bits = 0;
    while ((1 << tile_bits) < tiles) ++tile_bits;
    return (32 + tile_bits + RADIX_BITS - 1) / RADIX_BITS;
}

cudaError_t sgs_launch_sort_and_ranges(sgs_ctx* c, cudaStream_t s) {
    const int tiles = c->camd.tiles_x * c->camd.tiles_y;
    const int passes = sgs_sort_passes(tiles);
    const unsigned long long e_cap = (unsigned long long)c->e_cap;
    const int64_t bound = c->launch_entries;  // upper bound on E used to size the grids
    const int sort_tiles = (int)((bound + SGS_SORT_TILE - 1) / SGS_SORT_TILE);
    SgsStage stg(c, SGS_STAGE_SORT, s);
    cudaError_t e;
    e = cudaMemsetAsync(c->ranges, 0, sizeof(uint32_t) * 2 * (size_t)tiles, s);
    if (e != cudaSuccess) return e;
    c->sorted_buf = 0;
    if (sort_tiles > 0) {
        e = cudaMemsetAsync(c->sort_hist, 0, sizeof(uint32_t) * (size_t)(passes * RADIX + MAX_PASSES), s);
        if (e != cudaSuccess) return e;
        e = cudaMemsetAsync(c->sort_state, 0, sizeof(uint32_t) * (size_t)passes * sort_tiles * RADIX, s);
        if (e != cudaSuccess) return e;
        int hb = (int)((bound + 1023) / 1024);
        if (hb > 148 * 8) hb = 148 * 8;
        c->launches += 2 + passes;
        k_histogram<<<hb, 256, 0, s>>>(c->keys[0], c->counters, e_cap, passes, c->sort_hist);
        int cur = 0;
        for (int p = 0; p < passes; ++p) {
            k_onesweep<<<sort_tiles, 256, 0, s>>>(c->keys[cur], c->vals[cur], c->keys[cur ^ 1], c->vals[cur ^ 1], c->counters,
                                                  e_cap, p, c->sort_hist + p * RADIX,
                                                  c->sort_state + (size_t)p * sort_tiles * RADIX,
                                                  c->sort_hist + passes * RADIX + p);
            cur ^= 1;
        }
        c->sorted_buf = cur;
        int rb = (int)((bound + 255) / 256);
        if (rb > 148 * 8) rb = 148 * 8;
        k_ranges<<<rb, 256, 0, s>>>(c->keys[cur], c->counters, e_cap, c->ranges);
    }
    c->list_vals = c->vals[c->sorted_buf];
    c->list_stride = 1;
    return cudaGetLastError();
}

cudaError_t sgs_launch_export_idx(sgs_ctx* c, cudaStream_t s) {
    int b = (int)((c->launch_entries + 255) / 256);
    if (b > 148 * 8) b = 148 * 8;
    if (b > 0)
        c->launches += 1, k_export_idx<<<b, 256, 0, s>>>(c->vals[c->sorted_buf], c->vis_to_surfel, c->counters, (unsigned long long)c->e_cap,
                                       c->idx_export);
    return cudaGetLastError();
}
