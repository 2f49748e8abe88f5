// window.cu -- sparse hand-over of a mapping window's gradients (sgs_fetch_grads_sparse_host, include/sgs.h).
// A window of N_a + N_i views touches the surfels its views see: in the 2 M-surfel map of C4 a view
// sees 134 k, so the dense n x 13 floats per window that sgs_fetch_grads_host copies are mostly zeros, and that copy
// (104 MB per window over PCIe) is what bounds the host-buffer path.  Here the device picks the rows that hold anything,
// in ascending surfel order, and packs them into a staging buffer, zeroing the accumulator rows behind the read:
//   k_win_flag : one thread per surfel, any of its 13 accumulated floats != 0 -> one bit; bits per block of 1024 counted
//   k_win_scan : one block, exclusive scan of the block counts; the total goes to the host through mapped memory
//   k_win_ids  : rank of every flagged surfel -> compact ascending id list
//   k_win_pack : flat loops over the compact rows: gather from the accumulator, re-zero, store row-compact
// The host learns the row count from the mapped word and enqueues copy commands of exactly that many rows later, from
// whichever call of the window API finds the pack complete (api_host.cu).  A first version let the device write the
// rows into mapped host memory itself; measured on C4 (profiles/r02_rejected.md): that kernel lives 0.5 ms at the PCIe
// write rate, and the next view's k_forward, launched beside it, made no progress until it had ended.
// No arithmetic on the gradients: the values are moved bit for bit.
#include "sgs_internal.h"

namespace {

constexpr int WB = 1024;

__global__ void __launch_bounds__(WB)
k_win_flag(const float* __restrict__ acc, int64_t n, uint32_t* __restrict__ flags, uint32_t* __restrict__ block_count) {
    __shared__ uint32_t s_cnt[WB / 32];
    const int64_t i = (int64_t)blockIdx.x * WB + threadIdx.x;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    uint32_t any = 0;
    if (i < n) {
        const uint32_t* a = reinterpret_cast<const uint32_t*>(acc);
        const uint32_t* m = a + 3 * i; const uint32_t* sc = a + 3 * n + 2 * i; const uint32_t* q = a + 5 * n + 4 * i;
        const uint32_t* c = a + 10 * n + 3 * i;
        any = m[0] | m[1] | m[2] | sc[0] | sc[1] | q[0] | q[1] | q[2] | q[3] | a[9 * n + i] | c[0] | c[1] | c[2];
        any &= 0x7fffffffu;   // (-0 is zero; a NaN row is kept and reaches the caller)
    }
    const uint32_t b = __ballot_sync(0xffffffffu, any != 0u);
    if (lane == 0) { if (i < n) flags[i >> 5] = b; s_cnt[w] = (uint32_t)__popc(b); }
    __syncthreads();
    if (w == 0) {
        uint32_t t = s_cnt[lane];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
        if (lane == 0) block_count[blockIdx.x] = t;
    }
}

__global__ void __launch_bounds__(1024)
k_win_scan(const uint32_t* __restrict__ block_count, int nb, uint32_t* __restrict__ block_off, uint32_t* __restrict__ count_dev,
           uint32_t* __restrict__ count_mapped) {
    __shared__ uint32_t s_w[32];
    __shared__ uint32_t s_carry;
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    if (tid == 0) s_carry = 0;
    __syncthreads();
    for (int b0 = 0; b0 < nb; b0 += 1024) {
        const int b = b0 + tid;
        const uint32_t v = b < nb ? block_count[b] : 0u;
        uint32_t x = v;   // inclusive scan in the warp
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
        if (lane == 31) s_w[w] = x;
        __syncthreads();
        if (w == 0) {
            uint32_t t = s_w[lane];
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, t, o); if (lane >= o) t += y; }
            s_w[lane] = t;   // inclusive over warps
        }
        __syncthreads();
        const uint32_t carry = s_carry, before = w ? s_w[w - 1] : 0u;
        if (b < nb) block_off[b] = carry + before + x - v;
        __syncthreads();
        if (tid == 1023) s_carry = carry + before + x;
        __syncthreads();
    }
    if (tid == 0) { *count_dev = s_carry; *count_mapped = s_carry; }
}

__global__ void __launch_bounds__(WB)
k_win_ids(const uint32_t* __restrict__ flags, const uint32_t* __restrict__ block_off, int64_t n, uint32_t* __restrict__ ids) {
    __shared__ uint32_t s_cnt[WB / 32];
    const int64_t i = (int64_t)blockIdx.x * WB + threadIdx.x;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int64_t base_i = (int64_t)blockIdx.x * WB + (int64_t)w * 32;
    const uint32_t b = base_i < n ? flags[base_i >> 5] : 0u;
    if (lane == 0) s_cnt[w] = (uint32_t)__popc(b);
    __syncthreads();
    uint32_t before = 0;
    for (int k = 0; k < w; ++k) before += s_cnt[k];
    if ((b >> lane) & 1u) ids[block_off[blockIdx.x] + before + (uint32_t)__popc(b & ((1u << lane) - 1u))] = (uint32_t)i;
}

template <int K>
__device__ __forceinline__ void pack_group(float* __restrict__ acc_group, float* __restrict__ out, const uint32_t* __restrict__ ids,
                                           uint32_t count, uint32_t gtid, uint32_t gsz) {
    const uint64_t total = (uint64_t)count * K;
    for (uint64_t j = gtid; j < total; j += gsz) {
        const uint32_t k = (uint32_t)(j / K), comp = (uint32_t)(j - (uint64_t)k * K);
        float* src = acc_group + (size_t)ids[k] * K + comp;
        out[j] = *src;
        *src = 0.f;
    }
}

// stage: ids [n] | mean [3n] | scale [2n] | quat [4n] | opacity [n] | rgb [3n], each group row-compact from its start
__global__ void __launch_bounds__(256)
k_win_pack(float* __restrict__ acc, int64_t n, const uint32_t* __restrict__ count_dev, uint32_t* __restrict__ stage) {
    const uint32_t count = *count_dev, gtid = blockIdx.x * blockDim.x + threadIdx.x, gsz = gridDim.x * blockDim.x;
    const uint32_t* ids = stage;
    float* out = reinterpret_cast<float*>(stage) + n;
    pack_group<3>(acc, out, ids, count, gtid, gsz);
    pack_group<2>(acc + 3 * n, out + 3 * n, ids, count, gtid, gsz);
    pack_group<4>(acc + 5 * n, out + 5 * n, ids, count, gtid, gsz);
    pack_group<1>(acc + 9 * n, out + 9 * n, ids, count, gtid, gsz);
    pack_group<3>(acc + 10 * n, out + 10 * n, ids, count, gtid, gsz);
}

}  // namespace

// words of scratch the compaction needs for n surfels (flags, block counts, block offsets, count) and of staging (ids + rows)
int64_t sgs_window_scratch_words(int64_t n) {
    const int64_t nb = (n + WB - 1) / WB;
    return (n + 31) / 32 + 2 * nb + 4;
}
int64_t sgs_window_stage_words(int64_t n) { return 14 * n + 4; }

cudaError_t sgs_launch_window_compact(sgs_ctx* c, float* acc, int64_t n, uint32_t* scratch, uint32_t* stage, uint32_t* count_mapped,
                                      cudaStream_t s) {
    const int nb = (int)((n + WB - 1) / WB);
    uint32_t* flags = scratch;
    uint32_t* block_count = flags + (n + 31) / 32;
    uint32_t* block_off = block_count + nb;
    uint32_t* count_dev = block_off + nb;
    c->launches += 4;
    if (nb > 0) k_win_flag<<<nb, WB, 0, s>>>(acc, n, flags, block_count);
    k_win_scan<<<1, 1024, 0, s>>>(block_count, nb, block_off, count_dev, count_mapped);
    if (nb > 0) k_win_ids<<<nb, WB, 0, s>>>(flags, block_off, n, stage);
    int grid = (int)((n * 13 / 8 + 255) / 256);   // (a short kernel: enough threads for every row word of an eighth of the map)
    if (grid > 148 * 8) grid = 148 * 8;
    if (grid < 1) grid = 1;
    k_win_pack<<<grid, 256, 0, s>>>(acc, n, count_dev, stage);
    return cudaGetLastError();
}
