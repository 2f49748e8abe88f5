// probe.cu -- sgs_probe_staging: a measurement, not a step of the path.  north_star asks for "TMA bulk copies where that pays"
// in the compositing kernels' staging; the payload is one contiguous, 16-byte-aligned 128-byte record per surfel, so a staged
// batch can be fetched either by one thread per entry gathering seven LDG.128 (what k_forward / k_backward / k_track do) or by
// one cp.async.bulk per entry into shared memory, completed through an mbarrier, followed by the same re-basing arithmetic
// read from shared memory.  This kernel does exactly the staging of k_track (gather, stage_entry, seven 16-byte planes) over
// the real tile lists and payload of the ctx's last render, in both ways, so the two can be timed and profiled side by side.
#include "pair.cuh"
#include "sgs_internal.h"

namespace {

__device__ __forceinline__ void mbar_init(uint64_t* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_addr(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_addr(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_addr(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, unsigned parity) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}" ::"r"(smem_addr(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_copy_g2s(void* dst_smem, const void* src_gmem, unsigned bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_addr(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_addr(bar))
                 : "memory");
}

// MODE 0: seven LDG.128 per entry (registers) -> stage_entry -> seven STS.128.
// MODE 1: one 128-byte cp.async.bulk per entry -> mbarrier -> seven LDS.128 of the raw record -> stage_entry -> seven STS.128.
template <int MODE>
__global__ void __launch_bounds__(SGS_BLOCK)
k_stage_probe(const uint32_t* __restrict__ ranges, const uint32_t* __restrict__ vals, int vstride, SgsPayload pay, int tiles_x,
              float* __restrict__ sink) {
    __shared__ float4 sh[7][SGS_BLOCK];
    extern __shared__ __align__(128) float4 raw[];   // MODE 1: 256 raw records of 128 B (32 KB of dynamic shared memory on top of the 28 KB staged)
    __shared__ uint64_t bar;
    const int tile = blockIdx.x, tid = threadIdx.x;
    const int tx = tile % tiles_x, ty = tile / tiles_x;
    const double px0 = (double)(tx * SGS_TILE) + 0.5, py0 = (double)(ty * SGS_TILE) + 0.5;
    const uint32_t start = ranges[2 * tile], end = ranges[2 * tile + 1];
    float acc = 0.f;
    unsigned phase = 0;
    if (MODE == 1) {
        if (tid == 0) mbar_init(&bar, SGS_BLOCK);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        __syncthreads();
    }
    for (uint32_t base = start; base < end; base += SGS_BLOCK) {
        const uint32_t nb = min((uint32_t)SGS_BLOCK, end - base);
        float4 g0, g1, g3, g4, g5, g6;
        double2 g2;
        if (MODE == 0) {
            if ((uint32_t)tid < nb) {
                const uint32_t v = vals[(size_t)(base + tid) * vstride];
                g0 = pay.g0[v]; g1 = pay.g1[v]; g3 = pay.g3[v]; g4 = pay.g4[v]; g5 = pay.g5[v]; g6 = pay.g6[v]; g2 = pay.g2[v];
            }
        } else {
            if ((uint32_t)tid < nb) {
                const uint32_t v = vals[(size_t)(base + tid) * vstride];
                mbar_expect_tx(&bar, 128u);
                bulk_copy_g2s(&raw[tid * 8], pay.store + (size_t)v * 8, 128u, &bar);
            } else {
                mbar_arrive(&bar);
            }
            mbar_wait(&bar, phase);
            phase ^= 1u;
            if ((uint32_t)tid < nb) {
                const float4* r = &raw[tid * 8];
                g0 = r[0]; g1 = r[1]; g3 = r[3]; g4 = r[4]; g5 = r[5]; g6 = r[6];
                g2 = *reinterpret_cast<const double2*>(&r[2]);
            }
        }
        if ((uint32_t)tid < nb) {
            float4 s0, s1, s2;
            stage_entry(g0, g1, g2, g3, px0, py0, s0, s1, s2);
            sh[0][tid] = s0; sh[1][tid] = s1; sh[2][tid] = s2;
            sh[3][tid] = make_float4(g1.w, g3.w, g4.x, g4.y);
            const float aux = g5.y, auy = g5.z, auz = g5.w, avx = g6.x, avy = g6.y, avz = g6.z;
            sh[5][tid] = make_float4(aux, auy, auz, avx);
            sh[6][tid] = make_float4(avy, avz, auy * avz - auz * avy, auz * avx - aux * avz);
            sh[4][tid] = make_float4(g4.z, g4.w, g5.x, aux * avy - auy * avx);
        }
        __syncthreads();
        if (nb > 0) {   // consume something of every plane so that nothing above is dead
            const uint32_t j = ((uint32_t)tid * 7u + 3u) % nb;
            acc += sh[0][j].x + sh[1][j].y + sh[2][j].z + sh[3][j].w + sh[4][j].x + sh[5][j].y + sh[6][j].z;
        }
        __syncthreads();
    }
    if (acc == 1.2345678e30f) sink[tile] = acc;
}

}  // namespace

extern "C" int sgs_probe_staging(sgs_ctx* c, int mode, int reps, double* us_per_launch, void* stream) {
    if (!c || !us_per_launch || reps <= 0 || (mode != 0 && mode != 1)) return SGS_INVALID_ARGUMENT;
    if (!c->have_forward) return SGS_NO_FORWARD_STATE;
    cudaStream_t s = (cudaStream_t)stream;
    const int tiles = c->camd.tiles_x * c->camd.tiles_y;
    if (sgs_ensure_partials(c, tiles, s) != SGS_OK) return SGS_OUT_OF_MEMORY;
    if (cudaFuncSetAttribute(k_stage_probe<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, SGS_BLOCK * 128) != cudaSuccess) return SGS_CUDA_ERROR;
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return SGS_CUDA_ERROR;
    for (int r = -2; r < reps; ++r) {   // two untimed launches first
        if (r == 0) cudaEventRecord(e0, s);
        c->launches += 1;
        if (mode == 0) k_stage_probe<0><<<tiles, SGS_BLOCK, 0, s>>>(c->ranges, c->list_vals, c->list_stride, c->pay, c->camd.tiles_x, c->pose_partial);
        else k_stage_probe<1><<<tiles, SGS_BLOCK, SGS_BLOCK * 128, s>>>(c->ranges, c->list_vals, c->list_stride, c->pay, c->camd.tiles_x, c->pose_partial);
    }
    cudaEventRecord(e1, s);
    float ms = 0.f;
    const bool ok = cudaEventSynchronize(e1) == cudaSuccess && cudaEventElapsedTime(&ms, e0, e1) == cudaSuccess;
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    if (!ok || cudaGetLastError() != cudaSuccess) return SGS_CUDA_ERROR;
    *us_per_launch = 1e3 * (double)ms / reps;
    return SGS_OK;
}
