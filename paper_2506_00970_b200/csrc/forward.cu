// forward.cu -- K-fwd: per-tile front-to-back alpha compositing (Eq. 8;
// SURVEY §8(a) step 3).  One block per 16x16 tile, one thread per pixel, a warp covers an 8x4 pixel
// patch (better footprint coherence than 32x1).  The tile's depth-sorted entries are staged through
// shared memory in batches of 256: one thread per entry gathers the surfel's payload (float4 loads,
// L2-resident), converts it to the tile-relative form of pair.cuh and records which of the 8 warp
// patches the surfel's screen AABB reaches; each warp then walks only its own entries (a ballot over
// the mask bytes, then find-first-set), reading the staged records as warp-wide broadcasts.  A warp leaves the batch loop when all its pixels are
// saturated; the block stops fetching batches when every pixel is.
#include "pair.cuh"
#include "regsort.cuh"
#include "histsort.cuh"
#include "sgs_internal.h"

namespace {

struct Planes { float* p[8]; };

template <bool CONTRIB, bool NDEPTH, bool MEDIAN, bool LOWPASS = false>
__global__ void __launch_bounds__(SGS_BLOCK, 4)  // 64 registers, four blocks per SM: the D_n variant would take 72 and lose one (measured: with a bound of 1 block the default variant takes 89 registers and C4's forward goes from 246 to 289 us)
k_forward(const uint32_t* __restrict__ tile_order, uint32_t* __restrict__ ranges, const uint32_t* __restrict__ vals, int vstride, SgsPayload pay, int W, int H,
          int tiles_x, SgsCfgDev cfg, Planes out, float* __restrict__ T_final, uint32_t* __restrict__ n_last,
          const uint32_t* __restrict__ cursor, unsigned long long* bucket, uint32_t tile_cap,
          float* __restrict__ contrib, const uint32_t* __restrict__ contrib_map, float2* __restrict__ dn_state,
          float* __restrict__ median_out) {
    // staged batch, structure of float4 arrays (one base register, immediate offsets, broadcast reads)
    __shared__ float4 sh[LOWPASS ? 6 : 5][SGS_BLOCK];   // (R28: plane 5 = pixel-minus-centre offsets of the tile's first pixel)
    __shared__ __align__(16) unsigned char sh_mask[SGS_BLOCK];
    const uint32_t sa = smem_addr(&sh[0][0]), sm_a = smem_addr(sh_mask);
    constexpr uint32_t PL = SGS_BLOCK * 16;  // bytes per staged plane
    const int tile = tile_order ? (int)tile_order[blockIdx.x] : (int)blockIdx.x;  // longest tiles first
    const int tx = tile % tiles_x, ty = tile / tiles_x;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int lxi = (wid & 1) * 8 + (lane & 7), lyi = (wid >> 1) * 4 + (lane >> 3);
    const int px = tx * SGS_TILE + lxi, py = ty * SGS_TILE + lyi;
    const bool inside = px < W && py < H;
    const float lx = (float)lxi, ly = (float)lyi;
    const double px0 = (double)(tx * SGS_TILE) + 0.5, py0 = (double)(ty * SGS_TILE) + 0.5;
    uint32_t start, end;
    if (cursor != nullptr) {
        // Fused in-tile sort (bucket binning, tile_cap <= 2048): order this tile's bucket by the unique key
        // depth_bits << 32 | index in the staging memory before compositing, write it back for the
        // backward pass and publish the range.  See tilesort.cu for the rationale and the large-bucket path.
        const uint32_t raw = cursor[tile];
        const uint32_t n = raw < tile_cap ? raw : tile_cap;
        start = tile * tile_cap; end = start + n;
        if (tid == 0) { ranges[2 * tile] = start; ranges[2 * tile + 1] = end; }
        unsigned long long* g = bucket + (size_t)start;
        unsigned long long* sk = reinterpret_cast<unsigned long long*>(&sh[0][0]);
        // more than 128 keys: counting pass over the depth + rank inside each depth bin (histsort.cuh; linear in n); it declines
        // buckets whose depths crowd into one bin, which take the networks below like the short ones
        static_assert(sizeof(sh) >= 2048 * 8 + HS_SCRATCH_WORDS * 4 && SGS_BLOCK >= 32 * 4 && HS_BINS == 4 * SGS_BLOCK, "");
        const bool sorted = n > 128 && hist_sort_keys(g, n, sk, reinterpret_cast<uint32_t*>(sk + 2048), reinterpret_cast<uint32_t*>(sh_mask), tid, g);
        if (sorted) {
        } else if (n >= 2 && n <= 512) {   // keys in registers: shuffles + a few shared-memory exchanges (regsort.cuh)
            uint32_t npad = 32;
            while (npad < n) npad <<= 1;
            if (n <= 256) {
                unsigned long long key[1] = {(uint32_t)tid < n ? g[tid] : ~0ull};
                block_sort_keys<1>(key, sk, tid, npad);
                if ((uint32_t)tid < n) g[tid] = key[0];
            } else {
                unsigned long long key[2] = {g[tid], (uint32_t)tid + 256u < n ? g[tid + 256] : ~0ull};
                block_sort_keys<2>(key, sk, tid, npad);
                g[tid] = key[0];
                if ((uint32_t)tid + 256u < n) g[tid + 256] = key[1];
            }
        } else if (n > 512) {
            uint32_t npad = 512;
            while (npad < n) npad <<= 1;
            for (uint32_t i = tid; i < npad; i += SGS_BLOCK) sk[i] = i < n ? g[i] : ~0ull;
            __syncthreads();
            for (uint32_t k = 2; k <= npad; k <<= 1)
                for (uint32_t j = k >> 1; j > 0; j >>= 1) {
                    for (uint32_t t = tid; t < (npad >> 1); t += SGS_BLOCK) {
                        const uint32_t i = ((t & ~(j - 1)) << 1) | (t & (j - 1)), p = i | j;
                        const unsigned long long a = sk[i], b = sk[p];
                        if ((a > b) == ((i & k) == 0)) { sk[i] = b; sk[p] = a; }
                    }
                    __syncthreads();
                }
            for (uint32_t i = tid; i < n; i += SGS_BLOCK) g[i] = sk[i];
        }
        __syncthreads();  // sorted bucket visible to the block; staging memory free again
    } else {
        start = ranges[2 * tile]; end = ranges[2 * tile + 1];
    }

    float T = 1.f, C0 = 0.f, C1 = 0.f, C2 = 0.f, Dp = 0.f, N0 = 0.f, N1 = 0.f, N2 = 0.f, O = 0.f;
    float med = 0.f;    // MEDIAN (R9m): depth of the splat that takes T across 1/2
    uint32_t last = 0;  // entries [0, last) of the tile list contain every composited pair of this pixel
    bool done = !inside;

    for (uint32_t base = start; base < end; base += SGS_BLOCK) {
        if (__syncthreads_and(done)) break;
        const uint32_t nb = min((uint32_t)SGS_BLOCK, end - base);
        unsigned mask = 0;
        if ((uint32_t)tid < nb) {
            // fused mode: the bucket was just rewritten by this block -- plain loads, not the read-only path
            const uint32_t v = cursor != nullptr ? (uint32_t)bucket[base + tid] : vals[(size_t)(base + tid) * vstride];
            const float4 g0 = pay.g0[v], g1 = pay.g1[v], g3 = pay.g3[v], g4 = pay.g4[v], g5 = pay.g5[v], g7 = pay.g7[v];
            const double2 g2 = pay.g2[v];
            float4 s0, s1, s2;
            float xy0[2];
            stage_entry(g0, g1, g2, g3, px0, py0, s0, s1, s2, xy0);
            sh[0][tid] = s0; sh[1][tid] = s1; sh[2][tid] = s2;
            sh[3][tid] = make_float4(g1.w, g3.w, g4.x, g4.y);
            sh[4][tid] = make_float4(g4.z, g4.w, g5.x, __uint_as_float(v));
            mask = warp_patch_mask(g7, (float)(tx * SGS_TILE), (float)(ty * SGS_TILE));
            if (LOWPASS) sh[LOWPASS ? 5 : 0][tid] = make_float4(xy0[0], xy0[1], 0.f, 0.f);   // (the conic test knows nothing of the disc)
            else mask = refine_patch_mask(mask, s0, s1, s2, g1.w, cfg.cutoff2, cfg.alpha_min);
        }
        sh_mask[tid] = (unsigned char)mask;
        __syncthreads();
        for (uint32_t c0 = 0; c0 < nb; c0 += 32) {
            if (__all_sync(0xffffffffu, done)) break;  // per-warp early stop on saturation
            // entries of this chunk whose AABB reaches this warp's 8x4 patch, in list order
            unsigned m = __ballot_sync(0xffffffffu, (lds_u8(sm_a + c0 + lane) >> wid) & 1u);
            while (m) {
                const uint32_t j = c0 + (uint32_t)__ffs(m) - 1u;
                m &= m - 1u;
                const uint32_t ea = sa + j * 16u;
                const float4 s0 = lds128(ea), s1 = lds128(ea + PL), s2 = lds128(ea + 2 * PL);
                // pair test (pair.cuh sequence); control flow is kept warp-uniform: one vote, no divergence
                const float un = __fmaf_rn(ly, s0.y, __fmaf_rn(lx, s0.x, s0.z));
                const float vn = __fmaf_rn(ly, s1.y, __fmaf_rn(lx, s1.x, s1.z));
                const float dn = __fmaf_rn(ly, s1.w, __fmaf_rn(lx, s0.w, s2.x));
                const float inv = fast_rcp(dn);
                const float u = __fmul_rn(un, inv), v = __fmul_rn(vn, inv);
                float rho2 = __fmaf_rn(v, v, __fmul_rn(u, u));
                bool use2d = false;
                if (LOWPASS) {   // R28: rho^2 = min(u^2 + v^2, 2 |x - x_c|^2); the screen term also where the intersection is undefined
                    const float4 s5 = lds128(ea + 5 * PL);
                    const float ddx = __fadd_rn(lx, s5.x), ddy = __fadd_rn(ly, s5.y);
                    const float r2 = __fmul_rn(2.f, __fmaf_rn(ddy, ddy, __fmul_rn(ddx, ddx)));
                    use2d = !(rho2 <= r2);
                    rho2 = use2d ? r2 : rho2;
                }
                bool pass = !done && (rho2 <= cfg.cutoff2);
                if (!__any_sync(0xffffffffu, pass)) continue;
                const float4 s3 = lds128(ea + 3 * PL), s4 = lds128(ea + 4 * PL);
                const float z = (LOWPASS && use2d) ? s2.w : __fmaf_rn(s2.z, v, __fmaf_rn(s2.y, u, s2.w));
                const float G = fast_ex2(__fmul_rn(rho2, -0.72134752044448170368f));
                const float a = fminf(cfg.alpha_max, __fmul_rn(s3.x, G));
                pass = pass && (z > cfg.z_near) && (a >= cfg.alpha_min);
                const float Tn = __fmul_rn(T, 1.f - a);
                const bool stop = pass && (Tn < cfg.t_min);  // R6: stop, this splat is not composited
                done = done || stop;
                pass = pass && !stop;
                const float w = pass ? __fmul_rn(a, T) : 0.f;
                C0 = __fmaf_rn(w, s3.y, C0); C1 = __fmaf_rn(w, s3.z, C1); C2 = __fmaf_rn(w, s3.w, C2);
                Dp = __fmaf_rn(w, z, Dp);
                N0 = __fmaf_rn(w, s4.x, N0); N1 = __fmaf_rn(w, s4.y, N1); N2 = __fmaf_rn(w, s4.z, N2);
                O += w;
                if (CONTRIB) {  // Eq. 20-21: C_k += sum over the warp's pixels of w_k(p); one atomic per (warp, entry)
                    // w in [0, 1] as 24-bit fixed point: the warp sum is ONE redux.sync instead of five shuffle-adds
                    // (quantisation 6e-8 per pixel, far below the 1e-4 bar); 32 x 2^24 fits 32 bits
                    const unsigned ws = __reduce_add_sync(0xffffffffu, (unsigned)__float2uint_rn(w * 16777216.f));
                    // the staged list value is the surfel itself (bucket binning) or its compact visible index (radix
                    // binning, SGS_FLAG_RADIX_BINNING: contrib_map = vis_to_surfel takes it back to the surfel)
                    if (lane == 0 && ws != 0u) {
                        const uint32_t lv = __float_as_uint(s4.w);
                        atomicAdd(contrib + (contrib_map ? contrib_map[lv] : lv), (float)ws * (1.f / 16777216.f));
                    }
                }
                if (MEDIAN) med = (pass && T > 0.5f && Tn <= 0.5f) ? z : med;
                T = pass ? Tn : T;
                last = pass ? base - start + j + 1 : last;
            }
        }
    }
    if (inside) {
        const size_t pix = (size_t)py * W + px;
        if (NDEPTH) {  // SGS_FLAG_NORMALISED_DEPTH: D_n = D / O, kept with 1 / O for the backward's prologue
            const float io = O > 0.f ? __frcp_rn(O) : 0.f;
            Dp = __fmul_rn(Dp, io);
            dn_state[pix] = make_float2(Dp, io);
        }
        if (out.p[0]) out.p[0][pix] = C0;
        if (out.p[1]) out.p[1][pix] = C1;
        if (out.p[2]) out.p[2][pix] = C2;
        if (out.p[3]) out.p[3][pix] = Dp;
        if (out.p[4]) out.p[4][pix] = N0;
        if (out.p[5]) out.p[5][pix] = N1;
        if (out.p[6]) out.p[6][pix] = N2;
        if (out.p[7]) out.p[7][pix] = O;
        if (MEDIAN) median_out[pix] = med;
        T_final[pix] = T;
        n_last[pix] = last;
    }
}

}  // namespace

cudaError_t sgs_launch_forward(sgs_ctx* c, float* const planes[8], cudaStream_t s) {
    const int tiles = c->camd.tiles_x * c->camd.tiles_y;
    Planes out;
    for (int i = 0; i < 8; ++i) out.p[i] = planes[i];
    SgsStage st(c, SGS_STAGE_FORWARD, s);
    c->launches += 1;
#define SGS_FWD_ARGS c->render_order_valid ? c->render_order : nullptr, c->ranges, c->list_vals, c->list_stride, c->pay, c->camd.W, \
                     c->camd.H, c->camd.tiles_x, c->cfgd, out, c->T_final, c->n_last, c->fused_sort ? c->cursor : nullptr,     \
                     reinterpret_cast<unsigned long long*>(c->bucket), (uint32_t)c->tile_cap, c->contrib_out, \
                     (c->list_stride == 2 ? nullptr : c->vis_to_surfel), \
                     (c->cfg.flags & SGS_FLAG_NORMALISED_DEPTH) ? c->dn_state : nullptr, c->median_out
    const bool nd = (c->cfg.flags & SGS_FLAG_NORMALISED_DEPTH) != 0;
    if (c->cfgd.lowpass) {   // (sgs_render only: the contribution / median outputs are refused under the flag, api_run.cu)
        k_forward<false, false, false, true><<<tiles, SGS_BLOCK, 0, s>>>(SGS_FWD_ARGS);
    } else if (c->median_out) {  // (sgs_render_median; never together with the contribution output)
        if (nd) k_forward<false, true, true><<<tiles, SGS_BLOCK, 0, s>>>(SGS_FWD_ARGS);
        else k_forward<false, false, true><<<tiles, SGS_BLOCK, 0, s>>>(SGS_FWD_ARGS);
    } else if (c->contrib_out) {
        if (nd) k_forward<true, true, false><<<tiles, SGS_BLOCK, 0, s>>>(SGS_FWD_ARGS);
        else k_forward<true, false, false><<<tiles, SGS_BLOCK, 0, s>>>(SGS_FWD_ARGS);
    } else {
        if (nd) k_forward<false, true, false><<<tiles, SGS_BLOCK, 0, s>>>(SGS_FWD_ARGS);
        else k_forward<false, false, false><<<tiles, SGS_BLOCK, 0, s>>>(SGS_FWD_ARGS);
    }
#undef SGS_FWD_ARGS
    return cudaGetLastError();
}
