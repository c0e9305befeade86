// Rows a4-a8, host side of the tensor-core path: operand geometry, TMA tensor maps for both input
// layouts, the repack fallback for cubes TMA cannot address, launch of the CTA-pair kernel
// (tc_gemm2.cu) and of the peak-record combiner (peaks.cu).
//
//   [FQ | FU](pixels x 2n depths)  =  Q(pixels x Nchan) [Bc | -Bs]  +  U(pixels x Nchan) [Bs | Bc]
//   Bc = K w_i cos th_ik, Bs = K w_i sin th_ik                       (Eqs. 15-16 / 18-19)
#include <cuda.h>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include "common.cuh"
#include "tc_common.cuh"

namespace rms {

constexpr int TC_M = 128;            // pixels per CTA tile (UMMA M = 256 per CTA pair)
constexpr int TC_NMAX = 128;         // depths per tile (n); UMMA N = 2n <= 256

// ------------------------------------------------------------------------------------------------
// Host side
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn get_encode_fn() {
    static EncodeTiledFn fn = [] {
        void* f = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &q) != cudaSuccess) f = nullptr;
        return (EncodeTiledFn)f;
    }();
    return fn;
}

constexpr int TC_KS = 8;   // channels per pipeline stage (one UMMA K step; 32-byte swizzle rows)

rmsynth_status tc_plan_init(rmsynth_plan* p) {
    TcGeom& g = p->tc;
    g.kb = TC_KS;
    g.n_phi_tiles = (p->n_phi + TC_NMAX - 1) / TC_NMAX;
    int per = (p->n_phi + g.n_phi_tiles - 1) / g.n_phi_tiles;
    g.n_tile = (per + 7) & ~7;                         // UMMA N = 2n must be a multiple of 16
    const int n_stages = (p->n_chan + TC_KS - 1) / TC_KS;
    g.k_pad = n_stages * TC_KS;
    g.ctas = 2;
    if (!get_encode_fn()) return fail(RMSYNTH_ECUDA, "cuTensorMapEncodeTiled entry point not found");
    // reading A13: channels with w = 0 are removed -- both tensor kernels zero their samples on the way in
    const int n_words = (p->n_chan + 31) / 32;
    std::vector<uint32_t> mask(n_words, 0u);
    for (int i = 0; i < p->n_chan; ++i)
        if (p->w[i] > 0.0) mask[i / 32] |= 1u << (i % 32);
    RMS_CUDA(cudaMalloc(&p->d_chanmask, sizeof(uint32_t) * n_words));
    RMS_CUDA(cudaMemcpy(p->d_chanmask, mask.data(), sizeof(uint32_t) * n_words, cudaMemcpyHostToDevice));
    return p->scheme == RMSYNTH_SCHEME_F16X3 ? tc3_plan_init(p) : tc2_plan_init(p);
}

void tc_plan_free(rmsynth_plan* p) {
    if (p->d_tcB2) cudaFree(p->d_tcB2);
    if (p->d_tcB3) cudaFree(p->d_tcB3);
    if (p->d_chanmask) cudaFree(p->d_chanmask);
    p->d_tcB2 = nullptr;
    p->d_tcB3 = nullptr;
    p->d_chanmask = nullptr;
}

// Copy a cube into a buffer whose row pitch is a multiple of 4 floats (TMA needs 16-byte strides).
__global__ void tc_repack_kernel(const float* __restrict__ src, float* __restrict__ dst, long long rows, long long cols,
                                 long long pitch) {
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= rows * pitch) return;
    long long r = i / pitch, c = i % pitch;
    dst[i] = c < cols ? src[r * cols + c] : 0.f;
}

static rmsynth_status make_map3(CUtensorMap* m, const float* base, uint64_t n_chan, uint64_t n_pix, uint64_t pitch_floats,
                                uint32_t ks, CUtensorMapSwizzle sw = CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B) {
    cuuint64_t dims[3] = {32, n_chan, n_pix / 32};
    cuuint64_t strides[2] = {pitch_floats * 4, 128};
    cuuint32_t box[3] = {32, ks, 4};
    cuuint32_t es[3] = {1, 1, 1};
    CUresult r = get_encode_fn()(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<float*>(base), dims, strides, box, es,
                                 CU_TENSOR_MAP_INTERLEAVE_NONE, sw,
                                 CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(RMSYNTH_ECUDA, "cuTensorMapEncodeTiled(3d) failed with code " + std::to_string((int)r));
    return RMSYNTH_OK;
}

static rmsynth_status make_map(CUtensorMap* m, const float* base, uint64_t inner, uint64_t outer, uint64_t pitch_floats,
                               uint32_t box_in, uint32_t box_out, CUtensorMapSwizzle sw) {
    cuuint64_t dims[2] = {inner, outer};
    cuuint64_t strides[1] = {pitch_floats * 4};
    cuuint32_t box[2] = {box_in, box_out};
    cuuint32_t es[2] = {1, 1};
    CUresult r = get_encode_fn()(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<float*>(base), dims, strides, box, es,
                                 CU_TENSOR_MAP_INTERLEAVE_NONE, sw, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                                 CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(RMSYNTH_ECUDA, "cuTensorMapEncodeTiled failed with code " + std::to_string((int)r));
    return RMSYNTH_OK;
}


rmsynth_status tc_execute(const rmsynth_plan* p, const float* Q, const float* U, long long n_pix, int layout,
                          float* FQ, float* FU, float* FA, float* amp, float* phi, float* pa0, float* paz, int* idx,
                          cudaStream_t st) {
    const bool in_freq = layout & RMSYNTH_IN_FREQ_MAJOR, out_phi = layout & RMSYNTH_OUT_PHI_MAJOR;
    const bool want_maps = amp || phi || pa0 || paz || idx;
    rmsynth_status s;
    // TMA wants a 16-byte aligned base and row pitch; otherwise stage a padded copy (rare: odd shapes)
    const long long rows = in_freq ? p->n_chan : n_pix, cols = in_freq ? n_pix : p->n_chan;
    long long pitch = cols;
    if ((cols & 3) || ((uintptr_t)Q & 15) || ((uintptr_t)U & 15)) {
        pitch = (cols + 3) & ~3LL;
        float *q2, *u2;
        size_t bytes = sizeof(float) * (size_t)rows * pitch;
        if ((s = stream_scratch(p, st, SCR_REPACK_Q, bytes, &q2)) || (s = stream_scratch(p, st, SCR_REPACK_U, bytes, &u2)))
            return s;
        long long total = rows * pitch;
        unsigned blocks = (unsigned)((total + 255) / 256);
        tc_repack_kernel<<<blocks, 256, 0, st>>>(Q, q2, rows, cols, pitch);
        RMS_LAUNCH_CHECK("tc_repack_kernel");
        tc_repack_kernel<<<blocks, 256, 0, st>>>(U, u2, rows, cols, pitch);
        RMS_LAUNCH_CHECK("tc_repack_kernel");
        Q = q2;
        U = u2;
    }
    CUtensorMap mq, mu_;
    const bool a3d = in_freq && (n_pix % 32 == 0);
    const bool f16 = p->scheme == RMSYNTH_SCHEME_F16X3;
    // channels per TMA box: one 8-channel MMA stage (3xTF32) or one 32-channel chunk (FP16 split, raw tile)
    const uint32_t kbox = f16 ? 32 : TC_KS;
    const CUtensorMapSwizzle sw_mn = f16 ? CU_TENSOR_MAP_SWIZZLE_NONE : CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B;
    const CUtensorMapSwizzle sw_k = f16 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_32B;
    if (a3d) {
        if ((s = make_map3(&mq, Q, p->n_chan, n_pix, pitch, kbox, sw_mn)) || (s = make_map3(&mu_, U, p->n_chan, n_pix, pitch, kbox, sw_mn)))
            return s;
    } else if (in_freq) {
        if ((s = make_map(&mq, Q, n_pix, p->n_chan, pitch, 32, kbox, sw_mn)) ||
            (s = make_map(&mu_, U, n_pix, p->n_chan, pitch, 32, kbox, sw_mn)))
            return s;
    } else {
        if ((s = make_map(&mq, Q, p->n_chan, n_pix, pitch, kbox, TC_M, sw_k)) ||
            (s = make_map(&mu_, U, p->n_chan, n_pix, pitch, kbox, TC_M, sw_k)))
            return s;
    }
    // Fused peak search (a7): the epilogue warps write one record per (pixel, 64-depth segment); a small
    // second kernel merges a pixel's segments and refines.  No cube is re-read, none is needed (maps only).
    float* rec = nullptr;
    const int n_seg = 2 * (f16 ? p->tc3.n_phi_tiles : p->tc.n_phi_tiles);
    if (want_maps) {
        size_t bytes = sizeof(float) * 8 * (size_t)n_seg * (size_t)n_pix;
        if ((s = stream_scratch(p, st, SCR_PEAK_REC, bytes, &rec))) return s;
    }
    // check-in counters for the soft lock-step of the CTAs sharing a pixel-tile pair (tc_common.cuh: tile_checkin)
    int* tile_sync = nullptr;
    const long long n_pairs = ((n_pix + TC_M - 1) / TC_M + 1) / 2;
    if ((f16 ? p->tc3.n_phi_tiles : p->tc.n_phi_tiles) > 1 && n_pairs > p->sm_count / 2) {
        float* buf;
        if ((s = stream_scratch(p, st, SCR_TILE_SYNC, sizeof(int) * (size_t)n_pairs, &buf))) return s;
        tile_sync = reinterpret_cast<int*>(buf);
        RMS_CUDA(cudaMemsetAsync(tile_sync, 0, sizeof(int) * (size_t)n_pairs, st));
    }
    const int T = f16 ? p->tc3.n_phi_tiles : p->tc.n_phi_tiles;
    const char* lag_env = experiment_env("RMSYNTH_SYNC_LAG");   // compiled out of the product build (tc_common.cuh)
    const char* gang_env = experiment_env("RMSYNTH_GANG");
    const int sync_lag = lag_env ? atoi(lag_env) : 0;
    int gang = gang_env ? atoi(gang_env) : T;
    if (gang < 1 || gang > T || T % gang) gang = T;
    if (gang > p->sm_count / 2) gang = 1;                    // more depth tiles than CTA pairs: every cluster on its own
    if (sync_lag < 0 || gang == 1) tile_sync = nullptr;
    // Tile end of the FP16 kernel for phi-major cubes (tc_epilogue.cuh).  One SM stores 32 B/clk at most from registers, so a
    // 106 KB tile is >= 3.3 k cycles of store-port time against 2.5 k cycles of accumulator slack: the tile goes through a
    // shared-memory ring and TMA box stores (1) whenever TMA can address the cubes (16-byte aligned rows); else the epilogue
    // warps store it themselves with 8-byte vectors (2) or scalars (0).  With 1 and 2 the peak search records only
    // (max |F|^2, k) per segment and peaks_gather_kernel reads the three samples around k* back from the cubes.
    int ring_out = 0;
    CUtensorMap mfq, mfu;
    if (f16 && out_phi && FQ && !FA && !experiment_env("RMSYNTH_NO_RING_OUT")) {
        const char* force = experiment_env("RMSYNTH_RING_OUT");   // experiment build only: 1 = ring + TMA stores, 2 = vector stores
        const int want = force ? atoi(force) : 1;
        if (want == 1 && n_pix % 4 == 0 && n_pix < (1LL << 31) && !((uintptr_t)FQ & 15) && !((uintptr_t)FU & 15)) ring_out = 1;
        else if (n_pix % 2 == 0 && !((uintptr_t)FQ & 7) && !((uintptr_t)FU & 7)) ring_out = 2;
        if (ring_out == 1 && ((s = make_map(&mfq, FQ, n_pix, p->n_phi, n_pix, 128, 8, CU_TENSOR_MAP_SWIZZLE_NONE)) ||
                              (s = make_map(&mfu, FU, n_pix, p->n_phi, n_pix, 128, 8, CU_TENSOR_MAP_SWIZZLE_NONE))))
            return s;
    }
    s = f16 ? tc3_launch(p, &mq, &mu_, &mfq, &mfu, a3d, in_freq, out_phi, ring_out, n_pix, FQ, FU, FA, rec, tile_sync, gang, sync_lag, st)
            : tc2_launch(p, &mq, &mu_, a3d, in_freq, out_phi, n_pix, FQ, FU, FA, rec, tile_sync, gang, sync_lag, st);
    if (s) return s;
    if (!want_maps) return RMSYNTH_OK;
    if (ring_out) return peaks_gather(p, rec, n_seg, n_pix, FQ, FU, out_phi, amp, phi, pa0, paz, idx, st);
    return peaks_combine(p, rec, n_seg, n_pix, amp, phi, pa0, paz, idx, st);
}

}  // namespace rms
