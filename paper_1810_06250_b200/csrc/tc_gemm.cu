// Rows a4-a6, a8: the contraction on 5th-generation tensor cores (tcgen05 / TMEM / TMA), 3xTF32.
//
//   [FQ | FU](128 pixels x 2n depths)  =  Q(128 x Nchan) [Bc | -Bs]  +  U(128 x Nchan) [Bs | Bc]
//   Bc = K w_i cos th_ik, Bs = K w_i sin th_ik                       (Eqs. 15-16 / 18-19)
//
// Split precision (measured on B200, profiles/r01_tcgen05_probe.md): kind::tf32 TRUNCATES the low 13
// mantissa bits of FP32 operands, so the raw TMA tile of Q/U *is* A_hi and only
// A_lo = a - trunc(a) is produced on the SM (element-wise, layout-agnostic: same smem offset in a
// second buffer).  B_hi/B_lo are rounded in FP64 at plan time.  Per 8 channels, 6 MMAs:
//   Q_hi B1_hi, Q_lo B1_hi, Q_hi B1_lo, U_hi B2_hi, U_lo B2_hi, U_hi B2_lo,   B1=[Bc|-Bs], B2=[Bs|Bc]
// B1 and B2 are two windows into one smem block [Bs; Bc; -Bs].
// The TMEM FP32 accumulator rounds toward zero on every MMA (measured bias 5.6e-8 of the running sum
// per MMA), so a chain over all channels would drift past the 1e-5 budget on coherent sources; the
// accumulator is therefore drained every 32 channels (24 MMAs) into FP32 registers (round-to-nearest)
// by the epilogue warps, double-buffered in TMEM so the drain overlaps the next chunk's MMAs.
//
// Warp roles (512 threads, 1 CTA/SM, persistent over pixel tiles x depth tiles):
//   warp 0 TMA producer | warp 1 MMA issuer | warp 2 TMEM allocator | warps 4-7 A_lo transform |
//   warps 8-15 epilogue (TMEM -> registers -> global, either output layout)
// Frequency-major (FITS-order) cubes are consumed directly as an MN-major A operand
// (SWIZZLE_128B_ATOM_32B TMA boxes, UMMA layout SWIZZLE_128B_BASE32B): no transpose pass exists.
#include <cuda.h>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include "common.cuh"
#include "tc_common.cuh"

namespace rms {

constexpr int TC_M = 128;            // pixels per tile (UMMA M, cta_group::1)
constexpr int TC_NMAX = 128;         // depths per tile (n); UMMA N = 2n <= 256
constexpr int TC_CHUNK = 32;         // channels per accumulator drain
constexpr int TC_THREADS = 512;
constexpr int TC_SMEM_LIMIT = 227 * 1024;

template <int KS> struct TcCfg {
    static constexpr int kRowBytes = KS * 4;                      // K-major row = swizzle span
    static constexpr int kAPart = TC_M * KS * 4;                  // one of Qraw,Uraw,Qlo,Ulo
    static constexpr int kBPartMax = 3 * TC_NMAX * KS * 4;        // [Bs;Bc;-Bs] of one split part
    static constexpr int kStageBytes = 4 * kAPart + 2 * kBPartMax;
    static constexpr int kStages = (TC_SMEM_LIMIT - 2048) / kStageBytes;
    static constexpr int kSmemBytes = kStages * kStageBytes + 2048;   // + 1 KB align slack + barriers
    static constexpr uint32_t kLayoutK = KS == 8 ? 6u : (KS == 16 ? 4u : 2u);  // SWIZZLE_32B/64B/128B
    static constexpr uint32_t kSboK = 8 * kRowBytes;              // 8-row swizzle atom
    static constexpr int kStagesPerChunk = TC_CHUNK / KS;
    static constexpr int kKSteps = KS / 8;                        // MMAs (K=8) per operand pair per stage
};

// ------------------------------------------------------------------------------------------------
// Plan time: the pre-split, pre-swizzled B operand.  One blob per (depth tile j, K stage s):
//   [part hi|lo][block Bs | Bc | -Bs][row r < n][KS channels], K-major rows swizzled exactly as the
//   UMMA descriptor expects, so a stage is ONE 1-D bulk copy.  Values are formed in FP64 (a2).
template <int KS>
__global__ void tc_build_b_kernel(const double* __restrict__ delta, const double* __restrict__ kw,
                                  const double* __restrict__ phi, int n_chan, int n_phi, int n, int n_stages,
                                  float* __restrict__ blob) {
    const int r = blockIdx.x * blockDim.x + threadIdx.x;   // row within the depth tile
    const int s = blockIdx.y, j = blockIdx.z;
    if (r >= n) return;
    const int k_phi = j * n + r;
    const size_t part_floats = (size_t)3 * n * KS;
    float* base = blob + ((size_t)j * n_stages + s) * 2 * part_floats;
    const int row_bytes = KS * 4;
    for (int k = 0; k < KS; ++k) {
        const int i = s * KS + k;
        double c = 0.0, sn = 0.0;
        if (i < n_chan && k_phi < n_phi) {
            sincos(2.0 * phi[k_phi] * delta[i], &sn, &c);
            c *= kw[i];
            sn *= kw[i];
        }
        const float chi = rn_tf32((float)c), shi = rn_tf32((float)sn);
        const float clo = rn_tf32((float)(c - (double)chi)), slo = rn_tf32((float)(sn - (double)shi));
        // K-major swizzled offset of (row, k) inside a block whose rows are row_bytes long
        auto off = [&](int row) {
            uint32_t chunk = k / 4;
            if (KS == 8) chunk ^= (row >> 2) & 1; else if (KS == 16) chunk ^= (row >> 1) & 3; else chunk ^= row & 7;
            return ((size_t)row * row_bytes + chunk * 16 + (k % 4) * 4) / 4;
        };
        float* hi = base;
        float* lo = base + part_floats;
        hi[off(r)] = shi;          lo[off(r)] = slo;            // block 0: Bs
        hi[off(n + r)] = chi;      lo[off(n + r)] = clo;        // block 1: Bc
        hi[off(2 * n + r)] = -shi; lo[off(2 * n + r)] = -slo;   // block 2: -Bs
    }
}

// ------------------------------------------------------------------------------------------------
struct TcParams {
    long long n_pix;
    int n_chan, n_phi;
    int n;               // depths per tile
    int n_phi_tiles;
    int n_stages;        // ceil(n_chan / KS)
    int n_pix_tiles;
    int out_phi_major;   // 1: F[k*n_pix+p], 0: F[p*n_phi+k]
    int a3d;             // frequency-major input addressed through a 3-D map (32 pix, chan, pix/32)
    int n_items;         // n_pix_tiles * n_phi_tiles
    long long* prof;     // debug (RMSYNTH_TC_PROFILE=1): per-CTA cycles the MMA thread waited on {full, ready, acc_empty}, total
    const float* blob;
    float* FQ;
    float* FU;
};

template <int KS, int IN_MN, int OUT_LOS>
__global__ void __launch_bounds__(TC_THREADS, 1)
tc_rmsynth_kernel(const __grid_constant__ CUtensorMap mapQ, const __grid_constant__ CUtensorMap mapU, const TcParams prm) {
    using Cfg = TcCfg<KS>;
    // LOS-major output gives one ring stage to the per-warp transpose buffers of the epilogue
    constexpr int S = OUT_LOS ? Cfg::kStages - 1 : Cfg::kStages;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t* smem_gen = smem_raw + (smem_base - smem_u32(smem_raw));
    // stage layout: [Qraw][Uraw][Qlo][Ulo][B hi part][B lo part]
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem_gen + (size_t)S * Cfg::kStageBytes);
    uint64_t* full = bars;               // TMA bytes landed            (count 1 + tx)
    uint64_t* ready = bars + S;          // A_lo written                (count 4: one per transform warp)
    uint64_t* empty = bars + 2 * S;      // MMAs that read the stage done (count 1, tcgen05.commit)
    uint64_t* acc_full = bars + 3 * S;   // [2] chunk accumulated       (count 1, tcgen05.commit)
    uint64_t* acc_empty = acc_full + 2;  // [2] chunk drained           (count 8: one per epilogue warp)
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(acc_empty + 2);
    float* stage_t = reinterpret_cast<float*>(smem_gen + (size_t)S * Cfg::kStageBytes + 1024);   // 8 x [32][33] floats

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n = prm.n, N2 = 2 * prm.n;
    const uint32_t b_part_bytes = 3u * n * Cfg::kRowBytes;
    const uint32_t stage_tx = 2u * Cfg::kAPart + 2u * b_part_bytes;
    const int n_chunks = (prm.n_stages + Cfg::kStagesPerChunk - 1) / Cfg::kStagesPerChunk;

    if (threadIdx.x == 0) {
        for (int s = 0; s < S; ++s) { mbar_init(&full[s], 1); mbar_init(&ready[s], 4); mbar_init(&empty[s], 1); }
        for (int b = 0; b < 2; ++b) { mbar_init(&acc_full[b], 1); mbar_init(&acc_empty[b], 8); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 2) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(tmem_slot)));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;

    if (warp < 4) {
      asm volatile("setmaxnreg.dec.sync.aligned.u32 48;");
      if (warp == 0) {
        // ===================== TMA producer =====================
        if (lane == 0) {
            uint32_t st = 0, ph = 0;
            // Work items are (pixel tile, depth tile) pairs dealt round-robin, so the CTAs running at
            // any moment share ~grid/n_phi_tiles pixel tiles: A is fetched from HBM once and re-read from L2.
            for (int item = blockIdx.x; item < prm.n_items; item += gridDim.x) {
                const int t = item / prm.n_phi_tiles, j = item - t * prm.n_phi_tiles;
                const int pix0 = t * TC_M;
                const uint8_t* bsrc = reinterpret_cast<const uint8_t*>(prm.blob) + (size_t)j * prm.n_stages * 2 * b_part_bytes;
                for (int s = 0; s < prm.n_stages; ++s) {
                    mbar_wait(&empty[st], ph ^ 1);
                    mbar_expect_tx(&full[st], stage_tx);
                    const uint32_t sb = smem_base + st * Cfg::kStageBytes;
                    if (IN_MN) {
                        if (prm.a3d) {   // one box: 32 pixels x KS channels x 4 pixel groups
                            tma_load_3d(sb, &mapQ, 0, s * KS, pix0 / 32, &full[st]);
                            tma_load_3d(sb + Cfg::kAPart, &mapU, 0, s * KS, pix0 / 32, &full[st]);
                        } else {         // four boxes of 32 pixels x KS channels per operand
#pragma unroll
                            for (int g = 0; g < 4; ++g) {
                                tma_load_2d(sb + g * (KS * 128), &mapQ, pix0 + 32 * g, s * KS, &full[st]);
                                tma_load_2d(sb + Cfg::kAPart + g * (KS * 128), &mapU, pix0 + 32 * g, s * KS, &full[st]);
                            }
                        }
                    } else {             // [pix][chan]: one box of KS channels x 128 pixels per operand
                        tma_load_2d(sb, &mapQ, s * KS, pix0, &full[st]);
                        tma_load_2d(sb + Cfg::kAPart, &mapU, s * KS, pix0, &full[st]);
                    }
                    bulk_load(sb + 4 * Cfg::kAPart, bsrc + (size_t)s * 2 * b_part_bytes, 2 * b_part_bytes, &full[st]);
                    if (++st == S) { st = 0; ph ^= 1; }
                }
            }
        }
        __syncwarp();
      } else if (warp == 1) {
        // ===================== MMA issuer =====================
        if (lane == 0) {
            const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)IN_MN << 15) |
                                   ((uint32_t)(N2 >> 3) << 17) | ((uint32_t)(TC_M >> 4) << 24);
            uint32_t st = 0, ph = 0, ab = 0, aph = 0;
            long long w_full = 0, w_ready = 0, w_acc = 0, t_begin = clock64(), t0 = 0;
            const bool prof = prm.prof != nullptr;
            for (int item = blockIdx.x; item < prm.n_items; item += gridDim.x)
                    for (int c = 0; c < n_chunks; ++c) {
                        if (prof) t0 = clock64();
                        mbar_wait(&acc_empty[ab], aph ^ 1);
                        if (prof) w_acc += clock64() - t0;
                        tc_fence_after();
                        const uint32_t d_tmem = tmem + ab * 256;
                        const int s_end = min(prm.n_stages, (c + 1) * Cfg::kStagesPerChunk);
                        uint32_t first = 1;
                        for (int s = c * Cfg::kStagesPerChunk; s < s_end; ++s) {
                            if (prof) t0 = clock64();
                            mbar_wait(&full[st], ph);
                            if (prof) { long long t1 = clock64(); w_full += t1 - t0; t0 = t1; }
                            mbar_wait(&ready[st], ph);
                            if (prof) w_ready += clock64() - t0;
                            tc_fence_after();
                            const uint32_t sb = smem_base + st * Cfg::kStageBytes;
                            const uint32_t aQ = sb, aU = sb + Cfg::kAPart, aQl = sb + 2 * Cfg::kAPart, aUl = sb + 3 * Cfg::kAPart;
                            const uint32_t bh = sb + 4 * Cfg::kAPart, bl = bh + b_part_bytes;
                            const uint32_t b1 = n * Cfg::kRowBytes;   // [Bc|-Bs] window starts at block 1
#pragma unroll
                            for (int ks = 0; ks < Cfg::kKSteps; ++ks) {
                                const uint32_t ao = IN_MN ? ks * 1024 : ks * 32, bo = ks * 32;
                                auto adesc = [&](uint32_t a) {
                                    return IN_MN ? make_desc(a + ao, KS * 128, 512, 1u) : make_desc(a + ao, 16, Cfg::kSboK, Cfg::kLayoutK);
                                };
                                auto bdesc = [&](uint32_t b) { return make_desc(b + bo, 16, Cfg::kSboK, Cfg::kLayoutK); };
                                umma_tf32(d_tmem, adesc(aQ), bdesc(bh + b1), idesc, first ^ 1u);   // Q_hi [Bc|-Bs]_hi
                                first = 0;
                                umma_tf32(d_tmem, adesc(aQl), bdesc(bh + b1), idesc, 1u);          // Q_lo [Bc|-Bs]_hi
                                umma_tf32(d_tmem, adesc(aQ), bdesc(bl + b1), idesc, 1u);           // Q_hi [Bc|-Bs]_lo
                                umma_tf32(d_tmem, adesc(aU), bdesc(bh), idesc, 1u);                // U_hi [Bs|Bc]_hi
                                umma_tf32(d_tmem, adesc(aUl), bdesc(bh), idesc, 1u);               // U_lo [Bs|Bc]_hi
                                umma_tf32(d_tmem, adesc(aU), bdesc(bl), idesc, 1u);                // U_hi [Bs|Bc]_lo
                            }
                            umma_commit(&empty[st]);
                            if (++st == S) { st = 0; ph ^= 1; }
                        }
                        umma_commit(&acc_full[ab]);
                        if (++ab == 2) { ab = 0; aph ^= 1; }
                    }
            if (prof) {
                prm.prof[blockIdx.x * 4 + 0] = w_full; prm.prof[blockIdx.x * 4 + 1] = w_ready;
                prm.prof[blockIdx.x * 4 + 2] = w_acc;  prm.prof[blockIdx.x * 4 + 3] = clock64() - t_begin;
            }
        }
        __syncwarp();
      }
    } else if (warp < 8) {
        // ===================== A_lo transform: lo = a - trunc_tf32(a), rounded to tf32 =====================
        asm volatile("setmaxnreg.dec.sync.aligned.u32 48;");
        const int tt = threadIdx.x - 128;   // 0..127
        uint32_t st = 0, ph = 0;
        const long long total = (long long)((prm.n_items - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x) * prm.n_stages;
        for (long long it = 0; it < total; ++it) {
            mbar_wait(&full[st], ph);
            uint8_t* sg = smem_gen + (size_t)st * Cfg::kStageBytes;
#pragma unroll
            for (int v = 0; v < 2 * Cfg::kAPart / 16 / 128; ++v) {
                const int o = (v * 128 + tt) * 16;   // covers Qraw then Uraw; lo parts sit 2*kAPart further
                float4 a = *reinterpret_cast<const float4*>(sg + o);
                float4 l;
                auto lo = [](float x) {
                    float h = __uint_as_float(__float_as_uint(x) & 0xFFFFE000u);
                    return __uint_as_float(__float_as_uint(x - h) + 0x1000u);   // hardware truncation then rounds half up
                };
                l.x = lo(a.x); l.y = lo(a.y); l.z = lo(a.z); l.w = lo(a.w);
                *reinterpret_cast<float4*>(sg + 2 * Cfg::kAPart + o) = l;
            }
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            __syncwarp();
            if (lane == 0) mbar_arrive(&ready[st]);
            if (++st == S) { st = 0; ph ^= 1; }
        }
    } else {
        // ===================== epilogue: drain chunks into registers, store at tile end =====================
        asm volatile("setmaxnreg.inc.sync.aligned.u32 208;");
        const int q = warp & 3;                       // TMEM lane quarter this warp may access
        const int cbase = warp >= 12 ? 128 : 0;       // my 128 accumulator columns
        const uint32_t lane_addr = (uint32_t)(q * 32) << 16;
        uint32_t ab = 0, aph = 0;
        float acc[128];
        for (int item = blockIdx.x; item < prm.n_items; item += gridDim.x) {
            const int t = item / prm.n_phi_tiles, j = item - t * prm.n_phi_tiles;
            const long long p = (long long)t * TC_M + q * 32 + lane;
            {
                for (int c = 0; c < n_chunks; ++c) {
                    mbar_wait(&acc_full[ab], aph);
                    tc_fence_after();
#pragma unroll
                    for (int g = 0; g < 4; ++g) {
                        if (cbase + g * 32 < N2) {     // warp-uniform
                            uint32_t r[32];
                            tmem_ld32(tmem + lane_addr + ab * 256 + cbase + g * 32, r);
                            tmem_ld_wait();
                            if (c == 0) {
#pragma unroll
                                for (int i = 0; i < 32; ++i) acc[g * 32 + i] = __uint_as_float(r[i]);
                            } else {
#pragma unroll
                                for (int i = 0; i < 32; ++i) acc[g * 32 + i] += __uint_as_float(r[i]);
                            }
                        }
                    }
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&acc_empty[ab]);
                    if (++ab == 2) { ab = 0; aph ^= 1; }
                }
                // my columns cbase..cbase+127 of [FQ(0..n) | FU(n..2n)]; nv depths of this tile are real.
                const int nv = min(n, prm.n_phi - j * n);
                const int q_end = nv - cbase, u_beg = n - cbase, u_end = n + nv - cbase;
                const long long kq = (long long)j * n + cbase, ku = kq - n;
                if (!OUT_LOS) {
                  if (p < prm.n_pix) {
                    // phi-major: a warp writes 128 contiguous bytes per depth.  All bounds are warp-uniform;
                    // addresses are base + i*stride with compile-time i, stores predicated (no branches).
                    const long long sb = 4LL * prm.n_pix;   // byte stride between depths
                    unsigned long long aq = (unsigned long long)(prm.FQ + kq * prm.n_pix + p);
                    unsigned long long au = (unsigned long long)(prm.FU + ku * prm.n_pix + p);
                    asm volatile("" : "+l"(aq), "+l"(au));   // keep the bases in registers (no rematerialisation)
#pragma unroll
                    for (int g = 0; g < 4; ++g) {
                        if (g * 32 < q_end) {              // warp-uniform
#pragma unroll
                            for (int i = g * 32; i < g * 32 + 32; ++i)
                                st_global_pred(aq + i * sb, acc[i], i < q_end);
                        }
                        if (g * 32 + 32 > u_beg && g * 32 < u_end) {
#pragma unroll
                            for (int i = g * 32; i < g * 32 + 32; ++i)
                                st_global_pred(au + i * sb, acc[i], (unsigned)(i - u_beg) < (unsigned)nv);
                        }
                    }
                  }
                } else {
                    // LOS-major: transpose 32x32 blocks through a private smem buffer so that each store
                    // instruction writes 32 consecutive depths of ONE pixel row (128 contiguous bytes).
                    float* sT = stage_t + (warp - 8) * (32 * 33);
                    const long long P0 = (long long)t * TC_M + q * 32;              // first pixel of this warp
                    const int rows = (int)min(32LL, prm.n_pix - P0);                // ragged last tile (may be <= 0)
                    const long long rb = 4LL * prm.n_phi;                           // byte stride between pixel rows
#pragma unroll
                    for (int g = 0; g < 4; ++g) {
                        const int i = g * 32 + lane;                                 // the column this lane stores
                        const bool is_q = i < q_end, is_u = (unsigned)(i - u_beg) < (unsigned)nv;
                        if (g * 32 < q_end || (g * 32 + 32 > u_beg && g * 32 < u_end)) {   // warp-uniform
#pragma unroll
                            for (int c = 0; c < 32; ++c) sT[lane * 33 + c] = acc[g * 32 + c];
                            __syncwarp();
                            unsigned long long a = (unsigned long long)((is_u ? prm.FU + ku : prm.FQ + kq) + P0 * prm.n_phi + i);
#pragma unroll 8
                            for (int r = 0; r < 32; ++r)
                                st_global_pred(a + r * rb, sT[r * 33 + lane], (is_q || is_u) && r < rows);
                            __syncwarp();
                        }
                    }
                }
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 2) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem));
}

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
    using Cfg = TcCfg<TC_KS>;
    TcGeom& g = p->tc;
    g.kb = TC_KS;
    g.n_phi_tiles = (p->n_phi + TC_NMAX - 1) / TC_NMAX;
    int per = (p->n_phi + g.n_phi_tiles - 1) / g.n_phi_tiles;
    g.n_tile = (per + 7) & ~7;                         // UMMA N = 2n must be a multiple of 16
    const int n_stages = (p->n_chan + TC_KS - 1) / TC_KS;
    g.k_pad = n_stages * TC_KS;
    if (!get_encode_fn()) return fail(RMSYNTH_ECUDA, "cuTensorMapEncodeTiled entry point not found");
    size_t floats = (size_t)g.n_phi_tiles * n_stages * 2 * 3 * g.n_tile * TC_KS;
    RMS_CUDA(cudaMalloc(&p->d_tcB, floats * sizeof(float)));
    dim3 grid((g.n_tile + 63) / 64, n_stages, g.n_phi_tiles);
    tc_build_b_kernel<TC_KS><<<grid, 64>>>(p->d_delta, p->d_kw, p->d_phi, p->n_chan, p->n_phi, g.n_tile, n_stages, p->d_tcB);
    RMS_LAUNCH_CHECK("tc_build_b_kernel");
    RMS_CUDA(cudaFuncSetAttribute(tc_rmsynth_kernel<TC_KS, 0, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg::kSmemBytes));
    RMS_CUDA(cudaFuncSetAttribute(tc_rmsynth_kernel<TC_KS, 1, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg::kSmemBytes));
    RMS_CUDA(cudaFuncSetAttribute(tc_rmsynth_kernel<TC_KS, 0, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg::kSmemBytes));
    RMS_CUDA(cudaFuncSetAttribute(tc_rmsynth_kernel<TC_KS, 1, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg::kSmemBytes));
    const char* mode = getenv("RMSYNTH_TC_CTAS");      // "1" = single-CTA kernel, default = CTA pairs
    g.ctas = (mode && mode[0] == '1') ? 1 : 2;
    if (g.ctas == 2) return tc2_plan_init(p);
    return RMSYNTH_OK;
}

void tc_plan_free(rmsynth_plan* p) {
    if (p->d_tcB) cudaFree(p->d_tcB);
    if (p->d_tcB2) cudaFree(p->d_tcB2);
    p->d_tcB = p->d_tcB2 = nullptr;
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
                                uint32_t ks) {
    cuuint64_t dims[3] = {32, n_chan, n_pix / 32};
    cuuint64_t strides[2] = {pitch_floats * 4, 128};
    cuuint32_t box[3] = {32, ks, 4};
    cuuint32_t es[3] = {1, 1, 1};
    CUresult r = get_encode_fn()(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<float*>(base), dims, strides, box, es,
                                 CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B,
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
                          float* FQ, float* FU, float* amp, float* phi, float* pa0, float* paz, int* idx,
                          cudaStream_t st) {
    using Cfg = TcCfg<TC_KS>;
    const bool in_freq = layout & RMSYNTH_IN_FREQ_MAJOR, out_phi = layout & RMSYNTH_OUT_PHI_MAJOR;
    const bool want_maps = amp || phi || pa0 || paz || idx;
    rmsynth_status s;
    if (!FQ) {   // maps only: cubes go to plan-owned scratch
        std::lock_guard<std::mutex> g(p->mu);
        size_t bytes = sizeof(float) * (size_t)n_pix * p->n_phi;
        if ((s = ensure_scratch(p, 10, bytes, &FQ)) || (s = ensure_scratch(p, 11, bytes, &FU))) return s;
    }
    // TMA wants a 16-byte aligned base and row pitch; otherwise stage a padded copy (rare: odd shapes)
    const long long rows = in_freq ? p->n_chan : n_pix, cols = in_freq ? n_pix : p->n_chan;
    long long pitch = cols;
    if ((cols & 3) || ((uintptr_t)Q & 15) || ((uintptr_t)U & 15)) {
        pitch = (cols + 3) & ~3LL;
        std::lock_guard<std::mutex> g(p->mu);
        float *q2, *u2;
        size_t bytes = sizeof(float) * (size_t)rows * pitch;
        if ((s = ensure_scratch(p, 12, bytes, &q2)) || (s = ensure_scratch(p, 13, bytes, &u2))) return s;
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
    if (a3d) {
        if ((s = make_map3(&mq, Q, p->n_chan, n_pix, pitch, TC_KS)) || (s = make_map3(&mu_, U, p->n_chan, n_pix, pitch, TC_KS)))
            return s;
    } else if (in_freq) {
        if ((s = make_map(&mq, Q, n_pix, p->n_chan, pitch, 32, TC_KS, CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B)) ||
            (s = make_map(&mu_, U, n_pix, p->n_chan, pitch, 32, TC_KS, CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B)))
            return s;
    } else {
        const CUtensorMapSwizzle sw = TC_KS == 8 ? CU_TENSOR_MAP_SWIZZLE_32B
                                                 : (TC_KS == 16 ? CU_TENSOR_MAP_SWIZZLE_64B : CU_TENSOR_MAP_SWIZZLE_128B);
        if ((s = make_map(&mq, Q, p->n_chan, n_pix, pitch, TC_KS, TC_M, sw)) ||
            (s = make_map(&mu_, U, p->n_chan, n_pix, pitch, TC_KS, TC_M, sw)))
            return s;
    }
    if (p->tc.ctas == 2) {
        if ((s = tc2_launch(p, &mq, &mu_, a3d, in_freq, out_phi, n_pix, FQ, FU, st))) return s;
        if (!want_maps) return RMSYNTH_OK;
        return peaks_from_cubes(p, FQ, FU, n_pix, layout & RMSYNTH_OUT_PHI_MAJOR, amp, phi, pa0, paz, idx, st);
    }
    TcParams prm;
    prm.n_pix = n_pix;
    prm.n_chan = p->n_chan;
    prm.n_phi = p->n_phi;
    prm.n = p->tc.n_tile;
    prm.n_phi_tiles = p->tc.n_phi_tiles;
    prm.n_stages = p->tc.k_pad / TC_KS;
    prm.n_pix_tiles = (int)((n_pix + TC_M - 1) / TC_M);
    prm.out_phi_major = out_phi ? 1 : 0;
    prm.a3d = a3d ? 1 : 0;
    prm.n_items = prm.n_pix_tiles * prm.n_phi_tiles;
    prm.blob = p->d_tcB;
    prm.FQ = FQ;
    prm.FU = FU;
    const int grid = prm.n_items < p->sm_count ? prm.n_items : p->sm_count;
    prm.prof = nullptr;
    static const bool want_prof = getenv("RMSYNTH_TC_PROFILE") != nullptr;
    if (want_prof) {
        RMS_CUDA(cudaMalloc(&prm.prof, sizeof(long long) * 4 * grid));
    }
    if (in_freq && out_phi) tc_rmsynth_kernel<TC_KS, 1, 0><<<grid, TC_THREADS, Cfg::kSmemBytes, st>>>(mq, mu_, prm);
    else if (in_freq) tc_rmsynth_kernel<TC_KS, 1, 1><<<grid, TC_THREADS, Cfg::kSmemBytes, st>>>(mq, mu_, prm);
    else if (out_phi) tc_rmsynth_kernel<TC_KS, 0, 0><<<grid, TC_THREADS, Cfg::kSmemBytes, st>>>(mq, mu_, prm);
    else tc_rmsynth_kernel<TC_KS, 0, 1><<<grid, TC_THREADS, Cfg::kSmemBytes, st>>>(mq, mu_, prm);
    RMS_LAUNCH_CHECK("tc_rmsynth_kernel");
    if (want_prof) {   // debug only: synchronises
        std::vector<long long> h(4 * grid);
        RMS_CUDA(cudaMemcpy(h.data(), prm.prof, sizeof(long long) * 4 * grid, cudaMemcpyDeviceToHost));
        cudaFree(prm.prof);
        double a[4] = {0, 0, 0, 0};
        for (int i = 0; i < grid; ++i) for (int j = 0; j < 4; ++j) a[j] += (double)h[4 * i + j] / grid;
        fprintf(stderr, "[rmsynth tc profile] MMA thread: total %.0f cyc; waiting full %.1f%% ready %.1f%% acc_empty %.1f%%\n",
                a[3], 100 * a[0] / a[3], 100 * a[1] / a[3], 100 * a[2] / a[3]);
    }
    if (!want_maps) return RMSYNTH_OK;
    return peaks_from_cubes(p, FQ, FU, n_pix, layout & RMSYNTH_OUT_PHI_MAJOR, amp, phi, pa0, paz, idx, st);
}

}  // namespace rms
