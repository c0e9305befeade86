// Rows a4-a8, scheme FP16X3: the contraction of Eqs. 15-16 on tcgen05 tensor cores with a
// block-scaled FP16 split, twice the tensor rate of the 3xTF32 scheme (tc_gemm2.cu) at the same accuracy.
//
//   [FQ | FU](256 pixels x 2n depths)  =  Q [Bc | -Bs]  +  U [Bs | Bc],   per CTA pair (cta_group::2, M = 256)
//
// Split precision.  kind::f16 multiplies 11-bit significands exactly and honours FP16 subnormals (measured on the
// box), so a scaled value is carried as hi + lo (two FP16 numbers):
//   x s = hi + lo,  F = sum (hi_a hi_b + lo_a hi_b + hi_a lo_b).
//   * B = K w cos/sin is scaled once at plan time by a power of two (FP64 split).
//   * Q, U are scaled per (pixel, 32-channel chunk) by a power of two s that brings the chunk's largest |sample|
//     over the channels with w > 0 into [2^14, 2^15); zero-weight channels are replaced by zeros (they contribute
//     nothing, A13), so a flagged channel full of interference cannot crush the scale of its neighbours.
//     hi = x s rounded to a multiple of 16 (11 bits below 2^15: exact in FP16), lo = x s - hi (|lo| <= 8, exact in
//     FP32, then rounded to FP16: error <= 2^-9, i.e. 2^-23 of the chunk's largest sample).  Three packed FP32
//     instructions per PAIR of samples: hi' = fma(x, s, C) with C = 1.5 2^27 (one rounding, to a multiple of 16),
//     hi = hi' - C, lo = fma(x, s, -hi).
//   * The TMEM FP32 accumulator is drained after every chunk (12 MMAs) into FP32 registers with
//     acc += drained * 2^-e(pixel, chunk): the drains the accumulator's round-toward-zero already demands
//     (tc_gemm2.cu) are what makes a per-chunk scale free.
// A operands never touch shared memory as MMA operands: the transform warps convert the raw TMA tile in
// registers and write hi/lo straight into TENSOR MEMORY (tcgen05.st); the MMAs take A from TMEM (".ts" form).
// Shared memory carries only the raw FP32 tile (written by TMA, read once) and the B operand.
//
// TMEM (512 columns): accumulator buffers at columns 0 and 208 (2n <= 208 columns each), A ring of three
// 16-channel slots at 416 + 32 s: [Q_hi 8 | Q_lo 8 | U_hi 8 | U_lo 8] columns, two FP16 per column.
//
// Warps (512 threads, 1 CTA/SM, CTA pairs, persistent over (pixel-tile pair, depth tile) items):
//   0 raw-tile TMA producer | 1 MMA issuer (leader CTA) | 2 TMEM allocator + B producer |
//   4-11 epilogue (tc_epilogue.cuh: stores in either layout, |F| cube, fused peak search) | 12-15 transform
#include <cuda.h>
#include <cuda_fp16.h>
#include <cstdio>
#include <cstdlib>
#include <type_traits>
#include "common.cuh"
#include "tc_common.cuh"
#include "tc_epilogue.cuh"

namespace rms {

constexpr int T3_M = 128;                        // pixels per CTA (UMMA M = 256 per pair)
constexpr int T3_NMAX = 104;                     // depths per tile: 2 x 2n accumulator columns + 96 A columns = 512
constexpr int T3_KC = 32;                        // channels per chunk (scale and drain granularity)
constexpr int T3_RAW = 2 * T3_M * T3_KC * 4;     // 32 KB: raw Q tile + raw U tile of one chunk
constexpr int T3_BSTAGE = 256 * T3_NMAX;         // 26 KB: [hi|lo][slot0|slot1][4 k-cores][n rows][8 halves]
constexpr int T3_S = 3, T3_NA = 3;               // B ring (chunks); A ring in TMEM (16-channel slots)
constexpr int T3_SCALES = 8;                     // ring of per-pixel chunk scales (transform -> epilogue)
constexpr int T3_ACC_COLS = 208, T3_A_COL0 = 416;
constexpr int T3_MASKS = 48;                     // channel masks of the first 48 chunks live in shared memory
constexpr int T3_THREADS = 512;
// Shared-memory layout.  The raw ring has three stages, except in the ring-output variant (OUT == 2), where the third
// stage's 32 KB go to the output ring: a raw stage is held only from the TMA landing to the transform's read at the
// start of its chunk, so with two stages a load still has two chunk periods (~4 k cycles) to arrive.
template <int OUT>
struct T3Lay {
    static constexpr int R = OUT == 2 ? 2 : 3;                        // raw ring stages (chunks)
    static constexpr int OFF_B = R * T3_RAW;
    static constexpr int OFF_SCALE = OFF_B + T3_S * T3_BSTAGE;
    static constexpr int OFF_BARS = OFF_SCALE + T3_SCALES * T3_M * 2;  // scales are powers of two: kept as bf16 bit patterns
    static constexpr int OFF_MASK = OFF_BARS + 384;                    // <= 44 barriers + the TMEM address word come first
    static constexpr int OFF_STAGE = OFF_BARS + 640;                   // 128-byte aligned (TMA store source)
    static constexpr int STAGE_BYTES = OUT == 2 ? kRingSlots * 8192    // output ring (ten pairs x 8 KB)
                                     : OUT == 1 ? 8 * 32 * 33 * 4      // LOS-major transpose buffers
                                     : OUT == 3 ? 8 * 1024 * 4 : 0;    // per-warp turn-around buffers of the vectorised stores
    static constexpr int SMEM = OFF_STAGE + STAGE_BYTES + 1024;        // + alignment slack
    static_assert(OFF_STAGE % 128 == 0, "stage alignment");
    static_assert(2 * T3_S + 2 * T3_NA + 4 + 2 * 3 + 2 * kRingSlots <= 48, "barrier area");
    static_assert(SMEM <= 227 * 1024, "shared memory budget");
};

__device__ __forceinline__ void umma2_f16_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t bdesc, uint32_t idesc, uint32_t acc) {
    asm volatile(
        "{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::2.kind::f16 [%0], [%1], %2, %3, p;\n}" ::"r"(d_tmem), "r"(a_tmem), "l"(bdesc), "r"(idesc),
        "r"(acc) : "memory");
}
__device__ __forceinline__ void tmem_st32(uint32_t taddr, const uint32_t* r) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,"
        "%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31,%32};" ::"r"(taddr),
        "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]), "r"(r[9]),
        "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]), "r"(r[16]), "r"(r[17]), "r"(r[18]),
        "r"(r[19]), "r"(r[20]), "r"(r[21]), "r"(r[22]), "r"(r[23]), "r"(r[24]), "r"(r[25]), "r"(r[26]), "r"(r[27]),
        "r"(r[28]), "r"(r[29]), "r"(r[30]), "r"(r[31]) : "memory");
}
__device__ __forceinline__ void tmem_st_wait() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

// ------------------------------------------------------------------------------------------------
// Plan time (a2): the scaled FP16 hi/lo B operand.  One blob per (depth tile j, chunk c, CTA rank):
//   [part hi|lo][slot0 | slot1][k-core kc < 4][row < n][8 channels]   (no-swizzle K-major core matrices)
// slot0 feeds the Q MMAs, slot1 the U MMAs; accumulator column order as in tc_epilogue.cuh:
//   depth d -> FQ column cq = (d/8)*16 + d%8, FU column cu = cq + 8;  rank r holds columns [r n, r n + n)
//   slot0[cq] = Bc, slot0[cu] = -Bs, slot1[cq] = Bs, slot1[cu] = Bc.     Values: FP64 sincos, scaled by 2^eB.
__global__ void tc3_build_b_kernel(const double* __restrict__ delta, const double* __restrict__ kw,
                                   const double* __restrict__ phi, int n_chan, int n_phi, int n, int n_chunks,
                                   double scale_b, __half* __restrict__ blob) {
    const int d = blockIdx.x * blockDim.x + threadIdx.x;   // depth within the tile
    const int c = blockIdx.y, j = blockIdx.z;
    if (d >= n) return;
    const int k_phi = j * n + d;
    const size_t rank_halves = (size_t)128 * n;           // 256 n bytes per rank
    __half* base = blob + ((size_t)j * n_chunks + c) * 2 * rank_halves;
    const int cq = (d >> 3) * 16 + (d & 7), cu = cq + 8;
    for (int k = 0; k < T3_KC; ++k) {
        const int i = c * T3_KC + k;
        double cs = 0.0, sn = 0.0;
        if (i < n_chan && k_phi < n_phi) {
            sincos(2.0 * phi[k_phi] * delta[i], &sn, &cs);
            cs *= kw[i] * scale_b;
            sn *= kw[i] * scale_b;
        }
        const __half chi = __double2half(cs), shi = __double2half(sn);
        const __half clo = __double2half(cs - (double)__half2float(chi)), slo = __double2half(sn - (double)__half2float(shi));
        auto put = [&](int col, int slot, __half hi, __half lo) {
            const int rank = col >= n, row = col - rank * n;
            const size_t off = (size_t)rank * rank_halves + (size_t)slot * 32 * n + (size_t)(k >> 3) * 8 * n + (size_t)row * 8 + (k & 7);
            base[off] = hi;
            base[off + (size_t)64 * n] = lo;
        };
        put(cq, 0, chi, clo);
        put(cu, 0, __hneg(shi), __hneg(slo));
        put(cq, 1, shi, slo);
        put(cu, 1, chi, clo);
    }
}

struct Tc3Params {
    long long n_pix;
    int n_chan, n_phi, n, n_phi_tiles, n_chunks, n_items, n_pairs, a3d;
    float inv_scale_b;            // 2^-eB
    int e_min;                    // 15 + eB: lowest chunk exponent whose drain factor 2^(e - 141 - eB) is a normal FP32
    const __half* blob;
    const uint32_t* chan_mask;    // [n_chunks] bit i: channel 32 c + i exists and has w > 0
    float* FQ;                    // may be NULL
    float* FU;
    float* FA;                    // |F| cube, may be NULL
    float* rec;                   // peak-segment records, NULL = no peak search
    int* tile_sync;               // [pixel-tile pairs] check-in counters (gang_checkin), NULL = off
    int gang;                     // gang size G of the work schedule (tc_common.cuh: WorkIter)
    int sync_lag;                 // gang members may drift this many work items apart
    int stagger;                  // cycles by which consecutive gangs delay their start (de-phases the tile-end store bursts)
    long long* tl;                // timeline buffer (debug build), else NULL
};

// ------------------------------------------------------------------------------------------------
// Transform (a4): one thread per pixel row.  v[0..31] = Q, v[32..63] = U of the chunk's 32 channels.
__device__ __forceinline__ void t3_load_raw(const uint8_t* raw, int row, bool in_mn, float (&v)[64]) {
    if (in_mn) {        // [operand][pixel group][channel][32 pixels]: a warp reads 128 contiguous bytes per channel
        const float* q = reinterpret_cast<const float*>(raw) + (row >> 5) * 1024 + (row & 31);
#pragma unroll
        for (int c = 0; c < 32; ++c) { v[c] = q[c * 32]; v[32 + c] = q[4096 + c * 32]; }
    } else {            // [operand][pixel][32 channels], 128-byte rows, SWIZZLE_128B: 16-byte unit i sits at i ^ (row & 7)
        const uint8_t* q = raw + row * 128;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const int o = (i ^ (row & 7)) * 16;
            const float4 a = *reinterpret_cast<const float4*>(q + o), b = *reinterpret_cast<const float4*>(q + 16384 + o);
            v[4 * i] = a.x; v[4 * i + 1] = a.y; v[4 * i + 2] = a.z; v[4 * i + 3] = a.w;
            v[32 + 4 * i] = b.x; v[32 + 4 * i + 1] = b.y; v[32 + 4 * i + 2] = b.z; v[32 + 4 * i + 3] = b.w;
        }
    }
}

// Packed FP32 arithmetic (sm_100: FFMA2 / FADD2 work on register pairs; one issue slot for two lanes of work).
__device__ __forceinline__ uint64_t pack2(float a, float b) {
    uint64_t r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b)); return r;
}
__device__ __forceinline__ void unpack2(uint64_t v, float& a, float& b) { asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); }
__device__ __forceinline__ uint64_t fma2(uint64_t a, uint64_t b, uint64_t c) {
    uint64_t d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d;
}
__device__ __forceinline__ uint64_t mul2(uint64_t a, uint64_t b) {
    uint64_t d; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d;
}
__device__ __forceinline__ uint64_t add2(uint64_t a, uint64_t b) {
    uint64_t d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d;
}

// Two channels per call: hi = x s rounded to a multiple of 16 (exact in FP16 for |x s| < 2^15), lo = x s - hi.
__device__ __forceinline__ void t3_split(float x0, float x1, uint64_t scale2, uint32_t& hi, uint32_t& lo) {
    constexpr float C = 201326592.f;                         // 1.5 2^27: ulp 16
    const uint64_t x = pack2(x0, x1);
    const uint64_t h = add2(fma2(x, scale2, pack2(C, C)), pack2(-C, -C));
    float h0, h1, l0, l1;
    unpack2(h, h0, h1);
    unpack2(fma2(x, scale2, pack2(-h0, -h1)), l0, l1);
    const __half2 hh = __floats2half2_rn(h0, h1), ll = __floats2half2_rn(l0, l1);
    hi = *reinterpret_cast<const uint32_t*>(&hh);
    lo = *reinterpret_cast<const uint32_t*>(&ll);
}

// acc2[0..N/2) += drained[0..N) * inv: the accumulators live as register PAIRS, two columns per FFMA2
template <int N>
__device__ __forceinline__ void t3_accumulate(uint64_t* acc2, const uint32_t* r, uint64_t inv2) {
#pragma unroll
    for (int i = 0; i < N / 2; ++i)
        asm("{\n.reg .b64 t;\nmov.b64 t, {%1, %2};\nfma.rn.f32x2 %0, t, %3, %0;\n}" : "+l"(acc2[i]) : "r"(r[2 * i]), "r"(r[2 * i + 1]), "l"(inv2));
}

// OUT: 0 = phi-major cubes, scalar stores (any shape; also |F| cube and maps-only calls), 1 = LOS-major cubes,
//      2 = phi-major through the output ring and TMA stores, 3 = phi-major, vectorised stores (tc_epilogue.cuh)
// TAIL: the last chunk holds at most 16 real channels (0 < n_chan % 32 <= 16): its second, all-zero K step is neither
//      transformed nor multiplied (configs[4]: 400 channels = 12.5 chunks -> 6 of 156 MMAs per work item).  A separate
//      instantiation with the last chunk peeled off the loop, so the other shapes do not pay a branch per chunk.
template <int IN_MN, int OUT, bool TAIL>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(T3_THREADS, 1)
tc3_rmsynth_kernel(const __grid_constant__ CUtensorMap mapQ, const __grid_constant__ CUtensorMap mapU,
                   const __grid_constant__ CUtensorMap mapFQ, const __grid_constant__ CUtensorMap mapFU, const Tc3Params prm) {
    constexpr bool OUT_LOS = OUT == 1;
    using L = T3Lay<OUT>;
    constexpr int T3_R = L::R;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t* smem_gen = smem_raw + (smem_base - smem_u32(smem_raw));
    uint16_t* scales = reinterpret_cast<uint16_t*>(smem_gen + L::OFF_SCALE);      // [T3_SCALES][128] upper halves of FP32 powers of two
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem_gen + L::OFF_BARS);
    uint64_t* raw_full = bars;                    // [R] raw tile landed                     (1 + tx)
    uint64_t* raw_empty = raw_full + T3_R;        // [R] raw tile read by the transform      (4 warps)
    uint64_t* b_full = raw_empty + T3_R;          // [S] B chunk landed                      (1 + tx)
    uint64_t* b_empty = b_full + T3_S;            // [S] MMAs of the chunk done, both CTAs   (multicast commit)
    uint64_t* a_ready = b_empty + T3_S;           // [NA] LEADER's: slot written in both CTAs (4 local + 4 remote warps)
    uint64_t* a_empty = a_ready + T3_NA;          // [NA] MMAs that read the slot done        (multicast commit)
    uint64_t* acc_full = a_empty + T3_NA;         // [2] chunk accumulated, both CTAs         (multicast commit)
    uint64_t* acc_empty = acc_full + 2;           // [2] LEADER's: chunk drained by both epilogues (8 + 8 warps)
    uint64_t* ring_full = acc_empty + 2;          // [10] output pair staged                          (4 epilogue warps)
    uint64_t* ring_empty = ring_full + kRingSlots; // [10] output pair read by the TMA engine          (store thread)
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(ring_empty + kRingSlots);
    uint32_t* smask = reinterpret_cast<uint32_t*>(smem_gen + L::OFF_MASK);        // [T3_MASKS]
    float* stage_t = reinterpret_cast<float*>(smem_gen + L::OFF_STAGE);         // LOS-major transpose buffers

    // warp index through a shuffle: provably warp-uniform, so role branches are uniform and MMA operands stay in uniform registers
    const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0), lane = threadIdx.x & 31;
    const uint32_t rank = cluster_ctarank();
    const int cluster_id = blockIdx.x >> 1, n_clusters = gridDim.x >> 1;
    const int n = prm.n, N2 = 2 * prm.n;
    const uint32_t b_bytes = 256u * n;
    const int n_chunks = prm.n_chunks;
    const int n_full = TAIL ? n_chunks - 1 : n_chunks;      // chunks with two K steps

    if (threadIdx.x == 0) {
        for (int s = 0; s < T3_R; ++s) { mbar_init(&raw_full[s], 1); mbar_init(&raw_empty[s], 4); }
        for (int s = 0; s < T3_S; ++s) { mbar_init(&b_full[s], 1); mbar_init(&b_empty[s], 1); }
        for (int s = 0; s < T3_NA; ++s) { mbar_init(&a_ready[s], 8); mbar_init(&a_empty[s], 1); }
        for (int b = 0; b < 2; ++b) { mbar_init(&acc_full[b], 1); mbar_init(&acc_empty[b], 16); }
        for (int s = 0; s < kRingSlots; ++s) { mbar_init(&ring_full[s], 4); mbar_init(&ring_empty[s], 1); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (threadIdx.x >= 64 && threadIdx.x < 64 + T3_MASKS)   // T3_MASKS <= 64
        smask[threadIdx.x - 64] = (int)threadIdx.x - 64 < n_chunks ? prm.chan_mask[threadIdx.x - 64] : 0u;
    if (warp == 2) {
        asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(tmem_slot)));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;");
    }
    tc_fence_before();
    cluster_sync_all();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;

    if (warp < 4) {
      asm volatile("setmaxnreg.dec.sync.aligned.u32 32;");
      if (warp == 0) {
        // ===================== raw-tile TMA producer (both CTAs) =====================
        if (lane == 0) {
            const uint64_t pol = l2_policy_evict_last();
            uint32_t st = 0, ph = 0;
            TlRole tl;
            tl.init(prm.tl, TL_PRODUCER);
            WorkIter wi;
            wi.init(cluster_id, n_clusters, prm.n_phi_tiles, prm.n_pairs, prm.gang);
            // Every work item costs the same, so CTAs that start together reach their tile ends together and all 148
            // SMs store their 106 KB tiles at the same moment: 15.7 MB at the ~3.8 TB/s the memory system absorbs is
            // ~6.5 k cycles during which no epilogue warp drains (measured, profiles/r02_tile_timeline_cfg5.txt), then
            // nobody writes for the rest of the item.  Gang g therefore starts g x stagger cycles late; the phases then
            // stay spread over the item period and a tile's stores find the memory system idle.
            if (prm.stagger > 0) {
                const int G = prm.gang, S = (n_clusters / G) * G;
                const long long wait = (long long)(cluster_id < S ? cluster_id / G : S / G + cluster_id - S) * prm.stagger;
                const long long t0 = clock64();
                while (clock64() - t0 < wait) __nanosleep(64);
            }
            int tp, j;
            while (wi.next(tp, j)) {
                const int pix0 = (2 * tp + (int)rank) * T3_M;       // may lie past n_pix: TMA zero-fills
                tl.stamp(0);
                gang_checkin(prm.tile_sync, wi, tp, prm.sync_lag, 2 * prm.gang);
                tl.stamp(1);
                for (int c = 0; c < n_chunks; ++c) {
                    tl.begin();
                    mbar_wait(&raw_empty[st], ph ^ 1);
                    tl.add(3);
                    mbar_expect_tx(&raw_full[st], T3_RAW);
                    const uint32_t sb = smem_base + st * T3_RAW;
                    if (IN_MN) {
                        if (prm.a3d) {   // one box per operand: 32 pixels x 32 channels x 4 pixel groups
                            tma_load_3d(sb, &mapQ, 0, c * T3_KC, pix0 / 32, &raw_full[st], pol);
                            tma_load_3d(sb + T3_RAW / 2, &mapU, 0, c * T3_KC, pix0 / 32, &raw_full[st], pol);
                        } else {
#pragma unroll
                            for (int g = 0; g < 4; ++g) {
                                tma_load_2d(sb + g * 4096, &mapQ, pix0 + 32 * g, c * T3_KC, &raw_full[st], pol);
                                tma_load_2d(sb + T3_RAW / 2 + g * 4096, &mapU, pix0 + 32 * g, c * T3_KC, &raw_full[st], pol);
                            }
                        }
                    } else {             // [pix][chan]: one box of 32 channels x 128 pixels per operand
                        tma_load_2d(sb, &mapQ, c * T3_KC, pix0, &raw_full[st], pol);
                        tma_load_2d(sb + T3_RAW / 2, &mapU, c * T3_KC, pix0, &raw_full[st], pol);
                    }
                    if (++st == T3_R) { st = 0; ph ^= 1; }
                }
                tl.stamp(2);
                tl.next();
            }
        }
        __syncwarp();
      } else if (warp == 2) {
        // ===================== B producer (both CTAs): one bulk copy per chunk =====================
        if (lane == 0) {
            const uint64_t pol = l2_policy_evict_last();
            uint32_t st = 0, ph = 0;
            WorkIter wi;
            wi.init(cluster_id, n_clusters, prm.n_phi_tiles, prm.n_pairs, prm.gang);
            int tp, j;
            while (wi.next(tp, j)) {
                const uint8_t* bsrc = reinterpret_cast<const uint8_t*>(prm.blob) + ((size_t)j * n_chunks * 2 + rank) * b_bytes;
                for (int c = 0; c < n_chunks; ++c) {
                    mbar_wait(&b_empty[st], ph ^ 1);
                    mbar_expect_tx(&b_full[st], b_bytes);
                    bulk_load(smem_base + L::OFF_B + st * T3_BSTAGE, bsrc + (size_t)c * 2 * b_bytes, b_bytes, &b_full[st], pol);
                    if (++st == T3_S) { st = 0; ph ^= 1; }
                }
            }
        }
        __syncwarp();
      } else if (warp == 1) {
        // ===================== MMA issuer (leader CTA only; the whole warp runs the loop, lane 0 issues) =====================
        if (rank == 0) {
            // kind::f16: D = F32 (bit 4), A = B = F16 (0), K-major, N = 2n, M = 256.  One B descriptor per (stage, K step);
            // the other three differ by constants in the 16-byte address field.
            // The whole warp runs the loop (warp index from a shuffle = provably uniform) and one elected lane issues: the
            // MMA operands then stay in uniform registers and six UTCHMMA go out back to back.  Issued from inside an
            // `if (lane == 0)` region, nvcc wraps every MMA in an ELECT / R2UR "waterfall" of ~15 instructions.
            uint32_t lead;
            asm volatile("{\n.reg .pred p;\nelect.sync _|p, 0xffffffff;\nselp.u32 %0, 1, 0, p;\n}" : "=r"(lead));
            const uint32_t tmem_u = __shfl_sync(0xffffffffu, tmem, 0), smem_u = __shfl_sync(0xffffffffu, smem_base, 0);   // provably warp-uniform
            const uint32_t idesc = (1u << 4) | ((uint32_t)(N2 >> 3) << 17) | ((uint32_t)(256 >> 4) << 24);
            const uint64_t dhi = make_desc(0u, 16u * n, 128u, 0u);
            const uint32_t o_part = (128u * n) >> 4, o_slot = (64u * n) >> 4, o_ks = (32u * n) >> 4;
            uint32_t sa = 0, pa = 0, sb = 0, ab = 0, aph = 0;
            TlRole tl;
            tl.init(prm.tl, TL_ISSUER);
            WorkIter wi;
            wi.init(cluster_id, n_clusters, prm.n_phi_tiles, prm.n_pairs, prm.gang);
            int tp, j;
            while (wi.next(tp, j)) {
                tl.stamp(0);
                auto chunk = [&](int c, auto two_steps) {
                    tl.begin();
                    mbar_wait(&acc_empty[ab], aph ^ 1);
                    tl.add(c < 2 ? 4 : 1);                 // slot 4: the first two chunks of an item (the tile-end bubble)
                    tc_fence_after();
                    const uint32_t d_tmem = tmem_u + ab * T3_ACC_COLS;
                    const uint32_t baddr = (smem_u + L::OFF_B + sb * T3_BSTAGE) >> 4;
#pragma unroll
                    for (int ks = 0; ks < (decltype(two_steps)::value ? 2 : 1); ++ks) {
                        tl.begin();
                        mbar_wait(&a_ready[sa], pa);       // A slot written and (ks == 0) B chunk landed, in both CTAs
                        tl.add(c == 0 && ks == 0 ? 5 : 2); // slot 5: the first A slot of an item
                        tc_fence_after();
                        const uint32_t a0 = tmem_u + T3_A_COL0 + sa * 32;
                        const uint64_t d0 = dhi | (uint64_t)(baddr + ks * o_ks);             // hi part, slot 0
                        if (lead) {
                            umma2_f16_ts(d_tmem, a0 + 0, d0, idesc, ks);                      // Q_hi [Bc|-Bs]_hi
                            umma2_f16_ts(d_tmem, a0 + 8, d0, idesc, 1u);                      // Q_lo [Bc|-Bs]_hi
                            umma2_f16_ts(d_tmem, a0 + 0, d0 + o_part, idesc, 1u);             // Q_hi [Bc|-Bs]_lo
                            umma2_f16_ts(d_tmem, a0 + 16, d0 + o_slot, idesc, 1u);            // U_hi [Bs|Bc]_hi
                            umma2_f16_ts(d_tmem, a0 + 24, d0 + o_slot, idesc, 1u);            // U_lo [Bs|Bc]_hi
                            umma2_f16_ts(d_tmem, a0 + 16, d0 + o_part + o_slot, idesc, 1u);   // U_hi [Bs|Bc]_lo
                            umma2_commit_mc(&a_empty[sa]);
                        }
                        __syncwarp();
                        if (++sa == T3_NA) { sa = 0; pa ^= 1; }
                    }
                    if (lead) { umma2_commit_mc(&b_empty[sb]); umma2_commit_mc(&acc_full[ab]); }
                    __syncwarp();
                    if (++sb == T3_S) sb = 0;
                    if (++ab == 2) { ab = 0; aph ^= 1; }
                };
                for (int c = 0; c < n_full; ++c) chunk(c, std::true_type());
                if (TAIL) chunk(n_full, std::false_type());
                tl.stamp(3);
                tl.next();
            }
        }
        __syncwarp();
      } else if (OUT == 2) {
        // ===================== store thread (both CTAs): output ring -> TMA box stores (tc_epilogue.cuh) =====================
        if (lane == 0) {
            const uint64_t pol = l2_policy_evict_first();
            TileRing ring;
            ring.init(stage_t, ring_full, ring_empty);
            WorkIter wi;
            wi.init(cluster_id, n_clusters, prm.n_phi_tiles, prm.n_pairs, prm.gang);
            int tp, j;
            while (wi.next(tp, j))
                ring_store_item(ring, &mapFQ, &mapFU, (2 * tp + (int)rank) * T3_M, j * n, min(n, prm.n_phi - j * n), pol);
            ring_store_flush();
        }
        __syncwarp();
      }
    } else if (warp >= 12) {
        // ===================== transform (both CTAs): raw FP32 tile -> scaled FP16 hi/lo in TMEM =====================
        // The highest warp ids: the scheduler favours them over the epilogue warps of the same sub-partition, and this
        // role is the latency-critical one (the MMA issuer waits for every A slot; the epilogue has slack).
        asm volatile("setmaxnreg.dec.sync.aligned.u32 96;");
        const int row = threadIdx.x - 384;                          // pixel row of the tile = TMEM lane
        const uint32_t lane_addr = (uint32_t)((warp & 3) * 32) << 16;
        uint32_t sr = 0, pr = 0, sa = 0, pa = 0, sb = 0, pb = 0, seq = 0;
        const uint32_t ready0 = mapa_u32(smem_u32(&a_ready[0]), 0);
        TlRole tl;
        tl.init(warp == 12 ? prm.tl : nullptr, TL_TRANSFORM);
        WorkIter wi;
        wi.init(cluster_id, n_clusters, prm.n_phi_tiles, prm.n_pairs, prm.gang);
        int tp, j;
        while (wi.next(tp, j)) {
            tl.stamp(0);
            auto chunk = [&](int c, auto two_steps) {
                constexpr bool TWO = decltype(two_steps)::value;    // false: the half-filled last chunk (TAIL), one 16-channel slot
                float v[64];
                tl.begin();
                mbar_wait(&raw_full[sr], pr);
                tl.lap(c == 0 ? 5 : 1);
                t3_load_raw(smem_gen + sr * T3_RAW, row, IN_MN, v);
                const uint32_t mask = c < T3_MASKS ? smask[c] : __ldg(prm.chan_mask + c);
                if (mask != 0xFFFFFFFFu) {                          // warp-uniform: zero the zero-weight channels
#pragma unroll
                    for (int i = 0; i < 32; ++i)
                        if (!((mask >> i) & 1u)) { v[i] = 0.f; v[32 + i] = 0.f; }
                }
                float m4[4] = {0.f, 0.f, 0.f, 0.f};                  // four independent chains, not one of 64 dependent maxima
#pragma unroll
                for (int i = 0; i < 64; ++i) m4[i & 3] = fmaxf(m4[i & 3], fabsf(v[i]));
                const float m = fmaxf(fmaxf(m4[0], m4[1]), fmaxf(m4[2], m4[3]));
                __syncwarp();
                if (lane == 0) mbar_arrive(&raw_empty[sr]);         // every lane's loads have completed (values used above)
                if (++sr == T3_R) { sr = 0; pr ^= 1; }
                // scale 2^(141 - e) brings the chunk's largest sample into [2^14, 2^15); e clamped so that both powers AND the
                // drain factor below are normal FP32 numbers.  A chunk whose maximum lies under the clamp (2^(eB - 112),
                // ~1e-27) is scaled by the clamp's power instead: its halves sit lower in the FP16 range and lose
                // precision gradually (2^-24 of the scaled value 1) instead of being flushed to zero by the factor.
                int e = (int)(__float_as_uint(m) >> 23);
                e = min(max(e, prm.e_min), 254);
                const float scale = __uint_as_float((uint32_t)(268 - e) << 23);
                const uint64_t scale2 = pack2(scale, scale);
                // what the epilogue multiplies the drained chunk with: 2^(e - 141) 2^-eB (B's plan-time scale folded in)
                scales[(seq & (T3_SCALES - 1)) * T3_M + row] =
                    (uint16_t)(__float_as_uint(__uint_as_float((uint32_t)(e - 14) << 23) * prm.inv_scale_b) >> 16);
                ++seq;
                // The two 16-channel slots are published separately.  The first slot of a chunk was released long ago
                // (by the chunk before the previous one), the second only half-way through the previous chunk's MMAs:
                // published together, the chain  commit -> a_empty -> tcgen05.st -> wait::st -> remote arrive -> issuer
                // (~800 cycles) had to fit into the 624 cycles the previous chunk's second K step lasts, and the tensor
                // pipe idled ~250 cycles per chunk (profiles/r02_tile_timeline_cfg5.txt).  Published separately, the
                // first K step never waits for it and the second has a whole K step more of slack.
                const uint32_t s0 = sa, s1 = sa + 1 == T3_NA ? 0 : sa + 1;
                const uint32_t p0 = pa, p1 = sa + 1 == T3_NA ? pa ^ 1 : pa;
                uint32_t r0[32], r1[32];
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    t3_split(v[2 * i], v[2 * i + 1], scale2, r0[i], r0[8 + i]);
                    t3_split(v[32 + 2 * i], v[32 + 2 * i + 1], scale2, r0[16 + i], r0[24 + i]);
                }
                tl.lap(6);                                           // loads, chunk maximum, split arithmetic
                mbar_wait(&a_empty[s0], p0 ^ 1);
                tl.lap(2);
                tc_fence_after();
                tmem_st32(tmem + lane_addr + T3_A_COL0 + s0 * 32, r0);
                if (TWO) {
#pragma unroll
                    for (int i = 0; i < 8; ++i) {                    // the second conversion overlaps the first store
                        t3_split(v[16 + 2 * i], v[16 + 2 * i + 1], scale2, r1[i], r1[8 + i]);
                        t3_split(v[48 + 2 * i], v[48 + 2 * i + 1], scale2, r1[16 + i], r1[24 + i]);
                    }
                }
                tl.lap(6);
                tmem_st_wait();
                tl.lap(7);                                           // TMEM store round trip
                mbar_wait(&b_full[sb], pb);                          // the B chunk of this CTA must have landed too
                tl.lap(3);
                if (++sb == T3_S) { sb = 0; pb ^= 1; }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive_remote(ready0 + s0 * 8);
                if (!TWO) { sa = s1; pa = p1; return; }
                mbar_wait(&a_empty[s1], p1 ^ 1);
                tl.lap(2);
                tc_fence_after();
                tmem_st32(tmem + lane_addr + T3_A_COL0 + s1 * 32, r1);
                tmem_st_wait();
                tl.lap(7);
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive_remote(ready0 + s1 * 8);
                pa = p1;
                sa = s1 + 1 == T3_NA ? 0 : s1 + 1;
                if (sa == 0) pa ^= 1;
            };
            for (int c = 0; c < n_full; ++c) chunk(c, std::true_type());
            if (TAIL) chunk(n_full, std::false_type());
            tl.stamp(4);
            tl.next();
        }
    } else {
        // ===================== epilogue (both CTAs, own TMEM lanes = own 128 pixels) =====================
        asm volatile("setmaxnreg.inc.sync.aligned.u32 192;");
        const int q = warp & 3;
        // Columns are split 112 / 96 (7 / 6 depth groups) between the two warps of a lane quarter, so that 64 staging
        // registers fit next to the accumulators and a drain is two TMEM load round trips (~230 cycles each) instead of four.
        const int half = warp >= 8 ? 1 : 0;
        const int cbase = half ? 112 : 0;
        const uint32_t lane_addr = (uint32_t)(q * 32) << 16;
        const uint32_t empty0 = mapa_u32(smem_u32(&acc_empty[0]), 0);
        uint32_t ab = 0, aph = 0, seq = 0;
        uint64_t acc2[64];                                          // column pairs; 56 (half 0) or 48 (half 1) in use
        TileRing ring;
        ring.init(stage_t, ring_full, ring_empty);
        TlRole tl;
        tl.init(warp == 4 || warp == 8 ? prm.tl : nullptr, warp == 4 ? TL_EPI0 : TL_EPI1);
        WorkIter wi;
        wi.init(cluster_id, n_clusters, prm.n_phi_tiles, prm.n_pairs, prm.gang);
        int tp, j;
        while (wi.next(tp, j)) {
            tl.stamp(0);
#pragma unroll
            for (int i = 0; i < 64; ++i) acc2[i] = 0ull;
            for (int c = 0; c < n_chunks; ++c) {
                tl.begin();
                mbar_wait(&acc_full[ab], aph);
                tl.add(c == 0 ? 4 : 1);
                tc_fence_after();
                const float inv = __uint_as_float((uint32_t)scales[(seq & (T3_SCALES - 1)) * T3_M + q * 32 + lane] << 16);   // 2^-e of this pixel's chunk, times 2^-eB
                const uint64_t inv2 = pack2(inv, inv);
                ++seq;
                const uint32_t tbase = tmem + lane_addr + ab * T3_ACC_COLS + cbase;
                {
                    uint32_t r[64];
                    tmem_ld64(tbase, r);
                    tmem_ld_wait();
                    t3_accumulate<64>(acc2, r, inv2);
                }
                if (!half) {
                    uint32_t r[48];
                    tmem_ld32(tbase + 64, r);
                    tmem_ld16(tbase + 96, r + 32);
                    tmem_ld_wait();
                    t3_accumulate<48>(acc2 + 32, r, inv2);
                } else {
                    uint32_t r[32];
                    tmem_ld32(tbase + 64, r);
                    tmem_ld_wait();
                    t3_accumulate<32>(acc2 + 32, r, inv2);
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive_remote(empty0 + ab * 8);
                if (++ab == 2) { ab = 0; aph ^= 1; }
            }
            tl.stamp(2);
            float acc[128];
#pragma unroll
            for (int i = 0; i < 64; ++i) unpack2(acc2[i], acc[2 * i], acc[2 * i + 1]);
            asm volatile("" : "+r"(tp), "+r"(j));       // keep the tile-end address arithmetic out of the drain loop's live ranges
            const long long P0 = (long long)(2 * tp + (int)rank) * T3_M + q * 32;   // first pixel of this warp
            EpiTile et;
            et.n_pix = prm.n_pix;
            et.P0 = P0;
            et.n_phi = prm.n_phi;
            et.k0 = j * n + (cbase >> 1);
            et.nv = min(min(n, prm.n_phi - j * n) - (cbase >> 1), half ? 48 : 56);
            et.seg = 2 * j + half;
            float* sT = stage_t + (warp - 4) * (32 * 33);
            if (OUT == 2) {
                const int nv_tile = min(n, prm.n_phi - j * n);
                if (prm.rec) epi_tile_phi_major_ring<true>(acc, et, lane, q, half, nv_tile, ring, prm.rec);
                else epi_tile_phi_major_ring<false>(acc, et, lane, q, half, nv_tile, ring, nullptr);
            } else if (OUT == 3) {
                float* sV = stage_t + (warp - 4) * 1024;
                if (prm.rec) epi_tile_phi_major_vec<true>(acc, et, lane, sV, prm.FQ, prm.FU, prm.rec);
                else epi_tile_phi_major_vec<false>(acc, et, lane, sV, prm.FQ, prm.FU, nullptr);
            } else if (prm.rec) {
                if (!OUT_LOS) epi_tile_phi_major<true>(acc, et, lane, prm.FQ, prm.FU, prm.FA, prm.rec);
                else epi_tile_los_major<true>(acc, et, lane, sT, prm.FQ, prm.FU, prm.FA, prm.rec);
            } else {
                if (!OUT_LOS) epi_tile_phi_major<false>(acc, et, lane, prm.FQ, prm.FU, prm.FA, nullptr);
                else epi_tile_los_major<false>(acc, et, lane, sT, prm.FQ, prm.FU, prm.FA, nullptr);
            }
            tl.stamp(3);
            tl.next();
        }
    }
    tc_fence_before();
    cluster_sync_all();
    if (warp == 2) asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, 512;" ::"r"(tmem));
}

// ------------------------------------------------------------------------------------------------
// Host side
#ifdef RMSYNTH_TIMELINE
static long long* g_tl_buf = nullptr;
constexpr size_t kTlCount = (size_t)TL_CTAS * TL_ROLES * TL_ITEMS * TL_SLOTS;
// Debug build only (not part of include/rmsynth.h): copy out the timeline of the last tc3 launch; synchronises.
extern "C" int rmsynth_timeline_read(long long* out, int max_count) {
    if (!g_tl_buf || !out || max_count < (int)kTlCount) return -1;
    if (cudaDeviceSynchronize() != cudaSuccess) return -2;
    if (cudaMemcpy(out, g_tl_buf, kTlCount * sizeof(long long), cudaMemcpyDeviceToHost) != cudaSuccess) return -3;
    return (int)kTlCount;
}
#endif

rmsynth_status tc3_plan_init(rmsynth_plan* p) {
    TcGeom& g = p->tc3;
    g.kb = T3_KC;
    g.n_phi_tiles = (p->n_phi + T3_NMAX - 1) / T3_NMAX;
    const int per = (p->n_phi + g.n_phi_tiles - 1) / g.n_phi_tiles;
    g.n_tile = (per + 7) & ~7;
    const int n_chunks = (p->n_chan + T3_KC - 1) / T3_KC;
    g.k_pad = n_chunks * T3_KC;
    g.ctas = 2;
    // power-of-two scale bringing max |B| = K max(w) into [2^14, 2^15)
    double bmax = 0.0;
    for (int i = 0; i < p->n_chan; ++i) bmax = std::max(bmax, p->K * p->w[i]);
    int eb;
    std::frexp(bmax, &eb);                       // bmax = f 2^eb, f in [0.5, 1)
    p->tc3_eb = 15 - eb;                         // bmax 2^(15 - eb) in [2^14, 2^15)
    const size_t halves = (size_t)g.n_phi_tiles * n_chunks * 2 * 128 * g.n_tile;
    RMS_CUDA(cudaMalloc(&p->d_tcB3, halves * sizeof(__half)));
    dim3 grid((g.n_tile + 63) / 64, n_chunks, g.n_phi_tiles);
    tc3_build_b_kernel<<<grid, 64>>>(p->d_delta, p->d_kw, p->d_phi, p->n_chan, p->n_phi, g.n_tile, n_chunks,
                                     std::ldexp(1.0, p->tc3_eb), reinterpret_cast<__half*>(p->d_tcB3));
    RMS_LAUNCH_CHECK("tc3_build_b_kernel");
#define T3_ATTR(IN, O, BYTES)                                                                                                        \
    RMS_CUDA(cudaFuncSetAttribute(tc3_rmsynth_kernel<IN, O, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, BYTES)); \
    RMS_CUDA(cudaFuncSetAttribute(tc3_rmsynth_kernel<IN, O, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, BYTES))
    T3_ATTR(0, 0, T3Lay<0>::SMEM); T3_ATTR(1, 0, T3Lay<0>::SMEM); T3_ATTR(0, 1, T3Lay<1>::SMEM); T3_ATTR(1, 1, T3Lay<1>::SMEM);
    T3_ATTR(0, 2, T3Lay<2>::SMEM); T3_ATTR(1, 2, T3Lay<2>::SMEM); T3_ATTR(0, 3, T3Lay<3>::SMEM); T3_ATTR(1, 3, T3Lay<3>::SMEM);
#undef T3_ATTR
    return RMSYNTH_OK;
}

rmsynth_status tc3_launch(const rmsynth_plan* p, const void* map_q, const void* map_u, const void* map_fq, const void* map_fu,
                          bool a3d, bool in_freq, bool out_phi, int ring_out, long long n_pix, float* FQ, float* FU, float* FA, float* rec, int* tile_sync, int gang,
                          int sync_lag, cudaStream_t st) {
    Tc3Params prm;
    prm.n_pix = n_pix;
    prm.n_chan = p->n_chan;
    prm.n_phi = p->n_phi;
    prm.n = p->tc3.n_tile;
    prm.n_phi_tiles = p->tc3.n_phi_tiles;
    prm.n_chunks = p->tc3.k_pad / T3_KC;
    const long long pix_tiles = (n_pix + T3_M - 1) / T3_M;
    prm.n_pairs = (int)((pix_tiles + 1) / 2);
    prm.n_items = prm.n_pairs * prm.n_phi_tiles;
    prm.a3d = a3d ? 1 : 0;
    prm.inv_scale_b = (float)std::ldexp(1.0, -p->tc3_eb);
    prm.e_min = 15 + (p->tc3_eb > 0 ? p->tc3_eb : 0);
    prm.blob = reinterpret_cast<const __half*>(p->d_tcB3);
    prm.chan_mask = p->d_chanmask;
    prm.FQ = FQ;
    prm.FU = FU;
    prm.FA = FA;
    prm.rec = rec;
    prm.tile_sync = tile_sync;
    prm.gang = gang;
    prm.sync_lag = sync_lag;
    {
        // one item lasts ~ n_chunks x 1350 cycles (12 MMAs of 104 cycles + overheads); spread the gangs over one item
        const int max_cl = p->sm_count / 2;
        const int S = (max_cl / gang) * gang, n_groups = S / gang + (max_cl - S);
        const char* e = experiment_env("RMSYNTH_STAGGER");     // experiment build only: percent of the default, 0 = off
        const double scale = e ? atof(e) / 100.0 : 1.0;
        prm.stagger = (FQ || FA) && n_groups > 1 ? (int)(scale * prm.n_chunks * 1350.0 / n_groups) : 0;
    }
    prm.tl = nullptr;
#ifdef RMSYNTH_TIMELINE
    if (!g_tl_buf) RMS_CUDA(cudaMalloc(&g_tl_buf, kTlCount * sizeof(long long)));
    RMS_CUDA(cudaMemsetAsync(g_tl_buf, 0, kTlCount * sizeof(long long), st));
    prm.tl = g_tl_buf;
#endif
    const int max_clusters = p->sm_count / 2;
    const int clusters = prm.n_items < max_clusters ? prm.n_items : max_clusters;
    const int grid = 2 * clusters;
    const CUtensorMap& mq = *static_cast<const CUtensorMap*>(map_q);
    const CUtensorMap& mu = *static_cast<const CUtensorMap*>(map_u);
    const int out = !out_phi ? 1 : ring_out == 1 ? 2 : ring_out == 2 ? 3 : 0;
    // output tensor maps are read by the ring variant only; the others get the input maps as placeholders
    const CUtensorMap& mfq = *static_cast<const CUtensorMap*>(out == 2 ? map_fq : map_q);
    const CUtensorMap& mfu = *static_cast<const CUtensorMap*>(out == 2 ? map_fu : map_u);
    const bool tail = p->n_chan % T3_KC != 0 && p->n_chan % T3_KC <= T3_KC / 2;   // the last chunk's second K step is all padding
#define T3_LAUNCH(IN, O)                                                                                   \
    if (tail) tc3_rmsynth_kernel<IN, O, true><<<grid, T3_THREADS, T3Lay<O>::SMEM, st>>>(mq, mu, mfq, mfu, prm); \
    else tc3_rmsynth_kernel<IN, O, false><<<grid, T3_THREADS, T3Lay<O>::SMEM, st>>>(mq, mu, mfq, mfu, prm)
    switch (out * 2 + (in_freq ? 1 : 0)) {
        case 0: T3_LAUNCH(0, 0); break;
        case 1: T3_LAUNCH(1, 0); break;
        case 2: T3_LAUNCH(0, 1); break;
        case 3: T3_LAUNCH(1, 1); break;
        case 4: T3_LAUNCH(0, 2); break;
        case 5: T3_LAUNCH(1, 2); break;
        case 6: T3_LAUNCH(0, 3); break;
        default: T3_LAUNCH(1, 3); break;
    }
#undef T3_LAUNCH
    RMS_LAUNCH_CHECK("tc3_rmsynth_kernel");
    return RMSYNTH_OK;
}

}  // namespace rms
