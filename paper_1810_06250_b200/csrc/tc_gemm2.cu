// Rows a4-a6, a8, CTA-pair version: the same 3xTF32 contraction as tc_gemm.cu with
// tcgen05.mma.cta_group::2 (UMMA M = 256 = two 128-pixel tiles, one per SM of the pair).
//
// Why: with one CTA per tile the shared-memory port is the limit, not the tensor pipe.  Per 8-channel
// stage (768 MMA cycles at N=256) a lone CTA moves 72 KB of MMA operand reads + 32 KB of TMA writes +
// 16 KB of A_lo traffic = 120 KB through a 128 B/cycle port (~940 cycles).  In a pair each SM supplies
// only half of the B rows: [Bc|-Bs] splits into Bc (rank 0) and -Bs (rank 1), [Bs|Bc] into Bs and Bc,
// so a CTA stages 2 blocks instead of 3, reads 8 KB instead of 12 KB per MMA, and the ring gets 7 stages
// of 32 KB instead of 5 of 40 KB.
//
// Protocol (S-stage ring, per CTA unless noted; rank 0 = leader issues every MMA):
//   full[s]      own TMA bytes landed                         (1 arrival + tx)
//   ready[s]     LEADER's: A_lo written in BOTH CTAs          (4 local + 4 remote warp arrivals)
//   empty[s]     stage consumed, in both CTAs                 (tcgen05.commit ... multicast::cluster)
//   acc_full[b]  32-channel chunk accumulated, both CTAs      (multicast commit)
//   acc_empty[b] LEADER's: chunk drained by BOTH epilogues    (8 local + 8 remote warp arrivals)
// Remote arrivals use mbarrier.arrive.shared::cluster with default semantics, as NVIDIA's 2-SM kernels do;
// a .release.cluster arrival was measured at ~1000 cycles each and starved the MMA thread (50 % idle).
#include "common.cuh"
#include "tc_common.cuh"
#include "tc_epilogue.cuh"

namespace rms {

constexpr int T2_M = 128;                       // pixels per CTA (UMMA M = 256 per pair)
constexpr int T2_NMAX = 128;
constexpr int T2_KS = 8;
constexpr int T2_ROW = T2_KS * 4;               // 32-byte K-major rows (SWIZZLE_32B)
constexpr int T2_APART = T2_M * T2_ROW;         // 4 KB: one of Qraw, Uraw, Qlo, Ulo
constexpr int T2_BPART_MAX = 2 * T2_NMAX * T2_ROW;   // 8 KB: [slot0; slot1] of one split part
constexpr int T2_STAGE = 4 * T2_APART + 2 * T2_BPART_MAX;   // 32 KB
constexpr int T2_STAGES_PHI = 7, T2_STAGES_LOS = 6;
constexpr int T2_SMEM = T2_STAGES_PHI * T2_STAGE + 2048;
constexpr int T2_THREADS = 512;
constexpr int T2_CHUNK_STAGES = 8;              // 64 channels per accumulator drain

// Plan time (a2): per (depth tile j, stage s, CTA rank): [part hi|lo][slot0 | slot1][row < n][8 channels].
// slot0 feeds the Q MMAs, slot1 the U MMAs; each rank holds n of the 2n accumulator columns.  Column order
// (tc_epilogue.cuh): depth d of the tile -> FQ column cq = (d/8)*16 + d%8, FU column cu = cq + 8, and
//   FQ = Q.Bc + U.Bs,  FU = U.Bc - Q.Bs   =>   slot0[cq] = Bc, slot0[cu] = -Bs, slot1[cq] = Bs, slot1[cu] = Bc
// Values are formed in FP64 (sincos of the FP64 phase) and split hi/lo at TF32 precision.
__global__ void tc2_build_b_kernel(const double* __restrict__ delta, const double* __restrict__ kw,
                                   const double* __restrict__ phi, int n_chan, int n_phi, int n, int n_stages,
                                   float* __restrict__ blob) {
    const int d = blockIdx.x * blockDim.x + threadIdx.x;   // depth within the tile
    const int s = blockIdx.y, j = blockIdx.z;
    if (d >= n) return;
    const int k_phi = j * n + d;
    const size_t part = (size_t)2 * n * T2_KS;            // floats per split part
    float* base = blob + ((size_t)j * n_stages + s) * 2 * 2 * part;   // [rank][part][slot][row][8]
    const int cq = (d >> 3) * 16 + (d & 7), cu = cq + 8;
    for (int k = 0; k < T2_KS; ++k) {
        const int i = s * T2_KS + k;
        double c = 0.0, sn = 0.0;
        if (i < n_chan && k_phi < n_phi) {
            sincos(2.0 * phi[k_phi] * delta[i], &sn, &c);
            c *= kw[i];
            sn *= kw[i];
        }
        const float chi = rn_tf32((float)c), shi = rn_tf32((float)sn);
        const float clo = rn_tf32((float)(c - (double)chi)), slo = rn_tf32((float)(sn - (double)shi));
        auto put = [&](int col, int slot, float hi, float lo) {
            const int rank = col >= n, row = col - rank * n + slot * n;
            // SWIZZLE_32B K-major: 16-byte chunk index ^= bit 2 of the row
            const size_t off = ((size_t)row * T2_ROW + (((k / 4) ^ ((row >> 2) & 1)) * 16) + (k % 4) * 4) / 4;
            float* b = base + (size_t)rank * 2 * part;
            b[off] = hi;
            b[part + off] = lo;
        };
        put(cq, 0, chi, clo);
        put(cu, 0, -shi, -slo);
        put(cq, 1, shi, slo);
        put(cu, 1, chi, clo);
    }
}

struct Tc2Params {
    long long n_pix;
    int n_chan, n_phi, n, n_phi_tiles, n_stages, n_items, n_pairs, a3d;
    const float* blob;
    float* FQ;           // may be NULL (maps only)
    float* FU;
    float* FA;           // |F| cube (Eq. 17), may be NULL
    float* rec;          // peak-segment records (tc_epilogue.cuh), NULL = no peak search
    int* tile_sync;      // [pixel-tile pairs] check-in counters (gang_checkin), NULL = off
    int gang;                     // gang size G of the work schedule (tc_common.cuh: WorkIter)
    int sync_lag;        // gang members may drift this many work items apart
    const uint32_t* chan_mask;   // per 32 channels: bit i set = channel exists and has w > 0
};

template <int IN_MN, int OUT_LOS>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(T2_THREADS, 1)
tc2_rmsynth_kernel(const __grid_constant__ CUtensorMap mapQ, const __grid_constant__ CUtensorMap mapU, const Tc2Params prm) {
    constexpr int S = OUT_LOS ? T2_STAGES_LOS : T2_STAGES_PHI;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t* smem_gen = smem_raw + (smem_base - smem_u32(smem_raw));
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem_gen + (size_t)S * T2_STAGE);
    uint64_t* full = bars;
    uint64_t* ready = bars + S;
    uint64_t* empty = bars + 2 * S;
    uint64_t* acc_full = bars + 3 * S;
    uint64_t* acc_empty = acc_full + 2;
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(acc_empty + 2);
    float* stage_t = reinterpret_cast<float*>(smem_gen + (size_t)S * T2_STAGE + 1024);   // LOS-major transpose buffers

    // warp index through a shuffle: provably warp-uniform, so role branches are uniform and MMA operands stay in uniform registers
    const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0), lane = threadIdx.x & 31;
    const uint32_t rank = cluster_ctarank();
    const int cluster_id = blockIdx.x >> 1, n_clusters = gridDim.x >> 1;
    const int n = prm.n, N2 = 2 * prm.n;
    const uint32_t b_part_bytes = 2u * n * T2_ROW;
    const uint32_t stage_tx = 2u * T2_APART + 2u * b_part_bytes;
    const int n_chunks = (prm.n_stages + T2_CHUNK_STAGES - 1) / T2_CHUNK_STAGES;

    if (threadIdx.x == 0) {
        for (int s = 0; s < S; ++s) { mbar_init(&full[s], 1); mbar_init(&ready[s], 8); mbar_init(&empty[s], 1); }
        for (int b = 0; b < 2; ++b) { mbar_init(&acc_full[b], 1); mbar_init(&acc_empty[b], 16); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 2) {
        asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(tmem_slot)));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;");
    }
    tc_fence_before();
    cluster_sync_all();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;

    if (warp < 4) {
      asm volatile("setmaxnreg.dec.sync.aligned.u32 56;");
      if (warp == 0) {
        // ===================== TMA producer (both CTAs) =====================
        if (lane == 0) {
            const uint64_t pol = l2_policy_evict_last();
            uint32_t st = 0, ph = 0;
            WorkIter wi;
            wi.init(cluster_id, n_clusters, prm.n_phi_tiles, prm.n_pairs, prm.gang);
            int tp, j;
            while (wi.next(tp, j)) {
                const int pix0 = (2 * tp + (int)rank) * T2_M;       // may lie past n_pix: TMA zero-fills
                gang_checkin(prm.tile_sync, wi, tp, prm.sync_lag, 2 * prm.gang);
                const uint8_t* bsrc = reinterpret_cast<const uint8_t*>(prm.blob) +
                                      ((size_t)j * prm.n_stages * 2 + rank) * 2 * b_part_bytes;
                for (int s = 0; s < prm.n_stages; ++s) {
                    mbar_wait(&empty[st], ph ^ 1);
                    mbar_expect_tx(&full[st], stage_tx);
                    const uint32_t sb = smem_base + st * T2_STAGE;
                    if (IN_MN) {
                        if (prm.a3d) {
                            tma_load_3d(sb, &mapQ, 0, s * T2_KS, pix0 / 32, &full[st], pol);
                            tma_load_3d(sb + T2_APART, &mapU, 0, s * T2_KS, pix0 / 32, &full[st], pol);
                        } else {
#pragma unroll
                            for (int g = 0; g < 4; ++g) {
                                tma_load_2d(sb + g * (T2_KS * 128), &mapQ, pix0 + 32 * g, s * T2_KS, &full[st], pol);
                                tma_load_2d(sb + T2_APART + g * (T2_KS * 128), &mapU, pix0 + 32 * g, s * T2_KS, &full[st], pol);
                            }
                        }
                    } else {
                        tma_load_2d(sb, &mapQ, s * T2_KS, pix0, &full[st], pol);
                        tma_load_2d(sb + T2_APART, &mapU, s * T2_KS, pix0, &full[st], pol);
                    }
                    bulk_load(sb + 4 * T2_APART, bsrc + (size_t)s * 4 * b_part_bytes, 2 * b_part_bytes, &full[st], pol);
                    if (++st == S) { st = 0; ph ^= 1; }
                }
            }
        }
        __syncwarp();
      } else if (warp == 1) {
        // ===================== MMA issuer (leader CTA only) =====================
        if (rank == 0) {
            uint32_t lead;                                       // one elected lane issues; the whole warp runs the loop
            asm volatile("{\n.reg .pred p;\nelect.sync _|p, 0xffffffff;\nselp.u32 %0, 1, 0, p;\n}" : "=r"(lead));
            const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)IN_MN << 15) |
                                   ((uint32_t)(N2 >> 3) << 17) | ((uint32_t)(256 >> 4) << 24);
            uint32_t st = 0, ph = 0, ab = 0, aph = 0;
            WorkIter wi;
            wi.init(cluster_id, n_clusters, prm.n_phi_tiles, prm.n_pairs, prm.gang);
            int tp, j;
            while (wi.next(tp, j))
                for (int c = 0; c < n_chunks; ++c) {
                    mbar_wait(&acc_empty[ab], aph ^ 1);
                    tc_fence_after();
                    const uint32_t d_tmem = tmem + ab * 256;
                    const int s_end = min(prm.n_stages, (c + 1) * T2_CHUNK_STAGES);
                    uint32_t first = 1;
                    for (int s = c * T2_CHUNK_STAGES; s < s_end; ++s) {
                        mbar_wait(&ready[st], ph);
                        tc_fence_after();
                        const uint32_t sb = smem_base + st * T2_STAGE;
                        const uint32_t aQ = sb, aU = sb + T2_APART, aQl = sb + 2 * T2_APART, aUl = sb + 3 * T2_APART;
                        const uint32_t bh = sb + 4 * T2_APART, bl = bh + b_part_bytes;
                        const uint32_t s1 = n * T2_ROW;    // slot1 offset
                        auto adesc = [&](uint32_t a) {
                            return IN_MN ? make_desc(a, T2_KS * 128, 512, 1u) : make_desc(a, 16, 8 * T2_ROW, 6u);
                        };
                        auto bdesc = [&](uint32_t b) { return make_desc(b, 16, 8 * T2_ROW, 6u); };
                        if (lead) {
                            umma2_tf32(d_tmem, adesc(aQ), bdesc(bh), idesc, first ^ 1u);    // Q_hi [Bc|-Bs]_hi
                            umma2_tf32(d_tmem, adesc(aQl), bdesc(bh), idesc, 1u);           // Q_lo [Bc|-Bs]_hi
                            umma2_tf32(d_tmem, adesc(aQ), bdesc(bl), idesc, 1u);            // Q_hi [Bc|-Bs]_lo
                            umma2_tf32(d_tmem, adesc(aU), bdesc(bh + s1), idesc, 1u);       // U_hi [Bs|Bc]_hi
                            umma2_tf32(d_tmem, adesc(aUl), bdesc(bh + s1), idesc, 1u);      // U_lo [Bs|Bc]_hi
                            umma2_tf32(d_tmem, adesc(aU), bdesc(bl + s1), idesc, 1u);       // U_hi [Bs|Bc]_lo
                            umma2_commit_mc(&empty[st]);
                        }
                        __syncwarp();
                        first = 0;
                        if (++st == S) { st = 0; ph ^= 1; }
                    }
                    if (lead) umma2_commit_mc(&acc_full[ab]);
                    __syncwarp();
                    if (++ab == 2) { ab = 0; aph ^= 1; }
                }
        }
        __syncwarp();
      }
    } else if (warp < 8) {
        // ===================== A_lo transform (both CTAs); signals the LEADER's ready barrier =====================
        asm volatile("setmaxnreg.dec.sync.aligned.u32 56;");
        const int tt = threadIdx.x - 128;
        uint32_t st = 0, ph = 0;
        long long total = 0;                                 // stages this cluster will see = its work items x n_stages
        {
            WorkIter wi;
            wi.init(cluster_id, n_clusters, prm.n_phi_tiles, prm.n_pairs, prm.gang);
            int tp, j;
            while (wi.next(tp, j)) total += prm.n_stages;
        }
        int stage = 0;                                       // 8-channel stage within the work item
        for (long long it = 0; it < total; ++it) {
            mbar_wait(&full[st], ph);
            uint8_t* sg = smem_gen + (size_t)st * T2_STAGE;
            // reading A13: zero-weight channels are removed -- their samples (NaN-blanked planes included) become zeros
            // in the raw tile (= A_hi) and in A_lo.  Warp-uniform: stages without a flagged channel skip all of it.
            const uint32_t m8 = (__ldg(prm.chan_mask + (stage >> 2)) >> ((stage & 3) * 8)) & 0xFFu;
            if (++stage == prm.n_stages) stage = 0;
#pragma unroll
            for (int v = 0; v < 2 * T2_APART / 16 / 128; ++v) {
                const int o = (v * 128 + tt) * 16;
                float4 a = *reinterpret_cast<const float4*>(sg + o);
                if (m8 != 0xFFu) {
                    const int oo = o & (T2_APART - 1);           // offset inside the Q or the U part
                    if (IN_MN) {                                 // [pixel group][channel][32 pixels]: a unit belongs to one channel
                        if (!((m8 >> ((oo >> 7) & 7)) & 1u)) a = make_float4(0.f, 0.f, 0.f, 0.f);
                    } else {                                     // [pixel][8 channels], SWIZZLE_32B: unit j' holds channels 4 (j' ^ bit 2 of the row) ..
                        const int c0 = ((((oo >> 4) & 1) ^ ((oo >> 7) & 1)) << 2);
                        if (!((m8 >> c0) & 1u)) a.x = 0.f;
                        if (!((m8 >> (c0 + 1)) & 1u)) a.y = 0.f;
                        if (!((m8 >> (c0 + 2)) & 1u)) a.z = 0.f;
                        if (!((m8 >> (c0 + 3)) & 1u)) a.w = 0.f;
                    }
                    *reinterpret_cast<float4*>(sg + o) = a;
                }
                float4 l;
                auto lo = [](float x) {
                    float h = __uint_as_float(__float_as_uint(x) & 0xFFFFE000u);
                    return __uint_as_float(__float_as_uint(x - h) + 0x1000u);
                };
                l.x = lo(a.x); l.y = lo(a.y); l.z = lo(a.z); l.w = lo(a.w);
                *reinterpret_cast<float4*>(sg + 2 * T2_APART + o) = l;
            }
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            __syncwarp();                                   // one (remote) arrival per warp, not per thread
            if (lane == 0) mbar_arrive_remote(mapa_u32(smem_u32(&ready[st]), 0));
            if (++st == S) { st = 0; ph ^= 1; }
        }
    } else {
        // ===================== epilogue (both CTAs, own TMEM lanes = own 128 pixels) =====================
        asm volatile("setmaxnreg.inc.sync.aligned.u32 200;");
        const int q = warp & 3;
        const int cbase = warp >= 12 ? 128 : 0;
        const uint32_t lane_addr = (uint32_t)(q * 32) << 16;
        uint32_t ab = 0, aph = 0;
        float acc[128];
        WorkIter wi;
        wi.init(cluster_id, n_clusters, prm.n_phi_tiles, prm.n_pairs, prm.gang);
        int tp, j;
        while (wi.next(tp, j)) {
            const long long P0 = (long long)(2 * tp + (int)rank) * T2_M + q * 32;   // first pixel of this warp
            for (int c = 0; c < n_chunks; ++c) {
                mbar_wait(&acc_full[ab], aph);
                tc_fence_after();
#pragma unroll
                for (int g = 0; g < 4; ++g) {
                    if (cbase + g * 32 < N2) {
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
                if (lane == 0) mbar_arrive_remote(mapa_u32(smem_u32(&acc_empty[ab]), 0));
                if (++ab == 2) { ab = 0; aph ^= 1; }
            }
            EpiTile et;
            et.n_pix = prm.n_pix;
            et.P0 = P0;
            et.n_phi = prm.n_phi;
            et.k0 = j * n + (cbase >> 1);
            et.nv = min(n, prm.n_phi - j * n) - (cbase >> 1);
            et.seg = 2 * j + (cbase >> 7);
            float* sT = stage_t + (warp - 8) * (32 * 33);
            if (prm.rec) {
                if (!OUT_LOS) epi_tile_phi_major<true>(acc, et, lane, prm.FQ, prm.FU, prm.FA, prm.rec);
                else epi_tile_los_major<true>(acc, et, lane, sT, prm.FQ, prm.FU, prm.FA, prm.rec);
            } else {
                if (!OUT_LOS) epi_tile_phi_major<false>(acc, et, lane, prm.FQ, prm.FU, prm.FA, nullptr);
                else epi_tile_los_major<false>(acc, et, lane, sT, prm.FQ, prm.FU, prm.FA, nullptr);
            }
        }
    }
    tc_fence_before();
    cluster_sync_all();
    if (warp == 2) asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, 512;" ::"r"(tmem));
}

// ------------------------------------------------------------------------------------------------
rmsynth_status tc2_plan_init(rmsynth_plan* p) {
    const TcGeom& g = p->tc;
    const int n_stages = g.k_pad / T2_KS;
    size_t floats = (size_t)g.n_phi_tiles * n_stages * 2 * 2 * 2 * g.n_tile * T2_KS;
    RMS_CUDA(cudaMalloc(&p->d_tcB2, floats * sizeof(float)));
    dim3 grid((g.n_tile + 63) / 64, n_stages, g.n_phi_tiles);
    tc2_build_b_kernel<<<grid, 64>>>(p->d_delta, p->d_kw, p->d_phi, p->n_chan, p->n_phi, g.n_tile, n_stages, p->d_tcB2);
    RMS_LAUNCH_CHECK("tc2_build_b_kernel");
    RMS_CUDA(cudaFuncSetAttribute(tc2_rmsynth_kernel<0, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, T2_SMEM));
    RMS_CUDA(cudaFuncSetAttribute(tc2_rmsynth_kernel<1, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, T2_SMEM));
    RMS_CUDA(cudaFuncSetAttribute(tc2_rmsynth_kernel<0, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, T2_SMEM));
    RMS_CUDA(cudaFuncSetAttribute(tc2_rmsynth_kernel<1, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, T2_SMEM));
    return RMSYNTH_OK;
}

rmsynth_status tc2_launch(const rmsynth_plan* p, const void* map_q, const void* map_u, bool a3d, bool in_freq,
                          bool out_phi, long long n_pix, float* FQ, float* FU, float* FA, float* rec, int* tile_sync,
                          int gang, int sync_lag, cudaStream_t st) {
    Tc2Params prm;
    prm.n_pix = n_pix;
    prm.n_chan = p->n_chan;
    prm.n_phi = p->n_phi;
    prm.n = p->tc.n_tile;
    prm.n_phi_tiles = p->tc.n_phi_tiles;
    prm.n_stages = p->tc.k_pad / T2_KS;
    const long long pix_tiles = (n_pix + T2_M - 1) / T2_M;
    prm.n_pairs = (int)((pix_tiles + 1) / 2);
    prm.n_items = prm.n_pairs * prm.n_phi_tiles;
    prm.a3d = a3d ? 1 : 0;
    prm.blob = p->d_tcB2;
    prm.FQ = FQ;
    prm.FU = FU;
    prm.FA = FA;
    prm.rec = rec;
    prm.tile_sync = tile_sync;
    prm.gang = gang;
    prm.sync_lag = sync_lag;
    prm.chan_mask = p->d_chanmask;
    const int max_clusters = p->sm_count / 2;
    const int clusters = prm.n_items < max_clusters ? prm.n_items : max_clusters;
    const int grid = 2 * clusters;
    const CUtensorMap& mq = *static_cast<const CUtensorMap*>(map_q);
    const CUtensorMap& mu = *static_cast<const CUtensorMap*>(map_u);
    if (in_freq && out_phi) tc2_rmsynth_kernel<1, 0><<<grid, T2_THREADS, T2_SMEM, st>>>(mq, mu, prm);
    else if (in_freq) tc2_rmsynth_kernel<1, 1><<<grid, T2_THREADS, T2_SMEM, st>>>(mq, mu, prm);
    else if (out_phi) tc2_rmsynth_kernel<0, 0><<<grid, T2_THREADS, T2_SMEM, st>>>(mq, mu, prm);
    else tc2_rmsynth_kernel<0, 1><<<grid, T2_THREADS, T2_SMEM, st>>>(mq, mu, prm);
    RMS_LAUNCH_CHECK("tc2_rmsynth_kernel");
    return RMSYNTH_OK;
}

}  // namespace rms
