// Epilogue of the tensor-core kernels (rows a6, a7): what an epilogue warp does with its 128 drained
// accumulator columns of one (pixel tile, depth tile) work item.
//
// Column order of the accumulator tile (fixed at plan time by the B-operand builders): depths are
// interleaved in groups of eight,  [FQ d0..d7 | FU d0..d7 | FQ d8..d15 | FU d8..d15 | ...],  so a thread
// (= one pixel) holds FQ and FU of the same depth in registers i and i+8 and can form |F|^2 (Eq. 17,
// P:L134) for the fused peak search without exchanging data with another warp.
// Warps 8-11 of a CTA own columns [0,128) = local depths [0,64), warps 12-15 own [128,256) = [64,128).
#pragma once
#include "peak_refine.cuh"
#include "tc_common.cuh"

namespace rms {

// Per-(pixel, segment) record of the fused peak search; a segment = the <= 64 depths one epilogue warp
// sees of one work item (segment index = 2 * depth tile + warp half).  Stored field-major:
//   rec[(seg * kPeakFields + field) * n_pix + p]
// peaks_combine_kernel (peaks.cu) merges the segments of a pixel in ascending depth order.
constexpr int kPeakFields = 8;   // best_y2, best_k, best_q, best_u, ym2, yp2, first_y2, last_y2

struct EpiTile {
    long long n_pix;     // lines of sight in the cube
    long long P0;        // first pixel of this warp (lane l owns pixel P0 + l)
    int n_phi;           // depths in the cube
    int k0;              // first global depth of this warp's columns (depth tile start + 0 or 64)
    int nv;              // valid local depths of this warp: element (g, e) is real iff g*8+e < nv
    int seg;             // segment index for the peak records
};

// ---- fused peak search (a7) -------------------------------------------------------------------------------
// Branch-free streaming arg-max over one thread's depths, same decisions as PeakState::push (strict >, lowest
// index on ties, neighbours of the best sample tracked).  A warp's 64 depths are scanned as two independent
// chains (depth groups 0-3 and 4-7) so that consecutive steps are not one long dependency chain.
struct ScanChain {
    float best, ym2, yp2, q, u, prev, first, nf;
    int k;          // local depth index of the best sample
    bool wn;        // the next sample is the right-hand neighbour of the best
    __device__ __forceinline__ void init() { best = ym2 = yp2 = prev = first = -1.f; q = u = nf = 0.f; k = 0; wn = false; }
    __device__ __forceinline__ void step(int kl, float qq, float uu) {
        const float y2 = fmaf(qq, qq, uu * uu);
        nf = fmaf(y2, 0.f, nf);              // sticky NaN once |F|^2 is not finite (reading A17)
        yp2 = wn ? y2 : yp2;
        const bool gt = y2 > best;
        best = gt ? y2 : best;
        k = gt ? kl : k;
        q = gt ? qq : q;
        u = gt ? uu : u;
        ym2 = gt ? prev : ym2;
        yp2 = gt ? -1.f : yp2;
        wn = gt;
        prev = y2;
    }
};

struct SegScan {
    ScanChain a, b;
    __device__ __forceinline__ void init() { a.init(); b.init(); }
    // depth group g (eight depths) of this warp's columns; call with g = 0..7 in ascending order
    __device__ __forceinline__ void group(const float (&acc)[128], int g, int nv) {
        ScanChain& c = g < 4 ? a : b;
        if (g * 8 + 8 <= nv) {               // warp-uniform: a full group needs no per-sample bound check
#pragma unroll
            for (int e = 0; e < 8; ++e) {
                c.step(g * 8 + e, acc[g * 16 + e], acc[g * 16 + 8 + e]);
                if ((g & 3) == 0 && e == 0) c.first = c.prev;
            }
        } else if (g * 8 < nv) {             // the ragged group of the cube's last depth tile
#pragma unroll
            for (int e = 0; e < 8; ++e) {
                if (g * 8 + e < nv) {
                    c.step(g * 8 + e, acc[g * 16 + e], acc[g * 16 + 8 + e]);
                    if ((g & 3) == 0 && e == 0) c.first = c.prev;
                }
            }
        }
    }
    // merge the two chains and write the segment record
    __device__ __forceinline__ void finish(const EpiTile& t, int lane, float* __restrict__ rec) {
        const bool b_any = b.first != -1.f;          // chain b saw at least one sample
        if (b_any && a.yp2 == -1.f) a.yp2 = b.first;  // a's best was its last sample
        if (b_any && b.best > a.best) {
            a.best = b.best; a.k = b.k; a.q = b.q; a.u = b.u;
            a.ym2 = b.ym2 == -1.f ? a.prev : b.ym2;  // b's best was its first sample
            a.yp2 = b.yp2;
        }
        const float last = b_any ? b.prev : a.prev;
        const long long p = t.P0 + lane;
        if (p >= t.n_pix) return;
        float* r = rec + (long long)t.seg * kPeakFields * t.n_pix + p;
        r[0 * t.n_pix] = a.best + (a.nf + b.nf);     // NaN marks a segment that saw a non-finite |F|^2
        r[1 * t.n_pix] = __int_as_float(t.k0 + a.k);
        r[2 * t.n_pix] = a.q;
        r[3 * t.n_pix] = a.u;
        r[4 * t.n_pix] = a.ym2;
        r[5 * t.n_pix] = a.yp2;
        r[6 * t.n_pix] = a.first;                    // -1 marks an empty segment (a real |F|^2 is >= 0 or NaN)
        r[7 * t.n_pix] = last;
    }
};

// ---- output stores (a6) and the tile-end driver ---------------------------------------------------------
// phi-major cubes F[k*n_pix + p]: a warp writes 128 contiguous bytes per depth.  Bounds are warp-uniform per
// group of eight depths; inside a group the stores are predicated with compile-time offsets (no branches).
// The peak scan of group g is issued right after the stores of group g so that its arithmetic overlaps the
// store queue draining (the stores of a tile are a burst of ~100 KB per CTA).
template <bool WITH_SCAN>
__device__ __forceinline__ void epi_tile_phi_major(const float (&acc)[128], const EpiTile& t, int lane,
                                                   float* __restrict__ FQ, float* __restrict__ FU,
                                                   float* __restrict__ FA, float* __restrict__ rec) {
    const long long p = t.P0 + lane;
    const bool in = p < t.n_pix;
    const long long sb = 4LL * t.n_pix;   // byte stride between depths
    unsigned long long aq = (unsigned long long)(FQ + (long long)t.k0 * t.n_pix + p);
    unsigned long long au = (unsigned long long)(FU + (long long)t.k0 * t.n_pix + p);
    unsigned long long aa = (unsigned long long)(FA + (long long)t.k0 * t.n_pix + p);
    asm volatile("" : "+l"(aq), "+l"(au), "+l"(aa));   // keep the bases in registers (no rematerialisation)
    const uint64_t pol = l2_policy_evict_first();
    SegScan sc;
    if (WITH_SCAN) sc.init();
#pragma unroll
    for (int g = 0; g < 8; ++g) {
        if (g * 8 < t.nv) {                  // warp-uniform
            if (FQ) {
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    st_global_pred(aq + (g * 8 + e) * sb, acc[g * 16 + e], in && g * 8 + e < t.nv, pol);
                    st_global_pred(au + (g * 8 + e) * sb, acc[g * 16 + 8 + e], in && g * 8 + e < t.nv, pol);
                }
            }
            if (FA) {
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    const float q = acc[g * 16 + e], u = acc[g * 16 + 8 + e];
                    st_global_pred(aa + (g * 8 + e) * sb, sqrtf(fmaf(q, q, u * u)), in && g * 8 + e < t.nv, pol);
                }
            }
            if (WITH_SCAN) sc.group(acc, g, t.nv);
        }
    }
    if (WITH_SCAN) sc.finish(t, lane, rec);
}

// LOS-major cubes F[p*n_phi + k]: 32x32 blocks go through a private [32][33] smem buffer so that one store
// instruction writes, for ONE pixel row, 16 consecutive depths of FQ (lanes 0-15) and of FU (lanes 16-31):
// two contiguous 64-byte segments.  FA (|F| cube, may be NULL) is written by the same pass.
template <bool WITH_SCAN>
__device__ __forceinline__ void epi_tile_los_major(const float (&acc)[128], const EpiTile& t, int lane, float* sT,
                                                   float* __restrict__ FQ, float* __restrict__ FU,
                                                   float* __restrict__ FA, float* __restrict__ rec) {
    const int rows = (int)max(0LL, min(32LL, t.n_pix - t.P0));   // ragged last tile
    const long long rb = 4LL * t.n_phi;                           // byte stride between pixel rows
    const int e16 = lane & 15;                                    // depth within the block this lane stores
    const bool is_u = lane >= 16;
    const int src = (e16 >> 3) * 16 + (e16 & 7) + (is_u ? 8 : 0); // its column inside the 32-column block
    const uint64_t pol = l2_policy_evict_first();
    SegScan sc;
    if (WITH_SCAN) sc.init();
#pragma unroll
    for (int b = 0; b < 4; ++b) {                                 // 32 columns = 16 depths of FQ and FU
        if (b * 16 < t.nv) {                                      // warp-uniform
            const bool ok = b * 16 + e16 < t.nv;
            if (FQ) {
#pragma unroll
                for (int c = 0; c < 32; ++c) sT[lane * 33 + c] = acc[b * 32 + c];
                __syncwarp();
                unsigned long long a = (unsigned long long)((is_u ? FU : FQ) + t.P0 * t.n_phi + t.k0 + b * 16 + e16);
#pragma unroll 8
                for (int r = 0; r < 32; ++r) st_global_pred(a + r * rb, sT[r * 33 + src], ok && r < rows, pol);
                __syncwarp();
            }
            if (FA) {   // |F|: 16 depths per block -> lanes 0-15 store rows r, lanes 16-31 rows r+16
#pragma unroll
                for (int c = 0; c < 16; ++c) {
                    const float q = acc[b * 32 + (c >> 3) * 16 + (c & 7)], u = acc[b * 32 + (c >> 3) * 16 + 8 + (c & 7)];
                    sT[lane * 33 + c] = sqrtf(fmaf(q, q, u * u));
                }
                __syncwarp();
                unsigned long long a = (unsigned long long)(FA + t.P0 * t.n_phi + t.k0 + b * 16 + e16);
#pragma unroll 8
                for (int r = 0; r < 16; ++r) {
                    const int rr = r + (is_u ? 16 : 0);
                    st_global_pred(a + rr * rb, sT[rr * 33 + e16], ok && rr < rows, pol);
                }
                __syncwarp();
            }
            if (WITH_SCAN) { sc.group(acc, 2 * b, t.nv); sc.group(acc, 2 * b + 1, t.nv); }
        }
    }
    if (WITH_SCAN) sc.finish(t, lane, rec);
}

// ---- light peak search + TMA tile stores: the tile end of the FP16 kernel when cubes are written ----------------
// When the cubes go to memory anyway, the peak search only has to find (max |F|^2, k) per segment: the values at
// k*, k* - 1, k* + 1 are read back from the cubes by peaks_gather_kernel (peaks.cu), 24 bytes per pixel, instead of
// being tracked through eight selects per depth.  A group of eight depths costs 8 FFMA (|F|^2), 8 FFMA (non-finite
// flag) and a 7-match tournament (strict >, the left = lower depth wins ties), i.e. ~5 instructions per depth.
struct LightScan {
    float best, nf;
    int k;
    __device__ __forceinline__ void init() { best = -1.f; nf = 0.f; k = 0; }
    __device__ __forceinline__ void group(const float (&acc)[128], int g, int nv) {
        float y[8];
#pragma unroll
        for (int e = 0; e < 8; ++e) {
            const float q = acc[g * 16 + e], u = acc[g * 16 + 8 + e];
            const float v = fmaf(q, q, u * u);
            const bool ok = g * 8 + e < nv;                  // all true except in the cube's last, ragged group
            y[e] = ok ? v : -2.f;
            nf = fmaf(ok ? v : 0.f, 0.f, nf);
        }
        int i01 = y[1] > y[0], i23 = y[3] > y[2], i45 = y[5] > y[4], i67 = y[7] > y[6];
        const float m01 = i01 ? y[1] : y[0], m23 = i23 ? y[3] : y[2], m45 = i45 ? y[5] : y[4], m67 = i67 ? y[7] : y[6];
        const bool r03 = m23 > m01, r47 = m67 > m45;
        const float m03 = r03 ? m23 : m01, m47 = r47 ? m67 : m45;
        const int i03 = r03 ? 2 + i23 : i01, i47 = r47 ? 6 + i67 : 4 + i45;
        const bool r07 = m47 > m03;
        const float m = r07 ? m47 : m03;
        const int i = r07 ? i47 : i03;
        const bool gt = m > best;
        best = gt ? m : best;
        k = gt ? g * 8 + i : k;
    }
    __device__ __forceinline__ void finish(const EpiTile& t, int lane, float* __restrict__ rec) {
        const long long p = t.P0 + lane;
        if (p >= t.n_pix) return;
        float* r = rec + (long long)t.seg * kPeakFields * t.n_pix + p;
        r[0 * t.n_pix] = best + nf;                          // NaN marks a segment that saw a non-finite |F|^2
        r[1 * t.n_pix] = __int_as_float(t.k0 + k);
    }
};

// phi-major cubes, vectorised: with one pixel per lane a store instruction moves 4 bytes per lane and needs its own
// 64-bit address (208 stores and ~450 address instructions per thread and tile).  Here each warp turns a group of
// eight depths x 32 pixels of FQ and FU around in its own slice of shared memory ([FQ|FU][8 depths][32 pixels],
// double-buffered, only __syncwarp between the phases) so that lane l holds two consecutive pixels of depths
// l/16 + {0, 2, 4, 6}: one st.global.cs.v2 writes two full 128-byte lines per warp.  Per group 16 STS + 8 LDS.64 +
// 8 STG.64.  (Four pixels per lane would halve that again, but 128-bit register quads next to the 64-register TMEM
// loads and the accumulator pairs make ptxas spill seven accumulator pairs in the drain loop.)
// Needs n_pix % 2 == 0 and 8-byte aligned cubes (else the scalar path above).  sbuf: this warp's 2 x 512 floats.
template <bool WITH_SCAN>
__device__ __forceinline__ void epi_tile_phi_major_vec(const float (&acc)[128], const EpiTile& t, int lane, float* sbuf,
                                                       float* __restrict__ FQ, float* __restrict__ FU,
                                                       float* __restrict__ rec) {
    const int dl = lane >> 4, px = (lane & 15) * 2;             // this lane stores depths dl + {0,2,4,6} of a group, pixels px, px+1
    const bool pin = t.P0 + px < t.n_pix;                        // n_pix % 2 == 0: both pixels in range or none
    const long long row0 = (long long)(t.k0 + dl) * t.n_pix + t.P0 + px;
    float* gq = FQ + row0;
    float* gu = FU + row0;
    const long long r2 = 2 * t.n_pix;
    LightScan sc;
    if (WITH_SCAN) sc.init();
#pragma unroll
    for (int g = 0; g < 7; ++g) {
        if (g * 8 < t.nv) {                                      // warp-uniform
            float* b = sbuf + (g & 1) * 512;
#pragma unroll
            for (int e = 0; e < 8; ++e) {
                b[e * 32 + lane] = acc[g * 16 + e];
                b[256 + e * 32 + lane] = acc[g * 16 + 8 + e];
            }
            __syncwarp();
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const float2 q = *reinterpret_cast<const float2*>(b + (dl + 2 * i) * 32 + px);
                const float2 u = *reinterpret_cast<const float2*>(b + 256 + (dl + 2 * i) * 32 + px);
                if (pin && g * 8 + dl + 2 * i < t.nv) {
                    __stcs(reinterpret_cast<float2*>(gq), q);
                    __stcs(reinterpret_cast<float2*>(gu), u);
                }
                gq += r2;
                gu += r2;
            }
            if (WITH_SCAN) sc.group(acc, g, t.nv);
        }
    }
    if (WITH_SCAN) sc.finish(t, lane, rec);
}

// phi-major cubes through a shared-memory ring and TMA stores.  One SM stores at most 32 bytes per clock from registers
// (measured: 106 KB in 3.2 k cycles whatever the vector width and however many SMs store), and inside this kernel, next to
// ~46 B/clk of inbound TMA traffic, a 106 KB tile took 6.5-10 k cycles of the epilogue warps' time while the two TMEM
// accumulator buffers give the MMA issuer only 2.5 k cycles of slack (profiles/r02_tile_timeline_cfg5_before.txt: issuer
// blocked on acc_empty 6.6-9.5 k cycles of a 35 k-cycle item).  So the epilogue warps do not store: the four warps of a
// column half (128 pixels) stage a group of eight depths of FQ and of FU -- two [8 depths][128 pixels] slabs, 8 KB -- in
// a ring of ten such pairs (80 KB of the 106 KB tile: the raw-tile ring gives up its third stage for it) and go back to
// draining accumulators; one thread of an otherwise idle warp hands every pair to the TMA engine as two box stores
// (cp.async.bulk.tensor, 128 pixels x 8 depths; the tensor map clips ragged pixel and depth edges) and recycles a slot
// as soon as the engine has READ it (wait_group.read).  The stores then drain in the background during the next item.
// Pairs are used in a fixed order known to both sides: per work item, for g = 0..6: [half 0, group g] if g < ng0, then
// [half 1, group g] if g < ng1.  full[slot]: 4 warp arrivals; empty[slot]: 1 arrival by the store thread.
constexpr int kRingSlots = 10, kRingSlotFloats = 2048;
struct TileRing {
    float* base;          // kRingSlots x 2048 floats
    uint64_t* full;       // [kRingSlots]
    uint64_t* empty;      // [kRingSlots]
    uint32_t seq;         // pairs pushed / popped so far by this thread's role (slot = seq % kRingSlots, phase = seq / kRingSlots & 1)
    uint32_t released;    // store thread only: slots handed back so far
    __device__ __forceinline__ void init(float* b, uint64_t* f, uint64_t* e) { base = b; full = f; empty = e; seq = 0; released = 0; }
};
// number of 8-depth groups the two column halves hold of a depth tile with nv_tile valid depths
__device__ __forceinline__ void ring_groups(int nv_tile, int& ng0, int& ng1) {
    ng0 = (min(nv_tile, 56) + 7) >> 3;
    ng1 = (max(min(nv_tile - 56, 48), 0) + 7) >> 3;
}

template <bool WITH_SCAN>
__device__ __forceinline__ void epi_tile_phi_major_ring(const float (&acc)[128], const EpiTile& t, int lane, int q, int half,
                                                        int nv_tile, TileRing& ring, float* __restrict__ rec) {
    int ng0, ng1;
    ring_groups(nv_tile, ng0, ng1);
    LightScan sc;
    if (WITH_SCAN) sc.init();
#pragma unroll
    for (int g = 0; g < 7; ++g) {
        if (g < (half ? ng1 : ng0)) {                            // uniform over the four warps of the half
            const uint32_t n = ring.seq + (half ? min(g + 1, ng0) + g : g + min(g, ng1));   // position in the item's pair order
            const uint32_t slot = n % kRingSlots, phase = (n / kRingSlots) & 1u;
            mbar_wait(&ring.empty[slot], phase ^ 1u);
            float* b = ring.base + slot * kRingSlotFloats;
#pragma unroll
            for (int e = 0; e < 8; ++e) {
                b[e * 128 + q * 32 + lane] = acc[g * 16 + e];
                b[1024 + e * 128 + q * 32 + lane] = acc[g * 16 + 8 + e];
            }
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic-proxy writes -> visible to the TMA engine
            __syncwarp();
            if (lane == 0) mbar_arrive(&ring.full[slot]);
            if (WITH_SCAN) sc.group(acc, g, t.nv);
        }
    }
    ring.seq += ng0 + ng1;
    if (WITH_SCAN) sc.finish(t, lane, rec);
}

// The store thread's side: one work item = ng0 + ng1 pairs.  pix_tile: first pixel of the CTA's 128-pixel tile;
// k_tile: first depth of the depth tile.  Called by ONE thread.
__device__ __forceinline__ void tma_store_2d(const CUtensorMap* map, uint32_t src, int c0, int c1, uint64_t pol) {
    asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group.L2::cache_hint [%0, {%2, %3}], [%1], %4;" ::"l"(map), "r"(src),
                 "r"(c0), "r"(c1), "l"(pol) : "memory");
}
constexpr int kRingPending = 6;   // bulk groups that may still be reading their slot when the store thread moves on
__device__ __forceinline__ void ring_release(TileRing& ring, uint32_t upto) {      // slots of the groups < upto go back
    for (; ring.released < upto; ++ring.released) mbar_arrive(&ring.empty[ring.released % kRingSlots]);
}
__device__ __forceinline__ void ring_store_item(TileRing& ring, const CUtensorMap* mapFQ, const CUtensorMap* mapFU, int pix_tile,
                                                int k_tile, int nv_tile, uint64_t pol) {
    int ng0, ng1;
    ring_groups(nv_tile, ng0, ng1);
    for (int g = 0; g < 7; ++g) {
#pragma unroll
        for (int half = 0; half < 2; ++half) {
            if (g >= (half ? ng1 : ng0)) continue;
            const uint32_t slot = ring.seq % kRingSlots, phase = (ring.seq / kRingSlots) & 1u;
            ++ring.seq;
            mbar_wait(&ring.full[slot], phase);
            const uint32_t src = smem_u32(ring.base + slot * kRingSlotFloats);
            const int d0 = k_tile + half * 56 + g * 8;           // first depth of the pair
            tma_store_2d(mapFQ, src, pix_tile, d0, pol);
            tma_store_2d(mapFU, src + 4096, pix_tile, d0, pol);
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
            asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(kRingPending) : "memory");
            if (ring.seq > (uint32_t)kRingPending) ring_release(ring, ring.seq - kRingPending);
        }
    }
    // nothing else to do until the next tile end: wait until the engine has read the item's last slots, hand them all back
    asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
    ring_release(ring, ring.seq);
}
// before the kernel exits: every bulk store has been performed (written), not merely read
__device__ __forceinline__ void ring_store_flush() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }

}  // namespace rms
