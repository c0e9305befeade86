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
    float best, ym2, yp2, q, u, prev, first;
    int k;          // local depth index of the best sample
    bool wn;        // the next sample is the right-hand neighbour of the best
    __device__ __forceinline__ void init() { best = ym2 = yp2 = prev = first = -1.f; q = u = 0.f; k = 0; wn = false; }
    __device__ __forceinline__ void step(int kl, float qq, float uu) {
        const float y2 = fmaf(qq, qq, uu * uu);
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
        r[0 * t.n_pix] = a.best;
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

}  // namespace rms
