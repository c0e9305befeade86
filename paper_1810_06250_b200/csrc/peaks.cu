// Row a7 (stand-alone form): peak maps from FQ/FU cubes already in device memory.
//   k* = argmax_k |F_k|, |F| = sqrt(FQ^2+FU^2) (Eq. 17), lowest k on ties;
//   3-point parabolic refinement on amplitudes (reading A8; from BASELINE.json, not the paper);
//   pa_lambda0 = 0.5 atan2(FU_k*, FQ_k*), pa_zero = pa_lambda0 - phi_peak lambda_0^2 wrapped to
//   [-pi/2, pi/2) (Eq. 14 P:L121 is garbled -> reading A9/A10).
// Comparison is on |F|^2 in FP32 (monotone in |F|); the tensor kernel's fused epilogue uses the
// same refine_and_store() so both paths take the integer decision in the same precision.
#include "common.cuh"
#include "peak_refine.cuh"
#include "tc_epilogue.cuh"

namespace rms {

// phi-major cubes F[k*n_pix + p]: one thread per pixel, a warp reads 32 consecutive pixels.
__global__ void __launch_bounds__(256) peaks_phi_major_kernel(
    const float* __restrict__ FQ, const float* __restrict__ FU, long long n_pix, int n_phi,
    const float* __restrict__ phif, double lambda0_sq, float* amp, float* phi, float* pa0, float* paz, int* idx) {
    long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n_pix) return;
    PeakState s;
    s.init();
    for (int k = 0; k < n_phi; ++k) {
        float q = FQ[(size_t)k * n_pix + p], u = FU[(size_t)k * n_pix + p];
        s.push(k, q, u);
    }
    refine_and_store(s, n_phi, phif, lambda0_sq, p, amp, phi, pa0, paz, idx);
}

// LOS-major cubes F[p*n_phi + k]: one warp per pixel, lanes stride over phi, shuffle argmax.
__global__ void __launch_bounds__(256) peaks_los_major_kernel(
    const float* __restrict__ FQ, const float* __restrict__ FU, long long n_pix, int n_phi,
    const float* __restrict__ phif, double lambda0_sq, float* amp, float* phi, float* pa0, float* paz, int* idx) {
    long long p = (long long)blockIdx.x * (blockDim.x / 32) + threadIdx.x / 32;
    int lane = threadIdx.x % 32;
    if (p >= n_pix) return;
    const float* fq = FQ + (size_t)p * n_phi;
    const float* fu = FU + (size_t)p * n_phi;
    float best = -1.f, nf = 0.f;
    int kb = 0x7fffffff;
    for (int k = lane; k < n_phi; k += 32) {
        float q = fq[k], u = fu[k];
        float y2 = fmaf(q, q, u * u);
        nf = fmaf(y2, 0.f, nf);                    // sticky NaN once |F|^2 is not finite (reading A17)
        if (y2 > best) { best = y2; kb = k; }      // strict > keeps the lowest k per lane
    }
    for (int o = 16; o > 0; o >>= 1) {
        float ob = __shfl_xor_sync(0xffffffffu, best, o);
        int ok = __shfl_xor_sync(0xffffffffu, kb, o);
        nf += __shfl_xor_sync(0xffffffffu, nf, o);
        if (ob > best || (ob == best && ok < kb)) { best = ob; kb = ok; }
    }
    if (lane != 0) return;
    if (kb >= n_phi) kb = 0;                        // all-NaN row: flagged below
    PeakState s;
    s.init();
    s.nonfinite = nf;
    s.best_k = kb;
    s.best_q = fq[kb];
    s.best_u = fu[kb];
    s.best_y2 = fmaf(s.best_q, s.best_q, s.best_u * s.best_u);
    if (kb > 0) { float q = fq[kb - 1], u = fu[kb - 1]; s.best_ym2 = fmaf(q, q, u * u); }
    if (kb < n_phi - 1) { float q = fq[kb + 1], u = fu[kb + 1]; s.best_yp2 = fmaf(q, q, u * u); }
    refine_and_store(s, n_phi, phif, lambda0_sq, p, amp, phi, pa0, paz, idx);
}

// Row a7, fused form: merge the per-segment records the tensor kernel's epilogue wrote (tc_epilogue.cuh) --
// segments of a pixel are visited in ascending depth order with a strict >, so the decision sequence is the
// one a single scan over all depths would take (lowest k on ties); a best sample sitting on a segment edge
// takes its missing neighbour from the adjacent segment's first / last |F|^2.  One thread per pixel.
__global__ void __launch_bounds__(256) peaks_combine_kernel(
    const float* __restrict__ rec, int n_seg, long long n_pix, int n_phi, const float* __restrict__ phif,
    double lambda0_sq, float* amp, float* phi, float* pa0, float* paz, int* idx) {
    const long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n_pix) return;
    PeakState s;
    s.init();
    float last = -1.f;
    bool need_next = false;
    for (int g = 0; g < n_seg; ++g) {
        const float* r = rec + (long long)g * kPeakFields * n_pix + p;
        const float first = r[6 * n_pix];
        if (first == -1.f) continue;                       // empty segment (ragged last depth tile)
        if (need_next) { s.best_yp2 = first; need_next = false; }
        const float by2 = r[0];
        s.nonfinite += by2 * 0.f;                          // NaN: the segment saw a non-finite |F|^2
        if (by2 > s.best_y2) {
            s.best_y2 = by2;
            s.best_k = __float_as_int(r[1 * n_pix]);
            s.best_q = r[2 * n_pix];
            s.best_u = r[3 * n_pix];
            const float ym2 = r[4 * n_pix], yp2 = r[5 * n_pix];
            s.best_ym2 = ym2 == -1.f ? last : ym2;         // -1: the best was the segment's first sample
            s.best_yp2 = yp2;
            need_next = yp2 == -1.f;                       // -1: the best was the segment's last sample
        }
        last = r[7 * n_pix];
    }
    refine_and_store(s, n_phi, phif, lambda0_sq, p, amp, phi, pa0, paz, idx);
}

// Row a7, fused form when the cubes were written (tc_epilogue.cuh: LightScan): the segment records hold only
// (max |F|^2, k); k* is the first segment maximum in ascending depth order (strict >), and the samples at k*, k* - 1,
// k* + 1 are read back from the cubes the same launch sequence has just written -- the very FP32 values the epilogue
// held in registers, so |F|^2 = fma(q, q, u u) reproduces the recorded maximum bit for bit.  One thread per pixel.
__global__ void __launch_bounds__(256) peaks_gather_kernel(
    const float* __restrict__ rec, int n_seg, long long n_pix, int n_phi, const float* __restrict__ FQ,
    const float* __restrict__ FU, int out_phi, const float* __restrict__ phif, double lambda0_sq, float* amp, float* phi,
    float* pa0, float* paz, int* idx) {
    const long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n_pix) return;
    PeakState s;
    s.init();
    // Two memory round trips per pixel, not n_seg + 1: the segment records are fetched eight at a time with
    // unconditional, independent loads (a load of k guarded by the comparison would chain the segments), then the three
    // samples around k* with clamped indices.
    for (int g0 = 0; g0 < n_seg; g0 += 8) {
        float y[8];
        int kk[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const bool ok = g0 + i < n_seg;
            const float* r = rec + (long long)(ok ? g0 + i : g0) * kPeakFields * n_pix + p;
            const float v = __ldcs(r);
            kk[i] = __float_as_int(__ldcs(r + n_pix));
            y[i] = ok ? v : -2.f;                              // a padding slot never wins and is finite
        }
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            s.nonfinite += y[i] * 0.f;
            if (y[i] > s.best_y2) { s.best_y2 = y[i]; s.best_k = kk[i]; }
        }
    }
    const int k = s.best_k, km = max(k - 1, 0), kp = min(k + 1, n_phi - 1);
    auto at = [&](int kk) { return out_phi ? (size_t)kk * n_pix + p : (size_t)p * n_phi + kk; };
    const float q0 = FQ[at(k)], u0 = FU[at(k)], qm = FQ[at(km)], um = FU[at(km)], qp = FQ[at(kp)], up = FU[at(kp)];
    s.best_q = q0;
    s.best_u = u0;
    s.best_y2 = fmaf(q0, q0, u0 * u0);
    if (k > 0) s.best_ym2 = fmaf(qm, qm, um * um);
    if (k < n_phi - 1) s.best_yp2 = fmaf(qp, qp, up * up);
    refine_and_store(s, n_phi, phif, lambda0_sq, p, amp, phi, pa0, paz, idx);
}

rmsynth_status peaks_gather(const rmsynth_plan* p, const float* rec, int n_seg, long long n_pix, const float* FQ, const float* FU,
                            bool out_phi, float* amp, float* phi, float* pa0, float* paz, int* idx, cudaStream_t st) {
    if (n_pix == 0) return RMSYNTH_OK;
    peaks_gather_kernel<<<(unsigned)((n_pix + 255) / 256), 256, 0, st>>>(rec, n_seg, n_pix, p->n_phi, FQ, FU, out_phi ? 1 : 0,
                                                                          p->d_phif, p->lambda0_sq, amp, phi, pa0, paz, idx);
    RMS_LAUNCH_CHECK("peaks_gather_kernel");
    return RMSYNTH_OK;
}

rmsynth_status peaks_combine(const rmsynth_plan* p, const float* rec, int n_seg, long long n_pix, float* amp, float* phi,
                             float* pa0, float* paz, int* idx, cudaStream_t st) {
    if (n_pix == 0) return RMSYNTH_OK;
    peaks_combine_kernel<<<(unsigned)((n_pix + 255) / 256), 256, 0, st>>>(rec, n_seg, n_pix, p->n_phi, p->d_phif,
                                                                           p->lambda0_sq, amp, phi, pa0, paz, idx);
    RMS_LAUNCH_CHECK("peaks_combine_kernel");
    return RMSYNTH_OK;
}

// |F| cube (Eq. 17) from FQ/FU cubes, element-wise (used by the FP32 comparison schemes; the tensor
// kernel writes |F| from its epilogue registers).
__global__ void __launch_bounds__(256) abs_cube_kernel(const float* __restrict__ FQ, const float* __restrict__ FU,
                                                       long long n, float* __restrict__ FA) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const float q = FQ[i], u = FU[i];
        FA[i] = sqrtf(fmaf(q, q, u * u));
    }
}

rmsynth_status abs_from_cubes(const float* FQ, const float* FU, long long n, float* FA, cudaStream_t st) {
    if (n == 0) return RMSYNTH_OK;
    long long blocks = (n + 255) / 256;
    if (blocks > 148 * 32) blocks = 148 * 32;
    abs_cube_kernel<<<(unsigned)blocks, 256, 0, st>>>(FQ, FU, n, FA);
    RMS_LAUNCH_CHECK("abs_cube_kernel");
    return RMSYNTH_OK;
}

rmsynth_status peaks_from_cubes(const rmsynth_plan* p, const float* FQ, const float* FU, long long n_pix,
                                int out_layout, float* amp, float* phi, float* pa0, float* paz, int* idx,
                                cudaStream_t st) {
    if (n_pix == 0) return RMSYNTH_OK;
    if (out_layout == RMSYNTH_OUT_PHI_MAJOR) {
        long long g = (n_pix + 255) / 256;
        peaks_phi_major_kernel<<<(unsigned)g, 256, 0, st>>>(FQ, FU, n_pix, p->n_phi, p->d_phif,
                                                             p->lambda0_sq, amp, phi, pa0, paz, idx);
    } else {
        long long g = (n_pix + 7) / 8;
        peaks_los_major_kernel<<<(unsigned)g, 256, 0, st>>>(FQ, FU, n_pix, p->n_phi, p->d_phif,
                                                             p->lambda0_sq, amp, phi, pa0, paz, idx);
    }
    RMS_LAUNCH_CHECK("peaks kernel");
    return RMSYNTH_OK;
}

}  // namespace rms
