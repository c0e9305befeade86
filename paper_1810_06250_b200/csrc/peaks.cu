// Row a7 (stand-alone form): peak maps from FQ/FU cubes already in device memory.
//   k* = argmax_k |F_k|, |F| = sqrt(FQ^2+FU^2) (Eq. 17), lowest k on ties;
//   3-point parabolic refinement on amplitudes (reading A8; from BASELINE.json, not the paper);
//   pa_lambda0 = 0.5 atan2(FU_k*, FQ_k*), pa_zero = pa_lambda0 - phi_peak lambda_0^2 wrapped to
//   [-pi/2, pi/2) (Eq. 14 P:L121 is garbled -> reading A9/A10).
// Comparison is on |F|^2 in FP32 (monotone in |F|); the tensor kernel's fused epilogue uses the
// same refine_and_store() so both paths take the integer decision in the same precision.
#include "common.cuh"
#include "peak_refine.cuh"

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
    float best = -1.f;
    int kb = 0x7fffffff;
    for (int k = lane; k < n_phi; k += 32) {
        float q = fq[k], u = fu[k];
        float y2 = fmaf(q, q, u * u);
        if (y2 > best) { best = y2; kb = k; }      // strict > keeps the lowest k per lane
    }
    for (int o = 16; o > 0; o >>= 1) {
        float ob = __shfl_xor_sync(0xffffffffu, best, o);
        int ok = __shfl_xor_sync(0xffffffffu, kb, o);
        if (ob > best || (ob == best && ok < kb)) { best = ob; kb = ok; }
    }
    if (lane != 0) return;
    if (kb >= n_phi) kb = 0;                        // all-NaN row: report index 0
    PeakState s;
    s.init();
    s.best_k = kb;
    s.best_q = fq[kb];
    s.best_u = fu[kb];
    s.best_y2 = fmaf(s.best_q, s.best_q, s.best_u * s.best_u);
    if (kb > 0) { float q = fq[kb - 1], u = fu[kb - 1]; s.best_ym2 = fmaf(q, q, u * u); }
    if (kb < n_phi - 1) { float q = fq[kb + 1], u = fu[kb + 1]; s.best_yp2 = fmaf(q, q, u * u); }
    refine_and_store(s, n_phi, phif, lambda0_sq, p, amp, phi, pa0, paz, idx);
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
