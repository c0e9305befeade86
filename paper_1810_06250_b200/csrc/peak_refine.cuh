// Streaming arg-max state and the shared refinement/PA arithmetic of row a7 (readings A8-A10).
#pragma once
#include <cuda_runtime.h>

namespace rms {

struct PeakState {
    float best_y2, best_ym2, best_yp2, best_q, best_u, prev_y2;
    float nonfinite;   // 0, or NaN once a sample with a non-finite |F|^2 has been seen (reading A17)
    int best_k;
    bool want_next;

    __device__ __forceinline__ void init() {
        best_y2 = -1.f; best_ym2 = -1.f; best_yp2 = -1.f; best_q = 0.f; best_u = 0.f; prev_y2 = -1.f;
        nonfinite = 0.f; best_k = 0; want_next = false;
    }
    // samples must arrive in increasing k; strict > keeps the lowest index on ties
    __device__ __forceinline__ void push(int k, float q, float u) {
        float y2 = fmaf(q, q, u * u);
        nonfinite = fmaf(y2, 0.f, nonfinite);          // 0 x finite = 0, 0 x Inf = 0 x NaN = NaN: sticky
        if (want_next) { best_yp2 = y2; want_next = false; }
        if (y2 > best_y2) {
            best_y2 = y2; best_k = k; best_q = q; best_u = u;
            best_ym2 = prev_y2; best_yp2 = -1.f; want_next = true;
        }
        prev_y2 = y2;
    }
};

__device__ __forceinline__ void refine_and_store(const PeakState& s, int n_phi, const float* __restrict__ phif,
                                                 double lambda0_sq, long long p, float* amp, float* phi,
                                                 float* pa0, float* paz, int* idx) {
    if (!(s.nonfinite == 0.f)) {
        // Reading A17: a line of sight whose |F|^2 is not finite at some depth (non-finite input samples, or |F| beyond
        // 1.8e19 where |F|^2 overflows FP32) has no defined peak: index -1, NaN in every map.
        const float nan = __int_as_float(0x7fc00000);
        if (idx) idx[p] = -1;
        if (amp) amp[p] = nan;
        if (phi) phi[p] = nan;
        if (pa0) pa0[p] = nan;
        if (paz) paz[p] = nan;
        return;
    }
    const int k = s.best_k;
    float y0 = sqrtf(fmaxf(s.best_y2, 0.f));
    float a_out = y0, ph = phif[k];
    if (k > 0 && k < n_phi - 1 && s.best_ym2 >= 0.f && s.best_yp2 >= 0.f) {
        float ym = sqrtf(s.best_ym2), yp = sqrtf(s.best_yp2);
        float x0 = phif[k - 1] - ph, x2 = phif[k + 1] - ph;
        float d0 = (ym - y0) / x0, d2 = (yp - y0) / x2;
        float a = (d2 - d0) / (x2 - x0);
        float b = d0 - a * x0;
        if (a < 0.f) {
            float xv = -b / (2.f * a);
            ph += xv;
            a_out = y0 + 0.5f * b * xv;
        }
    }
    float pa = 0.5f * atan2f(s.best_u, s.best_q);
    if (idx) idx[p] = k;
    if (amp) amp[p] = a_out;
    if (phi) phi[p] = ph;
    if (pa0) pa0[p] = pa;
    if (paz) {
        const double pi = 3.14159265358979323846;
        double r = fmod((double)pa - (double)ph * lambda0_sq + 0.5 * pi, pi);
        if (r < 0.0) r += pi;
        paz[p] = (float)(r - 0.5 * pi);
    }
}

}  // namespace rms
