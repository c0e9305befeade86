// rmsynth_execute / rmsynth_execute_peaks / rmsynth_execute_ex / rmsynth_execute_host: argument checks,
// scheme dispatch (rows a4-a9) and the host-streaming loop (the paper's "each datum crosses the bus
// once" rule, with pixel chunks instead of LOS batches sized from GPU memory P:L210).
#include <cstdlib>
#include <cstring>
#include "common.cuh"

namespace rms {

struct Outs {
    float *FQ = nullptr, *FU = nullptr, *FA = nullptr;
    float *amp = nullptr, *phi = nullptr, *pa0 = nullptr, *paz = nullptr;
    int* idx = nullptr;
    bool maps() const { return amp || phi || pa0 || paz || idx; }
    bool any() const { return FQ || FA || maps(); }
};

static rmsynth_status check_args(const rmsynth_plan* p, const float* Q, const float* U, long long n_pix,
                                 int layout, bool need_cubes, const Outs& o) {
    if (!p) return fail(RMSYNTH_EINVAL, "plan is NULL");
    if (n_pix < 0) return fail(RMSYNTH_EINVAL, "n_pix < 0");
    if (layout & ~3) return fail(RMSYNTH_EINVAL, "unknown layout flags");
    if (n_pix == 0) return RMSYNTH_OK;
    if (!Q || !U) return fail(RMSYNTH_EINVAL, "Q/U is NULL");
    if ((o.FQ == nullptr) != (o.FU == nullptr)) return fail(RMSYNTH_EINVAL, "FQ and FU must both be given or both NULL");
    if (need_cubes && !o.FQ) return fail(RMSYNTH_EINVAL, "FQ/FU is NULL");
    if (!o.any()) return fail(RMSYNTH_EINVAL, "no output requested");
    if (n_pix > (1LL << 40)) return fail(RMSYNTH_EINVAL, "n_pix too large");
    return RMSYNTH_OK;
}

// Device-resident contraction + optional |F| cube and maps on one stream; never synchronises.
static rmsynth_status run_device(const rmsynth_plan* p, const float* Q, const float* U, long long n_pix, int layout,
                                 Outs o, cudaStream_t st) {
    if (p->scheme == RMSYNTH_SCHEME_TF32X3 || p->scheme == RMSYNTH_SCHEME_F16X3)
        return tc_execute(p, Q, U, n_pix, layout, o.FQ, o.FU, o.FA, o.amp, o.phi, o.pa0, o.paz, o.idx, st);
    // FP32 CUDA-core comparison paths: cubes first, then the stand-alone |F| and peak kernels.
    rmsynth_status s;
    if (!o.FQ) {
        size_t bytes = sizeof(float) * (size_t)n_pix * p->n_phi;
        if ((s = stream_scratch(p, st, SCR_CUBE_Q, bytes, &o.FQ)) || (s = stream_scratch(p, st, SCR_CUBE_U, bytes, &o.FU)))
            return s;
    }
    s = p->scheme == RMSYNTH_SCHEME_FP32_TABLE ? fp32_table_execute(p, Q, U, n_pix, layout, o.FQ, o.FU, st)
                                               : fp32_sincos_execute(p, Q, U, n_pix, layout, o.FQ, o.FU, st);
    if (s == RMSYNTH_OK && o.FA) s = abs_from_cubes(o.FQ, o.FU, n_pix * p->n_phi, o.FA, st);
    if (s != RMSYNTH_OK || !o.maps()) return s;
    return peaks_from_cubes(p, o.FQ, o.FU, n_pix, layout & RMSYNTH_OUT_PHI_MAJOR, o.amp, o.phi, o.pa0, o.paz, o.idx, st);
}

}  // namespace rms

using namespace rms;

extern "C" {

rmsynth_status rmsynth_execute(const rmsynth_plan* plan, const float* Q, const float* U, long long n_pix,
                               int layout, float* FQ, float* FU, void* stream) {
    Outs o;
    o.FQ = FQ;
    o.FU = FU;
    rmsynth_status s = check_args(plan, Q, U, n_pix, layout, true, o);
    if (s != RMSYNTH_OK || n_pix == 0) return s;
    return run_device(plan, Q, U, n_pix, layout, o, (cudaStream_t)stream);
}

rmsynth_status rmsynth_execute_peaks(const rmsynth_plan* plan, const float* Q, const float* U, long long n_pix,
                                     int layout, float* FQ, float* FU, float* peak_amp, float* peak_phi,
                                     float* pa_lambda0, float* pa_zero, int* peak_index, void* stream) {
    Outs o;
    o.FQ = FQ; o.FU = FU; o.amp = peak_amp; o.phi = peak_phi; o.pa0 = pa_lambda0; o.paz = pa_zero; o.idx = peak_index;
    rmsynth_status s = check_args(plan, Q, U, n_pix, layout, false, o);
    if (s != RMSYNTH_OK || n_pix == 0) return s;
    return run_device(plan, Q, U, n_pix, layout, o, (cudaStream_t)stream);
}

rmsynth_status rmsynth_execute_ex(const rmsynth_plan* plan, const float* Q, const float* U, long long n_pix,
                                  int layout, const rmsynth_outputs* out, void* stream) {
    if (!out || out->struct_size != (int)sizeof(rmsynth_outputs)) return fail(RMSYNTH_EINVAL, "outputs.struct_size");
    Outs o;
    o.FQ = out->FQ; o.FU = out->FU; o.FA = out->F_abs; o.amp = out->peak_amp; o.phi = out->peak_phi;
    o.pa0 = out->pa_lambda0; o.paz = out->pa_zero; o.idx = out->peak_index;
    rmsynth_status s = check_args(plan, Q, U, n_pix, layout, false, o);
    if (s != RMSYNTH_OK || n_pix == 0) return s;
    return run_device(plan, Q, U, n_pix, layout, o, (cudaStream_t)stream);
}

rmsynth_status rmsynth_execute_host(const rmsynth_plan* plan, const float* Q, const float* U, long long n_pix,
                                    int layout, float* FQ, float* FU, float* peak_amp, float* peak_phi,
                                    float* pa_lambda0, float* pa_zero, int* peak_index) {
    Outs ho;
    ho.FQ = FQ; ho.FU = FU; ho.amp = peak_amp; ho.phi = peak_phi; ho.pa0 = pa_lambda0; ho.paz = pa_zero; ho.idx = peak_index;
    rmsynth_status s = check_args(plan, Q, U, n_pix, layout, false, ho);
    if (s != RMSYNTH_OK || n_pix == 0) return s;
    const rmsynth_plan* p = plan;
    RMS_CUDA(cudaSetDevice(p->device));
    std::lock_guard<std::mutex> g(p->mu);
    const int nc = p->n_chan, np = p->n_phi;
    const bool in_freq = layout & RMSYNTH_IN_FREQ_MAJOR, out_phi = layout & RMSYNTH_OUT_PHI_MAJOR;
    // ~256 MB of device buffers per slot, two slots in flight
    static const long long chunk_mb = getenv("RMSYNTH_HOST_CHUNK_MB") ? atoll(getenv("RMSYNTH_HOST_CHUNK_MB")) : 256;
    long long chunk = ((chunk_mb > 0 ? chunk_mb : 256) << 20) / (8LL * (nc + np));
    chunk = chunk / 1024 * 1024;
    if (chunk < 1024) chunk = 1024;
    if (chunk > n_pix) chunk = n_pix;
    float *dQ[2], *dU[2], *dFQ[2], *dFU[2], *dM[2];
    for (int b = 0; b < 2; ++b) {
        if (!p->hs[b]) RMS_CUDA(cudaStreamCreateWithFlags(&p->hs[b], cudaStreamNonBlocking));
        if ((s = ensure_scratch(p, 4 * b + 0, sizeof(float) * chunk * nc, &dQ[b])) ||
            (s = ensure_scratch(p, 4 * b + 1, sizeof(float) * chunk * nc, &dU[b])) ||
            (s = ensure_scratch(p, 4 * b + 2, FQ ? sizeof(float) * chunk * np : 0, &dFQ[b])) ||    // maps only: no cube buffers
            (s = ensure_scratch(p, 4 * b + 3, FQ ? sizeof(float) * chunk * np : 0, &dFU[b])) ||
            (s = ensure_scratch(p, 8 + b, sizeof(float) * chunk * 5, &dM[b])))
            return s;
    }
    int it = 0;
    for (long long p0 = 0; p0 < n_pix; p0 += chunk, ++it) {
        const int b = it & 1;
        const long long n = n_pix - p0 < chunk ? n_pix - p0 : chunk;
        cudaStream_t st = p->hs[b];
        if (in_freq) {   // columns [p0, p0+n) of [chan][pix] -> compact [chan][n]
            RMS_CUDA(cudaMemcpy2DAsync(dQ[b], n * 4, Q + p0, n_pix * 4, n * 4, nc, cudaMemcpyHostToDevice, st));
            RMS_CUDA(cudaMemcpy2DAsync(dU[b], n * 4, U + p0, n_pix * 4, n * 4, nc, cudaMemcpyHostToDevice, st));
        } else {
            RMS_CUDA(cudaMemcpyAsync(dQ[b], Q + p0 * nc, sizeof(float) * n * nc, cudaMemcpyHostToDevice, st));
            RMS_CUDA(cudaMemcpyAsync(dU[b], U + p0 * nc, sizeof(float) * n * nc, cudaMemcpyHostToDevice, st));
        }
        float* m = dM[b];
        Outs o;
        if (FQ) { o.FQ = dFQ[b]; o.FU = dFU[b]; }
        o.amp = peak_amp ? m : nullptr;
        o.phi = peak_phi ? m + chunk : nullptr;
        o.pa0 = pa_lambda0 ? m + 2 * chunk : nullptr;
        o.paz = pa_zero ? m + 3 * chunk : nullptr;
        o.idx = peak_index ? (int*)(m + 4 * chunk) : nullptr;
        s = run_device(p, dQ[b], dU[b], n, layout, o, st);
        if (s != RMSYNTH_OK) return s;
        if (FQ) {
            if (out_phi) {
                RMS_CUDA(cudaMemcpy2DAsync(FQ + p0, n_pix * 4, dFQ[b], n * 4, n * 4, np, cudaMemcpyDeviceToHost, st));
                RMS_CUDA(cudaMemcpy2DAsync(FU + p0, n_pix * 4, dFU[b], n * 4, n * 4, np, cudaMemcpyDeviceToHost, st));
            } else {
                RMS_CUDA(cudaMemcpyAsync(FQ + p0 * np, dFQ[b], sizeof(float) * n * np, cudaMemcpyDeviceToHost, st));
                RMS_CUDA(cudaMemcpyAsync(FU + p0 * np, dFU[b], sizeof(float) * n * np, cudaMemcpyDeviceToHost, st));
            }
        }
        float* outs[5] = {peak_amp, peak_phi, pa_lambda0, pa_zero, (float*)peak_index};
        for (int j = 0; j < 5; ++j)
            if (outs[j])
                RMS_CUDA(cudaMemcpyAsync(outs[j] + p0, m + j * chunk, sizeof(float) * n, cudaMemcpyDeviceToHost, st));
    }
    RMS_CUDA(cudaStreamSynchronize(p->hs[0]));
    RMS_CUDA(cudaStreamSynchronize(p->hs[1]));
    return RMSYNTH_OK;
}

}  // extern "C"
