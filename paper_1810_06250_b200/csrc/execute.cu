// rmsynth_execute / rmsynth_execute_peaks / rmsynth_execute_ex: argument checks and scheme dispatch (rows a4-a9);
// rmsynth_execute_host / rmsynth_execute_stream: the out-of-core host-streaming engine (scope row NEXT-2) -- the paper's
// "a given piece of data is moved between the CPU and the GPU only once" rule with pixel chunks instead of
// LOS batches sized from GPU memory: three device slots, one stream per direction and one for the kernels, so
// that H2D(i+1), compute(i) and D2H(i-1) overlap.
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
    DeviceGuard g(p->device);
    RMS_CUDA(g.err);
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

// ------------------------------------------------------------------------------------------------
// Host streaming engine.  Slot b holds one pixel chunk: inputs dQ,dU [chunk x n_chan], cubes dFQ,dFU [chunk x n_phi]
// (only if cubes are wanted) and five maps.  Per chunk i in slot b = i % 3:
//   s_in : wait run_done[b] (the chunk that last used these input buffers has been computed) -> H2D -> in_done[b]
//   s_run: wait in_done[b], out_done[b] (the slot's previous outputs have left)               -> kernels -> run_done[b]
//   s_out: wait run_done[b]                                                                   -> D2H -> out_done[b]
constexpr int kSlots = 3;

struct HostPipe {
    cudaStream_t s_in = nullptr, s_run = nullptr, s_out = nullptr;
    cudaEvent_t in_done[kSlots] = {}, run_done[kSlots] = {}, out_done[kSlots] = {};
    float *dQ[kSlots] = {}, *dU[kSlots] = {}, *dFQ[kSlots] = {}, *dFU[kSlots] = {}, *dM[kSlots] = {};
    float* hIn[kSlots] = {};    // pinned staging of rmsynth_execute_stream: Q then U
    float* hOut[kSlots] = {};   //                                             FQ, FU, then five maps
    size_t in_bytes = 0, out_bytes = 0;
};

// Streams and events of the host pipeline, created on first use.  The HostPipe is attached to the plan only once every
// create has succeeded: a failure half-way releases what exists and leaves the plan without one, so the next call starts
// over instead of running with null streams (the legacy default stream) and null events.
static rmsynth_status pipe_get(const rmsynth_plan* p, HostPipe** out) {
    if (!p->host_pipe) {
        HostPipe* hp = new HostPipe;
        cudaError_t e = cudaStreamCreateWithFlags(&hp->s_in, cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&hp->s_run, cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&hp->s_out, cudaStreamNonBlocking);
        for (int b = 0; b < kSlots && e == cudaSuccess; ++b) {
            e = cudaEventCreateWithFlags(&hp->in_done[b], cudaEventDisableTiming);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&hp->run_done[b], cudaEventDisableTiming);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&hp->out_done[b], cudaEventDisableTiming);
        }
        if (e != cudaSuccess) {
            p->host_pipe = hp;                                // host_pipe_free releases whatever was created and detaches it
            host_pipe_free(const_cast<rmsynth_plan*>(p));
            RMS_CUDA(e);
        }
        p->host_pipe = hp;
    }
    *out = static_cast<HostPipe*>(p->host_pipe);
    return RMSYNTH_OK;
}

void host_pipe_free(rmsynth_plan* p) {
    HostPipe* hp = static_cast<HostPipe*>(p->host_pipe);
    if (!hp) return;
    for (int b = 0; b < kSlots; ++b) {
        if (hp->in_done[b]) cudaEventDestroy(hp->in_done[b]);
        if (hp->run_done[b]) cudaEventDestroy(hp->run_done[b]);
        if (hp->out_done[b]) cudaEventDestroy(hp->out_done[b]);
        if (hp->hIn[b]) cudaFreeHost(hp->hIn[b]);
        if (hp->hOut[b]) cudaFreeHost(hp->hOut[b]);
    }
    if (hp->s_in) cudaStreamDestroy(hp->s_in);
    if (hp->s_run) cudaStreamDestroy(hp->s_run);
    if (hp->s_out) cudaStreamDestroy(hp->s_out);
    delete hp;
    p->host_pipe = nullptr;
}

// pixels per chunk: the plan option, else ~256 MB of device buffers per slot; a multiple of 4 (the FP16 kernel's
// fast paths want 16-byte rows), at least 4, at most n_pix
static long long chunk_pixels(const rmsynth_plan* p, long long n_pix, bool cubes) {
    long long chunk = p->host_chunk_pixels;
    if (chunk <= 0) {
        chunk = (256LL << 20) / (8LL * (p->n_chan + (cubes ? p->n_phi : 0)));
        chunk = chunk / 1024 * 1024;
        if (chunk < 1024) chunk = 1024;
    }
    chunk = (chunk + 3) & ~3LL;
    if (n_pix > 0 && chunk > n_pix) chunk = n_pix;
    return chunk;
}

static rmsynth_status pipe_buffers(const rmsynth_plan* p, HostPipe* hp, long long chunk, bool cubes) {
    rmsynth_status s;
    for (int b = 0; b < kSlots; ++b)
        if ((s = ensure_scratch(p, 5 * b + 0, sizeof(float) * chunk * p->n_chan, &hp->dQ[b])) ||
            (s = ensure_scratch(p, 5 * b + 1, sizeof(float) * chunk * p->n_chan, &hp->dU[b])) ||
            (s = ensure_scratch(p, 5 * b + 2, cubes ? sizeof(float) * chunk * p->n_phi : 0, &hp->dFQ[b])) ||   // maps only: no cube buffers
            (s = ensure_scratch(p, 5 * b + 3, cubes ? sizeof(float) * chunk * p->n_phi : 0, &hp->dFU[b])) ||
            (s = ensure_scratch(p, 5 * b + 4, sizeof(float) * chunk * 5, &hp->dM[b])))
            return s;
    return RMSYNTH_OK;
}

// One chunk through slot b.  hQ/hU point at the chunk's first pixel in HOST memory; for frequency-major input in_pitch is
// the host row pitch in pixels (n_pix of the whole cube, or the chunk's own pixel count for compact staging buffers);
// likewise out_pitch for phi-major cubes.  Maps go to ho.amp.. (already offset to the chunk's first pixel).
static rmsynth_status pipe_chunk(const rmsynth_plan* p, HostPipe* hp, int b, long long chunk, long long n, int layout,
                                 const float* hQ, const float* hU, long long in_pitch, const Outs& ho, long long out_pitch) {
    const int nc = p->n_chan, np = p->n_phi;
    const bool in_freq = layout & RMSYNTH_IN_FREQ_MAJOR, out_phi = layout & RMSYNTH_OUT_PHI_MAJOR;
    RMS_CUDA(cudaStreamWaitEvent(hp->s_in, hp->run_done[b], 0));
    if (in_freq) {   // columns of [chan][pitch] -> compact [chan][n]
        RMS_CUDA(cudaMemcpy2DAsync(hp->dQ[b], n * 4, hQ, in_pitch * 4, n * 4, nc, cudaMemcpyHostToDevice, hp->s_in));
        RMS_CUDA(cudaMemcpy2DAsync(hp->dU[b], n * 4, hU, in_pitch * 4, n * 4, nc, cudaMemcpyHostToDevice, hp->s_in));
    } else {
        RMS_CUDA(cudaMemcpyAsync(hp->dQ[b], hQ, sizeof(float) * n * nc, cudaMemcpyHostToDevice, hp->s_in));
        RMS_CUDA(cudaMemcpyAsync(hp->dU[b], hU, sizeof(float) * n * nc, cudaMemcpyHostToDevice, hp->s_in));
    }
    RMS_CUDA(cudaEventRecord(hp->in_done[b], hp->s_in));
    RMS_CUDA(cudaStreamWaitEvent(hp->s_run, hp->in_done[b], 0));
    RMS_CUDA(cudaStreamWaitEvent(hp->s_run, hp->out_done[b], 0));
    float* m = hp->dM[b];
    Outs o;
    if (ho.FQ) { o.FQ = hp->dFQ[b]; o.FU = hp->dFU[b]; }
    o.amp = ho.amp ? m : nullptr;
    o.phi = ho.phi ? m + chunk : nullptr;
    o.pa0 = ho.pa0 ? m + 2 * chunk : nullptr;
    o.paz = ho.paz ? m + 3 * chunk : nullptr;
    o.idx = ho.idx ? (int*)(m + 4 * chunk) : nullptr;
    rmsynth_status s = run_device(p, hp->dQ[b], hp->dU[b], n, layout, o, hp->s_run);
    if (s != RMSYNTH_OK) return s;
    RMS_CUDA(cudaEventRecord(hp->run_done[b], hp->s_run));
    RMS_CUDA(cudaStreamWaitEvent(hp->s_out, hp->run_done[b], 0));
    if (ho.FQ) {
        if (out_phi) {
            RMS_CUDA(cudaMemcpy2DAsync(ho.FQ, out_pitch * 4, hp->dFQ[b], n * 4, n * 4, np, cudaMemcpyDeviceToHost, hp->s_out));
            RMS_CUDA(cudaMemcpy2DAsync(ho.FU, out_pitch * 4, hp->dFU[b], n * 4, n * 4, np, cudaMemcpyDeviceToHost, hp->s_out));
        } else {
            RMS_CUDA(cudaMemcpyAsync(ho.FQ, hp->dFQ[b], sizeof(float) * n * np, cudaMemcpyDeviceToHost, hp->s_out));
            RMS_CUDA(cudaMemcpyAsync(ho.FU, hp->dFU[b], sizeof(float) * n * np, cudaMemcpyDeviceToHost, hp->s_out));
        }
    }
    float* outs[5] = {ho.amp, ho.phi, ho.pa0, ho.paz, (float*)ho.idx};
    for (int j = 0; j < 5; ++j)
        if (outs[j]) RMS_CUDA(cudaMemcpyAsync(outs[j], m + j * chunk, sizeof(float) * n, cudaMemcpyDeviceToHost, hp->s_out));
    RMS_CUDA(cudaEventRecord(hp->out_done[b], hp->s_out));
    return RMSYNTH_OK;
}

static rmsynth_status pipe_drain(HostPipe* hp) {
    RMS_CUDA(cudaStreamSynchronize(hp->s_in));
    RMS_CUDA(cudaStreamSynchronize(hp->s_run));
    RMS_CUDA(cudaStreamSynchronize(hp->s_out));
    return RMSYNTH_OK;
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
    DeviceGuard g(p->device);
    RMS_CUDA(g.err);
    std::lock_guard<std::mutex> lock(p->mu);
    const int nc = p->n_chan, np = p->n_phi;
    const bool in_freq = layout & RMSYNTH_IN_FREQ_MAJOR, out_phi = layout & RMSYNTH_OUT_PHI_MAJOR;
    const long long chunk = chunk_pixels(p, n_pix, FQ != nullptr);
    HostPipe* hp;
    if ((s = pipe_get(p, &hp)) || (s = pipe_buffers(p, hp, chunk, FQ != nullptr))) return s;
    int it = 0;
    for (long long p0 = 0; p0 < n_pix; p0 += chunk, ++it) {
        const long long n = n_pix - p0 < chunk ? n_pix - p0 : chunk;
        Outs o;
        if (FQ) {
            o.FQ = out_phi ? FQ + p0 : FQ + p0 * np;
            o.FU = out_phi ? FU + p0 : FU + p0 * np;
        }
        o.amp = peak_amp ? peak_amp + p0 : nullptr;
        o.phi = peak_phi ? peak_phi + p0 : nullptr;
        o.pa0 = pa_lambda0 ? pa_lambda0 + p0 : nullptr;
        o.paz = pa_zero ? pa_zero + p0 : nullptr;
        o.idx = peak_index ? peak_index + p0 : nullptr;
        s = pipe_chunk(p, hp, it % kSlots, chunk, n, layout, in_freq ? Q + p0 : Q + p0 * nc, in_freq ? U + p0 : U + p0 * nc, n_pix, o, n_pix);
        if (s != RMSYNTH_OK) {
            pipe_drain(hp);
            return s;
        }
    }
    return pipe_drain(hp);
}

rmsynth_status rmsynth_execute_stream(const rmsynth_plan* plan, int layout, int outputs, rmsynth_fill_fn fill,
                                      rmsynth_drain_fn drain, void* user, long long* n_pix_done) {
    if (n_pix_done) *n_pix_done = 0;
    if (!plan) return fail(RMSYNTH_EINVAL, "plan is NULL");
    if (layout & ~3) return fail(RMSYNTH_EINVAL, "unknown layout flags");
    if (!fill || !drain) return fail(RMSYNTH_EINVAL, "fill/drain callback is NULL");
    if (!(outputs & (RMSYNTH_WANT_CUBES | RMSYNTH_WANT_MAPS)) || (outputs & ~(RMSYNTH_WANT_CUBES | RMSYNTH_WANT_MAPS)))
        return fail(RMSYNTH_EINVAL, "outputs must be RMSYNTH_WANT_CUBES and/or RMSYNTH_WANT_MAPS");
    const rmsynth_plan* p = plan;
    DeviceGuard g(p->device);
    RMS_CUDA(g.err);
    std::lock_guard<std::mutex> lock(p->mu);
    const int nc = p->n_chan, np = p->n_phi;
    const bool cubes = outputs & RMSYNTH_WANT_CUBES, maps = outputs & RMSYNTH_WANT_MAPS;
    const long long chunk = chunk_pixels(p, 0, cubes);
    rmsynth_status s;
    HostPipe* hp;
    if ((s = pipe_get(p, &hp)) || (s = pipe_buffers(p, hp, chunk, cubes))) return s;
    const size_t in_bytes = sizeof(float) * 2 * (size_t)chunk * nc;
    const size_t out_bytes = sizeof(float) * (size_t)chunk * ((cubes ? 2 * (size_t)np : 0) + 5);
    if (hp->in_bytes < in_bytes || hp->out_bytes < out_bytes) {
        for (int b = 0; b < kSlots; ++b) {
            if (hp->hIn[b]) cudaFreeHost(hp->hIn[b]);
            if (hp->hOut[b]) cudaFreeHost(hp->hOut[b]);
            hp->hIn[b] = hp->hOut[b] = nullptr;
        }
        hp->in_bytes = hp->out_bytes = 0;
        for (int b = 0; b < kSlots; ++b) {
            RMS_CUDA(cudaMallocHost(&hp->hIn[b], in_bytes));
            RMS_CUDA(cudaMallocHost(&hp->hOut[b], out_bytes));
        }
        hp->in_bytes = in_bytes;
        hp->out_bytes = out_bytes;
    }
    long long count[kSlots] = {0, 0, 0}, total = 0;
    auto finish = [&](long long i) -> rmsynth_status {       // chunk i's outputs are in host staging: hand them over
        const int b = (int)(i % kSlots);
        RMS_CUDA(cudaEventSynchronize(hp->out_done[b]));
        const long long n = count[b];
        float* o = hp->hOut[b];
        rmsynth_outputs ro;
        std::memset(&ro, 0, sizeof(ro));
        ro.struct_size = (int)sizeof(ro);
        if (cubes) { ro.FQ = o; ro.FU = o + (size_t)n * np; o += 2 * (size_t)n * np; }
        if (maps) { ro.peak_amp = o; ro.peak_phi = o + n; ro.pa_lambda0 = o + 2 * n; ro.pa_zero = o + 3 * n; ro.peak_index = (int*)(o + 4 * n); }
        drain(user, i, n, &ro);
        total += n;
        return RMSYNTH_OK;
    };
    long long i = 0;
    for (;; ++i) {
        const int b = (int)(i % kSlots);
        if (i >= kSlots && (s = finish(i - kSlots))) break;   // frees slot b's staging buffers
        float* hq = hp->hIn[b];
        const long long n = fill(user, i, hq, hq + (size_t)chunk * nc, chunk);
        if (n <= 0) break;
        if (n > chunk) { s = fail(RMSYNTH_EINVAL, "fill callback returned more pixels than the chunk holds"); break; }
        count[b] = n;
        // staging is compact: [chan][n] / [n][chan] with U starting at Q + chunk*n_chan; outputs [phi][n] / [n][phi]
        float* o = hp->hOut[b];
        Outs ho;
        if (cubes) { ho.FQ = o; ho.FU = o + (size_t)n * np; o += 2 * (size_t)n * np; }
        if (maps) { ho.amp = o; ho.phi = o + n; ho.pa0 = o + 2 * n; ho.paz = o + 3 * n; ho.idx = (int*)(o + 4 * n); }
        if ((s = pipe_chunk(p, hp, b, chunk, n, layout, hq, hq + (size_t)chunk * nc, n, ho, n))) break;
    }
    // chunks 0 .. i-1 were submitted; the loop has handed over all but the last kSlots - 1 of them
    for (long long j = i > kSlots - 1 ? i - (kSlots - 1) : 0; j < i && s == RMSYNTH_OK; ++j) s = finish(j);
    pipe_drain(hp);
    if (n_pix_done) *n_pix_done = total;
    return s;
}

}  // extern "C"
