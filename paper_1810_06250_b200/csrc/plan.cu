// Plan builder (rows a1-a3 of the scope table) and the C-ABI entry points.
//   a1: lambda_i^2 = (c/nu_i)^2, K = 1/sum w (Eq. 13), lambda_0^2   host, FP64
//   a2: phase matrix K w_i cos/sin(2 phi_k (lambda_i^2-lambda_0^2))                  device, FP64 -> FP32
//   a3: R(phi) (Eq. 12)                                                      device, FP64
// The paper evaluates two trig functions per (LOS, channel, phi) term; they do not
// depend on the LOS, so they are hoisted into this plan (N_pix-fold fewer trig calls).
#include <cmath>
#include <cstring>
#include <new>
#include "common.cuh"

namespace rms {

static thread_local std::string t_last_error;
std::atomic<long long> g_launches{0};

void set_error(const std::string& s) { t_last_error = s; }
rmsynth_status fail(rmsynth_status st, const std::string& s) {
    t_last_error = s;
    return st;
}

rmsynth_status ensure_scratch(const rmsynth_plan* p, int slot, size_t bytes, float** out) {
    if (p->scratch_bytes[slot] < bytes) {
        if (p->scratch[slot]) cudaFree(p->scratch[slot]);
        p->scratch[slot] = nullptr;
        p->scratch_bytes[slot] = 0;
        RMS_CUDA(cudaMalloc(&p->scratch[slot], bytes));
        p->scratch_bytes[slot] = bytes;
    }
    *out = p->scratch[slot];
    return RMSYNTH_OK;
}

rmsynth_status stream_scratch(const rmsynth_plan* p, cudaStream_t st, int tag, size_t bytes, float** out) {
    std::lock_guard<std::mutex> g(p->pool_mu);
    rmsynth_plan::StreamScratch* e = nullptr;
    for (auto& x : p->pool)
        if (x.st == st && x.tag == tag) e = &x;
    if (!e) {
        p->pool.push_back({st, tag, nullptr, 0});
        e = &p->pool.back();
    }
    if (e->bytes < bytes) {
        // Growing never frees: work already enqueued on this stream, or a CUDA graph captured from an earlier call, may
        // still reference the old buffer, so it is retired and lives until the plan is destroyed.  An allocation cannot
        // happen inside a stream capture: the caller must run the shape once (or a larger one) before capturing.
        cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
        if (cudaStreamIsCapturing(st, &cap) == cudaSuccess && cap != cudaStreamCaptureStatusNone)
            return fail(RMSYNTH_EINVAL, "workspace must grow during a stream capture: execute this shape once before capturing");
        if (e->ptr) p->retired.push_back(e->ptr);
        e->ptr = nullptr;
        e->bytes = 0;
        RMS_CUDA(cudaMalloc(&e->ptr, bytes));
        e->bytes = bytes;
    }
    *out = e->ptr;
    return RMSYNTH_OK;
}

// ---- a2: one thread per (channel i, depth k).  theta and its sincos are formed in FP64
// (max|theta| reaches 713 rad in config 5; an FP32 theta would already miss the 1e-5 budget)
// and only the product K w_i cos/sin is rounded to FP32.
__global__ void phase_matrix_kernel(const double* __restrict__ delta, const double* __restrict__ kw,
                                    const double* __restrict__ phi, int n_chan, int n_phi, int ldb,
                                    float* __restrict__ c_out, float* __restrict__ s_out) {
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    int i = blockIdx.y;
    if (k >= ldb || i >= n_chan) return;
    float c = 0.f, s = 0.f;
    if (k < n_phi) {
        double sn, cs;
        sincos(2.0 * phi[k] * delta[i], &sn, &cs);
        c = (float)(kw[i] * cs);
        s = (float)(kw[i] * sn);
    }
    c_out[(size_t)i * ldb + k] = c;
    s_out[(size_t)i * ldb + k] = s;
}

// ---- a3: R(phi_k) = sum_i K w_i (cos th - i sin th); one warp per depth, FP64.
__global__ void rmsf_kernel(const double* __restrict__ delta, const double* __restrict__ kw,
                            const double* __restrict__ phi, int n_chan, int n,
                            double* __restrict__ re, double* __restrict__ im) {
    int k = blockIdx.x * (blockDim.x / 32) + threadIdx.x / 32;
    int lane = threadIdx.x % 32;
    if (k >= n) return;
    double sr = 0.0, si = 0.0;
    for (int i = lane; i < n_chan; i += 32) {
        double sn, cs;
        sincos(2.0 * phi[k] * delta[i], &sn, &cs);
        sr += kw[i] * cs;
        si -= kw[i] * sn;
    }
    for (int o = 16; o > 0; o >>= 1) {
        sr += __shfl_xor_sync(0xffffffffu, sr, o);
        si += __shfl_xor_sync(0xffffffffu, si, o);
    }
    if (lane == 0) { re[k] = sr; im[k] = si; }
}

// R(phi) for n device-resident depths into device arrays (used by rmclean.cu for the double-width beam)
rmsynth_status device_rmsf_to(const rmsynth_plan* p, const double* d_phi, int n, double* d_re, double* d_im) {
    rmsf_kernel<<<(n + 3) / 4, 128>>>(p->d_delta, p->d_kw, d_phi, p->n_chan, n, d_re, d_im);
    RMS_LAUNCH_CHECK("rmsf_kernel");
    return RMSYNTH_OK;
}

static rmsynth_status device_rmsf(const rmsynth_plan* p, const double* d_phi, int n, double* re, double* im) {
    double* d_out = nullptr;
    RMS_CUDA(cudaMalloc(&d_out, sizeof(double) * 2 * (size_t)n));
    rmsf_kernel<<<(n + 3) / 4, 128>>>(p->d_delta, p->d_kw, d_phi, p->n_chan, n, d_out, d_out + n);
    count_launch();
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaMemcpy(re, d_out, sizeof(double) * n, cudaMemcpyDeviceToHost);
    if (e == cudaSuccess) e = cudaMemcpy(im, d_out + n, sizeof(double) * n, cudaMemcpyDeviceToHost);
    cudaFree(d_out);
    if (e != cudaSuccess) return fail(RMSYNTH_ECUDA, std::string("rmsf: ") + cudaGetErrorString(e));
    return RMSYNTH_OK;
}

template <class T>
static rmsynth_status upload(T** dst, const std::vector<T>& v) {
    RMS_CUDA(cudaMalloc(dst, sizeof(T) * v.size()));
    RMS_CUDA(cudaMemcpy(*dst, v.data(), sizeof(T) * v.size(), cudaMemcpyHostToDevice));
    return RMSYNTH_OK;
}

static rmsynth_status build_plan(rmsynth_plan* p) {
    const int nc = p->n_chan, np = p->n_phi;
    std::vector<double> delta(nc), kw(nc);
    std::vector<float> kwf(nc), phif(np);
    std::vector<float2> dpi(nc), phi2(np);
    const double two_over_pi = 0.63661977236758134308;
    for (int i = 0; i < nc; ++i) {
        delta[i] = p->lam2[i] - p->lambda0_sq;
        kw[i] = p->K * p->w[i];
        kwf[i] = (float)kw[i];
        double d = two_over_pi * delta[i];
        float hi = (float)d;
        dpi[i] = make_float2(hi, (float)(d - (double)hi));
    }
    for (int k = 0; k < np; ++k) {
        float hi = (float)p->phi[k];
        phif[k] = hi;
        phi2[k] = make_float2(hi, (float)(p->phi[k] - (double)hi));
    }
    rmsynth_status st;
    if ((st = upload(&p->d_delta, delta)) || (st = upload(&p->d_kw, kw)) || (st = upload(&p->d_phi, p->phi)) ||
        (st = upload(&p->d_kwf, kwf)) || (st = upload(&p->d_phif, phif)) || (st = upload(&p->d_dpi, dpi)) ||
        (st = upload(&p->d_phi2, phi2)))
        return st;
    p->ldb = (np + 3) & ~3;
    size_t nb = sizeof(float) * (size_t)nc * p->ldb;
    RMS_CUDA(cudaMalloc(&p->d_cos, nb));
    RMS_CUDA(cudaMalloc(&p->d_sin, nb));
    dim3 grid((p->ldb + 127) / 128, nc);
    phase_matrix_kernel<<<grid, 128>>>(p->d_delta, p->d_kw, p->d_phi, nc, np, p->ldb, p->d_cos, p->d_sin);
    RMS_LAUNCH_CHECK("phase_matrix_kernel");
    p->R_re.resize(np);
    p->R_im.resize(np);
    if ((st = device_rmsf(p, p->d_phi, np, p->R_re.data(), p->R_im.data()))) return st;
    if ((p->scheme == RMSYNTH_SCHEME_TF32X3 || p->scheme == RMSYNTH_SCHEME_F16X3) && (st = tc_plan_init(p))) return st;
    RMS_CUDA(cudaDeviceSynchronize());
    return RMSYNTH_OK;
}

}  // namespace rms

using namespace rms;

extern "C" {

rmsynth_status rmsynth_plan_create(rmsynth_plan** plan, const double* nu_hz, const double* w, int n_chan,
                                   const double* phi, int n_phi, const rmsynth_options* opt) {
    if (!plan) return fail(RMSYNTH_EINVAL, "plan is NULL");
    *plan = nullptr;
    if (!nu_hz || !phi) return fail(RMSYNTH_EINVAL, "nu_hz/phi is NULL");
    if (n_chan < 1 || n_phi < 1) return fail(RMSYNTH_EINVAL, "n_chan and n_phi must be >= 1");
    rmsynth_options o;
    std::memset(&o, 0, sizeof(o));
    o.device = -1;
    if (opt) {
        if (opt->struct_size < (int)(4 * sizeof(int)) || opt->struct_size > (int)sizeof(o))
            return fail(RMSYNTH_EINVAL, "options.struct_size");
        std::memcpy(&o, opt, opt->struct_size);
    }
    int scheme = o.scheme;
    if (scheme == RMSYNTH_SCHEME_AUTO) {
        // FP16 split (twice the tensor rate) unless (a) the weights span more than 2^18: B = K w cos/sin carries one
        // power-of-two scale for the whole plan, and below 2^-18 of the largest weight its FP16 lo part goes
        // subnormal (3xTF32 has FP32's exponent range and no such limit); or (b) there are fewer than 384 channels:
        // the FP16 kernel's gain comes from the K loop while its per-tile costs (drains, stores) do not shrink --
        // measured on B200 it is 1.4x faster at 800-1000 channels and 1.14x at 400.
        double wmax = 0.0, wmin = 0.0;
        for (int i = 0; i < n_chan; ++i) {
            const double wi = w ? w[i] : 1.0;
            if (wi > wmax) wmax = wi;
            if (wi > 0.0 && (wmin == 0.0 || wi < wmin)) wmin = wi;
        }
        scheme = (n_chan >= 384 && wmax > 0.0 && wmin >= wmax * (1.0 / 262144.0)) ? RMSYNTH_SCHEME_F16X3 : RMSYNTH_SCHEME_TF32X3;
    }
    if (scheme != RMSYNTH_SCHEME_TF32X3 && scheme != RMSYNTH_SCHEME_F16X3 && scheme != RMSYNTH_SCHEME_FP32_TABLE && scheme != RMSYNTH_SCHEME_FP32_SINCOS)
        return fail(RMSYNTH_EINVAL, "unknown scheme");
    if (o.lambda0_mode < 0 || o.lambda0_mode > 2) return fail(RMSYNTH_EINVAL, "unknown lambda0_mode");
    if (o.lambda0_mode == 2 && !std::isfinite(o.lambda0_sq)) return fail(RMSYNTH_EINVAL, "lambda0_sq not finite");
    if (o.host_chunk_pixels < 0) return fail(RMSYNTH_EINVAL, "host_chunk_pixels < 0");

    rmsynth_plan* p = new (std::nothrow) rmsynth_plan;
    if (!p) return fail(RMSYNTH_ENOMEM, "plan");
    p->n_chan = n_chan;
    p->n_phi = n_phi;
    p->scheme = scheme;
    p->lambda0_mode = o.lambda0_mode;
    p->host_chunk_pixels = o.host_chunk_pixels;
    const double c = 299792458.0;
    double W = 0.0, S = 0.0, M = 0.0;
    p->lam2.resize(n_chan);
    p->w.resize(n_chan);
    for (int i = 0; i < n_chan; ++i) {
        double wi = w ? w[i] : 1.0;
        if (!std::isfinite(nu_hz[i]) || nu_hz[i] <= 0.0 || !std::isfinite(wi) || wi < 0.0) {
            delete p;
            return fail(RMSYNTH_EINVAL, "nu_hz must be finite and > 0, w finite and >= 0");
        }
        double lam = c / nu_hz[i];
        p->lam2[i] = lam * lam;
        p->w[i] = wi;
        W += wi;
        S += wi * p->lam2[i];
        M += p->lam2[i];
    }
    if (!(W > 0.0) || !std::isfinite(W)) {
        delete p;
        return fail(RMSYNTH_EINVAL, "sum of weights must be > 0");
    }
    p->phi.assign(phi, phi + n_phi);
    for (int k = 0; k < n_phi; ++k)
        if (!std::isfinite(phi[k])) {
            delete p;
            return fail(RMSYNTH_EINVAL, "phi must be finite");
        }
    // uniform grid? (RM-CLEAN shifts one beam along the grid, reading C1)
    p->dphi = n_phi > 1 ? (phi[n_phi - 1] - phi[0]) / (n_phi - 1) : 1.0;
    p->uniform_phi = p->dphi != 0.0;
    for (int k = 1; k < n_phi && p->uniform_phi; ++k)
        if (std::fabs((phi[k] - phi[k - 1]) - p->dphi) > 1e-9 * std::fabs(p->dphi)) p->uniform_phi = false;
    p->K = 1.0 / W;
    p->lambda0_sq = o.lambda0_mode == 0 ? S / W : (o.lambda0_mode == 1 ? M / n_chan : o.lambda0_sq);

    DeviceGuard guard(o.device);                       // the plan's device for the rest of this call, the caller's afterwards
    int dev = o.device;
    cudaError_t e = guard.err;
    if (e == cudaSuccess && dev < 0) e = cudaGetDevice(&dev);
    cudaDeviceProp prop;
    if (e == cudaSuccess) e = cudaGetDeviceProperties(&prop, dev);
    if (e != cudaSuccess) {
        delete p;
        return fail(RMSYNTH_ECUDA, std::string("no usable CUDA device: ") + cudaGetErrorString(e));
    }
    if (prop.major != 10) {
        delete p;
        return fail(RMSYNTH_EUNSUPPORTED, "librmsynth is built for sm_100a (B200) only");
    }
    p->device = dev;
    p->sm_count = prop.multiProcessorCount;
    rmsynth_status st = build_plan(p);
    if (st != RMSYNTH_OK) {
        std::string keep = t_last_error;
        rmsynth_plan_destroy(p);
        t_last_error = keep;
        return st;
    }
    *plan = p;
    return RMSYNTH_OK;
}

rmsynth_status rmsynth_plan_destroy(rmsynth_plan* p) {
    if (!p) return RMSYNTH_OK;
    DeviceGuard guard(p->device);
    tc_plan_free(p);
    void* ptrs[] = {p->d_delta, p->d_kw, p->d_phi, p->d_cos, p->d_sin, p->d_phif, p->d_kwf, p->d_dpi, p->d_phi2, p->d_Rdw, p->d_gauss};
    for (void* q : ptrs)
        if (q) cudaFree(q);
    for (int i = 0; i < rmsynth_plan::kScratch; ++i)
        if (p->scratch[i]) cudaFree(p->scratch[i]);
    for (auto& x : p->pool)
        if (x.ptr) cudaFree(x.ptr);
    for (float* q : p->retired) cudaFree(q);
    host_pipe_free(p);
    fft_tables_free(p);
    delete p;
    return RMSYNTH_OK;
}

rmsynth_status rmsynth_plan_info(const rmsynth_plan* p, double* lambda0_sq, double* K, int* n_chan, int* n_phi,
                                 int* scheme) {
    if (!p) return fail(RMSYNTH_EINVAL, "plan is NULL");
    if (lambda0_sq) *lambda0_sq = p->lambda0_sq;
    if (K) *K = p->K;
    if (n_chan) *n_chan = p->n_chan;
    if (n_phi) *n_phi = p->n_phi;
    if (scheme) *scheme = p->scheme;
    return RMSYNTH_OK;
}

rmsynth_status rmsynth_plan_phase_matrix(const rmsynth_plan* p, float* cos_kw, float* sin_kw) {
    if (!p) return fail(RMSYNTH_EINVAL, "plan is NULL");
    DeviceGuard guard(p->device);
    RMS_CUDA(guard.err);
    size_t row = sizeof(float) * p->n_phi;
    if (cos_kw)
        RMS_CUDA(cudaMemcpy2D(cos_kw, row, p->d_cos, sizeof(float) * p->ldb, row, p->n_chan, cudaMemcpyDeviceToHost));
    if (sin_kw)
        RMS_CUDA(cudaMemcpy2D(sin_kw, row, p->d_sin, sizeof(float) * p->ldb, row, p->n_chan, cudaMemcpyDeviceToHost));
    return RMSYNTH_OK;
}

rmsynth_status rmsynth_rmsf(const rmsynth_plan* p, const double* phi_eval, int n, double* R_re, double* R_im) {
    if (!p || !R_re || !R_im) return fail(RMSYNTH_EINVAL, "NULL argument");
    if (!phi_eval) {
        if (n != p->n_phi) return fail(RMSYNTH_EINVAL, "n must equal n_phi when phi_eval is NULL");
        std::memcpy(R_re, p->R_re.data(), sizeof(double) * n);
        std::memcpy(R_im, p->R_im.data(), sizeof(double) * n);
        return RMSYNTH_OK;
    }
    if (n < 0) return fail(RMSYNTH_EINVAL, "n < 0");
    if (n == 0) return RMSYNTH_OK;
    for (int k = 0; k < n; ++k)
        if (!std::isfinite(phi_eval[k])) return fail(RMSYNTH_EINVAL, "phi_eval must be finite");
    DeviceGuard guard(p->device);
    RMS_CUDA(guard.err);
    double* d_phi = nullptr;
    RMS_CUDA(cudaMalloc(&d_phi, sizeof(double) * n));
    cudaError_t e = cudaMemcpy(d_phi, phi_eval, sizeof(double) * n, cudaMemcpyHostToDevice);
    rmsynth_status st = e == cudaSuccess ? device_rmsf(p, d_phi, n, R_re, R_im)
                                         : fail(RMSYNTH_ECUDA, cudaGetErrorString(e));
    cudaFree(d_phi);
    return st;
}

long long rmsynth_launch_count(int reset) {
    return reset ? g_launches.exchange(0) : g_launches.load();
}

const char* rmsynth_strerror(rmsynth_status s) {
    switch (s) {
        case RMSYNTH_OK: return "ok";
        case RMSYNTH_EINVAL: return "invalid argument";
        case RMSYNTH_ENOMEM: return "out of memory";
        case RMSYNTH_ECUDA: return "CUDA error";
        case RMSYNTH_EUNSUPPORTED: return "unsupported device or configuration";
    }
    return "unknown status";
}

const char* rmsynth_last_error(void) { return t_last_error.c_str(); }
#ifndef RMSYNTH_SOURCE_HASH
#define RMSYNTH_SOURCE_HASH "unknown"
#endif
// the hash is the SHA-256 prefix of the sources this binary was compiled from (paper_1810_06250_b200/build.py)
const char* rmsynth_version(void) { return "rmsynth-b200 0.2 (sm_100a) src " RMSYNTH_SOURCE_HASH; }

}  // extern "C"
