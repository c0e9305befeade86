// Approximate fast path (scope row NEXT-4): "Further increase in speed can be achieved by using Fast Fourier
// Transforms (FFT) instead of Discrete Fourier Transforms (DFT) in equations 15 and 16".  Channels are not
// uniform in lambda^2, so this is a non-uniform FFT of type 1 per line of sight (readings F1-F6, DESIGN.md
// section 2c; Dutt & Rokhlin 1993, Greengard & Lee 2004, Kaiser-Bessel window as in Beatty et al. 2005):
//   F1  c_i = K w_i P_i exp(-2i phi_kc x_i), x_i = lambda_i^2 - lambda_0^2, kc = N/2:  F_k = sum_i c_i exp(-2 pi i (k - kc) t_i)
//   F2  fine grid of M = 2^ceil(log2(sigma N)) points, channel i at u_i = M t_i mod M, t_i = dphi x_i / pi
//   F3  g[m] = sum_i c_i psi(m - u_i), Kaiser-Bessel window of width W
//   F4  G = FFT_M(g)          F5  F_k = G[(k - kc) mod M] / psihat(k - kc)          F6  zero-weight channels skipped
// Everything that does not depend on the line of sight is tabulated at plan time in FP64: the pre-phase, the spreading
// matrix in gather form (for every fine-grid point the channels whose window covers it, CSR), the twiddles, 1/psihat.
// Kernel: a CTA of 256 threads takes a batch of B consecutive pixels (B = 8 .. 1, as many as fit in shared memory; B = 8
// makes 32-byte sectors of FITS-order cubes), forms c[B][n_chan], gathers g[B][M], runs an in-place radix-2
// decimation-in-frequency FFT in shared memory (bit-reversed output, read back through __brev -- no reorder pass),
// deapodises and stores.  Error against the exact contraction: the window's (tests: <= 2e-6 T_p at W = 6, sigma = 2, falling
// a decade per unit of W) plus FP32 rounding of the FFT (~1e-6 T_p).
#include <cmath>
#include "common.cuh"

namespace rms {

struct FftTables {
    int W = 0, M = 0, log2M = 0, kc = 0;
    float sigma = 0.f;
    float2* d_pre = nullptr;      // [n_chan]  K w_i exp(-2i phi_kc x_i)  (0 for flagged channels)
    int* d_row = nullptr;         // [M + 1]   CSR row pointers: entries of fine-grid point m
    int* d_col = nullptr;         // [nnz]     channel
    float* d_val = nullptr;       // [nnz]     psi(m - u_i)
    float2* d_tw = nullptr;       // [M / 2]   exp(-2 pi i j / M)
    float* d_hat_inv = nullptr;   // [n_phi]   1 / psihat(k - kc)
    void free_all() {
        void* ptrs[] = {d_pre, d_row, d_col, d_val, d_tw, d_hat_inv};
        for (void* q : ptrs)
            if (q) cudaFree(q);
        *this = FftTables();
    }
};

struct FftArgs {
    const float* Q; const float* U; float* FQ; float* FU;
    long long n_pix;
    int n_chan, n_phi, in_freq, out_phi, M, log2M, kc, B;
    const float2* pre; const int* row; const int* col; const float* val; const float2* tw; const float* hat_inv;
};

constexpr int FV_THREADS = 256;

__global__ void __launch_bounds__(FV_THREADS) fft_variant_kernel(const FftArgs a) {
    extern __shared__ float2 fv_smem[];
    const int nc = a.n_chan, M = a.M, B = a.B;
    float2* c = fv_smem;                    // [B][nc]
    float2* g = fv_smem + (size_t)B * nc;   // [B][M]
    const long long n_batches = (a.n_pix + B - 1) / B;
    for (long long batch = blockIdx.x; batch < n_batches; batch += gridDim.x) {
        const long long p0 = batch * B;
        // F1: c = pre * (Q + iU).  FITS order: B consecutive pixels of one channel are contiguous (a 32-byte sector for B = 8)
        for (int e = threadIdx.x; e < B * nc; e += FV_THREADS) {
            const int j = a.in_freq ? e % B : e / nc, i = a.in_freq ? e / B : e % nc;
            const long long p = p0 + j;
            float2 v = make_float2(0.f, 0.f);
            const float2 pr = a.pre[i];
            if (p < a.n_pix && (pr.x != 0.f || pr.y != 0.f)) {          // F6: flagged channels are never read
                const size_t o = a.in_freq ? (size_t)i * a.n_pix + p : (size_t)p * nc + i;
                const float q = a.Q[o], u = a.U[o];
                v = make_float2(pr.x * q - pr.y * u, pr.x * u + pr.y * q);
            }
            c[(size_t)j * nc + i] = v;
        }
        __syncthreads();
        // F3 in gather form: every fine-grid point sums the channels whose window covers it -- no atomics
        for (int m = threadIdx.x; m < M; m += FV_THREADS) {
            const int e0 = a.row[m], e1 = a.row[m + 1];
            for (int j = 0; j < B; ++j) {
                float sx = 0.f, sy = 0.f;
                for (int e = e0; e < e1; ++e) {
                    const float w = a.val[e];
                    const float2 v = c[(size_t)j * nc + a.col[e]];
                    sx = fmaf(w, v.x, sx);
                    sy = fmaf(w, v.y, sy);
                }
                g[(size_t)j * M + m] = make_float2(sx, sy);
            }
        }
        __syncthreads();
        // F4: in-place radix-2 DIF, natural order in, bit-reversed order out
        for (int s = 0; s < a.log2M; ++s) {
            const int span = M >> (s + 1);                                  // distance between the two legs
            for (int e = threadIdx.x; e < B * (M / 2); e += FV_THREADS) {
                const int j = e / (M / 2), t = e % (M / 2);
                const int lo = ((t / span) * 2 * span) + (t % span), hi = lo + span;
                float2* x = g + (size_t)j * M;
                const float2 u = x[lo], v = x[hi];
                const float2 w = __ldg(a.tw + (size_t)(t % span) * (M / (2 * span)));
                const float dx = u.x - v.x, dy = u.y - v.y;
                x[lo] = make_float2(u.x + v.x, u.y + v.y);
                x[hi] = make_float2(dx * w.x - dy * w.y, dx * w.y + dy * w.x);
            }
            __syncthreads();
        }
        // F5: F_k = G[(k - kc) mod M] / psihat(k - kc); G sits at the bit-reversed position
        for (int e = threadIdx.x; e < B * a.n_phi; e += FV_THREADS) {
            const int j = a.out_phi ? e % B : e / a.n_phi, k = a.out_phi ? e / B : e % a.n_phi;
            const long long p = p0 + j;
            if (p >= a.n_pix) continue;
            const unsigned idx = (unsigned)((k - a.kc) & (M - 1));
            const unsigned rev = __brev(idx) >> (32 - a.log2M);
            const float2 v = g[(size_t)j * M + rev];
            const float h = a.hat_inv[k];
            const size_t o = a.out_phi ? (size_t)k * a.n_pix + p : (size_t)p * a.n_phi + k;
            a.FQ[o] = v.x * h;
            a.FU[o] = v.y * h;
        }
        __syncthreads();
    }
}

static double bessel_i0(double x) {            // power series, converges for every x used here (beta <= ~40)
    double sum = 1.0, term = 1.0;
    const double q = x * x / 4.0;
    for (int k = 1; k < 500; ++k) {
        term *= q / ((double)k * k);
        sum += term;
        if (term < 1e-17 * sum) break;
    }
    return sum;
}

static rmsynth_status build_tables(const rmsynth_plan* p, int W, float sigma, FftTables& t) {
    const int n = p->n_phi, nc = p->n_chan;
    int M = 1, lg = 0;
    while (M < sigma * n) { M *= 2; ++lg; }
    if (M < 2) { M = 2; lg = 1; }
    const double s = (double)M / n;
    const double beta = M_PI * std::sqrt((double)W * W / (s * s) * (s - 0.5) * (s - 0.5) - 0.8);
    const double i0b = bessel_i0(beta);
    auto psi = [&](double z) {
        const double a = 1.0 - (2.0 * z / W) * (2.0 * z / W);
        return a >= 0.0 ? bessel_i0(beta * std::sqrt(a)) / i0b : 0.0;
    };
    const int kc = n / 2;
    std::vector<float2> pre(nc);
    std::vector<std::vector<std::pair<int, float>>> rows(M);
    for (int i = 0; i < nc; ++i) {
        const double x = p->lam2[i] - p->lambda0_sq;
        if (p->w[i] == 0.0) { pre[i] = make_float2(0.f, 0.f); continue; }
        const double kw = p->K * p->w[i], ang = -2.0 * p->phi[kc] * x;
        pre[i] = make_float2((float)(kw * std::cos(ang)), (float)(kw * std::sin(ang)));
        double u = std::fmod(M * (p->dphi * x / M_PI), (double)M);
        if (u < 0) u += M;
        const long long m0 = (long long)std::ceil(u - W / 2.0);
        for (int j = 0; j < W; ++j) {
            const long long m = m0 + j;
            const double v = psi((double)m - u);
            if (v != 0.0) rows[(size_t)(((m % M) + M) % M)].push_back({i, (float)v});
        }
    }
    std::vector<int> row(M + 1, 0), col;
    std::vector<float> val;
    for (int m = 0; m < M; ++m) {
        row[m + 1] = row[m] + (int)rows[m].size();
        for (auto& e : rows[m]) { col.push_back(e.first); val.push_back(e.second); }
    }
    if (col.empty()) { col.push_back(0); val.push_back(0.f); }
    std::vector<float2> tw(M / 2);
    for (int j = 0; j < M / 2; ++j) tw[j] = make_float2((float)std::cos(-2.0 * M_PI * j / M), (float)std::sin(-2.0 * M_PI * j / M));
    std::vector<float> hat_inv(n);
    const int nq = 2048;
    for (int k = 0; k < n; ++k) {                  // F5: window transform at (k - kc) / M by the midpoint rule
        double acc = 0.0;
        for (int q = 0; q < nq; ++q) {
            const double z = (q + 0.5) / nq * W - W / 2.0;
            acc += psi(z) * std::cos(2.0 * M_PI * (k - kc) * z / M);
        }
        hat_inv[k] = (float)(1.0 / (acc * W / nq));
    }
    t.free_all();
    t.W = W; t.M = M; t.log2M = lg; t.kc = kc; t.sigma = sigma;
    RMS_CUDA(cudaMalloc(&t.d_pre, sizeof(float2) * nc));
    RMS_CUDA(cudaMalloc(&t.d_row, sizeof(int) * (M + 1)));
    RMS_CUDA(cudaMalloc(&t.d_col, sizeof(int) * col.size()));
    RMS_CUDA(cudaMalloc(&t.d_val, sizeof(float) * val.size()));
    RMS_CUDA(cudaMalloc(&t.d_tw, sizeof(float2) * (M / 2)));
    RMS_CUDA(cudaMalloc(&t.d_hat_inv, sizeof(float) * n));
    RMS_CUDA(cudaMemcpy(t.d_pre, pre.data(), sizeof(float2) * nc, cudaMemcpyHostToDevice));
    RMS_CUDA(cudaMemcpy(t.d_row, row.data(), sizeof(int) * (M + 1), cudaMemcpyHostToDevice));
    RMS_CUDA(cudaMemcpy(t.d_col, col.data(), sizeof(int) * col.size(), cudaMemcpyHostToDevice));
    RMS_CUDA(cudaMemcpy(t.d_val, val.data(), sizeof(float) * val.size(), cudaMemcpyHostToDevice));
    RMS_CUDA(cudaMemcpy(t.d_tw, tw.data(), sizeof(float2) * (M / 2), cudaMemcpyHostToDevice));
    RMS_CUDA(cudaMemcpy(t.d_hat_inv, hat_inv.data(), sizeof(float) * n, cudaMemcpyHostToDevice));
    return RMSYNTH_OK;
}

void fft_tables_free(rmsynth_plan* p) {
    FftTables* t = static_cast<FftTables*>(p->fft_tables);
    if (!t) return;
    t->free_all();
    delete t;
    p->fft_tables = nullptr;
}

}  // namespace rms

using namespace rms;

extern "C" rmsynth_status rmsynth_execute_fft(const rmsynth_plan* plan, const float* Q, const float* U, long long n_pix, int layout,
                                              float* FQ, float* FU, const rmsynth_fft_params* prm, void* stream) {
    if (!plan) return fail(RMSYNTH_EINVAL, "plan is NULL");
    if (n_pix < 0) return fail(RMSYNTH_EINVAL, "n_pix < 0");
    if (layout & ~3) return fail(RMSYNTH_EINVAL, "unknown layout flags");
    int W = 6;
    float sigma = 2.f;
    if (prm) {
        if (prm->struct_size != (int)sizeof(rmsynth_fft_params)) return fail(RMSYNTH_EINVAL, "fft_params.struct_size");
        if (prm->window) W = prm->window;
        if (prm->oversampling > 0.f) sigma = prm->oversampling;
    }
    if (W < 2 || W > 16 || (W & 1)) return fail(RMSYNTH_EINVAL, "window must be even, 2..16");
    if (!(sigma >= 1.25f) || sigma > 8.f) return fail(RMSYNTH_EINVAL, "oversampling must be in [1.25, 8]");
    if (n_pix == 0) return RMSYNTH_OK;
    if (!Q || !U || !FQ || !FU) return fail(RMSYNTH_EINVAL, "NULL cube pointer");
    const rmsynth_plan* p = plan;
    if (!p->uniform_phi) return fail(RMSYNTH_EUNSUPPORTED, "the FFT variant needs a uniform depth grid (reading F1)");
    DeviceGuard g(p->device);
    RMS_CUDA(g.err);
    cudaStream_t st = (cudaStream_t)stream;
    FftTables* t;
    {
        std::lock_guard<std::mutex> lock(p->mu);
        if (!p->fft_tables) p->fft_tables = new FftTables;
        t = static_cast<FftTables*>(p->fft_tables);
        if (t->W != W || t->sigma != sigma) {
            RMS_CUDA(cudaStreamSynchronize(st));          // an earlier call on this stream may still read the old tables
            rmsynth_status s = build_tables(p, W, sigma, *t);
            if (s != RMSYNTH_OK) return s;
        }
    }
    FftArgs a;
    a.Q = Q; a.U = U; a.FQ = FQ; a.FU = FU; a.n_pix = n_pix; a.n_chan = p->n_chan; a.n_phi = p->n_phi;
    a.in_freq = (layout & RMSYNTH_IN_FREQ_MAJOR) ? 1 : 0; a.out_phi = (layout & RMSYNTH_OUT_PHI_MAJOR) ? 1 : 0;
    a.M = t->M; a.log2M = t->log2M; a.kc = t->kc;
    a.pre = t->d_pre; a.row = t->d_row; a.col = t->d_col; a.val = t->d_val; a.tw = t->d_tw; a.hat_inv = t->d_hat_inv;
    const size_t per_pix = sizeof(float2) * ((size_t)p->n_chan + t->M);
    int B = 8;
    while (B > 1 && per_pix * B > 100 * 1024) B >>= 1;       // <= 100 KB: two CTAs per SM
    if (per_pix * B > 220 * 1024) return fail(RMSYNTH_EUNSUPPORTED, "the FFT variant: fine grid does not fit in shared memory");
    a.B = B;
    const size_t smem = per_pix * B;
    RMS_CUDA(cudaFuncSetAttribute(fft_variant_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const long long n_batches = (n_pix + B - 1) / B;
    const int per_sm = smem <= 100 * 1024 ? 2 : 1;
    const long long grid = std::min<long long>(n_batches, (long long)p->sm_count * per_sm);
    fft_variant_kernel<<<(unsigned)grid, FV_THREADS, smem, st>>>(a);
    RMS_LAUNCH_CHECK("fft_variant_kernel");
    return RMSYNTH_OK;
}
