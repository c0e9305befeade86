// RM-CLEAN per line of sight (scope row NEXT-3): Hogbom CLEAN of the complex dirty Faraday spectrum F~(phi_k) with the
// complex RMSF R (Eq. 12) as the beam.  The paper only names the procedure ("a procedure called RM-CLEAN
// (Heald 2009)", footnote 6 P:L151); the loop is the reading C1-C8 of DESIGN.md section 2b:
//   C1 uniform depth grid; R on the double-width grid R((k - j) dphi), 2 n_phi - 1 samples
//   C2 residual r <- F~, model m <- 0
//   C3 k* = lowest index of max |r_k| (|r|^2 compared in FP32); stop before subtracting if |r_k*| < cutoff or after max_iter
//   C4 c = gain r_k*;  m_k* += c;  r_k -= c R[k - k*]
//   C5 restored = sum_j m_j G((k - j) dphi) + r_k, real Gaussian of the given FWHM
//   C7 a line of sight with a non-finite sample is passed through (model 0, residual = restored = input, 0 iterations)
// Two kernels.  (a) n_phi <= 1024: one warp per line of sight, the residual in registers (lane l holds depths l + 32 i),
// R, the Gaussian table and the eight warps' model arrays in shared memory, arg-max by warp shuffles; a CTA takes eight
// consecutive pixels so that phi-major cubes are read and written in 32-byte sectors through a staging buffer.
// (b) larger grids (the paper's 7000 depths): one CTA per line of sight, residual in registers, model in shared memory.
#include <cmath>
#include "common.cuh"

namespace rms {

struct CleanArgs {
    const float* FQ; const float* FU;
    float *mq, *mu, *rq, *ru, *sq, *su;       // model, residual, restored (sq/su may be NULL)
    int* n_iter;                              // may be NULL
    long long n_pix;
    int n_phi, out_phi, max_iter;
    float gain, cutoff2;                      // cutoff^2: compared with |r|^2
    const float2* Rdw;                        // [2 n_phi - 1], R(0) at index n_phi - 1
    const float* gauss;                       // [n_phi]  exp(-(m dphi)^2 / (2 sigma^2)), m = 0 .. n_phi - 1
    int gauss_reach;                          // beyond this many samples the Gaussian is < 1e-9 (6.5 sigma) and is skipped
};

__device__ __forceinline__ size_t cube_index(const CleanArgs& a, long long p, int k) {
    return a.out_phi ? (size_t)k * a.n_pix + p : (size_t)p * a.n_phi + k;
}

// ---- (a) warp per line of sight, NPL depths per lane ---------------------------------------------------------------
constexpr int CL_WARPS = 8;

template <int NPL>
__global__ void __launch_bounds__(CL_WARPS * 32, NPL <= 16 ? 3 : 1) rmclean_warp_kernel(const CleanArgs a) {
    extern __shared__ float2 smem2[];
    const int n = a.n_phi, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    float2* sR = smem2;                                   // [2n - 1]
    float2* sStage = sR + (2 * n - 1);                    // [CL_WARPS][n]: dirty in, then model, then the outputs
    float* sG = reinterpret_cast<float*>(sStage + (size_t)CL_WARPS * n);   // [n]
    for (int i = threadIdx.x; i < 2 * n - 1; i += blockDim.x) sR[i] = a.Rdw[i];
    for (int i = threadIdx.x; i < n; i += blockDim.x) sG[i] = a.gauss[i];
    const long long p0 = (long long)blockIdx.x * CL_WARPS;
    // stage the eight dirty spectra: phi-major cubes are read as 32-byte sectors (8 pixels of one depth)
    for (int i = threadIdx.x; i < CL_WARPS * n; i += blockDim.x) {
        const int j = a.out_phi ? i % CL_WARPS : i / n, k = a.out_phi ? i / CL_WARPS : i % n;
        const long long p = p0 + j;
        float2 v = make_float2(0.f, 0.f);
        if (p < a.n_pix) { const size_t o = cube_index(a, p, k); v = make_float2(a.FQ[o], a.FU[o]); }
        sStage[(size_t)j * n + k] = v;
    }
    __syncthreads();
    float2* mine = sStage + (size_t)warp * n;
    float rq[NPL], ru[NPL];
    float bad = 0.f;
#pragma unroll
    for (int i = 0; i < NPL; ++i) {
        const int k = lane + 32 * i;
        const float2 v = k < n ? mine[k] : make_float2(0.f, 0.f);
        rq[i] = v.x; ru[i] = v.y;
        bad = fmaf(v.x, 0.f, fmaf(v.y, 0.f, bad));        // sticky NaN for non-finite samples
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) bad += __shfl_xor_sync(0xffffffffu, bad, o);
    const bool finite = bad == 0.f;                       // warp-uniform after the reduction
    __syncwarp();
    for (int k = lane; k < n; k += 32) mine[k] = make_float2(0.f, 0.f);   // the staging row becomes the model (C2)
    __syncwarp();
    int it = 0;
    const int c0 = n - 1;
    while (finite && it < a.max_iter) {
        // C3: arg-max of |r|^2, lowest depth on ties: per lane over i (strict >), then across lanes on (value, depth)
        float y = -1.f, cq = 0.f, cu = 0.f;
        int kb = 0;
#pragma unroll
        for (int i = 0; i < NPL; ++i) {
            const float v = lane + 32 * i < n ? fmaf(rq[i], rq[i], ru[i] * ru[i]) : -1.f;
            if (v > y) { y = v; kb = lane + 32 * i; cq = rq[i]; cu = ru[i]; }
        }
        {   // two warp reductions (redux.sync) instead of five shuffle stages: |r|^2 >= 0, so its bit pattern orders like an
            // unsigned integer; among the lanes holding the maximum the lowest depth wins; its owner is lane kb & 31
            // a lane beyond the grid (n_phi < 32) holds no depth: its -1 sentinel would sort above every real value as an
            // unsigned integer, so it enters the reductions as the lowest value and never as a candidate depth
            const bool has = y >= 0.f;
            const unsigned yb = has ? __float_as_uint(y) : 0u, ymax = __reduce_max_sync(0xffffffffu, yb);
            kb = (int)__reduce_min_sync(0xffffffffu, has && yb == ymax ? (unsigned)kb : 0x7fffffffu);
            y = __uint_as_float(ymax);
            cq = __shfl_sync(0xffffffffu, cq, kb & 31);
            cu = __shfl_sync(0xffffffffu, cu, kb & 31);
        }
        if (y < a.cutoff2) break;
        cq *= a.gain; cu *= a.gain;                       // C4
        if (lane == (kb & 31)) { float2 m = mine[kb]; m.x += cq; m.y += cu; mine[kb] = m; }
        const float2* beam = sR + (c0 - kb);
#pragma unroll
        for (int i = 0; i < NPL; ++i) {
            const int k = lane + 32 * i;
            if (k < n) {
                const float2 b = beam[k];
                rq[i] -= cq * b.x - cu * b.y;
                ru[i] -= cq * b.y + cu * b.x;
            }
        }
        ++it;
    }
    __syncwarp();
    const long long p = p0 + warp;
    if (a.n_iter && lane == 0 && p < a.n_pix) a.n_iter[p] = it;
    // C5: restored = model convolved with the Gaussian + residual, component-driven (the model is sparse)
    float sq[NPL], su[NPL];
    if (a.sq) {
#pragma unroll
        for (int i = 0; i < NPL; ++i) { sq[i] = rq[i]; su[i] = ru[i]; }
        for (int kc = 0; kc < n; kc += 32) {
            const int k = kc + lane;
            const float2 m = k < n ? mine[k] : make_float2(0.f, 0.f);
            unsigned mask = __ballot_sync(0xffffffffu, m.x != 0.f || m.y != 0.f);
            while (mask) {
                const int src = __ffs(mask) - 1;
                mask &= mask - 1;
                const float cq = __shfl_sync(0xffffffffu, m.x, src), cu = __shfl_sync(0xffffffffu, m.y, src);
                const int j = kc + src;
#pragma unroll
                for (int i = 0; i < NPL; ++i) {
                    const int kk = lane + 32 * i, d = kk > j ? kk - j : j - kk;
                    if (kk < n && d <= a.gauss_reach) { const float g = sG[d]; sq[i] = fmaf(cq, g, sq[i]); su[i] = fmaf(cu, g, su[i]); }
                }
            }
        }
    }
    // outputs, one cube pair at a time through the staging rows (sector-sized accesses for phi-major cubes)
    auto flush = [&](float* oq, float* ou) {
        __syncthreads();
        for (int i = threadIdx.x; i < CL_WARPS * n; i += blockDim.x) {
            const int j = a.out_phi ? i % CL_WARPS : i / n, k = a.out_phi ? i / CL_WARPS : i % n;
            const long long pp = p0 + j;
            if (pp < a.n_pix) { const size_t o = cube_index(a, pp, k); const float2 v = sStage[(size_t)j * n + k]; oq[o] = v.x; ou[o] = v.y; }
        }
        __syncthreads();
    };
    flush(a.mq, a.mu);                                   // the model is in the staging rows already
#pragma unroll
    for (int i = 0; i < NPL; ++i) { const int k = lane + 32 * i; if (k < n) mine[k] = make_float2(rq[i], ru[i]); }
    flush(a.rq, a.ru);
    if (a.sq) {
#pragma unroll
        for (int i = 0; i < NPL; ++i) { const int k = lane + 32 * i; if (k < n) mine[k] = make_float2(sq[i], su[i]); }
        flush(a.sq, a.su);
    }
}

// ---- (b) CTA per line of sight: residual in registers (thread t holds depths t + 512 i), model in shared memory -------
// One pass over the residual per iteration: the subtraction of component j also finds the candidates for component
// j + 1 (each thread keeps the largest |r|^2 of its own depths, strict > while its depths ascend = lowest index on
// ties), so an iteration is NPT complex FMAs per thread, one block reduction and one __syncthreads (the per-warp
// candidates are double-buffered by iteration parity).  The loop is latency-bound (one dependent beam load per FMA), so
// the double-width beam sits in shared memory whenever it fits next to the model (n <= 9000: LDS instead of an L2 round
// trip) and the CTA has 16 warps.  The restoring convolution visits only the non-zero model components of its window,
// found through a bitmap of the model (one bit per depth), in ascending depth order (deterministic sums).
constexpr int CB_THREADS = 512;

template <int NPT, bool BEAM_SMEM>
__global__ void __launch_bounds__(CB_THREADS) rmclean_block_kernel(const CleanArgs a) {
    extern __shared__ float2 smem2[];
    const int n = a.n_phi, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    constexpr int NW = CB_THREADS / 32;
    float2* m = smem2;                                            // [n] model
    uint32_t* bits = reinterpret_cast<uint32_t*>(smem2 + n);      // [(n + 31) / 32 rounded up to even] bitmap of the model
    const int n_words = (n + 31) >> 5;
    float2* sR = smem2 + n + ((n_words + 1) >> 1);                // [2n - 1] beam (BEAM_SMEM)
    __shared__ float s_y[2][NW], s_q[2][NW], s_u[2][NW];
    __shared__ int s_k[2][NW];
    __shared__ float s_bad;
    const long long p = blockIdx.x;
    if (threadIdx.x == 0) s_bad = 0.f;
    for (int i = threadIdx.x; i < n_words; i += CB_THREADS) bits[i] = 0u;
    if (BEAM_SMEM)
        for (int i = threadIdx.x; i < 2 * n - 1; i += CB_THREADS) sR[i] = __ldg(a.Rdw + i);
    __syncthreads();
    float2 r[NPT];
    float bad = 0.f;
    float y = -1.f, cq = 0.f, cu = 0.f;     // this thread's candidate: largest |r|^2 of its depths
    int kb = 0;
#pragma unroll
    for (int i = 0; i < NPT; ++i) {
        const int k = threadIdx.x + i * CB_THREADS;
        float2 v = make_float2(0.f, 0.f);
        if (k < n) {
            const size_t o = cube_index(a, p, k);
            v = make_float2(a.FQ[o], a.FU[o]);
            m[k] = make_float2(0.f, 0.f);
            bad = fmaf(v.x, 0.f, fmaf(v.y, 0.f, bad));
            const float t = fmaf(v.x, v.x, v.y * v.y);
            if (t > y) { y = t; kb = k; cq = v.x; cu = v.y; }
        }
        r[i] = v;
    }
    if (!(bad == 0.f)) s_bad = 1.f;
    __syncthreads();
    const bool finite = s_bad == 0.f;
    const int c0 = n - 1;
    int it = 0;
    while (finite && it < a.max_iter) {
        const int par = it & 1;
        {   // warp level: two redux.sync reductions (|r|^2 >= 0 orders like its bit pattern; lowest depth among the maxima)
            const unsigned yb = __float_as_uint(y), ymax = __reduce_max_sync(0xffffffffu, yb);
            const unsigned kmin = __reduce_min_sync(0xffffffffu, yb == ymax ? (unsigned)kb : 0x7fffffffu);
            if (yb == ymax && (unsigned)kb == kmin) { s_y[par][warp] = y; s_k[par][warp] = kb; s_q[par][warp] = cq; s_u[par][warp] = cu; }
        }
        __syncthreads();
        {   // every warp merges the NW = 16 candidates the same way (lane l takes warp l & 15's)
            const int wsrc = lane & (NW - 1);
            const unsigned yb = __float_as_uint(s_y[par][wsrc]), ymax = __reduce_max_sync(0xffffffffu, yb);
            const unsigned kc = (unsigned)s_k[par][wsrc], kmin = __reduce_min_sync(0xffffffffu, yb == ymax ? kc : 0x7fffffffu);
            const int wb = __ffs(__ballot_sync(0xffffffffu, yb == ymax && kc == kmin)) - 1;
            y = __uint_as_float(ymax); kb = (int)kmin;
            cq = s_q[par][wb]; cu = s_u[par][wb];
        }
        if (y < a.cutoff2) break;                              // C3: stop before subtracting
        cq *= a.gain; cu *= a.gain;
        if (threadIdx.x == 0) { float2 v = m[kb]; v.x += cq; v.y += cu; m[kb] = v; bits[kb >> 5] |= 1u << (kb & 31); }
        const float2* beam = (BEAM_SMEM ? sR : a.Rdw) + (c0 - kb);
        const float gq = cq, gu = cu;
        y = -1.f; kb = 0; cq = 0.f; cu = 0.f;
#pragma unroll
        for (int i = 0; i < NPT; ++i) {
            const int k = threadIdx.x + i * CB_THREADS;
            if (k < n) {
                const float2 b = BEAM_SMEM ? beam[k] : __ldg(beam + k);
                float2 v = r[i];
                v.x -= gq * b.x - gu * b.y;
                v.y -= gq * b.y + gu * b.x;
                r[i] = v;
                const float t = fmaf(v.x, v.x, v.y * v.y);
                if (t > y) { y = t; kb = k; cq = v.x; cu = v.y; }
            }
        }
        ++it;
    }
    __syncthreads();                                           // the model and its bitmap are complete
    if (a.n_iter && threadIdx.x == 0) a.n_iter[p] = it;
#pragma unroll
    for (int i = 0; i < NPT; ++i) {
        const int k = threadIdx.x + i * CB_THREADS;
        if (k >= n) continue;
        const size_t o = cube_index(a, p, k);
        const float2 rv = r[i], mv = m[k];
        a.mq[o] = mv.x; a.mu[o] = mv.y; a.rq[o] = rv.x; a.ru[o] = rv.y;
        if (a.sq) {
            float sq = rv.x, su = rv.y;
            const int lo = max(0, k - a.gauss_reach), hi = min(n - 1, k + a.gauss_reach);
            for (int wd = lo >> 5; wd <= hi >> 5; ++wd) {
                uint32_t bb = bits[wd];
                if (wd == lo >> 5) bb &= 0xFFFFFFFFu << (lo & 31);
                if (wd == hi >> 5) bb &= 0xFFFFFFFFu >> (31 - (hi & 31));
                while (bb) {                                     // ascending depth order
                    const int j = wd * 32 + __ffs(bb) - 1;
                    bb &= bb - 1;
                    const float2 c = m[j];
                    const float g = __ldg(a.gauss + (j > k ? j - k : k - j));
                    sq = fmaf(c.x, g, sq);
                    su = fmaf(c.y, g, su);
                }
            }
            a.sq[o] = sq; a.su[o] = su;
        }
    }
}

// R on the double-width grid in FP64 (rmsf_kernel of plan.cu), rounded to FP32 pairs
__global__ void clean_pack_kernel(const double* __restrict__ re, const double* __restrict__ im, int n, float2* __restrict__ out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = make_float2((float)re[i], (float)im[i]);
}

rmsynth_status device_rmsf_to(const rmsynth_plan* p, const double* d_phi, int n, double* d_re, double* d_im);   // plan.cu

}  // namespace rms

using namespace rms;

extern "C" rmsynth_status rmsynth_rmclean(const rmsynth_plan* plan, const float* FQ, const float* FU, long long n_pix, int layout,
                                          const rmsynth_clean_params* prm, float* model_q, float* model_u, float* resid_q,
                                          float* resid_u, float* rest_q, float* rest_u, int* n_iter, void* stream) {
    if (!plan) return fail(RMSYNTH_EINVAL, "plan is NULL");
    if (!prm || prm->struct_size != (int)sizeof(rmsynth_clean_params)) return fail(RMSYNTH_EINVAL, "clean_params.struct_size");
    if (n_pix < 0) return fail(RMSYNTH_EINVAL, "n_pix < 0");
    if (layout & ~3) return fail(RMSYNTH_EINVAL, "unknown layout flags");
    if (!(prm->gain > 0.f) || prm->gain > 1.f) return fail(RMSYNTH_EINVAL, "gain must be in (0, 1]");
    if (!(prm->cutoff >= 0.f)) return fail(RMSYNTH_EINVAL, "cutoff must be >= 0");
    if (prm->max_iter < 0) return fail(RMSYNTH_EINVAL, "max_iter < 0");
    if (n_pix == 0) return RMSYNTH_OK;
    if (!FQ || !FU || !model_q || !model_u || !resid_q || !resid_u) return fail(RMSYNTH_EINVAL, "NULL cube pointer");
    if ((rest_q == nullptr) != (rest_u == nullptr)) return fail(RMSYNTH_EINVAL, "restored cubes: both or neither");
    const rmsynth_plan* p = plan;
    if (!p->uniform_phi) return fail(RMSYNTH_EUNSUPPORTED, "RM-CLEAN needs a uniform depth grid (reading C1)");
    DeviceGuard g(p->device);
    RMS_CUDA(g.err);
    cudaStream_t st = (cudaStream_t)stream;
    const int n = p->n_phi;
    {   // the double-width RMSF and the restoring Gaussian are built on first use and kept by the plan
        std::lock_guard<std::mutex> lock(p->mu);
        if (!p->d_Rdw) {
            const int m = 2 * n - 1;
            std::vector<double> ph(m);
            for (int i = 0; i < m; ++i) ph[i] = (double)(i - (n - 1)) * p->dphi;
            double *d_ph = nullptr, *d_out = nullptr;
            RMS_CUDA(cudaMalloc(&d_ph, sizeof(double) * m));
            RMS_CUDA(cudaMalloc(&d_out, sizeof(double) * 2 * m));
            RMS_CUDA(cudaMemcpy(d_ph, ph.data(), sizeof(double) * m, cudaMemcpyHostToDevice));
            rmsynth_status s = device_rmsf_to(p, d_ph, m, d_out, d_out + m);
            if (s == RMSYNTH_OK) {
                RMS_CUDA(cudaMalloc(&p->d_Rdw, sizeof(float2) * m));
                clean_pack_kernel<<<(m + 255) / 256, 256>>>(d_out, d_out + m, m, p->d_Rdw);
                count_launch();
                // FWHM of |R| on a fine grid around 0 (for fwhm <= 0): first crossing of 1/2 by linear interpolation
                std::vector<double> re(m), im(m);
                cudaMemcpy(re.data(), d_out, sizeof(double) * m, cudaMemcpyDeviceToHost);
                cudaMemcpy(im.data(), d_out + m, sizeof(double) * m, cudaMemcpyDeviceToHost);
                double half = 0.0;
                for (int i = 1; i < n; ++i) {
                    const double a0 = std::hypot(re[n - 1 + i - 1], im[n - 1 + i - 1]), a1 = std::hypot(re[n - 1 + i], im[n - 1 + i]);
                    if (a1 < 0.5) { half = ((i - 1) + (a0 - 0.5) / (a0 - a1)) * std::fabs(p->dphi); break; }
                }
                p->rmsf_fwhm = half > 0.0 ? 2.0 * half : 2.0 * std::fabs(p->dphi) * (n - 1);
            }
            cudaFree(d_ph);
            cudaFree(d_out);
            if (s != RMSYNTH_OK) return s;
            RMS_CUDA(cudaDeviceSynchronize());
        }
        const float fwhm = prm->fwhm > 0.f ? prm->fwhm : (float)p->rmsf_fwhm;
        if (!p->d_gauss || p->gauss_fwhm != fwhm) {
            if (!p->d_gauss) RMS_CUDA(cudaMalloc(&p->d_gauss, sizeof(float) * n));
            const double sigma = (double)fwhm / (2.0 * std::sqrt(2.0 * std::log(2.0)));
            std::vector<float> gt(n);
            for (int i = 0; i < n; ++i) { const double x = i * p->dphi; gt[i] = (float)std::exp(-x * x / (2.0 * sigma * sigma)); }
            RMS_CUDA(cudaStreamSynchronize(st));          // an earlier call on this stream may still read the old table
            RMS_CUDA(cudaMemcpy(p->d_gauss, gt.data(), sizeof(float) * n, cudaMemcpyHostToDevice));
            p->gauss_fwhm = fwhm;
            p->gauss_reach = (int)std::min<double>(n - 1, std::ceil(6.5 * sigma / std::fabs(p->dphi)));
        }
    }
    CleanArgs a;
    a.FQ = FQ; a.FU = FU; a.mq = model_q; a.mu = model_u; a.rq = resid_q; a.ru = resid_u; a.sq = rest_q; a.su = rest_u;
    a.n_iter = n_iter; a.n_pix = n_pix; a.n_phi = n; a.out_phi = (layout & RMSYNTH_OUT_PHI_MAJOR) ? 1 : 0;
    a.max_iter = prm->max_iter; a.gain = prm->gain; a.cutoff2 = prm->cutoff * prm->cutoff;
    a.Rdw = p->d_Rdw; a.gauss = p->d_gauss; a.gauss_reach = p->gauss_reach;
    if (n <= 1024) {
        const size_t smem = sizeof(float2) * ((size_t)(2 * n - 1) + (size_t)CL_WARPS * n) + sizeof(float) * n;
        const unsigned grid = (unsigned)((n_pix + CL_WARPS - 1) / CL_WARPS);
#define CL_GO(NPL)                                                                                                          \
        do {                                                                                                                \
            RMS_CUDA(cudaFuncSetAttribute(rmclean_warp_kernel<NPL>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)); \
            rmclean_warp_kernel<NPL><<<grid, CL_WARPS * 32, smem, st>>>(a);                                                 \
        } while (0)
        if (n <= 128) CL_GO(4);
        else if (n <= 256) CL_GO(8);
        else if (n <= 512) CL_GO(16);
        else CL_GO(32);
#undef CL_GO
        RMS_LAUNCH_CHECK("rmclean_warp_kernel");
    } else {
        const int n_words = (n + 31) >> 5;
        const size_t smem_small = sizeof(float2) * ((size_t)n + ((n_words + 1) >> 1));
        const size_t smem_beam = smem_small + sizeof(float2) * (size_t)(2 * n - 1);
        const bool beam_smem = smem_beam <= 220 * 1024;
        const size_t smem = beam_smem ? smem_beam : smem_small;
        if (n > 28 * CB_THREADS) return fail(RMSYNTH_EUNSUPPORTED, "RM-CLEAN: more than 14336 depths do not fit in the registers of a CTA");
        if (n_pix > 0x7fffffffLL) return fail(RMSYNTH_EINVAL, "n_pix too large");
#define CB_GO(NPT, BS)                                                                                                            \
        do {                                                                                                                      \
            RMS_CUDA(cudaFuncSetAttribute(rmclean_block_kernel<NPT, BS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)); \
            rmclean_block_kernel<NPT, BS><<<(unsigned)n_pix, CB_THREADS, smem, st>>>(a);                                          \
        } while (0)
        if (n <= 4 * CB_THREADS) CB_GO(4, true);
        else if (n <= 8 * CB_THREADS) CB_GO(8, true);
        else if (n <= 16 * CB_THREADS) { if (beam_smem) CB_GO(16, true); else CB_GO(16, false); }
        else CB_GO(28, false);
#undef CB_GO
        RMS_LAUNCH_CHECK("rmclean_block_kernel");
    }
    return RMSYNTH_OK;
}
