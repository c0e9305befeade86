// Row a9: FP32 CUDA-core comparison kernels (kept "for comparison" per north_star).
//  (i)  fp32_table:  register-tiled SIMT complex GEMM reading the plan's FP32 phase matrix.
//  (ii) fp32_sincos: one thread per (pixel, phi) looping over channels with two trig calls
//       per term -- the kernel shape the paper describes -- with an exact
//       double-float range reduction so theta = 2 phi (lambda^2-lambda_0^2) keeps FP32-grade
//       accuracy up to |theta| ~ 10^3 rad.
// Both compute Eqs. 15-16 / 18-19 with K w_i folded in (readings A3, A14).
#include "common.cuh"

namespace rms {

constexpr int TM = 64;   // pixels per block tile
constexpr int TN = 64;   // depths per block tile
constexpr int TK = 16;   // channels per step

// IN: 0 = LOS-major [pix][chan], 1 = frequency-major [chan][pix]
// OUT: 0 = LOS-major [pix][phi], 1 = phi-major [phi][pix]
template <int IN, int OUT>
__global__ void __launch_bounds__(256) fp32_table_kernel(
    const float* __restrict__ Q, const float* __restrict__ U, long long n_pix, int n_chan, int n_phi,
    const float* __restrict__ Bc, const float* __restrict__ Bs, int ldb, const float* __restrict__ kwf,
    float* __restrict__ FQ, float* __restrict__ FU) {
    __shared__ float sQ[TK][TM + 4], sU[TK][TM + 4], sC[TK][TN + 4], sS[TK][TN + 4];
    const int tid = threadIdx.x;
    // the thread index that varies fastest follows the contiguous output axis
    const int tn = OUT == 0 ? tid % 16 : tid / 16;   // depth group   (4 depths each)
    const int tm = OUT == 0 ? tid / 16 : tid % 16;   // pixel group   (4 pixels each)
    const long long p0 = (long long)blockIdx.x * TM;
    const int k0 = blockIdx.y * TN;
    float aq[4][4], au[4][4];
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) aq[a][b] = au[a][b] = 0.f;

    for (int c0 = 0; c0 < n_chan; c0 += TK) {
        // stage Q,U: TM x TK elements each, 4 per thread
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            int e = tid + 256 * r;
            int m, c;
            if (IN == 0) { c = e % TK; m = e / TK; } else { m = e % TM; c = e / TM; }
            long long p = p0 + m;
            int ch = c0 + c;
            float q = 0.f, u = 0.f;
            if (p < n_pix && ch < n_chan && kwf[ch] != 0.f) {   // reading A13: zero-weight channels are never read
                size_t off = IN == 0 ? (size_t)p * n_chan + ch : (size_t)ch * n_pix + p;
                q = Q[off];
                u = U[off];
            }
            sQ[c][m] = q;
            sU[c][m] = u;
        }
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            int e = tid + 256 * r;
            int n = e % TN, c = e / TN;
            int ch = c0 + c, k = k0 + n;
            float cc = 0.f, ss = 0.f;
            if (ch < n_chan && k < n_phi) {
                cc = Bc[(size_t)ch * ldb + k];
                ss = Bs[(size_t)ch * ldb + k];
            }
            sC[c][n] = cc;
            sS[c][n] = ss;
        }
        __syncthreads();
        // Partial sums per TK-channel step, flushed into the totals below: a plain sequential FP32
        // sum of ~2000 near-equal terms (coherent source on the grid) drifts by > 1e-5 of the norm.
        float pq[4][4], pu[4][4];
#pragma unroll
        for (int a = 0; a < 4; ++a)
#pragma unroll
            for (int b = 0; b < 4; ++b) pq[a][b] = pu[a][b] = 0.f;
#pragma unroll
        for (int c = 0; c < TK; ++c) {
            float4 q4 = *reinterpret_cast<const float4*>(&sQ[c][tm * 4]);
            float4 u4 = *reinterpret_cast<const float4*>(&sU[c][tm * 4]);
            float4 c4 = *reinterpret_cast<const float4*>(&sC[c][tn * 4]);
            float4 s4 = *reinterpret_cast<const float4*>(&sS[c][tn * 4]);
            const float q[4] = {q4.x, q4.y, q4.z, q4.w}, u[4] = {u4.x, u4.y, u4.z, u4.w};
            const float cs[4] = {c4.x, c4.y, c4.z, c4.w}, sn[4] = {s4.x, s4.y, s4.z, s4.w};
#pragma unroll
            for (int a = 0; a < 4; ++a)
#pragma unroll
                for (int b = 0; b < 4; ++b) {
                    pq[a][b] = fmaf(q[a], cs[b], pq[a][b]);   // Eq. 15: Q cos + U sin
                    pq[a][b] = fmaf(u[a], sn[b], pq[a][b]);
                    pu[a][b] = fmaf(u[a], cs[b], pu[a][b]);   // Eq. 16: U cos - Q sin
                    pu[a][b] = fmaf(-q[a], sn[b], pu[a][b]);
                }
        }
#pragma unroll
        for (int a = 0; a < 4; ++a)
#pragma unroll
            for (int b = 0; b < 4; ++b) { aq[a][b] += pq[a][b]; au[a][b] += pu[a][b]; }
        __syncthreads();
    }
#pragma unroll
    for (int a = 0; a < 4; ++a) {
        long long p = p0 + tm * 4 + a;
        if (p >= n_pix) continue;
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            int k = k0 + tn * 4 + b;
            if (k >= n_phi) continue;
            size_t off = OUT == 0 ? (size_t)p * n_phi + k : (size_t)k * n_pix + p;
            FQ[off] = aq[a][b];
            FU[off] = au[a][b];
        }
    }
}

rmsynth_status fp32_table_execute(const rmsynth_plan* p, const float* Q, const float* U, long long n_pix,
                                  int layout, float* FQ, float* FU, cudaStream_t st) {
    long long gx = (n_pix + TM - 1) / TM;
    if (gx > 0x7fffffffLL) return fail(RMSYNTH_EINVAL, "n_pix too large");
    dim3 grid((unsigned)gx, (p->n_phi + TN - 1) / TN);
    const int in = layout & 1, out = (layout >> 1) & 1;
#define RMS_GO(I, O)                                                                                       \
    fp32_table_kernel<I, O><<<grid, 256, 0, st>>>(Q, U, n_pix, p->n_chan, p->n_phi, p->d_cos, p->d_sin, \
                                                    p->ldb, p->d_kwf, FQ, FU)
    if (in == 0 && out == 0) RMS_GO(0, 0);
    else if (in == 0) RMS_GO(0, 1);
    else if (out == 0) RMS_GO(1, 0);
    else RMS_GO(1, 1);
#undef RMS_GO
    RMS_LAUNCH_CHECK("fp32_table_kernel");
    return RMSYNTH_OK;
}

// ---- (ii) the paper's kernel shape.  x = (2/pi) phi Delta is formed as a double-float:
//   p = phi_hi * d_hi (rounded), e = fma(phi_hi, d_hi, -p) (exact error), plus the cross terms;
//   p is reduced mod 2 exactly (p - 2 rint(p/2) is exact in FP32), then theta = pi x and
//   sincospif(x) evaluates cos/sin of theta with ~1 ulp error.
constexpr int SP = 8;     // pixels per block
constexpr int SCH = 128;  // channels staged per pass

template <int IN, int OUT>
__global__ void __launch_bounds__(128) fp32_sincos_kernel(
    const float* __restrict__ Q, const float* __restrict__ U, long long n_pix, int n_chan, int n_phi,
    const float2* __restrict__ dpi, const float* __restrict__ kwf, const float2* __restrict__ phi2,
    float* __restrict__ FQ, float* __restrict__ FU) {
    __shared__ float sQ[SP][SCH], sU[SP][SCH], sKw[SCH];
    __shared__ float2 sD[SCH];
    const int k = blockIdx.y * 128 + threadIdx.x;
    const long long p0 = (long long)blockIdx.x * SP;
    const float2 ph = k < n_phi ? phi2[k] : make_float2(0.f, 0.f);
    float aq[SP], au[SP];
#pragma unroll
    for (int j = 0; j < SP; ++j) aq[j] = au[j] = 0.f;
    for (int c0 = 0; c0 < n_chan; c0 += SCH) {
        __syncthreads();
        for (int e = threadIdx.x; e < SP * SCH; e += 128) {
            int j, c;
            if (IN == 0) { c = e % SCH; j = e / SCH; } else { j = e % SP; c = e / SP; }
            long long p = p0 + j;
            int ch = c0 + c;
            float q = 0.f, u = 0.f;
            if (p < n_pix && ch < n_chan && kwf[ch] != 0.f) {   // reading A13: zero-weight channels are never read
                size_t off = IN == 0 ? (size_t)p * n_chan + ch : (size_t)ch * n_pix + p;
                q = Q[off];
                u = U[off];
            }
            sQ[j][c] = q;
            sU[j][c] = u;
        }
        {
            int ch = c0 + threadIdx.x;
            sD[threadIdx.x] = ch < n_chan ? dpi[ch] : make_float2(0.f, 0.f);
            sKw[threadIdx.x] = ch < n_chan ? kwf[ch] : 0.f;
        }
        __syncthreads();
        const int cmax = min(SCH, n_chan - c0);
        for (int cc = 0; cc < cmax; cc += 32) {   // 32-channel partial sums (see fp32_table_kernel)
        float pq[SP], pu[SP];
#pragma unroll
        for (int j = 0; j < SP; ++j) pq[j] = pu[j] = 0.f;
        const int ce = min(cc + 32, cmax);
        for (int c = cc; c < ce; ++c) {
            const float2 d = sD[c];
            float pr = ph.x * d.x;
            float er = fmaf(ph.x, d.x, -pr);
            er = fmaf(ph.x, d.y, er);
            er = fmaf(ph.y, d.x, er);
            pr -= 2.0f * rintf(0.5f * pr);            // exact
            float sn, cs;
            sincospif(pr + er, &sn, &cs);             // theta = pi (pr+er)
            const float kw = sKw[c];
            cs *= kw;
            sn *= kw;
#pragma unroll
            for (int j = 0; j < SP; ++j) {
                float q = sQ[j][c], u = sU[j][c];
                pq[j] = fmaf(q, cs, pq[j]);
                pq[j] = fmaf(u, sn, pq[j]);
                pu[j] = fmaf(u, cs, pu[j]);
                pu[j] = fmaf(-q, sn, pu[j]);
            }
        }
#pragma unroll
        for (int j = 0; j < SP; ++j) { aq[j] += pq[j]; au[j] += pu[j]; }
        }
    }
    if (k >= n_phi) return;
#pragma unroll
    for (int j = 0; j < SP; ++j) {
        long long p = p0 + j;
        if (p >= n_pix) break;
        size_t off = OUT == 0 ? (size_t)p * n_phi + k : (size_t)k * n_pix + p;
        FQ[off] = aq[j];
        FU[off] = au[j];
    }
}

rmsynth_status fp32_sincos_execute(const rmsynth_plan* p, const float* Q, const float* U, long long n_pix,
                                   int layout, float* FQ, float* FU, cudaStream_t st) {
    const int in = layout & 1, out = (layout >> 1) & 1;
    long long gx = (n_pix + SP - 1) / SP;
    if (gx > 0x7fffffffLL) return fail(RMSYNTH_EINVAL, "n_pix too large");
    dim3 grid((unsigned)gx, (p->n_phi + 127) / 128);
#define RMS_GO(I, O)                                                                                      \
    fp32_sincos_kernel<I, O><<<grid, 128, 0, st>>>(Q, U, n_pix, p->n_chan, p->n_phi, p->d_dpi, p->d_kwf, \
                                                     p->d_phi2, FQ, FU)
    if (in == 0 && out == 0) RMS_GO(0, 0);
    else if (in == 0) RMS_GO(0, 1);
    else if (out == 0) RMS_GO(1, 0);
    else RMS_GO(1, 1);
#undef RMS_GO
    RMS_LAUNCH_CHECK("fp32_sincos_kernel");
    return RMSYNTH_OK;
}

}  // namespace rms
