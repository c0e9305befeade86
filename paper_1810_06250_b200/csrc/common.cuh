// Internal declarations shared by the translation units of librmsynth.so.
// Nothing here is visible across the C-ABI (include/rmsynth.h is the boundary).
#pragma once
#include <cuda_runtime.h>
#include <atomic>
#include <mutex>
#include <string>
#include <vector>
#include "rmsynth.h"

namespace rms {

void set_error(const std::string& s);
rmsynth_status fail(rmsynth_status st, const std::string& s);
extern std::atomic<long long> g_launches;
inline void count_launch(int n = 1) { g_launches.fetch_add(n, std::memory_order_relaxed); }

#define RMS_CUDA(expr)                                                                   \
    do {                                                                                 \
        cudaError_t e__ = (expr);                                                        \
        if (e__ != cudaSuccess)                                                          \
            return rms::fail(e__ == cudaErrorMemoryAllocation ? RMSYNTH_ENOMEM : RMSYNTH_ECUDA, \
                             std::string(#expr) + ": " + cudaGetErrorString(e__));       \
    } while (0)

#define RMS_LAUNCH_CHECK(name)                                                           \
    do {                                                                                 \
        rms::count_launch();                                                             \
        cudaError_t e__ = cudaGetLastError();                                            \
        if (e__ != cudaSuccess)                                                          \
            return rms::fail(RMSYNTH_ECUDA, std::string(name) + " launch: " + cudaGetErrorString(e__)); \
    } while (0)

// Every entry point that touches the device runs on the PLAN's device whatever the caller's current device is, and
// leaves the caller's current device as it found it.
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    cudaError_t err = cudaSuccess;
    explicit DeviceGuard(int dev) {
        err = cudaGetDevice(&prev);
        if (err == cudaSuccess && dev >= 0 && prev != dev) {
            err = cudaSetDevice(dev);
            switched = err == cudaSuccess;
        }
    }
    ~DeviceGuard() {
        if (switched) cudaSetDevice(prev);
    }
};

// Tensor-path operand geometry chosen at plan time (see tc_gemm.cu).
struct TcGeom {
    int n_tile = 0;      // phi columns per tile (n); UMMA N = 2n
    int n_phi_tiles = 0; // ceil(n_phi / n)
    int k_pad = 0;       // n_chan rounded up to the K block
    int kb = 0;          // channels per K block
    int ctas = 2;        // CTA pairs (tcgen05 cta_group::2)
};

}  // namespace rms

struct rmsynth_plan {
    int n_chan = 0, n_phi = 0, scheme = 0, device = 0, lambda0_mode = 0, sm_count = 0;
    double K = 0.0, lambda0_sq = 0.0;
    std::vector<double> lam2, w, phi;     // host copies
    std::vector<double> R_re, R_im;       // R(phi) on the plan grid (Eq. 12)
    // device, FP64 plan inputs
    double* d_delta = nullptr;            // lambda_i^2 - lambda_0^2          [n_chan]
    double* d_kw = nullptr;               // K w_i                            [n_chan]
    double* d_phi = nullptr;              //                                  [n_phi]
    // device, FP32 phase matrix  K w_i cos/sin(th_ik), row i, column k, pitch ldb
    int ldb = 0;
    float* d_cos = nullptr;
    float* d_sin = nullptr;
    // device, FP32 helpers
    float* d_phif = nullptr;              // phi as float                     [n_phi]
    float* d_kwf = nullptr;               // K w_i as float                   [n_chan]
    float2* d_dpi = nullptr;              // (2/pi)(lambda_i^2-lambda_0^2) as hi+lo floats [n_chan]
    float2* d_phi2 = nullptr;             // phi as hi+lo floats              [n_phi]
    // tensor path (tc_gemm.cu)
    rms::TcGeom tc;
    float* d_tcB2 = nullptr;              // pre-split, pre-swizzled B operand blobs (tc_gemm2.cu)
    // FP16 split tensor path (tc_gemm3.cu)
    rms::TcGeom tc3;
    void* d_tcB3 = nullptr;               // scaled FP16 hi/lo B operand blobs
    unsigned int* d_chanmask = nullptr;   // per 32 channels: bit i set = channel exists and has w > 0 (reading A13)
    int tc3_eb = 0;                       // B is scaled by 2^tc3_eb
    // scratch for maps-only calls and host streaming (grown on demand, guarded by mu)
    mutable std::mutex mu;
    static constexpr int kScratch = 15;   // host-streaming slots: (Q, U, FQ, FU, maps) x 3
    mutable float* scratch[kScratch] = {};
    mutable size_t scratch_bytes[kScratch] = {};
    // per-call workspace keyed by (stream, tag) so that concurrent calls on different streams never share it
    struct StreamScratch { cudaStream_t st; int tag; float* ptr; size_t bytes; };
    mutable std::mutex pool_mu;
    mutable std::vector<StreamScratch> pool;
    mutable std::vector<float*> retired;  // outgrown workspace buffers, kept until destroy (captured graphs may reference them)
    mutable void* host_pipe = nullptr;    // streams, events and staging of the host-streaming engine (execute.cu)
    long long host_chunk_pixels = 0;      // rmsynth_options.host_chunk_pixels (0 = automatic)
    // RM-CLEAN (rmclean.cu): needs a uniform depth grid; beam and restoring Gaussian are built on first use
    bool uniform_phi = false;
    double dphi = 0.0;
    mutable float2* d_Rdw = nullptr;      // R((k - j) dphi), 2 n_phi - 1 samples, R(0) at n_phi - 1
    mutable float* d_gauss = nullptr;     // restoring Gaussian at m dphi, m = 0 .. n_phi - 1
    mutable float gauss_fwhm = 0.f;
    mutable int gauss_reach = 0;
    mutable double rmsf_fwhm = 0.0;       // FWHM of |R| (used when the caller passes fwhm <= 0)
    mutable void* fft_tables = nullptr;   // tables of the FFT variant for the last (window, oversampling) used (fft_variant.cu)
};

namespace rms {

rmsynth_status ensure_scratch(const rmsynth_plan* p, int slot, size_t bytes, float** out);
enum { SCR_PEAK_REC = 0, SCR_CUBE_Q = 1, SCR_CUBE_U = 2, SCR_REPACK_Q = 3, SCR_REPACK_U = 4, SCR_TILE_SYNC = 5 };
rmsynth_status stream_scratch(const rmsynth_plan* p, cudaStream_t st, int tag, size_t bytes, float** out);

// fp32_kernels.cu
rmsynth_status fp32_table_execute(const rmsynth_plan* p, const float* Q, const float* U, long long n_pix,
                                  int layout, float* FQ, float* FU, cudaStream_t st);
rmsynth_status fp32_sincos_execute(const rmsynth_plan* p, const float* Q, const float* U, long long n_pix,
                                   int layout, float* FQ, float* FU, cudaStream_t st);
// execute.cu
void host_pipe_free(rmsynth_plan* p);
// fft_variant.cu
void fft_tables_free(rmsynth_plan* p);
// peaks.cu
rmsynth_status peaks_combine(const rmsynth_plan* p, const float* rec, int n_seg, long long n_pix, float* amp, float* phi,
                             float* pa0, float* paz, int* idx, cudaStream_t st);
rmsynth_status peaks_gather(const rmsynth_plan* p, const float* rec, int n_seg, long long n_pix, const float* FQ, const float* FU,
                            bool out_phi, float* amp, float* phi, float* pa0, float* paz, int* idx, cudaStream_t st);
rmsynth_status abs_from_cubes(const float* FQ, const float* FU, long long n, float* FA, cudaStream_t st);
rmsynth_status peaks_from_cubes(const rmsynth_plan* p, const float* FQ, const float* FU, long long n_pix,
                                int out_layout, float* amp, float* phi, float* pa0, float* paz, int* idx,
                                cudaStream_t st);
// tc_gemm.cu
rmsynth_status tc_plan_init(rmsynth_plan* p);
void tc_plan_free(rmsynth_plan* p);
rmsynth_status tc_execute(const rmsynth_plan* p, const float* Q, const float* U, long long n_pix, int layout,
                          float* FQ, float* FU, float* FA, float* amp, float* phi, float* pa0, float* paz, int* idx,
                          cudaStream_t st);

// tc_gemm3.cu
rmsynth_status tc3_plan_init(rmsynth_plan* p);
rmsynth_status tc3_launch(const rmsynth_plan* p, const void* map_q, const void* map_u, const void* map_fq, const void* map_fu,
                          bool a3d, bool in_freq, bool out_phi, int ring_out, long long n_pix, float* FQ, float* FU, float* FA, float* rec, int* tile_sync, int gang,
                          int sync_lag, cudaStream_t st);

// tc_gemm2.cu
rmsynth_status tc2_plan_init(rmsynth_plan* p);
rmsynth_status tc2_launch(const rmsynth_plan* p, const void* map_q, const void* map_u, bool a3d, bool in_freq,
                          bool out_phi, long long n_pix, float* FQ, float* FU, float* FA, float* rec, int* tile_sync,
                          int gang, int sync_lag, cudaStream_t st);

}  // namespace rms
