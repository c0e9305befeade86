// rmsynth_peaks_static: row a7 (peak |F|, peak phi and polarisation-angle maps; Eq. 14, Eq. 17)
// for FQ/FU cubes that already sit in device memory, as a call that ALLOCATES NOTHING.
//
// Who this is for.  Every other peak path of the library obtains its segment records from cudaMalloc the first time a
// (stream, size) is seen (stream_scratch, plan.cu).  Some callers cannot afford that, or cannot do it at all:
//   * a host framework that reserved the whole device for its own memory pool at start-up -- a later cudaMalloc from a
//     library it calls simply fails with out-of-memory;
//   * a client running under a fixed device-memory cap (an MPS or MIG share): what fits at start-up is all there is;
//   * an acquisition or real-time loop: cudaMalloc may synchronise the whole device and takes milliseconds at an
//     unpredictable moment, which is exactly what such a loop is built to avoid.
// For them the records live in a fixed array that is part of the library image itself.
//
// The method is the two-kernel peak search of the tensor path with the first kernel replaced by a plain scan: the depth
// axis is cut into n_seg segments, one thread (phi-major cubes) or one warp (LOS-major cubes) scans one segment of one
// line of sight and writes the same 8-float record the tensor kernel's epilogue writes (tc_epilogue.cuh: SegScan::finish),
// and peaks_combine_kernel (peaks.cu, unchanged) merges a pixel's records in ascending depth order and refines.  Cutting
// the depth axis is what gives a small image with a long depth axis (540^2 pixels x 7000 depths) enough threads.
#include <algorithm>
#include <climits>
#include <mutex>
#include "common.cuh"
#include "tc_epilogue.cuh"

namespace rms {

// ---- the static workspace ----------------------------------------------------------------------------------------
// 32 MiB = 1 048 576 records of kPeakFields floats.  It is a file-scope device array: every GPU on which this library's
// module is loaded sets the 32 MiB aside until the process exits, whether or not rmsynth_peaks_static is ever called.
constexpr long long kStaticRecords = 1LL << 20;
constexpr size_t kStaticBytes = (size_t)kStaticRecords * kPeakFields * sizeof(float);
static __device__ __align__(256) unsigned char g_static_rec[kStaticBytes];

// In HOST code the name g_static_rec is only a handle for the runtime, not an address the GPU understands: a kernel
// handed `g_static_rec` directly would fault (or, on a system where the GPU can reach host memory, quietly scribble over
// the host-side shadow).  The device address has to be asked for, per device, with that device current.
constexpr int kMaxDevices = 64;
static std::mutex g_static_mu;
static float* g_static_addr[kMaxDevices] = {};

// Caller holds a DeviceGuard: the plan's device is current.  The first call on a device does the look-up (and, with lazy
// module loading, makes the driver load this module -- the moment the 32 MiB are actually set aside); later calls only
// read the cached pointer.  No cudaMalloc / cudaFree anywhere.
static rmsynth_status static_workspace(float** out) {
    int dev = -1;
    RMS_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) return fail(RMSYNTH_EUNSUPPORTED, "rmsynth_peaks_static: device ordinal beyond 63");
    std::lock_guard<std::mutex> lk(g_static_mu);
    if (!g_static_addr[dev]) {
        void* ptr = nullptr;
        RMS_CUDA(cudaGetSymbolAddress(&ptr, g_static_rec));
        if (!ptr) return fail(RMSYNTH_ECUDA, "rmsynth_peaks_static: cudaGetSymbolAddress returned a null address");
        g_static_addr[dev] = static_cast<float*>(ptr);
    }
    *out = g_static_addr[dev];
    return RMSYNTH_OK;
}

// ---- first kernel: one record per (line of sight, depth segment) ---------------------------------------------------
__device__ __forceinline__ void write_record(float* __restrict__ rec, int g, long long n_pix, long long p, float best,
                                             int k, float q, float u, float ym2, float yp2, float first, float last) {
    float* r = rec + (long long)g * kPeakFields * n_pix + p;
    r[0 * n_pix] = best;                      // NaN marks a segment that saw a non-finite |F|^2 (reading A17)
    r[1 * n_pix] = __int_as_float(k);
    r[2 * n_pix] = q;
    r[3 * n_pix] = u;
    r[4 * n_pix] = ym2;                       // -1: the best sample was the segment's first
    r[5 * n_pix] = yp2;                       // -1: the best sample was the segment's last
    r[6 * n_pix] = first;                     // -1: empty segment
    r[7 * n_pix] = last;
}

// phi-major cubes F[k*ld + p]: thread = (pixel, segment); a warp reads 32 consecutive pixels of one depth.
__global__ void __launch_bounds__(256) peaks_static_scan_phi_kernel(
    const float* __restrict__ FQ, const float* __restrict__ FU, long long n_pix, long long ld, int n_phi, int seg_len,
    float* __restrict__ rec) {
    const long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n_pix) return;
    const int g = blockIdx.y, k0 = g * seg_len, k1 = min(n_phi, k0 + seg_len);
    PeakState s;
    s.init();
    float first = -1.f;
    for (int k = k0; k < k1; ++k) {
        s.push(k, FQ[(size_t)k * ld + p], FU[(size_t)k * ld + p]);
        if (k == k0) first = s.prev_y2;
    }
    write_record(rec, g, n_pix, p, s.best_y2 + s.nonfinite, s.best_k, s.best_q, s.best_u, s.best_ym2, s.best_yp2, first,
                 s.prev_y2);
}

// LOS-major cubes F[p*ld + k]: warp = (pixel, segment), lanes stride over the segment's depths (coalesced), shuffle
// arg-max with the lowest index winning ties, then lane 0 re-reads the winner and its neighbours inside the segment.
__global__ void __launch_bounds__(256) peaks_static_scan_los_kernel(
    const float* __restrict__ FQ, const float* __restrict__ FU, long long n_pix, long long ld, int n_phi, int seg_len,
    int n_seg, float* __restrict__ rec) {
    const long long w = (long long)blockIdx.x * (blockDim.x / 32) + threadIdx.x / 32;
    const int lane = threadIdx.x % 32;
    const long long p = w / n_seg;
    if (p >= n_pix) return;
    const int g = (int)(w % n_seg), k0 = g * seg_len, k1 = min(n_phi, k0 + seg_len);
    if (k0 >= k1) {
        if (lane == 0) write_record(rec, g, n_pix, p, -1.f, 0, 0.f, 0.f, -1.f, -1.f, -1.f, -1.f);
        return;
    }
    const float* fq = FQ + (size_t)p * ld;
    const float* fu = FU + (size_t)p * ld;
    float best = -1.f, nf = 0.f;
    int kb = INT_MAX;
    for (int k = k0 + lane; k < k1; k += 32) {
        const float q = fq[k], u = fu[k];
        const float y2 = fmaf(q, q, u * u);
        nf = fmaf(y2, 0.f, nf);
        if (y2 > best) { best = y2; kb = k; }
    }
    for (int o = 16; o > 0; o >>= 1) {
        const float ob = __shfl_xor_sync(0xffffffffu, best, o);
        const int ok = __shfl_xor_sync(0xffffffffu, kb, o);
        nf += __shfl_xor_sync(0xffffffffu, nf, o);
        if (ob > best || (ob == best && ok < kb)) { best = ob; kb = ok; }
    }
    if (lane != 0) return;
    if (kb >= k1) kb = k0;                                       // nothing but NaN in this segment: flagged through nf
    auto y2_at = [&](int k) { const float q = fq[k], u = fu[k]; return fmaf(q, q, u * u); };
    write_record(rec, g, n_pix, p, best + nf, kb, fq[kb], fu[kb], kb > k0 ? y2_at(kb - 1) : -1.f,
                 kb < k1 - 1 ? y2_at(kb + 1) : -1.f, y2_at(k0), y2_at(k1 - 1));
}

}  // namespace rms

using namespace rms;

extern "C" rmsynth_status rmsynth_peaks_static(const rmsynth_plan* plan, const float* FQ, const float* FU, long long n_pix,
                                               long long ld, int layout, float* peak_amp, float* peak_phi,
                                               float* pa_lambda0, float* pa_zero, int* peak_index, void* stream) {
    const rmsynth_plan* p = plan;
    if (!p) return fail(RMSYNTH_EINVAL, "plan is NULL");
    if (n_pix < 0) return fail(RMSYNTH_EINVAL, "n_pix < 0");
    if (layout & ~3) return fail(RMSYNTH_EINVAL, "unknown layout flags");
    if (n_pix == 0) return RMSYNTH_OK;
    if (!FQ || !FU) return fail(RMSYNTH_EINVAL, "FQ/FU is NULL");
    if (!(peak_amp || peak_phi || pa_lambda0 || pa_zero || peak_index)) return fail(RMSYNTH_EINVAL, "no map requested");
    const bool phi_major = layout & RMSYNTH_OUT_PHI_MAJOR;
    const long long dense = phi_major ? n_pix : p->n_phi;
    if (ld == 0) ld = dense;
    if (ld < dense) return fail(RMSYNTH_EINVAL, "ld is smaller than the dense row length");
    if (n_pix > kStaticRecords)
        return fail(RMSYNTH_EINVAL, "rmsynth_peaks_static: n_pix = " + std::to_string(n_pix) +
                                        " exceeds the static workspace (1048576 lines of sight per call); pass the cube in "
                                        "slabs of pixels (pointer offset + ld) or use rmsynth_execute_peaks");
    // Segments: enough (pixel, segment) work items to fill the machine, never shorter than 32 depths, never more records
    // than the array holds.
    const long long per_item = phi_major ? 1 : 32;                           // threads per work item
    const long long want_items = (148LL * 2048 * 2 + per_item - 1) / per_item;
    long long n_seg = (want_items + n_pix - 1) / n_pix;
    n_seg = std::min<long long>(n_seg, (p->n_phi + 31) / 32);
    n_seg = std::min<long long>(n_seg, kStaticRecords / n_pix);
    n_seg = std::min<long long>(n_seg, 65535);                               // gridDim.y
    n_seg = std::max<long long>(n_seg, 1);
    const int seg_len = (int)((p->n_phi + n_seg - 1) / n_seg);
    n_seg = (p->n_phi + seg_len - 1) / seg_len;                              // no empty trailing segment

    DeviceGuard g(p->device);
    RMS_CUDA(g.err);
    float* rec = nullptr;
    rmsynth_status s = static_workspace(&rec);
    if (s) return s;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    // Nothing is assumed about what an earlier call left in the array: the scan kernel writes every record the combine
    // kernel reads (n_seg x n_pix of them), and the two are ordered by the stream.
    if (phi_major) {
        dim3 grid((unsigned)((n_pix + 255) / 256), (unsigned)n_seg);
        peaks_static_scan_phi_kernel<<<grid, 256, 0, st>>>(FQ, FU, n_pix, ld, p->n_phi, seg_len, rec);
    } else {
        const long long warps = n_pix * n_seg;
        peaks_static_scan_los_kernel<<<(unsigned)((warps + 7) / 8), 256, 0, st>>>(FQ, FU, n_pix, ld, p->n_phi, seg_len,
                                                                                 (int)n_seg, rec);
    }
    RMS_LAUNCH_CHECK("peaks_static_scan_kernel");
    return peaks_combine(p, rec, (int)n_seg, n_pix, peak_amp, peak_phi, pa_lambda0, pa_zero, peak_index, st);
}
