// PTX wrappers (tcgen05 / TMEM / TMA / mbarrier) shared by the tensor-core kernels.
#pragma once
#include <cuda.h>
#include <cstdint>
#include <cstdlib>
#include <cuda_runtime.h>

namespace rms {

// ------------------------------------------------------------------------------------------------
// PTX wrappers
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n.reg .pred p;\nWAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\nbra WAIT_%=;\nDONE_%=:\n}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
// L2 eviction policies.  The operands (Q/U tiles re-read by every depth tile of a pixel tile, and the phase-matrix
// blobs) are loaded evict_last; the output cubes are a write-once stream and are stored evict_first, so that
// the 8 B x N_pix x N_phi going out do not push the inputs out of L2 between two depth tiles.
__device__ __forceinline__ uint64_t l2_policy_evict_last() {
    uint64_t p; asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p)); return p;
}
__device__ __forceinline__ uint64_t l2_policy_evict_first() {
    uint64_t p; asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p)); return p;
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* map, int c0, int c1, uint64_t* bar, uint64_t pol) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3}], [%4], %5;" ::"r"(dst),
        "l"(map), "r"(c0), "r"(c1), "r"(smem_u32(bar)), "l"(pol) : "memory");
}
__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap* map, int c0, int c1, int c2, uint64_t* bar, uint64_t pol) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3, %4}], [%5], %6;" ::"r"(dst),
        "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar)), "l"(pol) : "memory");
}
__device__ __forceinline__ void bulk_load(uint32_t dst, const void* src, uint32_t bytes, uint64_t* bar, uint64_t pol) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar)), "l"(pol) : "memory");
}
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t* r) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,"
        "%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
          "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]),
          "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]),
          "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
        : "r"(taddr));
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t* r) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
          "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
        : "r"(taddr));
}
__device__ __forceinline__ void tmem_ld64(uint32_t taddr, uint32_t* r) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x64.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31,%32,%33,%34,%35,%36,%37,%38,%39,%40,%41,%42,%43,%44,%45,%46,%47,%48,%49,%50,%51,%52,%53,%54,%55,%56,%57,%58,%59,%60,%61,%62,%63}, [%64];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31]), "=r"(r[32]), "=r"(r[33]), "=r"(r[34]), "=r"(r[35]), "=r"(r[36]), "=r"(r[37]), "=r"(r[38]), "=r"(r[39]), "=r"(r[40]), "=r"(r[41]), "=r"(r[42]), "=r"(r[43]), "=r"(r[44]), "=r"(r[45]), "=r"(r[46]), "=r"(r[47]), "=r"(r[48]), "=r"(r[49]), "=r"(r[50]), "=r"(r[51]), "=r"(r[52]), "=r"(r[53]), "=r"(r[54]), "=r"(r[55]), "=r"(r[56]), "=r"(r[57]), "=r"(r[58]), "=r"(r[59]), "=r"(r[60]), "=r"(r[61]), "=r"(r[62]), "=r"(r[63])
        : "r"(taddr));
}
__device__ __forceinline__ void st_global_pred(unsigned long long addr, float v, bool pred, uint64_t pol) {
    asm volatile("{\n.reg .pred p;\nsetp.ne.b32 p, %2, 0;\n@p st.global.L2::cache_hint.f32 [%0], %1, %3;\n}" ::"l"(addr), "f"(v),
                 "r"((int)pred), "l"(pol) : "memory");
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

// UMMA shared-memory matrix descriptor (version 1 = sm_100).  Offsets in bytes.
__device__ __forceinline__ uint64_t make_desc(uint32_t saddr, uint32_t lbo, uint32_t sbo, uint32_t layout_type) {
    uint64_t d = 0;
    d |= (uint64_t)((saddr >> 4) & 0x3FFF);
    d |= (uint64_t)((lbo >> 4) & 0x3FFF) << 16;
    d |= (uint64_t)((sbo >> 4) & 0x3FFF) << 32;
    d |= (uint64_t)1 << 46;
    d |= (uint64_t)layout_type << 61;
    return d;
}

__device__ __forceinline__ float rn_tf32(float x) {   // round-to-nearest(-even) to 10 explicit mantissa bits
    uint32_t u = __float_as_uint(x);
    if ((u & 0x7F800000u) == 0x7F800000u) return x;
    u += 0xFFFu + ((u >> 13) & 1u);
    return __uint_as_float(u & 0xFFFFE000u);
}


// Experiment knobs exist only in a -DRMSYNTH_EXPERIMENT build, which build() never makes: the product library reads no
// environment variable, so a call, a later call and a captured graph always take the same path.
#ifdef RMSYNTH_EXPERIMENT
static inline const char* experiment_env(const char* name) { return getenv(name); }
#else
static inline const char* experiment_env(const char*) { return nullptr; }
#endif

// Static "gang" schedule of the (pixel-tile pair, depth tile) work items over the CTA pairs of the grid.
// T = depth tiles per pixel-tile pair, G = gang size (a divisor of T).  The first S = floor(n_clusters / G) G clusters
// work in gangs of G: a gang takes one pair, member m = cid % G walks the depth tiles m, m + G, m + 2G, ... one after
// the other, all members at the same time, so the pair's Q/U tiles are fetched from HBM once and hit L2 for every other
// (member, depth tile) -- across members because gang_checkin keeps them together, within a member because it used the
// same tiles one item earlier.  G = T is "one depth tile per member" (smallest L2 footprint: n_clusters / T pairs in
// flight), G = 1 is "every cluster on its own" (no check-in at all, n_clusters pairs in flight).  The n_clusters - S
// left-over clusters take whole pairs and walk all T depth tiles.  Of every n_clusters consecutive pairs, S go to the
// gangs (S / G at a time) and one to each left-over cluster, so both kinds finish together.
// Every role of a CTA walks the same sequence.
struct WorkIter {
    int T, G, S, n_clusters, n_pairs, cid, k;
    __device__ __forceinline__ void init(int cluster_id, int n_clusters_, int T_, int n_pairs_, int G_) {
        T = T_; G = G_; n_clusters = n_clusters_; n_pairs = n_pairs_; cid = cluster_id; k = 0;
        S = (n_clusters / G) * G;
    }
    __device__ __forceinline__ bool ganged() const { return cid < S && G > 1; }
    __device__ __forceinline__ int walk() const { return cid < S ? T / G : T; }     // depth tiles this cluster walks per pair
    // pixel-tile pair of the r-th round of a ganged cluster
    __device__ __forceinline__ int gang_pair(int r) const {
        const int sg = r * (S / G) + cid / G;              // r-th gang round, gang cid / G
        return (sg / S) * n_clusters + sg % S;
    }
    // next work item of this cluster: pixel-tile pair tp, depth tile j; false when the cluster is done
    __device__ __forceinline__ bool next(int& tp, int& j) {
        int g;
        if (cid < S) {
            const int w = T / G;
            g = gang_pair(k / w);
            j = cid % G + (k % w) * G;
        } else {
            g = (k / T) * n_clusters + cid;
            j = k % T;
        }
        ++k;
        tp = g;
        return g < n_pairs;
    }
    __device__ __forceinline__ bool new_pair() const { return (k - 1) % walk() == 0; }   // the item next() just returned starts a pair
};

// Soft lock-step of the CTAs of a gang.  The work items are dealt statically and nothing else ties the members
// together; left alone they drift apart until the tiles a leader pulled in from HBM have left L2 by the time the
// laggards ask for them (measured on the 2048^2 cube without any check-in: 39.9 GB read for 13.4 GB algorithmic).
// Every TMA producer therefore checks in on a per-pair counter before it loads a new pair's first tile, and waits
// (bounded) until the whole gang has checked in for the pair it started `lag` rounds earlier: lag = 0 is a barrier
// per pair; lag >= 1 only bounds the drift.  A performance hint only: the spin is bounded, correctness never depends on it.
__device__ __forceinline__ void gang_checkin(int* counters, const WorkIter& wi, int tp, int lag, int expected) {
    if (!counters || !wi.ganged() || !wi.new_pair()) return;
    atomicAdd(counters + tp, 1);
    const int r = (wi.k - 1) / wi.walk() - lag;            // wi.next() has already advanced k past this item
    if (r < 0) return;
    const int* c = counters + wi.gang_pair(r);
    for (int tries = 0; tries < 256; ++tries) {
        int v;
        asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(c) : "memory");
        if (v >= expected) break;
        __nanosleep(200);
    }
}

// ---- per-role timeline (debug build only: python -m paper_1810_06250_b200.build --timeline) -----------------------
// clock64 stamps / accumulated waits of the first TL_ITEMS work items of a few CTAs, one row of TL_SLOTS values per
// (CTA, role, item); read back and tabulated by paper_1810_06250_b200/timeline.py.  In the product build every
// method is empty and the optimiser removes the calls.
constexpr int TL_ITEMS = 128, TL_SLOTS = 8, TL_ROLES = 5, TL_CTAS = 8;
enum { TL_PRODUCER = 0, TL_ISSUER = 1, TL_TRANSFORM = 2, TL_EPI0 = 3, TL_EPI1 = 4 };
struct TlRole {
#ifdef RMSYNTH_TIMELINE
    long long* base;
    long long t0;
    int item;
    __device__ __forceinline__ void init(long long* buf, int role) {
        const int b = blockIdx.x, g = gridDim.x;           // cluster 0, cluster 1, cluster 3 (same gang) and the last cluster
        const int slot = b < 4 ? b : (b == 6 || b == 7) ? b - 2 : (g >= 10 && b >= g - 2) ? 6 + b - (g - 2) : -1;
        base = (buf && slot >= 0 && (threadIdx.x & 31) == 0) ? buf + (size_t)(slot * TL_ROLES + role) * TL_ITEMS * TL_SLOTS : nullptr;
        item = 0;
        t0 = 0;
    }
    __device__ __forceinline__ bool on() const { return base && item < TL_ITEMS; }
    __device__ __forceinline__ void stamp(int s) { if (on()) base[item * TL_SLOTS + s] = clock64(); }
    __device__ __forceinline__ void begin() { if (on()) t0 = clock64(); }
    __device__ __forceinline__ void add(int s) { if (on()) base[item * TL_SLOTS + s] += clock64() - t0; }
    __device__ __forceinline__ void lap(int s) { if (on()) { const long long t = clock64(); base[item * TL_SLOTS + s] += t - t0; t0 = t; } }
    __device__ __forceinline__ void next() { ++item; }
#else
    __device__ __forceinline__ void init(long long*, int) {}
    __device__ __forceinline__ void stamp(int) {}
    __device__ __forceinline__ void begin() {}
    __device__ __forceinline__ void add(int) {}
    __device__ __forceinline__ void lap(int) {}
    __device__ __forceinline__ void next() {}
#endif
};

// ---- cluster / 2-CTA variants
__device__ __forceinline__ uint32_t cluster_ctarank() { uint32_t r; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;\nbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ uint32_t mapa_u32(uint32_t saddr, uint32_t rank) {
    uint32_t r; asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(saddr), "r"(rank)); return r;
}
// Remote arrival with the default (.release.cta) semantics -- the form NVIDIA's own 2-SM kernels use to signal
// the leader CTA's barrier.  A cluster-scope release (.release.cluster) costs ~1000 cycles per arrival (measured).
__device__ __forceinline__ void mbar_arrive_remote(uint32_t cluster_addr) {
    asm volatile("mbarrier.arrive.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}
__device__ __forceinline__ void umma2_tf32(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t acc) {
    asm volatile(
        "{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::2.kind::tf32 [%0], %1, %2, %3, p;\n}" ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc),
        "r"(acc) : "memory");
}
__device__ __forceinline__ void umma2_commit_mc(uint64_t* bar) {   // arrive on the same barrier in both CTAs of the pair
    asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(smem_u32(bar)),
                 "h"((uint16_t)3) : "memory");
}

}  // namespace rms
