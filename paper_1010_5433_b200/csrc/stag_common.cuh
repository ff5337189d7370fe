// stag_common.cuh — geometry, context and small device helpers shared by the kernels of
// libstag_b200.so (sm_100a).  Private to the CUDA path; the oracle includes none of this.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <condition_variable>
#include <mutex>

#include "../../include/stag.h"

namespace stag {

// ---- exact unsigned division by a runtime constant (n < 2^31) ------------------------------
struct FastDiv {
    uint32_t d, mul, shift;
    __host__ void init(uint32_t div) {
        d = div;
        shift = 0;
        while ((1u << shift) < div) ++shift;
        mul = (uint32_t)((((uint64_t)1 << (32 + shift)) + div - 1) / div - ((uint64_t)1 << 32));
    }
    __device__ __forceinline__ uint32_t div(uint32_t n) const {
        return (__umulhi(n, mul) + n) >> shift;
    }
};

// ---- lattice geometry, passed by value to every kernel ---------------------------------------
struct Geom {
    int L[4];
    int Lh0;      // L0 / 2: sites of one parity per x0-row
    int Vh;       // sites per parity
    int V;
    FastDiv dLh0, dL1, dL2;
};

// coordinates of the site with one-parity index e and parity par
struct Site {
    int x0, x1, x2, x3;
    int lex;
};

__device__ __forceinline__ Site site_of(const Geom &g, int e, int par) {
    Site s;
    const uint32_t row = g.dLh0.div((uint32_t)e);            // x1 + L1*(x2 + L2*x3)
    const int h = e - (int)row * g.Lh0;
    const uint32_t r2 = g.dL1.div(row);
    s.x1 = (int)row - (int)r2 * g.L[1];
    s.x3 = (int)g.dL2.div(r2);
    s.x2 = (int)r2 - s.x3 * g.L[2];
    s.x0 = 2 * h + ((s.x1 + s.x2 + s.x3 + par) & 1);
    s.lex = s.x0 + g.L[0] * (int)row;
    return s;
}

// ---- context -------------------------------------------------------------------------------
struct Options {
    int dslash_block;        // threads per CTA of the Dslash kernels: 64 | 128 | 256
    int dslash_regs;         // registers per thread: 64 (1024 resident threads / SM) | 128 (512) | 255 (256) | 0 auto
    int dslash_ctas_per_sm;  // 0: one CTA per block of sites; k > 0: persistent grid of k*SMs CTAs
    int dslash_pipe;         // stag_dslash_block: 1 = cp.async-ring kernel where it is the faster one (default); 0 = never
    int cg_check_every;      // iterations between convergence polls (= iterations per CUDA graph)
    int cg_graph;            // replay the iteration batch as a CUDA graph
    int cg_freeze;           // stop updating converged shifts (reading A10)
    int cg_ctas_per_sm;      // persistent grid size of the CG streaming kernels, per SM
    int cg_persistent_threads;  // persistent-kernel CTA: 1024 threads (64 regs) | 512 (128 regs) | 0 auto
    int cg_resident_slices;  // persistent kernel: at most this many of r, q, p_base resident in shared memory (0..3)
    int cg_mixed_reliable;   // stag_mshift_cg_mixed: inner stage = persistent kernel with residual replacement: 0 never | 1 single shift | 2 always
    int cg_mixed_delta_inv;  // ... which replaces the residual whenever ||r|| has fallen by this factor (default 10)
    int cg_mixed_fp64_from;  // stag_mshift_cg_mixed: from this many shifts on (and stop < 1e-6) the call is the fp64 multi-shift solve; 0 never
    int cg_persistent;       // 1: whole solve as one cooperative kernel when r,q,p fit in shared memory; 0: never
    int cg_l2_keep_mb;       // persistent kernel: MB of x_i, p_i (lightest shifts first) kept L2-resident (evict_last); 0: none
    int cg_fill;             // persistent kernel: 1 = deferred shift updates are worked off while waiting at sync points
    int cg_single_reduction; // persistent kernel, single source: 1 = one grid-wide reduction per iteration (stag_cg_persist_sr.cuh)
    int cg_nbflags;          // persistent kernel: 1 = neighbour epoch flags instead of grid barriers after phases A and D
    int cg_profile;          // multi-kernel path: 1 = no graph, CUDA events around every kernel of 32 iterations (stag_cg_profile)
};

}  // namespace stag

namespace stag {
// Host-side staging of ONE synchronising call (stag_mshift_cg*, stag_cg_polish, recon-12 stag_gauge_pack): pinned
// memory for the state upload / read-back and the convergence polls, and the cached CUDA graph of the multi-kernel
// CG path.  A context owns a small pool of these; a call leases one for its whole duration, so independent
// solves — the paper's several pseudo-fermions — may run concurrently on different streams of one
// context, and back-to-back solves with the same buffers replay the graph instead of re-capturing it.
struct GraphKey {                 // everything the captured launches depend on
    const void *packed; void *ws; void *x;
    int prec, recon, nshift, base, batch, dslash_block, dslash_regs, dslash_ctas_per_sm, cg_ctas_per_sm;
};
struct Slot {
    int *pinned_flags;            // 512 B pinned (mapped): status words, convergence polls; bytes 128.. = 16 doubles (N2 norms)
    void *pinned_info;            // pinned staging for the CG state upload / read-back (one CgState)
    cudaGraphExec_t gexec;        // multi-kernel path: one batch of cg_check_every iterations, for `key`
    GraphKey key;
    cudaEvent_t ev[2];            // poll events of the multi-kernel path
    bool busy;
};
static constexpr int kSlots = 4;
}  // namespace stag

struct stag_ctx {
    stag::Geom g;
    stag::Options opt;
    int device;
    int num_sms;
    mutable stag::Slot slots[stag::kSlots];
    mutable std::mutex mu;
    mutable std::condition_variable cv;
    // measurement aids (stag_kernel_log, stag_cg_profile): which kernels the calls on this ctx launched, and the
    // per-kernel times of the last profiled multi-kernel solve
    mutable const void *klog[32];
    mutable int nklog;
    mutable double prof_us[4];
    mutable int prof_iters;
};

namespace stag {

#define STAG_CUDA_OK(call)                                  \
    do {                                                    \
        cudaError_t e__ = (call);                           \
        if (e__ != cudaSuccess) return STAG_ERR_CUDA;       \
    } while (0)

// lease of one staging slot for the duration of a synchronising call (waits if all kSlots are in use)
class SlotLease {
    const stag_ctx *ctx_;
    Slot *s_;
public:
    explicit SlotLease(const stag_ctx *ctx) : ctx_(ctx), s_(nullptr) {
        std::unique_lock<std::mutex> lk(ctx->mu);
        for (;;) {
            for (int i = 0; i < kSlots; ++i)
                if (!ctx->slots[i].busy) { s_ = &ctx->slots[i]; break; }
            if (s_) break;
            ctx->cv.wait(lk);
        }
        s_->busy = true;
    }
    ~SlotLease() {
        { std::lock_guard<std::mutex> lk(ctx_->mu); s_->busy = false; }
        ctx_->cv.notify_one();
    }
    SlotLease(const SlotLease &) = delete;
    SlotLease &operator=(const SlotLease &) = delete;
    Slot &slot() const { return *s_; }
};

// remember that `func` (a __global__ function) was launched on behalf of ctx (stag_kernel_log)
inline void log_kernel(const stag_ctx *ctx, const void *func) {
    std::lock_guard<std::mutex> lk(ctx->mu);
    for (int i = 0; i < ctx->nklog; ++i)
        if (ctx->klog[i] == func) return;
    if (ctx->nklog < 32) ctx->klog[ctx->nklog++] = func;
}
// launch kern<<<...>>>(args) and log it; `kern` is an expression of function-pointer type
#define STAG_LAUNCH_K(ctx, kern, grid, block, smem, st, ...)             \
    do {                                                                  \
        auto k__ = kern;                                                  \
        stag::log_kernel(ctx, reinterpret_cast<const void *>(k__));       \
        k__<<<grid, block, smem, st>>>(__VA_ARGS__);                      \
    } while (0)

inline bool valid_prec(int p) { return p == STAG_F64 || p == STAG_F32 || p == STAG_F64_SPLIT; }
// precision of the colour vectors that go with a gauge format (split-double links carry fp64 vectors)
inline int vec_prec(int p) { return p == STAG_F32 ? STAG_F32 : STAG_F64; }
inline bool valid_recon(int r) { return r == STAG_RECON18 || r == STAG_RECON12; }

// bytes of one link set plane group: (recon reals) * sizeof(T) per site
inline size_t link_bytes_per_site(int prec, int recon) {
    return (size_t)recon * (prec == STAG_F32 ? 4 : 8);   // split-double: a float b plus a float c per real
}
inline size_t vec_bytes_per_site(int prec) { return (size_t)6 * (prec == STAG_F32 ? 4 : 8); }
inline size_t align256(size_t n) { return (n + 255) & ~(size_t)255; }

// ---- streaming / cached 128-bit and 64-bit loads ---------------------------------------------
// Links are read exactly once per Dslash: keep them out of L1 and first in line for L2
// eviction so that the (re-used) colour vectors stay cached.
__device__ __forceinline__ uint64_t policy_evict_first() {
    uint64_t pol;
    asm("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ double2 ld_stream(const double2 *p, uint64_t pol) {
    double2 r;
    asm("ld.global.nc.L1::no_allocate.L2::cache_hint.v2.f64 {%0,%1}, [%2], %3;"
        : "=d"(r.x), "=d"(r.y) : "l"(p), "l"(pol));
    return r;
}
__device__ __forceinline__ float4 ld_stream(const float4 *p, uint64_t pol) {
    float4 r;
    asm("ld.global.nc.L1::no_allocate.L2::cache_hint.v4.f32 {%0,%1,%2,%3}, [%4], %5;"
        : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w) : "l"(p), "l"(pol));
    return r;
}
__device__ __forceinline__ float2 ld_stream(const float2 *p, uint64_t pol) {
    float2 r;
    asm("ld.global.nc.L1::no_allocate.L2::cache_hint.v2.f32 {%0,%1}, [%2], %3;"
        : "=f"(r.x), "=f"(r.y) : "l"(p), "l"(pol));
    return r;
}
// Neighbour colour vectors are re-used by up to 8 output sites: read-only path, L1-allocating.
__device__ __forceinline__ double2 ld_reuse(const double2 *p) { return __ldg(p); }
__device__ __forceinline__ float4 ld_reuse(const float4 *p) { return __ldg(p); }
__device__ __forceinline__ float2 ld_reuse(const float2 *p) { return __ldg(p); }

// Coherent (weak, L1-allocating) loads for data that other CTAs rewrite inside the same kernel
// between grid barriers.  asm volatile: never turned into ld.global.nc, never hoisted over a barrier.
__device__ __forceinline__ double2 ld_coherent(const double2 *p) {
    double2 r;
    asm volatile("ld.global.v2.f64 {%0,%1}, [%2];" : "=d"(r.x), "=d"(r.y) : "l"(p) : "memory");
    return r;
}
__device__ __forceinline__ float4 ld_coherent(const float4 *p) {
    float4 r;
    asm volatile("ld.global.v4.f32 {%0,%1,%2,%3}, [%4];"
                 : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w) : "l"(p) : "memory");
    return r;
}
__device__ __forceinline__ float2 ld_coherent(const float2 *p) {
    float2 r;
    asm volatile("ld.global.v2.f32 {%0,%1}, [%2];" : "=f"(r.x), "=f"(r.y) : "l"(p) : "memory");
    return r;
}

// ---- block-wide sum of one double (deterministic for a fixed block size) ----------------------
template <int BLOCK>
__device__ __forceinline__ double block_sum(double v, double *smem /* BLOCK/32 doubles */) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    __syncthreads();
    if (lane == 0) smem[warp] = v;
    __syncthreads();
    double s = 0.0;
    if (warp == 0) {
        s = lane < BLOCK / 32 ? smem[lane] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    }
    return s;  // valid in warp 0 (all its lanes)
}

// ---- grid-wide sum, finished by the last CTA to arrive ------------------------------------------
// Every CTA writes its partial to partials[blockIdx.x]; the CTA that draws the last ticket adds
// all partials in index order (deterministic for a fixed grid) and gets `true` with the total in
// every lane of its warp 0.  One __threadfence per CTA, at its very end (a gpu-scope fence
// invalidates L1, so the kernels that use this are persistent: many tiles, one fence).
template <int BLOCK>
__device__ __forceinline__ bool grid_sum_last_cta(double v, double *partials, unsigned int *ticket,
                                                  double *smem /* BLOCK/32 + 1 doubles */,
                                                  double &total) {
    const double s = block_sum<BLOCK>(v, smem);
    int *flag = reinterpret_cast<int *>(smem + BLOCK / 32);
    if (threadIdx.x == 0) {
        __stcg(partials + blockIdx.x, s);
        __threadfence();
        const unsigned int t = atomicAdd(ticket, 1u);
        *flag = (t == gridDim.x - 1);
    }
    __syncthreads();
    if (!*flag) return false;
    __threadfence();
    double t = 0.0;
    for (unsigned int i = threadIdx.x; i < gridDim.x; i += BLOCK) t += __ldcg(partials + i);
    total = block_sum<BLOCK>(t, smem);
    if (threadIdx.x == 0) *ticket = 0u;
    return true;
}

}  // namespace stag
