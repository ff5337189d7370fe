// stag_dslash_pipe.cuh — the staggered hopping term with the hopping matrices streamed through a
// per-thread asynchronous shared-memory ring (cp.async), for R >= 1 sources per link read.
//
// Why (profiles/README.md, "N1"): with R sources per thread the R x 6 accumulators plus one 18-real
// matrix leave no registers to keep several directions' loads in flight, and the register-staged
// kernel (stag_dslash.cuh) drops to ~45 % of HBM bandwidth at R = 4 — every warp sits on a long
// scoreboard.  Here the loads need no registers at all: every thread copies ITS OWN site's matrix
// for direction d + STAGES - 1 (and, optionally, its R gathered neighbours) from global to its own
// shared-memory slots with cp.async while it multiplies direction d.  The slots are thread-private,
// so the only synchronisation is the thread's own cp.async.wait_group: no mbarrier, no CTA barrier,
// no producer warp.  Bytes in flight per SM = threads x (STAGES - 1) x stage bytes, set by shared
// memory (227 KB), not by the register file.
//
// Stage layout (per CTA, per stage): rows of BLOCK 16-byte chunks, row k of the matrix at
// (k * BLOCK + tid) * 16 — consecutive lanes read consecutive 16-byte words: conflict-free.
#pragma once

#include "stag_dslash.cuh"

namespace stag {

__device__ __forceinline__ void cp_async16_stream(uint32_t dst, const void *src, uint64_t pol) {
    asm volatile("cp.async.cg.shared.global.L2::cache_hint [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "l"(pol)
                 : "memory");
}
__device__ __forceinline__ void cp_async8_stream(uint32_t dst, const void *src, uint64_t pol) {
    asm volatile("cp.async.ca.shared.global.L2::cache_hint [%0], [%1], 8, %2;" ::"r"(dst), "l"(src), "l"(pol)
                 : "memory");
}
__device__ __forceinline__ void cp_async16_reuse(uint32_t dst, const void *src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async8_reuse(uint32_t dst, const void *src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// bytes of one stage of the ring for a CTA of BLOCK threads
template <typename T, int RECON, int R, int BLOCK, bool VA>
__host__ __device__ constexpr int pipe_stage_bytes() {
    return BLOCK * (RECON * (int)sizeof(T) + (VA ? R * 6 * (int)sizeof(T) : 0));
}

// ---- issue / read of one direction's matrix -----------------------------------------------------------
template <int RECON, int BLOCK>
__device__ __forceinline__ void pipe_issue_link(uint32_t st, const char *w, int Vh, int e, uint64_t pol, double) {
    const double2 *p = reinterpret_cast<const double2 *>(w) + e;
#pragma unroll
    for (int k = 0; k < RECON / 2; ++k)
        cp_async16_stream(st + (uint32_t)(k * BLOCK + threadIdx.x) * 16u, p + (size_t)k * Vh, pol);
}
template <int RECON, int BLOCK>
__device__ __forceinline__ void pipe_issue_link(uint32_t st, const char *w, int Vh, int e, uint64_t pol, float) {
    const float4 *p = reinterpret_cast<const float4 *>(w) + e;
#pragma unroll
    for (int k = 0; k < RECON / 4; ++k)
        cp_async16_stream(st + (uint32_t)(k * BLOCK + threadIdx.x) * 16u, p + (size_t)k * Vh, pol);
    if (RECON == 18)
        cp_async8_stream(st + (uint32_t)(4 * BLOCK * 16) + threadIdx.x * 8u,
                         reinterpret_cast<const float2 *>(w + (size_t)Vh * 64) + e, pol);
}
template <int RECON, int BLOCK>
__device__ __forceinline__ void pipe_read_link(const unsigned char *st, double (&u)[18], double c3) {
    const double2 *p = reinterpret_cast<const double2 *>(st) + threadIdx.x;
#pragma unroll
    for (int k = 0; k < RECON / 2; ++k) {
        const double2 t = p[k * BLOCK];
        u[2 * k] = t.x; u[2 * k + 1] = t.y;
    }
    if (RECON == 12) rebuild_row3(u, c3);
}
template <int RECON, int BLOCK>
__device__ __forceinline__ void pipe_read_link(const unsigned char *st, float (&u)[18], float c3) {
    const float4 *p = reinterpret_cast<const float4 *>(st) + threadIdx.x;
#pragma unroll
    for (int k = 0; k < RECON / 4; ++k) {
        const float4 t = p[k * BLOCK];
        u[4 * k] = t.x; u[4 * k + 1] = t.y; u[4 * k + 2] = t.z; u[4 * k + 3] = t.w;
    }
    if (RECON == 18) {
        const float2 t = reinterpret_cast<const float2 *>(st + 4 * BLOCK * 16)[threadIdx.x];
        u[16] = t.x; u[17] = t.y;
    } else {
        rebuild_row3(u, c3);
    }
}

// ---- issue / read of one gathered neighbour vector (VA = true) --------------------------------------------
template <int BLOCK>
__device__ __forceinline__ void pipe_issue_vec(uint32_t sv, const char *v, int Vh, int e, double) {
    const double2 *p = reinterpret_cast<const double2 *>(v) + e;
#pragma unroll
    for (int c = 0; c < 3; ++c)
        cp_async16_reuse(sv + (uint32_t)(c * BLOCK + threadIdx.x) * 16u, p + (size_t)c * Vh);
}
template <int BLOCK>
__device__ __forceinline__ void pipe_issue_vec(uint32_t sv, const char *v, int Vh, int e, float) {
    cp_async16_reuse(sv + threadIdx.x * 16u, reinterpret_cast<const float4 *>(v) + e);
    cp_async8_reuse(sv + (uint32_t)(BLOCK * 16) + threadIdx.x * 8u,
                    reinterpret_cast<const float2 *>(v + (size_t)Vh * 16) + e);
}
template <int BLOCK>
__device__ __forceinline__ void pipe_read_vec(const unsigned char *sv, double (&x)[6]) {
    const double2 *p = reinterpret_cast<const double2 *>(sv) + threadIdx.x;
#pragma unroll
    for (int c = 0; c < 3; ++c) { const double2 t = p[c * BLOCK]; x[2 * c] = t.x; x[2 * c + 1] = t.y; }
}
template <int BLOCK>
__device__ __forceinline__ void pipe_read_vec(const unsigned char *sv, float (&x)[6]) {
    const float4 a = reinterpret_cast<const float4 *>(sv)[threadIdx.x];
    const float2 b = reinterpret_cast<const float2 *>(sv + BLOCK * 16)[threadIdx.x];
    x[0] = a.x; x[1] = a.y; x[2] = a.z; x[3] = a.w; x[4] = b.x; x[5] = b.y;
}

// acc[r] = (D in_r)(x) for the output site (e, par), R sources, matrices through the ring.
// `ring`: STAGES * pipe_stage_bytes<T,RECON,R,BLOCK,VA>() bytes of shared memory, 16-byte aligned.
// VA: the gathered neighbours go through the ring too (cp.async.ca); else plain loads (NC as in
// stag_dslash.cuh).  The caller must not have outstanding cp.async groups of its own.
template <typename T, int RECON, int R, int BLOCK, int STAGES, bool VA, bool NC = true>
__device__ __forceinline__ void dslash_site_pipe(const Geom &g, const char *__restrict__ W,
                                                 const char *const (&in)[R], unsigned mask, int par, int e,
                                                 T (&acc)[R][6], unsigned char *ring) {
    static_assert(STAGES >= 2 && STAGES <= 8, "ring depth");
    constexpr int P = STAGES - 1;                       // prefetch distance (directions)
    constexpr int SB = pipe_stage_bytes<T, RECON, R, BLOCK, VA>();
    constexpr int LB = BLOCK * RECON * (int)sizeof(T);  // matrix part of a stage
    constexpr int VB = BLOCK * 6 * (int)sizeof(T);      // one vector
    const Site s = site_of(g, e, par);
    const int Vh = g.Vh;
    const uint64_t pol = policy_evict_first();
    const char *wp = W + (size_t)par * 8 * link_set_bytes<T, RECON>(Vh);
    const uint32_t ring32 = (uint32_t)__cvta_generic_to_shared(ring);
    const int x[4] = {s.x0, s.x1, s.x2, s.x3};

    int nb[8];
    T c3[8];
    {
        int stride = 1, phase_sum = 0;
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) {
            const int Lmu = g.L[mu];
            nb[2 * mu] = (s.lex + stride - (x[mu] == Lmu - 1 ? Lmu * stride : 0)) >> 1;
            nb[2 * mu + 1] = (s.lex - stride + (x[mu] == 0 ? Lmu * stride : 0)) >> 1;
            const T eta = (phase_sum & 1) ? T(-2) : T(2);
            c3[2 * mu] = (mu == 3 && x[3] == Lmu - 1) ? -eta : eta;
            c3[2 * mu + 1] = (mu == 3 && x[3] == 0) ? eta : -eta;
            stride *= Lmu;
            phase_sum += x[mu];
        }
    }
    auto issue = [&](int d) {
        const uint32_t st = ring32 + (uint32_t)((d % STAGES) * SB);
        pipe_issue_link<RECON, BLOCK>(st, wp + (size_t)d * link_set_bytes<T, RECON>(Vh), Vh, e, pol, T());
        if (VA) {
#pragma unroll
            for (int r = 0; r < R; ++r)
                if (R == 1 || ((mask >> r) & 1u))
                    pipe_issue_vec<BLOCK>(st + (uint32_t)(LB + r * VB), in[r], Vh, nb[d], T());
        }
    };
#pragma unroll
    for (int d = 0; d < P; ++d) { issue(d); cp_async_commit(); }
#pragma unroll
    for (int r = 0; r < R; ++r)
#pragma unroll
        for (int i = 0; i < 6; ++i) acc[r][i] = T(0);
#pragma unroll
    for (int d = 0; d < 8; ++d) {
        if (d + P < 8) issue(d + P);
        cp_async_commit();                               // (possibly empty) group: keeps the count uniform
        cp_async_wait<P>();                              // direction d has landed in this thread's slots
        const unsigned char *st = ring + (d % STAGES) * SB;
        T u[18], v[6];
        pipe_read_link<RECON, BLOCK>(st, u, c3[d]);
#pragma unroll
        for (int r = 0; r < R; ++r)
            if (R == 1 || ((mask >> r) & 1u)) {
                if (VA) pipe_read_vec<BLOCK>(st + LB + r * VB, v);
                else load_vec<NC>(in[r], Vh, nb[d], v);
                matvec_acc(u, v, acc[r]);
            }
    }
    cp_async_wait<0>();
}

}  // namespace stag
