// stag_dslash.cuh — the per-site body of the staggered hopping term ("a
// different thread is associated to every (even) site").
//
//   (D psi)(x) = sum_{d=0..7} W_d(x) psi(nbr_d(x)),   d = 2*mu (forward) | 2*mu+1 (backward)
//
// with the hopping matrices W_d packed by stag_gauge_pack (1/2, eta, boundary sign, the
// dagger and the minus of the backward term are already folded in).  8 x (3x3 complex
// mat-vec) + 7 vector adds = 570 flop / site (BASELINE.json:north_star).  Not a dense
// contraction (a different matrix per site and direction): CUDA cores, no tensor cores.
//
// Memory behaviour: every thread streams its 8 hopping matrices with aligned, fully
// coalesced 128-bit loads that bypass L1 and are marked evict-first in L2 (read exactly once
// per Dslash); the 8 neighbour colour vectors come through the read-only L1/L2 path, where
// the up-to-8-fold re-use between neighbouring sites is served.
#pragma once

#include "stag_common.cuh"

namespace stag {

template <typename T> struct Prec;
template <> struct Prec<double> {
    static constexpr int id = STAG_F64;
    static constexpr int vec_chunks = 3;   // full 16-byte chunks per colour vector
};
template <> struct Prec<float> {
    static constexpr int id = STAG_F32;
    static constexpr int vec_chunks = 1;   // + one 8-byte tail chunk
};

// ---- colour-vector load / store in the device format ----------------------------------------
// NC = true: the vector is constant for the whole kernel (read-only path, __ldg).  NC = false: it
// is rewritten inside the same (persistent) kernel between grid barriers, so the loads must stay
// inside the memory model: plain coherent ld.global (still L1-allocating).
template <bool NC = true>
__device__ __forceinline__ void load_vec(const char *v, int Vh, int e, double (&x)[6]) {
    const double2 *p = reinterpret_cast<const double2 *>(v) + e;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const double2 t = NC ? ld_reuse(p + (size_t)c * Vh) : ld_coherent(p + (size_t)c * Vh);
        x[2 * c] = t.x; x[2 * c + 1] = t.y;
    }
}
template <bool NC = true>
__device__ __forceinline__ void load_vec(const char *v, int Vh, int e, float (&x)[6]) {
    const float4 *pa = reinterpret_cast<const float4 *>(v) + e;
    const float2 *pb = reinterpret_cast<const float2 *>(v + (size_t)Vh * 16) + e;
    const float4 a = NC ? ld_reuse(pa) : ld_coherent(pa);
    const float2 b = NC ? ld_reuse(pb) : ld_coherent(pb);
    x[0] = a.x; x[1] = a.y; x[2] = a.z; x[3] = a.w; x[4] = b.x; x[5] = b.y;
}
__device__ __forceinline__ void store_vec(char *__restrict__ v, int Vh, int e, const double (&x)[6]) {
    double2 *p = reinterpret_cast<double2 *>(v) + e;
#pragma unroll
    for (int c = 0; c < 3; ++c) p[(size_t)c * Vh] = make_double2(x[2 * c], x[2 * c + 1]);
}
__device__ __forceinline__ void store_vec(char *__restrict__ v, int Vh, int e, const float (&x)[6]) {
    reinterpret_cast<float4 *>(v)[e] = make_float4(x[0], x[1], x[2], x[3]);
    reinterpret_cast<float2 *>(v + (size_t)Vh * 16)[e] = make_float2(x[4], x[5]);
}

// ---- hopping-matrix load: u[18] = row-major 3x3 complex (re,im interleaved) -------------------
// c3: factor of the rebuilt third row (recon 12 only).  Rows 1-2 carry the folded factor
// f = +-1/2, so conj(row1 x row2) = f^2 * row3_true = (1/4) row3_true and the stored matrix
// needs f * row3_true = (4f) * conj(row1 x row2):  c3 = 4f = +-2  (reading A6).
template <typename T>
__device__ __forceinline__ void rebuild_row3(T (&u)[18], T c3) {
#pragma unroll
    for (int j = 0; j < 3; ++j) {
        const int a = (j + 1) % 3, b = (j + 2) % 3;
        // z = r1[a]*r2[b] - r1[b]*r2[a];  row3[j] = c3 * conj(z)
        const T zr = u[2 * a] * u[6 + 2 * b] - u[2 * a + 1] * u[6 + 2 * b + 1]
                   - u[2 * b] * u[6 + 2 * a] + u[2 * b + 1] * u[6 + 2 * a + 1];
        const T zi = u[2 * a] * u[6 + 2 * b + 1] + u[2 * a + 1] * u[6 + 2 * b]
                   - u[2 * b] * u[6 + 2 * a + 1] - u[2 * b + 1] * u[6 + 2 * a];
        u[12 + 2 * j] = c3 * zr;
        u[12 + 2 * j + 1] = -c3 * zi;
    }
}

template <int RECON>
__device__ __forceinline__ void load_link(const char *__restrict__ w, int Vh, int e,
                                          double (&u)[18], double c3, uint64_t pol) {
    const double2 *p = reinterpret_cast<const double2 *>(w) + e;
#pragma unroll
    for (int k = 0; k < RECON / 2; ++k) {
        const double2 t = ld_stream(p + (size_t)k * Vh, pol);
        u[2 * k] = t.x; u[2 * k + 1] = t.y;
    }
    if (RECON == 12) rebuild_row3(u, c3);
}
template <int RECON>
__device__ __forceinline__ void load_link(const char *__restrict__ w, int Vh, int e,
                                          float (&u)[18], float c3, uint64_t pol) {
    const float4 *p = reinterpret_cast<const float4 *>(w) + e;
#pragma unroll
    for (int k = 0; k < RECON / 4; ++k) {
        const float4 t = ld_stream(p + (size_t)k * Vh, pol);
        u[4 * k] = t.x; u[4 * k + 1] = t.y; u[4 * k + 2] = t.z; u[4 * k + 3] = t.w;
    }
    if (RECON == 18) {
        const float2 t = ld_stream(reinterpret_cast<const float2 *>(w + (size_t)Vh * 64) + e, pol);
        u[16] = t.x; u[17] = t.y;
    } else {
        rebuild_row3(u, c3);
    }
}

// N3 split-double links ("write a double precision number a by using two single
// precision numbers b and c ... reconstruct the double precision number a to be used in
// calculations"): wb = this direction's b planes in the fp32 packed layout, wb + c_off = its c planes.
template <int RECON>
__device__ __forceinline__ void load_link_split(const char *__restrict__ wb, size_t c_off, int Vh, int e,
                                                double (&u)[18], double c3, uint64_t pol) {
    const float4 *pb = reinterpret_cast<const float4 *>(wb) + e;
    const float4 *pc = reinterpret_cast<const float4 *>(wb + c_off) + e;
#pragma unroll
    for (int k = 0; k < RECON / 4; ++k) {
        const float4 b = ld_stream(pb + (size_t)k * Vh, pol);
        const float4 c = ld_stream(pc + (size_t)k * Vh, pol);
        u[4 * k] = (double)b.x + (double)c.x; u[4 * k + 1] = (double)b.y + (double)c.y;
        u[4 * k + 2] = (double)b.z + (double)c.z; u[4 * k + 3] = (double)b.w + (double)c.w;
    }
    if (RECON == 18) {
        const float2 b = ld_stream(reinterpret_cast<const float2 *>(wb + (size_t)Vh * 64) + e, pol);
        const float2 c = ld_stream(reinterpret_cast<const float2 *>(wb + c_off + (size_t)Vh * 64) + e, pol);
        u[16] = (double)b.x + (double)c.x; u[17] = (double)b.y + (double)c.y;
    } else {
        rebuild_row3(u, c3);
    }
}

template <typename T>
__device__ __forceinline__ void matvec_acc(const T (&u)[18], const T (&v)[6], T (&acc)[6]) {
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            // four fused multiply-adds per complex multiply-accumulate (not mul + fma + add)
            const T ur = u[6 * i + 2 * j], ui = u[6 * i + 2 * j + 1];
            acc[2 * i] = fma(ur, v[2 * j], acc[2 * i]);
            acc[2 * i] = fma(-ui, v[2 * j + 1], acc[2 * i]);
            acc[2 * i + 1] = fma(ur, v[2 * j + 1], acc[2 * i + 1]);
            acc[2 * i + 1] = fma(ui, v[2 * j], acc[2 * i + 1]);
        }
}

// bytes of one (parity, direction) link set
template <typename T, int RECON>
__device__ __host__ __forceinline__ size_t link_set_bytes(int Vh) {
    return (size_t)Vh * RECON * sizeof(T);
}

// acc[r] = (D in_r)(x) for the output site (e, par) and R independent source vectors in_r, with
// ONE load of the 8 hopping matrices (N1: links are 92 % of the stencil's bytes;
// the paper's multiple pseudo-fermions).  W: packed gauge base (both parities).
// `mask` bit r = source r wanted (uniform over the CTA); the others cost nothing.
// SPLIT (T = double only): W is a split-double buffer (N3).
template <typename T, int RECON, int R, bool NC = true, bool SPLIT = false>
__device__ __forceinline__ void dslash_site_multi(const Geom &g, const char *__restrict__ W,
                                                  const char *const (&in)[R], unsigned mask, int par,
                                                  int e, T (&acc)[R][6]) {
    static_assert(!SPLIT || sizeof(T) == 8, "split-double links carry fp64 vectors");
    const Site s = site_of(g, e, par);
    const int Vh = g.Vh;
    const uint64_t pol = policy_evict_first();
    const size_t set = SPLIT ? link_set_bytes<float, RECON>(Vh) : link_set_bytes<T, RECON>(Vh);
    const size_t c_off = 16 * set;                       // split: the c planes follow the 16 b sets
    const char *wp = W + (size_t)par * 8 * set;
    const int x[4] = {s.x0, s.x1, s.x2, s.x3};
    int stride = 1;
    int phase_sum = 0;
#pragma unroll
    for (int r = 0; r < R; ++r)
#pragma unroll
        for (int i = 0; i < 6; ++i) acc[r][i] = T(0);
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) {
        const int Lmu = g.L[mu];
        const int ef = (s.lex + stride - (x[mu] == Lmu - 1 ? Lmu * stride : 0)) >> 1;
        const int eb = (s.lex - stride + (x[mu] == 0 ? Lmu * stride : 0)) >> 1;
        T c3f = T(0), c3b = T(0);
        if (RECON == 12) {
            const T eta = (phase_sum & 1) ? T(-2) : T(2);
            c3f = (mu == 3 && x[3] == Lmu - 1) ? -eta : eta;
            c3b = (mu == 3 && x[3] == 0) ? eta : -eta;
        }
        T u[18], v[6];
        if constexpr (SPLIT) load_link_split<RECON>(wp + (size_t)(2 * mu) * set, c_off, Vh, e, u, c3f, pol);
        else load_link<RECON>(wp + (size_t)(2 * mu) * set, Vh, e, u, c3f, pol);
#pragma unroll
        for (int r = 0; r < R; ++r)
            if (R == 1 || ((mask >> r) & 1u)) {
                load_vec<NC>(in[r], Vh, ef, v);
                matvec_acc(u, v, acc[r]);
            }
        if constexpr (SPLIT) load_link_split<RECON>(wp + (size_t)(2 * mu + 1) * set, c_off, Vh, e, u, c3b, pol);
        else load_link<RECON>(wp + (size_t)(2 * mu + 1) * set, Vh, e, u, c3b, pol);
#pragma unroll
        for (int r = 0; r < R; ++r)
            if (R == 1 || ((mask >> r) & 1u)) {
                load_vec<NC>(in[r], Vh, eb, v);
                matvec_acc(u, v, acc[r]);
            }
        stride *= Lmu;
        phase_sum += x[mu];
    }
}

// single source
template <typename T, int RECON, bool NC = true, bool SPLIT = false>
__device__ __forceinline__ void dslash_site(const Geom &g, const char *__restrict__ W,
                                            const char *in, int par, int e, T (&acc)[6]) {
    const char *const ins[1] = {in};
    T a[1][6];
    dslash_site_multi<T, RECON, 1, NC, SPLIT>(g, W, ins, 1u, par, e, a);
#pragma unroll
    for (int i = 0; i < 6; ++i) acc[i] = a[0][i];
}

}  // namespace stag
