// stag_cg_persist.cuh — the whole multi-shift CG solve of R independent sources as ONE persistent
// cooperative kernel (PAPER.md:125-129 shifted CG; "multiple pseudo-fermions" = the R
// independent right-hand sides).
//
// For the lattices of the paper's runs (4 x 16^3 ... 8 x 32^3, 4 x 48^3) one
// CG iteration moves only a few hundred MB, so four kernel launches per iteration — each with a
// fill/drain ramp and, twice, a serial "last CTA" reduction tail — cost as much as 15 % of the
// iteration.  Here one CTA per SM owns a fixed, contiguous range of sites for the whole solve:
//
//   phase A  w = D_oe p_base                on the CTA's odd sites   -> global (neighbours read it)
//            grid barrier
//   phase B  q = (m^2+sigma_0) p - D_eo w   on the CTA's even sites  -> q stays in SHARED memory
//            per-CTA partial of Re<p,q>     -> global;  grid barrier
//   phase C  every CTA adds the partials in the same order (bit-identical alpha everywhere),
//            runs the a4 recurrences in its own shared memory, then r -= alpha q with r and q
//            both in shared memory (a5 moves no HBM bytes at all); partial of <r,r>; grid barrier
//   phase D  every CTA: beta, beta_i, zeta_i, convergence latch, freezing (a4, a7); then the base shift of a6
//            (p_base is what the neighbours gather next).  The other live shifts' x_i, p_i updates are DEFERRED:
//            they are worked off, one CTA-wide pass at a time, while the CTA waits at the sync points of the
//            next iteration (a wait is skew + barrier latency during which HBM would idle), and whatever is left
//            is forced before phase D overwrites their coefficients.  r and q swap buffers every iteration so
//            that the old r stays readable until then.
//   sync     after B and C: grid-wide (the two reductions).  After A and D a CTA needs w / p_base only from the
//            CTAs that own its neighbouring sites: per-CTA epoch flags instead of a grid barrier.
//   L2       x_i, p_i of the lightest shifts (the longest-lived) are marked evict_last, the hopping matrices
//            evict_first: what fits of the shift vectors stays in the 126 MB L2 across iterations.
//
// r, q and the CTA's own slice of p_base live in shared memory for the whole solve when they fit
// (3 x 48 B x sites/SM x R: 129 KB at 32^3 x 8, R = 1); what does not fit (priority r, q, p) stays
// in the global workspace.  All scalars are fp64 and never leave the SM; the host sees one launch
// and one read-back.
//
// R > 1 (N1): in the stencil phases (A, B) a thread owns one output site and ALL R sources: the 8
// hopping matrices are loaded into registers once and applied to the R gathered neighbours, so the
// links — 92 % of the stencil's bytes and most of its load instructions — are paid once for R
// sources.  In the streaming phases (start, C, D, a7) the CTA's warps are split between the sources
// (warp-uniform source, 32 consecutive sites per warp).  Every source has its own scalars, shift
// list and convergence latch; a source that has converged stops issuing work while the others finish.
#pragma once

#include "stag_cg.cuh"
#include "stag_dslash.cuh"

// Per-phase timers (build with -DSTAG_PHASE_TIMERS: `STAG_PHASE_TIMERS=1 python -m paper_1010_5433_b200._build`
// writes libstag_b200_timers.so, which the binding loads when the same variable is set).  CTAs 0, 77 and the last
// one print, at the end of the solve, the mean microseconds per iteration they spent in each phase, at each sync
// point (arrive + deferred shift updates worked off while waiting + wait) and in the shift updates that had to be
// forced before phase D (%globaltimer, CTA-wide: a __syncthreads precedes every tick).  Compiles to nothing otherwise.
#ifdef STAG_PHASE_TIMERS
#include <cstdio>
#define STAG_T_DECL                                                                       \
    unsigned long long tt_[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0}, t0_, t1_;                    \
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0_));
#define STAG_TICK(k)                                                                      \
    do {                                                                                  \
        __syncthreads();                                                                  \
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1_));                           \
        tt_[k] += t1_ - t0_;                                                              \
        t0_ = t1_;                                                                        \
    } while (0)
#define STAG_T_REPORT(R_, iters_)                                                                          \
    if (threadIdx.x == 0 && (blockIdx.x == 0 || blockIdx.x == 77 || blockIdx.x == gridDim.x - 1 ||         \
                             STAG_PHASE_TIMERS > 1)) {                                                     \
        const double k_ = 1e-3 / ((iters_) > 0 ? (iters_) : 1);                                            \
        unsigned smid_;                                                                                    \
        asm volatile("mov.u32 %0, %%smid;" : "=r"(smid_));                                                 \
        printf("[stag timers] CTA %d sm %u R=%d iters %d  us/iter: A %.2f sync %.2f | B %.2f sync %.2f | C %.2f " \
               "sync %.2f | D %.2f sync %.2f\n", (int)blockIdx.x, smid_, R_, (int)(iters_),                 \
               tt_[0] * k_, tt_[1] * k_, tt_[2] * k_, tt_[3] * k_, tt_[4] * k_, tt_[5] * k_, tt_[6] * k_,  \
               tt_[7] * k_);                                                                               \
    }
#else
#define STAG_T_DECL
#define STAG_TICK(k) ((void)0)
#define STAG_T_REPORT(R_, iters_)
#endif

namespace stag {

// ---- grid barrier: monotone counter, arrive / wait split ---------------------------------------
// Safe only because the kernel is launched cooperatively (all CTAs co-resident).
__device__ __forceinline__ void grid_arrive(unsigned int *bar) {
    __syncthreads();                       // every thread's writes of this phase are issued
    if (threadIdx.x == 0) {
        __threadfence();                   // ... and ordered before the arrival (cumulative)
        atomicAdd(bar, 1u);
    }
}
__device__ __forceinline__ void grid_wait(unsigned int *bar, unsigned int target) {
    if (threadIdx.x == 0) {
        unsigned int v;
        do {
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(bar) : "memory");
        } while ((int)(v - target) < 0);
        // the acquire load orders everything after it (and, through the CTA barrier below, every other
        // thread's later loads) behind the arrivals it observed: no further fence needed
    }
    __syncthreads();
}

// ---- a vector slice resident in shared memory: `n` thread-private slots ---------------------------
template <typename T> struct SVec;
template <> struct SVec<double> {
    double2 *a; int n;
    __device__ __forceinline__ void init(unsigned char *base, int n_) { a = reinterpret_cast<double2 *>(base); n = n_; }
    __device__ __forceinline__ void load(int slot, double (&x)[6]) const {
#pragma unroll
        for (int c = 0; c < 3; ++c) { const double2 t = a[c * n + slot]; x[2 * c] = t.x; x[2 * c + 1] = t.y; }
    }
    __device__ __forceinline__ void store(int slot, const double (&x)[6]) {
#pragma unroll
        for (int c = 0; c < 3; ++c) a[c * n + slot] = make_double2(x[2 * c], x[2 * c + 1]);
    }
};
template <> struct SVec<float> {
    float4 *a; float2 *b;
    __device__ __forceinline__ void init(unsigned char *base, int n_) {
        a = reinterpret_cast<float4 *>(base); b = reinterpret_cast<float2 *>(base + (size_t)n_ * 16);
    }
    __device__ __forceinline__ void load(int slot, float (&x)[6]) const {
        const float4 u = a[slot]; const float2 v = b[slot];
        x[0] = u.x; x[1] = u.y; x[2] = u.z; x[3] = u.w; x[4] = v.x; x[5] = v.y;
    }
    __device__ __forceinline__ void store(int slot, const float (&x)[6]) {
        a[slot] = make_float4(x[0], x[1], x[2], x[3]); b[slot] = make_float2(x[4], x[5]);
    }
};

// A CTA-owned slice of one vector of each of the R sources: in shared memory when it fits (slot =
// source * S + local site), else in the global workspace (read and written only by this CTA, with
// a CTA barrier between phases, so plain loads and stores are coherent).
template <typename T>
struct Slice {
    SVec<T> s;
    char *g;          // global home of source 0 (device format)
    size_t gstride;   // bytes between the sources' global homes
    bool res;
    __device__ __forceinline__ void load(int slot, int r, int Vh, int e, T (&x)[6]) const {
        if (res) s.load(slot, x); else load_vec<false>(g + (size_t)r * gstride, Vh, e, x);
    }
    __device__ __forceinline__ void store(int slot, int r, int Vh, int e, const T (&x)[6]) {
        if (res) s.store(slot, x); else store_vec(g + (size_t)r * gstride, Vh, e, x);
    }
};

// ---- own-site access to x_i, p_i with an explicit L2 eviction policy -------------------------------
// Every x_i, p_i element is read and written by exactly one thread, once per iteration: L1 is bypassed.  In L2
// the vectors of the KEEP set (the lightest shifts, which stay live longest; PersistArgs::keep_mask) are marked
// evict_last so that they survive the 2 x 151 MB of hopping matrices (evict_first) that stream through the
// 126 MB L2 every iteration: their 192 B per site and iteration then never reach HBM.  All other shifts stream
// (evict_first).
__device__ __forceinline__ uint64_t policy_evict_last() {
    uint64_t pol;
    asm("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ void load_vec_pol(const char *v, int Vh, int e, double (&x)[6], uint64_t pol) {
    const double2 *p = reinterpret_cast<const double2 *>(v) + e;
#pragma unroll
    for (int c = 0; c < 3; ++c)
        asm volatile("ld.global.L1::no_allocate.L2::cache_hint.v2.f64 {%0,%1}, [%2], %3;"
                     : "=d"(x[2 * c]), "=d"(x[2 * c + 1]) : "l"(p + (size_t)c * Vh), "l"(pol) : "memory");
}
__device__ __forceinline__ void load_vec_pol(const char *v, int Vh, int e, float (&x)[6], uint64_t pol) {
    asm volatile("ld.global.L1::no_allocate.L2::cache_hint.v4.f32 {%0,%1,%2,%3}, [%4], %5;"
                 : "=f"(x[0]), "=f"(x[1]), "=f"(x[2]), "=f"(x[3])
                 : "l"(reinterpret_cast<const float4 *>(v) + e), "l"(pol) : "memory");
    asm volatile("ld.global.L1::no_allocate.L2::cache_hint.v2.f32 {%0,%1}, [%2], %3;"
                 : "=f"(x[4]), "=f"(x[5])
                 : "l"(reinterpret_cast<const float2 *>(v + (size_t)Vh * 16) + e), "l"(pol) : "memory");
}
__device__ __forceinline__ void store_vec_pol(char *v, int Vh, int e, const double (&x)[6], uint64_t pol) {
    double2 *p = reinterpret_cast<double2 *>(v) + e;
#pragma unroll
    for (int c = 0; c < 3; ++c)
        asm volatile("st.global.L1::no_allocate.L2::cache_hint.v2.f64 [%0], {%1,%2}, %3;"
                     :: "l"(p + (size_t)c * Vh), "d"(x[2 * c]), "d"(x[2 * c + 1]), "l"(pol) : "memory");
}
__device__ __forceinline__ void store_vec_pol(char *v, int Vh, int e, const float (&x)[6], uint64_t pol) {
    asm volatile("st.global.L1::no_allocate.L2::cache_hint.v4.f32 [%0], {%1,%2,%3,%4}, %5;"
                 :: "l"(reinterpret_cast<float4 *>(v) + e), "f"(x[0]), "f"(x[1]), "f"(x[2]), "f"(x[3]), "l"(pol)
                 : "memory");
    asm volatile("st.global.L1::no_allocate.L2::cache_hint.v2.f32 [%0], {%1,%2}, %3;"
                 :: "l"(reinterpret_cast<float2 *>(v + (size_t)Vh * 16) + e), "f"(x[4]), "f"(x[5]), "l"(pol)
                 : "memory");
}

// ---- streaming (evict-first) own-site access, used by the mixed-precision kernel ---------------------
__device__ __forceinline__ void load_vec_cs(const char *v, int Vh, int e, double (&x)[6]) {
    const double2 *p = reinterpret_cast<const double2 *>(v) + e;
#pragma unroll
    for (int c = 0; c < 3; ++c) { const double2 t = __ldcs(p + (size_t)c * Vh); x[2 * c] = t.x; x[2 * c + 1] = t.y; }
}
__device__ __forceinline__ void load_vec_cs(const char *v, int Vh, int e, float (&x)[6]) {
    const float4 a = __ldcs(reinterpret_cast<const float4 *>(v) + e);
    const float2 b = __ldcs(reinterpret_cast<const float2 *>(v + (size_t)Vh * 16) + e);
    x[0] = a.x; x[1] = a.y; x[2] = a.z; x[3] = a.w; x[4] = b.x; x[5] = b.y;
}
__device__ __forceinline__ void store_vec_cs(char *v, int Vh, int e, const double (&x)[6]) {
    double2 *p = reinterpret_cast<double2 *>(v) + e;
#pragma unroll
    for (int c = 0; c < 3; ++c) __stcs(p + (size_t)c * Vh, make_double2(x[2 * c], x[2 * c + 1]));
}
__device__ __forceinline__ void store_vec_cs(char *v, int Vh, int e, const float (&x)[6]) {
    __stcs(reinterpret_cast<float4 *>(v) + e, make_float4(x[0], x[1], x[2], x[3]));
    __stcs(reinterpret_cast<float2 *>(v + (size_t)Vh * 16) + e, make_float2(x[4], x[5]));
}

// ---- per-CTA copy of one source's scalar state (every CTA carries the same values) ------------------
template <typename T>
struct Scalars {
    double delta[STAG_MAX_SHIFTS], zeta[STAG_MAX_SHIFTS], theta[STAG_MAX_SHIFTS], theta_new[STAG_MAX_SHIFTS];
    double resid[STAG_MAX_SHIFTS];
    T ca[STAG_MAX_SHIFTS], cz[STAG_MAX_SHIFTS], cb[STAG_MAX_SHIFTS];   // alpha_i, zeta_i(new), beta_i of live shifts
    int live[STAG_MAX_SHIFTS];                                           // compacted list, base excluded
    int active[STAG_MAX_SHIFTS], iters_shift[STAG_MAX_SHIFTS];
    double bb, rr, alpha, alpha_old, beta_old, best_rr, pq;
    T a_base, z_base, b_base;
    T c0;                    // m^2 + sigma_0 of THIS source (N2: the polish solves one shift per source)
    double stop;             // on sqrt(rr/bb) of this source
    int nlive, iter, done, converged, breakdown, stagnated, since_best;
    // done: 0 running | 1 this iteration's x/p update is the last | 2 over
};

// sum of the G per-CTA partials, same order in every CTA => bit-identical result everywhere.
// Valid in every lane of the calling warp.
__device__ __forceinline__ double grid_total(const double *part, int G) {
    double t = 0.0;
    for (int i = threadIdx.x & 31; i < G; i += 32) t += __ldcg(part + i);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
    return t;
}

// per-source CTA sums -> slot[s * G].  Two thread mappings:
// "all": every thread holds one value per source (stencil phases)
template <int NT, int R>
__device__ __forceinline__ void cta_partials_all(const double (&v)[R], double *red /* (NT/32)*R */, double *slot, int G) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double w[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        w[r] = v[r];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) w[r] += __shfl_xor_sync(0xffffffffu, w[r], o);
    }
    __syncthreads();
    if (lane == 0) {
#pragma unroll
        for (int r = 0; r < R; ++r) red[warp * R + r] = w[r];
    }
    __syncthreads();
    if (warp == 0) {
#pragma unroll
        for (int s = 0; s < R; ++s) {
            double t = lane < NT / 32 ? red[lane * R + s] : 0.0;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
            if (lane == 0) __stcg(slot + (size_t)s * G, t);
        }
    }
}
// "stream": warp w works for source w / (NT/32/R) (streaming phases)
template <int NT, int R>
__device__ __forceinline__ void cta_partials_stream(double v, double *red /* NT/32 */, double *slot, int G) {
    constexpr int WPS = NT / 32 / R;             // warps per source
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    __syncthreads();
    if (lane == 0) red[warp] = v;
    __syncthreads();
    if (warp == 0) {
#pragma unroll
        for (int s = 0; s < R; ++s) {
            double t = lane < WPS ? red[s * WPS + lane] : 0.0;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
            if (lane == 0) __stcg(slot + (size_t)s * G, t);
        }
    }
}

struct PersistArgs {
    const char *W;        // packed gauge
    const char *b;        // R sources, stride b_stride
    size_t b_stride;
    char *w;              // R odd-site scratch vectors (global), stride vec_stride
    char *r_g, *q_g;      // R global homes of r, q (used when not resident), stride vec_stride
    size_t vec_stride;
    char *p;              // search directions [source][shift] (global), stride p_stride
    size_t p_stride;
    char *x;              // solutions [source][shift], stride x_stride
    size_t x_stride;
    char *y;              // nullable; R vectors, stride x_stride
    CgState *state;       // R states, stride state_stride bytes
    size_t state_stride;
    double *partials;     // 2 * R * gridDim.x doubles: per-CTA partials of <p,q>, then of <r,r>
    unsigned int *flags;  // gridDim.x epoch words, one per 128-byte line (zeroed by the host before the launch)
    int S;                // slots per CTA and source in a resident slice = the largest CTA's sites (multiple of 32)
    int nrhs;             // sources actually present (<= R)
    int res_r, res_q, res_p;   // which slices are resident in shared memory
    unsigned keep_mask;   // shifts whose x_i, p_i are kept L2-resident (evict_last); the others stream
    int fill;             // 1: deferred shift updates are worked off while the CTA waits at a sync point
    int nbflags;          // 1: phases A->B and D->A wait for the owners of the neighbouring sites only; 0: for every CTA
};

// The CTA's contiguous range of 32-site tiles: tiles [c T / G, (c+1) T / G) of T, so the sizes differ by at most
// one tile and no SM idles (32^3 x 8 on 148 SMs: 100 CTAs of 28 tiles, 48 of 27).
__host__ __device__ __forceinline__ int cta_first_tile(int c, int T, int G) { return (int)((long long)c * T / G); }
__device__ __forceinline__ int tile_owner(int t, int T, int G) { return (int)((((long long)t + 1) * G - 1) / T); }

static constexpr int kMaxPersistGrid = 256;          // CTAs (= SMs) the neighbour tables are sized for

template <typename T, int RECON, int NT, int R, bool SPLIT = false>
__global__ void __launch_bounds__(NT, 1)
cg_persistent_kernel(const Geom g, const PersistArgs a) {
    extern __shared__ __align__(16) unsigned char dyn[];
    __shared__ Scalars<T> sc[R];
    __shared__ double red[(NT / 32) * R];
    __shared__ int n_running;
    __shared__ unsigned int nb_mask[kMaxPersistGrid / 32];
    __shared__ int nb_list[kMaxPersistGrid];
    __shared__ int nb_n;
    __shared__ unsigned int sync_seen;               // number of the last sync point warp 0 has seen released

    constexpr int LS = NT / R;                       // streaming phases: sites per pass and source
    // deferred update: shifts per item = loads in flight per thread.  One: with two, the stencil phases of the same
    // kernel ran at 31 instead of 23 us (register pressure changes their schedule).
    constexpr int B = 1;
    const int tid = threadIdx.x, G = gridDim.x, Vh = g.Vh, S = a.S;
    const int rhs = tid / LS, l0 = tid % LS;         // streaming phases: this thread's source (warp-uniform)
    const int tiles = (Vh + 31) >> 5;
    const int e0 = min(Vh, cta_first_tile(blockIdx.x, tiles, G) << 5);
    const int ns = min(Vh, cta_first_tile(blockIdx.x + 1, tiles, G) << 5) - e0;
    unsigned int *bar = &a.state->ticket;
    double *part_pq = a.partials, *part_rr = a.partials + (size_t)R * G;

    CgState *st = reinterpret_cast<CgState *>(reinterpret_cast<char *>(a.state) + (size_t)rhs * a.state_stride);
    const int nshift = a.state->nshift, base = a.state->base, maxiter = a.state->maxiter;   // same for every source
    const int freeze = a.state->freeze, fp32 = a.state->fp32;

    const char *b_r = a.b + (size_t)rhs * a.b_stride;
    char *p_r = a.p + (size_t)rhs * nshift * a.p_stride;
    char *x_r = a.x + (size_t)rhs * nshift * a.x_stride;
    char *p_base = p_r + (size_t)base * a.p_stride;
    char *x_base = x_r + (size_t)base * a.x_stride;
    const size_t pb_stride = (size_t)nshift * a.p_stride;       // between the sources' p_base
    char *p_base0 = a.p + (size_t)base * a.p_stride;            // p_base of source 0
    // L2 policy of shift i's x_i, p_i (made where it is used: two registers less across the stencil phases)
    auto shift_policy = [&](int i) { return ((a.keep_mask >> i) & 1u) ? policy_evict_last() : policy_evict_first(); };

    // r and q swap roles every iteration when both live in the same kind of memory: phase C then writes the new
    // r over q and leaves the old r intact for the deferred shift updates still pending (see the sync point)
    const bool swap_rq = a.res_r == a.res_q;
    Slice<T> r_s, q_s, p_s;
    {
        const size_t slice = (size_t)S * R * 6 * sizeof(T);
        unsigned char *d = dyn;
        r_s.res = a.res_r != 0; r_s.g = a.r_g; r_s.gstride = a.vec_stride;
        if (r_s.res) { r_s.s.init(d, S * R); d += slice; }
        q_s.res = a.res_q != 0; q_s.g = a.q_g; q_s.gstride = a.vec_stride;
        if (q_s.res) { q_s.s.init(d, S * R); d += slice; }
        p_s.res = a.res_p != 0; p_s.g = p_base0; p_s.gstride = pb_stride;
        if (p_s.res) { p_s.s.init(d, S * R); d += slice; }
    }
    const bool present = rhs < a.nrhs;

    // ---- the CTAs that own a neighbour of one of this CTA's sites (either parity) ---------------------
    if (tid < kMaxPersistGrid / 32) nb_mask[tid] = 0u;
    if (tid == 0) { nb_n = 0; sync_seen = 0u; }
    __syncthreads();
    if (a.nbflags) {
        for (int ls = tid; ls < 2 * ns; ls += NT) {
            const int par = ls >= ns, e = e0 + (par ? ls - ns : ls);
            const Site s = site_of(g, e, par);
            const int x[4] = {s.x0, s.x1, s.x2, s.x3};
            int stride = 1;
#pragma unroll
            for (int mu = 0; mu < 4; ++mu) {
                const int Lmu = g.L[mu];
                const int ef = (s.lex + stride - (x[mu] == Lmu - 1 ? Lmu * stride : 0)) >> 1;
                const int eb = (s.lex - stride + (x[mu] == 0 ? Lmu * stride : 0)) >> 1;
                const int of = tile_owner(ef >> 5, tiles, G), ob = tile_owner(eb >> 5, tiles, G);
                if (of != (int)blockIdx.x) atomicOr(&nb_mask[of >> 5], 1u << (of & 31));
                if (ob != (int)blockIdx.x) atomicOr(&nb_mask[ob >> 5], 1u << (ob & 31));
                stride *= Lmu;
            }
        }
        __syncthreads();
    }
    for (int c = tid; c < G; c += NT)
        if (c != (int)blockIdx.x && (!a.nbflags || ((nb_mask[c >> 5] >> (c & 31)) & 1u))) nb_list[atomicAdd(&nb_n, 1)] = c;
    __syncthreads();
    const int nnb = nb_n;

    // ---- start: x_i = 0, r = p_i = b, bb = <b,b> ---------------------------------------------------
    if (tid < 32 * R && (tid & 31) < STAG_MAX_SHIFTS) {
        const int s = tid >> 5, i = tid & 31;
        const CgState *ss = reinterpret_cast<const CgState *>(reinterpret_cast<const char *>(a.state) + (size_t)s * a.state_stride);
        const bool on = i < nshift && s < a.nrhs;
        sc[s].delta[i] = on ? ss->delta[i] : 0.0;
        sc[s].zeta[i] = 1.0; sc[s].theta[i] = 1.0; sc[s].theta_new[i] = 1.0;
        sc[s].resid[i] = 1.0;
        sc[s].active[i] = on ? 1 : 0;
        sc[s].iters_shift[i] = 0;
    }
    {
        double acc = 0.0;
        if (present)
            for (int ls = l0; ls < ns; ls += LS) {
                const int e = e0 + ls, slot = rhs * S + ls;
                T v[6], z[6] = {T(0), T(0), T(0), T(0), T(0), T(0)};
                load_vec<true>(b_r, Vh, e, v);
#pragma unroll
                for (int k = 0; k < 6; ++k) acc += (double)v[k] * (double)v[k];
                r_s.store(slot, rhs, Vh, e, v);
                if (p_s.res) p_s.s.store(slot, v);
                for (int i = 0; i < nshift; ++i) {
                    const uint64_t pol = shift_policy(i);
                    if (i == base) store_vec(p_base, Vh, e, v);
                    else store_vec_pol(p_r + (size_t)i * a.p_stride, Vh, e, v, pol);
                    store_vec_pol(x_r + (size_t)i * a.x_stride, Vh, e, z, pol);
                }
            }
        cta_partials_stream<NT, R>(acc, red, part_rr + blockIdx.x, G);
    }
    grid_arrive(bar);                                  // grid-wide: bb, and every p_base is in place for phase A
    grid_wait(bar, (unsigned)G);
    if (tid < 32 * R) {
        const int s = tid >> 5;
        const double bb = grid_total(part_rr + (size_t)s * G, G);
        if ((tid & 31) == 0) {
            Scalars<T> &c = sc[s];
            const CgState *ss = reinterpret_cast<const CgState *>(reinterpret_cast<const char *>(a.state) + (size_t)min(s, a.nrhs - 1) * a.state_stride);
            c.c0 = (T)ss->c0; c.stop = ss->stop;
            c.bb = bb; c.rr = bb; c.best_rr = bb; c.alpha = 0.0; c.alpha_old = 1.0; c.beta_old = 0.0;
            c.pq = 0.0; c.iter = 0; c.done = 0; c.converged = 0; c.breakdown = 0; c.stagnated = 0;
            c.since_best = 0; c.nlive = 0;
            if (s >= a.nrhs) c.done = 2;
            else if (!(bb > 0.0)) { c.converged = (bb == 0.0); c.breakdown = !(bb == 0.0); c.done = 2; }
            else if (ss->zero_ok && ss->stop >= 1.0) { c.converged = 1; c.done = 2; }   // polish: x = 0 already meets it
            else if (maxiter <= 0) c.done = 2;
        }
    }
    __syncthreads();
    if (tid == 0) {
        int n = 0;
        for (int s = 0; s < R; ++s) n += sc[s].done == 0;
        n_running = n;
    }
    __syncthreads();

    // stencil phases: the R sources' input / output vectors
    const char *pin[R];
    const char *win[R];
    char *wout[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        pin[r] = p_base0 + (size_t)r * pb_stride;
        win[r] = a.w + (size_t)r * a.vec_stride;
        wout[r] = a.w + (size_t)r * a.vec_stride;
    }

    // ---- iterations: a four-phase state machine around ONE sync point -----------------------------------
    // (one copy of the sync-and-work-off code keeps the kernel inside its register budget: as a lambda called
    // from four places it was not inlined and every captured variable went to local memory.  The stencil's
    // instruction schedule — how many of a site's 96 loads are in flight — is sensitive to every register the
    // surrounding code keeps alive across it: with two shifts per item instead of one the same stencil ran at 31
    // instead of 23 us per phase.  profiles/README.md has the variants that were measured.)
    //
    // Deferred shift update (a6 of the iteration just finished), worked off in items: one item = one pass of
    // the CTA over its sites (one site per thread) x one live shift.  Its state is in registers, identical in
    // all threads of a source; the coefficients stay in sc[rhs] until phase D of the next iteration.  The r they
    // need is r_s at every sync point: phase C leaves it alone (swap) and the roles only flip in phase D.
    int pn = 0, pj = 0, ppass = 0, pnpass = 0;        // live shifts, next shift, next pass, passes (0: nothing pending)
    bool act = false, act2 = false;
    unsigned mask = 0;
    unsigned int gepoch = 1, nepoch = 0;              // grid-wide barriers / neighbour syncs so far
    int phase = 0;                                    // 0 A | 1 B | 2 C | 3 D
    STAG_T_DECL
    while (n_running > 0 || phase != 0) {
        if (phase == 0) {
            act = sc[rhs].done == 0;                 // streaming phases: this thread's source is still iterating
            mask = 0;                                // stencil phases: the sources still iterating
#pragma unroll
            for (int r = 0; r < R; ++r) mask |= (sc[r].done == 0 ? 1u : 0u) << r;
            // phase A (a2): w = D_oe p_base on this CTA's odd sites
            for (int ls = tid; ls < ns; ls += NT) {
                T acc[R][6];
                dslash_site_multi<T, RECON, R, false, SPLIT>(g, a.W, pin, mask, 1, e0 + ls, acc);
#pragma unroll
                for (int r = 0; r < R; ++r)
                    if (R == 1 || ((mask >> r) & 1u)) store_vec(wout[r], Vh, e0 + ls, acc[r]);
            }
        } else if (phase == 1) {
            // phase B (a3): q = c0 p - D_eo w, partial Re<p,q>
            double dot[R];
            T c0[R];
#pragma unroll
            for (int r = 0; r < R; ++r) { dot[r] = 0.0; c0[r] = sc[r].c0; }
            for (int ls = tid; ls < ns; ls += NT) {
                const int e = e0 + ls;
                T acc[R][6];
                dslash_site_multi<T, RECON, R, false, SPLIT>(g, a.W, win, mask, 0, e, acc);
#pragma unroll
                for (int r = 0; r < R; ++r)
                    if (R == 1 || ((mask >> r) & 1u)) {
                        T pv[6];
                        p_s.load(r * S + ls, r, Vh, e, pv);
#pragma unroll
                        for (int k = 0; k < 6; ++k) {
                            acc[r][k] = c0[r] * pv[k] - acc[r][k];
                            dot[r] += (double)pv[k] * (double)acc[r][k];
                        }
                        q_s.store(r * S + ls, r, Vh, e, acc[r]);
                    }
            }
            cta_partials_all<NT, R>(dot, red, part_pq + blockIdx.x, G);
        } else if (phase == 2) {
            // phase C (a4 after <p,q>, then a5): alpha, theta_new_i;  r_new = r - alpha q;  partial <r,r>
            if (tid < 32 * R) {
                const int s = tid >> 5, i = tid & 31;
                Scalars<T> &c = sc[s];
                if (c.done == 0) {
                    const double pq = grid_total(part_pq + (size_t)s * G, G);
                    const double alpha = c.rr / pq;
                    const bool bad = !(pq > 0.0) || !isfinite(alpha);
                    const double k = alpha * c.beta_old / c.alpha_old;
                    __syncwarp();
                    if (!bad && i < nshift) c.theta_new[i] = 1.0 / ((1.0 + c.delta[i] * alpha) + k * (1.0 - c.theta[i]));
                    if (i == 0) {
                        c.pq = pq;
                        if (bad) { c.breakdown = 1; c.done = 2; } else c.alpha = alpha;   // breakdown: no update
                    }
                }
            }
            __syncthreads();
            act2 = act && sc[rhs].done == 0;
            double acc = 0.0;
            if (act2) {
                const T na = (T)(-sc[rhs].alpha);
                for (int ls = l0; ls < ns; ls += LS) {
                    const int e = e0 + ls, slot = rhs * S + ls;
                    T rv[6], qv[6];
                    r_s.load(slot, rhs, Vh, e, rv);
                    q_s.load(slot, rhs, Vh, e, qv);
#pragma unroll
                    for (int k = 0; k < 6; ++k) {
                        rv[k] = fma(na, qv[k], rv[k]);
                        acc += (double)rv[k] * (double)rv[k];
                    }
                    // with the swap the new r goes where q was and the old r stays readable for the pending items
                    if (swap_rq) q_s.store(slot, rhs, Vh, e, rv); else r_s.store(slot, rhs, Vh, e, rv);
                }
            }
            cta_partials_stream<NT, R>(acc, red, part_rr + blockIdx.x, G);
        } else {
            // phase D (a4 after <r,r>, a7 latch, a6).  Nothing is pending here: the sync point before forced it.
            if (tid < 32 * R) {
                const int s = tid >> 5, i = tid & 31;
                Scalars<T> &c = sc[s];
                if (c.done == 0) {
                    const double rr_new = grid_total(part_rr + (size_t)s * G, G);
                    const double alpha = c.alpha;
                    const double beta = rr_new / c.rr;
                    const double rel = sqrt(rr_new / c.bb);
                    const int iter = c.iter + 1;
                    bool live = false;
                    double th = 1.0, z = 1.0;
                    __syncwarp();
                    if (i < nshift) {
                        if (c.active[i] == 2) c.active[i] = 0;            // frozen at the previous iteration
                        th = c.theta_new[i];
                        z = c.zeta[i] * th;
                        c.zeta[i] = z;
                        c.theta[i] = th;
                        if (c.active[i] != 0) {
                            live = true;
                            c.resid[i] = z * rel;
                            c.iters_shift[i] = iter;
                            if (freeze && i != base && z * rel <= 0.1 * c.stop) c.active[i] = 2;
                        }
                    }
                    const unsigned m = __ballot_sync(0xffffffffu, live && i != base);
                    if (live && i != base) {
                        const int j = __popc(m & ((1u << i) - 1u));
                        c.live[j] = i;
                        c.ca[j] = (T)(alpha * th);
                        c.cz[j] = (T)z;
                        c.cb[j] = (T)(beta * th * th);
                    }
                    if (i == base) { c.a_base = (T)(alpha * th); c.z_base = (T)z; c.b_base = (T)(beta * th * th); }
                    if (i == 0) {
                        c.nlive = __popc(m);
                        c.alpha_old = alpha;
                        c.beta_old = beta;
                        c.rr = rr_new;
                        c.iter = iter;
                        int done = 0;
                        if (rel <= c.stop) { c.converged = 1; done = 1; }
                        else if (iter >= maxiter) done = 1;
                        else if (!(rr_new == rr_new)) { c.breakdown = 1; done = 1; }
                        else if (fp32) {                                     // reading A9
                            if (rr_new < c.best_rr) { c.best_rr = rr_new; c.since_best = 0; }
                            else if (++c.since_best >= 50) { c.stagnated = 1; done = 1; }
                        }
                        c.done = done;
                    }
                }
            }
            __syncthreads();
            if (swap_rq) { const Slice<T> t = r_s; r_s = q_s; q_s = t; }       // the new r is where q was
            if (act2) {   // base shift first: its new p is what phase A of the next iteration gathers
                // (x_base += alpha p_base was already done while waiting at the sync point before: the base shift has
                // theta = 1, so its alpha_i is alpha itself and needs only the first reduction)
                const T zb = sc[rhs].z_base, bb_ = sc[rhs].b_base;
                for (int ls = l0; ls < ns; ls += LS) {
                    const int e = e0 + ls, slot = rhs * S + ls;
                    T rv[6], pv[6];
                    r_s.load(slot, rhs, Vh, e, rv);
                    p_s.load(slot, rhs, Vh, e, pv);
#pragma unroll
                    for (int k = 0; k < 6; ++k) pv[k] = fma(zb, rv[k], bb_ * pv[k]);
                    if (p_s.res) p_s.s.store(slot, pv);
                    store_vec(p_base, Vh, e, pv);
                }
                // the other live shifts of this iteration: deferred, worked off at the sync points that follow
                pn = sc[rhs].nlive; pj = 0; ppass = 0;
                pnpass = pn > 0 ? (ns + LS - 1) / LS : 0;
            }
            __syncthreads();                               // every thread has read sc[].done / coefficients
            if (tid == 0) {
                int n = 0;
                for (int s = 0; s < R; ++s) {
                    if (sc[s].done == 1) sc[s].done = 2;   // its last x/p update is queued
                    n += sc[s].done == 0;
                }
                n_running = n;
            }
        }
        STAG_TICK(2 * phase);

        // ---- sync point: arrive, then work off deferred items until everybody needed has arrived -----------
        // grid-wide after B and C (the two reductions): monotone counter `bar`.  After A and D a CTA needs w /
        // p_base only from the CTAs that own its neighbouring sites (nb_list; all CTAs if cg_nbflags = 0): their
        // epoch flags.  That is safe because two grid-wide barriers separate every write of w or p_base from the
        // previous iteration's reads of it.  Warp 0 polls (relaxed loads, one flag per lane), issues the acquire
        // fence once everybody needed has arrived (it also drops the SM's L1) and publishes the sync count in
        // shared memory; the other warps work off their own pending items — thread-private sites, so no CTA
        // barrier between items — until they see it or run out of items.  The closing CTA barrier hands warp 0's
        // acquire on to them.
        // Pending items MUST be finished (force) before phase D rewrites their coefficients, before phase C when
        // it overwrites the r they read (no swap), at the end of the solve — and at once if filling is off.
        // Arrivals are release operations (red.release / st.release: MEMBAR.ALL, no L1 invalidation) instead of
        // __threadfence() + a relaxed one (MEMBAR.SC + CCTL.IVALL).
        {
            const bool global = phase == 1 || phase == 2;
            __syncthreads();                               // this phase's writes are issued; n_running is visible
            const bool force = !a.fill || phase == 2 || (phase == 1 && !swap_rq) || (phase == 3 && n_running == 0);
            const unsigned int sync_id = gepoch + nepoch + 1u;
            unsigned int target;
            if (global) {
                target = ++gepoch * (unsigned)G;
                if (tid == 0) asm volatile("red.release.gpu.global.add.u32 [%0], %1;" :: "l"(bar), "r"(1u) : "memory");
            } else {
                target = ++nepoch;
                if (tid == 0) {
                    asm volatile("st.release.gpu.global.u32 [%0], %1;" :: "l"(a.flags + (size_t)blockIdx.x * 32), "r"(target) : "memory");
                }
            }
            const bool poll_warp = tid < 32;
            bool released = false;
            const int xbn = (phase == 2 && act2) ? (ns + LS - 1) / LS : 0;
            int xbpass = 0;
            while (!released || (force && ppass < pnpass) || xbpass < xbn) {
                unsigned int v = target;
                if (poll_warp && !released) {
                    if (global) {
                        if (tid == 0) asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(bar) : "memory");
                    } else {
                        for (int c = tid; c < nnb; c += 32) {      // wrapped unsigned min over this lane's flags
                            unsigned int f;
                            asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];"
                                         : "=r"(f) : "l"(a.flags + (size_t)nb_list[c] * 32) : "memory");
                            if ((int)(f - v) < 0) v = f;
                        }
                    }
                }
                if (ppass < pnpass) {                      // one item; the poll is in flight meanwhile
                    const Scalars<T> &c = sc[rhs];
                    const int ls = l0 + ppass * LS;
                    if (ls < ns) {
                        const int e = e0 + ls, slot = rhs * S + ls;
                        T rv[6], pv[B][6], xv[B][6];
                        r_s.load(slot, rhs, Vh, e, rv);
#pragma unroll
                        for (int u = 0; u < B; ++u)
                            if (B == 1 || pj + u < pn) {
                                const int i = c.live[pj + u];
                                const uint64_t pol = shift_policy(i);
                                load_vec_pol(p_r + (size_t)i * a.p_stride, Vh, e, pv[u], pol);
                                load_vec_pol(x_r + (size_t)i * a.x_stride, Vh, e, xv[u], pol);
                            }
#pragma unroll
                        for (int u = 0; u < B; ++u)
                            if (B == 1 || pj + u < pn) {
                                const int i = c.live[pj + u];
                                const uint64_t pol = shift_policy(i);
                                const T aj = c.ca[pj + u], zj = c.cz[pj + u], bj = c.cb[pj + u];
#pragma unroll
                                for (int k = 0; k < 6; ++k) {
                                    xv[u][k] = fma(aj, pv[u][k], xv[u][k]);
                                    pv[u][k] = fma(zj, rv[k], bj * pv[u][k]);
                                }
                                store_vec_pol(x_r + (size_t)i * a.x_stride, Vh, e, xv[u], pol);
                                store_vec_pol(p_r + (size_t)i * a.p_stride, Vh, e, pv[u], pol);
                            }
                    }
                    pj += B;
                    if (pj >= pn) { pj = 0; ++ppass; }
                }
                else if (xbpass < xbn) {                   // x_base += alpha p_base: needs alpha only (theta_base = 1), so it
                                                           // runs here, in the wait for <r,r>, instead of in phase D
                    const int ls = l0 + xbpass * LS;
                    if (ls < ns) {
                        const int e = e0 + ls, slot = rhs * S + ls;
                        const uint64_t pol = shift_policy(base);
                        const T ab = (T)sc[rhs].alpha;
                        T pv[6], xv[6];
                        load_vec_pol(x_base, Vh, e, xv, pol);
                        p_s.load(slot, rhs, Vh, e, pv);
#pragma unroll
                        for (int k = 0; k < 6; ++k) xv[k] = fma(ab, pv[k], xv[k]);
                        store_vec_pol(x_base, Vh, e, xv, pol);
                    }
                    ++xbpass;
                }
                if (poll_warp) {
                    if (!released && __all_sync(0xffffffffu, (int)(v - target) >= 0)) {
                        if (tid == 0) {
                            asm volatile("fence.acquire.gpu;" ::: "memory");
                            *reinterpret_cast<volatile unsigned int *>(&sync_seen) = sync_id;
                        }
                        released = true;
                    }
                } else {
                    // the other warps: released once warp 0 has seen the arrivals, or when out of items (the
                    // closing CTA barrier then waits in hardware instead of spinning)
                    released = (ppass >= pnpass && xbpass >= xbn) || *reinterpret_cast<volatile unsigned int *>(&sync_seen) == sync_id;
                }
            }
            __syncthreads();
        }
        STAG_TICK(2 * phase + 1);
        phase = (phase + 1) & 3;
    }

    STAG_T_REPORT(R, sc[0].iter)

    // ---- a7: y = residue0 b + sum_i residues_i x_i (own sites only: no barrier needed) ---------------
    if (a.y && present) {
        char *y_r = a.y + (size_t)rhs * a.x_stride;
        const T r0 = (T)st->residue0;
        for (int ls = l0; ls < ns; ls += LS) {
            const int e = e0 + ls;
            T bv[6], acc[6];
            load_vec<true>(b_r, Vh, e, bv);
#pragma unroll
            for (int k = 0; k < 6; ++k) acc[k] = r0 * bv[k];
            for (int i = 0; i < nshift; ++i) {
                const T ri = (T)st->residues[i];
                T xv[6];
                load_vec_pol(x_r + (size_t)i * a.x_stride, Vh, e, xv, policy_evict_first());
#pragma unroll
                for (int k = 0; k < 6; ++k) acc[k] = fma(ri, xv[k], acc[k]);
            }
            store_vec(y_r, Vh, e, acc);
        }
    }

    // ---- read-back state (every CTA holds the same scalars; CTA 0 writes them) -------------------------
    if (blockIdx.x == 0 && tid < 32 * R && (tid >> 5) < a.nrhs) {
        const int s = tid >> 5, i = tid & 31;
        CgState *o = reinterpret_cast<CgState *>(reinterpret_cast<char *>(a.state) + (size_t)s * a.state_stride);
        const Scalars<T> &c = sc[s];
        if (i < nshift) {
            o->zeta[i] = c.zeta[i];
            o->theta[i] = c.theta[i];
            o->resid_shift[i] = c.resid[i];
            o->iters_shift[i] = c.iters_shift[i];
            o->active[i] = c.active[i];
        }
        if (i == 0) {
            o->bb = c.bb; o->rr = c.rr; o->pq = c.pq; o->alpha = c.alpha;
            o->iter = c.iter; o->converged = c.converged; o->breakdown = c.breakdown;
            o->stagnated = c.stagnated; o->done = 2;
        }
    }
}

// ---- host side ---------------------------------------------------------------------------------------
static constexpr size_t kMaxDynSmem = 200 * 1024;     // of 227 KB; the rest: static scalars + L1

// sites per CTA for a grid of `grid` CTAs (multiple of 32: every CTA's slice starts on a 512-byte line);
// the slice layout of the mixed-precision kernel, and the slot count of a resident slice here (the largest CTA)
inline int sites_per_cta(int Vh, int grid) {
    const int s = (Vh + grid - 1) / grid;
    return (s + 31) & ~31;
}
inline int persist_grid(const stag_ctx *ctx) {
    const int tiles = (ctx->g.Vh + 31) / 32;
    return ctx->num_sms < tiles ? ctx->num_sms : tiles;
}
inline int persist_slots(const stag_ctx *ctx) {       // sites of the largest CTA
    const int tiles = (ctx->g.Vh + 31) / 32, grid = persist_grid(ctx);
    return 32 * ((tiles + grid - 1) / grid);
}

// The shifts whose x_i, p_i the kernel marks evict_last: lightest first (they stay live longest), as many as
// fit in `cg_l2_keep_mb` MB for all the sources of the launch.
inline unsigned persist_keep_mask(const stag_ctx *ctx, int prec, int nrhs, int nshift, const double *shifts) {
    const size_t per_shift = (size_t)2 * nrhs * ctx->g.Vh * vec_bytes_per_site(prec);
    long long budget = (long long)ctx->opt.cg_l2_keep_mb << 20;
    unsigned mask = 0;
    for (;;) {
        int best = -1;
        for (int i = 0; i < nshift; ++i)
            if (!((mask >> i) & 1u) && (best < 0 || shifts[i] < shifts[best])) best = i;
        if (best < 0 || (long long)per_shift > budget) break;
        budget -= (long long)per_shift;
        mask |= 1u << best;
    }
    return mask;
}

template <typename T, int RECON, int NT, int R, bool SPLIT = false>
int launch_persistent(const stag_ctx *ctx, const PersistArgs &args, cudaStream_t st) {
    const Geom &g = ctx->g;
    const int grid = persist_grid(ctx);
    if (grid > kMaxPersistGrid) return STAG_ERR_UNSUPPORTED;
    PersistArgs a = args;
    a.S = persist_slots(ctx);
    a.fill = ctx->opt.cg_fill != 0;
    a.nbflags = ctx->opt.cg_nbflags != 0;

    // residency: as many of r, q, p (in that order of bytes saved) as fit
    const size_t slice = (size_t)a.S * R * 6 * sizeof(T);
    // cg_resident_slices (test / tuning knob): cap on how many of r, q, p stay in shared memory (default 3)
    int fit = (int)(kMaxDynSmem / slice);
    if (fit > ctx->opt.cg_resident_slices) fit = ctx->opt.cg_resident_slices;
    a.res_r = fit >= 1; a.res_q = fit >= 2; a.res_p = fit >= 3;
    const size_t smem = slice * (size_t)(a.res_r + a.res_q + a.res_p);
    auto kern = cg_persistent_kernel<T, RECON, NT, R, SPLIT>;
    STAG_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int per_sm = 0;
    STAG_CUDA_OK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, NT, smem));
    if (per_sm < 1) return STAG_ERR_UNSUPPORTED;
    STAG_CUDA_OK(cudaMemsetAsync(a.flags, 0, (size_t)grid * 128, st));
    Geom gg = g;
    void *params[] = {(void *)&gg, (void *)&a};
    log_kernel(ctx, (const void *)kern);
    STAG_CUDA_OK(cudaLaunchCooperativeKernel((const void *)kern, dim3(grid), dim3(NT), params, smem, st));
    return STAG_OK;
}

// one explicit-instantiation translation unit per R (parallel compilation)
template <int R>
int cg_persistent_launch_r(const stag_ctx *ctx, int prec, int recon, const PersistArgs &a, cudaStream_t st);

// N3: split-double links (stag_cg_persist_split.cu); R = 1, 2 or 4 sources compiled in
int cg_persistent_launch_split(const stag_ctx *ctx, int recon, int R, const PersistArgs &a, cudaStream_t st);

#define STAG_DEFINE_PERSIST_R(RR)                                                                       \
    template <>                                                                                         \
    int cg_persistent_launch_r<RR>(const stag_ctx *ctx, int prec, int recon, const PersistArgs &a,      \
                                   cudaStream_t st) {                                                   \
        /* 1024 threads x 64 registers, 512 x 128 or (fp64) 256 x 255 per SM.  Measured at 32^3 x 8     \
           (profiles/README.md): fp64 is fastest with 512 x 128 (deeper per-thread load queue; fp64     \
           12-real needs ~100 registers anyway), fp32 with 1024 x 64, for R = 1 and R = 4 alike.        \
           cg_persistent_threads = 0 picks that. */                                                     \
        int nt = ctx->opt.cg_persistent_threads;                                                        \
        if (nt == 0) nt = prec == STAG_F64 ? 512 : 1024;                                                \
        if (prec == STAG_F64) {                                                                         \
            if (recon == 12)                                                                            \
                return nt == 256 ? launch_persistent<double, 12, 256, RR>(ctx, a, st)                   \
                                 : launch_persistent<double, 12, 512, RR>(ctx, a, st);                  \
            return nt == 1024  ? launch_persistent<double, 18, 1024, RR>(ctx, a, st)                    \
                   : nt == 256 ? launch_persistent<double, 18, 256, RR>(ctx, a, st)                     \
                               : launch_persistent<double, 18, 512, RR>(ctx, a, st);                    \
        }                                                                                               \
        if (recon == 18)                                                                                \
            return nt == 1024 ? launch_persistent<float, 18, 1024, RR>(ctx, a, st)                      \
                              : launch_persistent<float, 18, 512, RR>(ctx, a, st);                      \
        return nt == 1024 ? launch_persistent<float, 12, 1024, RR>(ctx, a, st)                          \
                          : launch_persistent<float, 12, 512, RR>(ctx, a, st);                          \
    }

}  // namespace stag
