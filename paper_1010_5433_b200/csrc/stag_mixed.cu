// stag_mixed.cu — N2: fp32 multi-shift CG + per-shift fp64 defect-correction polish.
//   PAPER.md:93      fp32 for the MD-force inversions, fp64 for the first and last (Metropolis) ones
//   PAPER.md:127     fp32 alone stalls at a true residual of 1e-2 .. 1e-3
//   PAPER.md:129     a SHIFTED solver starts from zero and cannot be restarted — but each single
//                    system (A + sigma_i) x_i = b can: the polish is ordinary CG with a non-zero start.
// The correction solves are the N1 persistent kernel with one shift per source (stag_cg_persist.cuh):
// up to STAG_MAX_RHS shifts share every read of the links.
#include <cmath>
#include <cstring>

#include "stag_cg_mixed_persist.cuh"

namespace stag {

// ---- device vector format conversion -------------------------------------------------------------------
// fp64: 3 planes of double2 [c][e];  fp32: float4 plane (c0,c1) + float2 plane (c2)
template <bool TO_F32>
__global__ void __launch_bounds__(256)
vector_convert_kernel(const int Vh, const char *__restrict__ src, char *__restrict__ dst, const size_t src_stride,
                      const size_t dst_stride) {
    const int e = blockIdx.x * 256 + threadIdx.x;
    if (e >= Vh) return;
    const char *s = src + (size_t)blockIdx.y * src_stride;
    char *d = dst + (size_t)blockIdx.y * dst_stride;
    if (TO_F32) {
        const double2 *p = reinterpret_cast<const double2 *>(s) + e;
        const double2 a = p[0], b = p[Vh], c = p[2 * (size_t)Vh];
        reinterpret_cast<float4 *>(d)[e] = make_float4((float)a.x, (float)a.y, (float)b.x, (float)b.y);
        reinterpret_cast<float2 *>(d + (size_t)Vh * 16)[e] = make_float2((float)c.x, (float)c.y);
    } else {
        const float4 a = reinterpret_cast<const float4 *>(s)[e];
        const float2 c = reinterpret_cast<const float2 *>(s + (size_t)Vh * 16)[e];
        double2 *p = reinterpret_cast<double2 *>(d) + e;
        p[0] = make_double2(a.x, a.y);
        p[Vh] = make_double2(a.z, a.w);
        p[2 * (size_t)Vh] = make_double2(c.x, c.y);
    }
}

// ---- defect: r = b - c0 x + t  (t = D_eo D_oe x, so r = b - (A + sigma) x) and ||r||^2, fp64 -------------
// x, t, r nullable: (x = t = r = null) gives ||b||^2.
template <int BLOCK>
__global__ void __launch_bounds__(BLOCK)
defect_kernel(const long nchunk, const double2 *__restrict__ b, const double2 *__restrict__ x,
              const double2 *__restrict__ t, const double c0, double2 *__restrict__ r,
              double *__restrict__ partials, unsigned int *__restrict__ ticket, double *__restrict__ out) {
    __shared__ double red[BLOCK / 32 + 1];
    double acc = 0.0;
    for (long k = (long)blockIdx.x * BLOCK + threadIdx.x; k < nchunk; k += (long)gridDim.x * BLOCK) {
        double2 v = b[k];
        if (x) {
            const double2 xv = x[k], tv = t[k];
            v.x = (v.x - c0 * xv.x) + tv.x;
            v.y = (v.y - c0 * xv.y) + tv.y;
        }
        if (r) r[k] = v;
        acc += v.x * v.x + v.y * v.y;
    }
    double total;
    if (grid_sum_last_cta<BLOCK>(acc, partials, ticket, red, total) && threadIdx.x == 0) *out = total;
}

// x += e
__global__ void __launch_bounds__(256)
add_kernel(const long nchunk, double2 *__restrict__ x, const double2 *__restrict__ e) {
    for (long k = (long)blockIdx.x * 256 + threadIdx.x; k < nchunk; k += (long)gridDim.x * 256) {
        double2 v = x[k];
        const double2 w = e[k];
        v.x += w.x; v.y += w.y;
        x[k] = v;
    }
}

struct PolishLayout {
    size_t scal, partials, w, r, e, cg, total;   // scal: 8 doubles + ticket; w, r, e: STAG_MAX_RHS vectors each
    size_t vec;
    int grid;
};

static PolishLayout polish_layout(const stag_ctx *ctx) {
    PolishLayout l;
    l.vec = align256((size_t)ctx->g.Vh * vec_bytes_per_site(STAG_F64));
    l.grid = ctx->num_sms * 8;
    size_t off = 0;
    l.scal = off;     off += 256;
    l.partials = off; off += align256(sizeof(double) * (size_t)l.grid);
    l.w = off;        off += l.vec * STAG_MAX_RHS;
    l.r = off;        off += l.vec * STAG_MAX_RHS;
    l.e = off;        off += l.vec * STAG_MAX_RHS;
    l.cg = off;       off += align256(stag_cg_block_workspace_bytes(ctx, STAG_F64, 1, STAG_MAX_RHS));
    l.total = off;
    return l;
}

// D on n contiguous fp64 vectors: the N1 block kernel (native fp64 or split-double links: one read of the links)
static int dslash_n(const stag_ctx *ctx, const void *packed, int prec, int recon, int par, int n, const char *in,
                    char *out, size_t stride, cudaStream_t st, int *launches) {
    (void)stride;
    ++*launches;
    return stag_dslash_block(ctx, packed, prec, recon, par, n, in, out, st);
}

static int polish(const stag_ctx *ctx, Slot &slot, const void *packed, int prec, int recon, const char *b, double mass,
                  int nshift, const double *shifts, double stop, int maxiter, char *x, char *ws,
                  stag_polish_info *info, cudaStream_t st) {
    const PolishLayout lay = polish_layout(ctx);
    const Geom &g = ctx->g;
    const size_t vbytes = (size_t)g.Vh * vec_bytes_per_site(STAG_F64);    // stride of x_i (ABI) and of w, r, e
    const long nchunk = (long)g.Vh * 3;
    const int grid = (int)((nchunk + 255) / 256 < lay.grid ? (nchunk + 255) / 256 : lay.grid);
    double *scal = reinterpret_cast<double *>(ws + lay.scal);
    unsigned int *ticket = reinterpret_cast<unsigned int *>(ws + lay.scal + 128);
    double *partials = reinterpret_cast<double *>(ws + lay.partials);
    volatile double *hn = reinterpret_cast<volatile double *>(reinterpret_cast<char *>(slot.pinned_flags) + 128);
    const int group = STAG_MAX_RHS;    // the defects of a split-double group are one Dslash launch per shift (dslash_n)
    stag_polish_info pi;
    std::memset(&pi, 0, sizeof(pi));
    int launches = 0;

    STAG_CUDA_OK(cudaMemsetAsync(ws + lay.scal, 0, 256, st));
    STAG_LAUNCH_K(ctx, defect_kernel<256>, grid, 256, 0, st, nchunk, reinterpret_cast<const double2 *>(b),
                  static_cast<const double2 *>(nullptr), static_cast<const double2 *>(nullptr), 0.0,
                  static_cast<double2 *>(nullptr), partials, ticket, scal + 7);
    ++launches;
    STAG_CUDA_OK(cudaMemcpyAsync((void *)hn, scal, 8 * sizeof(double), cudaMemcpyDeviceToHost, st));
    STAG_CUDA_OK(cudaStreamSynchronize(st));
    const double bb = hn[7];
    if (!(bb >= 0.0)) return STAG_ERR_BREAKDOWN;
    int worst = STAG_OK;

    // true residuals of n shifts starting at i0: r_s = b - (A + sigma_s) x_s -> ws.r, norms -> rel[]
    auto defects = [&](int i0, int n, double *rel) -> int {
        const char *xg = x + (size_t)i0 * vbytes;
        int rc = dslash_n(ctx, packed, prec, recon, 1, n, xg, ws + lay.w, vbytes, st, &launches);
        if (rc) return rc;
        rc = dslash_n(ctx, packed, prec, recon, 0, n, ws + lay.w, ws + lay.e, vbytes, st, &launches);   // e as scratch
        if (rc) return rc;
        for (int s = 0; s < n; ++s) {
            STAG_LAUNCH_K(ctx, defect_kernel<256>, grid, 256, 0, st,
                nchunk, reinterpret_cast<const double2 *>(b), reinterpret_cast<const double2 *>(xg + s * vbytes),
                reinterpret_cast<const double2 *>(ws + lay.e + s * vbytes), mass * mass + shifts[i0 + s],
                reinterpret_cast<double2 *>(ws + lay.r + s * vbytes), partials, ticket, scal + s);
            ++launches;
        }
        STAG_CUDA_OK(cudaGetLastError());
        STAG_CUDA_OK(cudaMemcpyAsync((void *)hn, scal, 8 * sizeof(double), cudaMemcpyDeviceToHost, st));
        STAG_CUDA_OK(cudaStreamSynchronize(st));
        for (int s = 0; s < n; ++s) rel[s] = bb > 0.0 ? std::sqrt(hn[s] / bb) : 0.0;
        return STAG_OK;
    };

    for (int i0 = 0; i0 < nshift; i0 += group) {
        const int n = nshift - i0 < group ? nshift - i0 : group;
        double rel[STAG_MAX_RHS];
        int rc = defects(i0, n, rel);
        if (rc) return rc;
        for (int s = 0; s < n; ++s) pi.resid_before[i0 + s] = pi.resid_after[i0 + s] = rel[s];
        for (int pass = 1; pass <= 3; ++pass) {
            bool any = false;
            double sstop[STAG_MAX_RHS], sigma[STAG_MAX_RHS];
            for (int s = 0; s < n; ++s) {
                if (!(rel[s] == rel[s])) return STAG_ERR_BREAKDOWN;
                any = any || rel[s] > stop;
                // correction to ||r_new|| <= stop ||b||, relative to its own source r_s; already-good shifts: 0 iterations
                sstop[s] = rel[s] > stop ? stop / rel[s] : 2.0;
                sigma[s] = shifts[i0 + s];
            }
            if (!any) break;
            if (pi.passes < pass) pi.passes = pass;
            stag_cg_info ci[STAG_MAX_RHS];
            rc = block_solve(ctx, slot, packed, prec, recon, n, ws + lay.r, mass, 1, sigma, sigma, sstop, nullptr, 0.0,
                             stop, maxiter, ws + lay.e, nullptr, ws + lay.cg, ci, st);
            ++launches;
            if (rc == STAG_ERR_BREAKDOWN) worst = rc;
            else if (rc != STAG_OK && rc != STAG_ERR_NOTCONV) return rc;
            for (int s = 0; s < n; ++s) {
                pi.iters[i0 + s] += ci[s].iters;
                if (ci[s].iters > 0) {
                    add_kernel<<<grid, 256, 0, st>>>(nchunk, reinterpret_cast<double2 *>(x + (size_t)(i0 + s) * vbytes),
                                                     reinterpret_cast<const double2 *>(ws + lay.e + s * vbytes));
                    ++launches;
                }
            }
            STAG_CUDA_OK(cudaGetLastError());
            rc = defects(i0, n, rel);
            if (rc) return rc;
            for (int s = 0; s < n; ++s) pi.resid_after[i0 + s] = rel[s];
            if (worst == STAG_ERR_BREAKDOWN) break;
        }
        for (int s = 0; s < n; ++s)
            if (rel[s] > stop && worst == STAG_OK) worst = STAG_ERR_NOTCONV;
    }
    pi.kernel_launches = launches;
    if (info) *info = pi;
    return worst;
}

// y = residue0 b + sum_i residues_i x_i, fp64
__global__ void __launch_bounds__(256)
partial_fraction64_kernel(const long nchunk, const double2 *__restrict__ b, const double2 *__restrict__ x,
                          const size_t x_stride_chunks, const int nshift, const double residue0,
                          const double *__restrict__ residues, double2 *__restrict__ y) {
    for (long k = (long)blockIdx.x * 256 + threadIdx.x; k < nchunk; k += (long)gridDim.x * 256) {
        const double2 bv = b[k];
        double2 acc = make_double2(residue0 * bv.x, residue0 * bv.y);
        for (int i = 0; i < nshift; ++i) {
            const double2 xv = x[(size_t)i * x_stride_chunks + k];
            acc.x = fma(residues[i], xv.x, acc.x);
            acc.y = fma(residues[i], xv.y, acc.y);
        }
        y[k] = acc;
    }
}

struct MixedLayout { size_t res, b32, x32, cg32, w64, polish, total; };   // cg32 also holds the fp64 CG workspace of route 3

static MixedLayout mixed_layout(const stag_ctx *ctx, int nshift) {
    MixedLayout l;
    const size_t v32 = (size_t)ctx->g.Vh * vec_bytes_per_site(STAG_F32);
    size_t off = 0;
    l.res = off;    off += 256;                                   // residues on the device
    l.b32 = off;    off += align256(v32);
    l.x32 = off;    off += align256(v32 * (size_t)nshift);
    l.cg32 = off;   off += align256(cg_workspace_layout(ctx, STAG_F64, nshift, nullptr));   // >= the fp32 layout
    l.w64 = off;    off += align256((size_t)ctx->g.Vh * vec_bytes_per_site(STAG_F64));
    l.polish = off; off += polish_layout(ctx).total;
    l.total = off;
    return l;
}

// The inner stage as ONE persistent kernel with residual replacement (stag_cg_mixed_persist.cuh): fp32 matrices
// and directions, fp64 solutions, true fp64 residual of the base system at every replacement.  Returns
// STAG_ERR_UNSUPPORTED when that kernel does not apply (the caller then runs the plain fp32 stage).
static int mixed_persistent(const stag_ctx *ctx, Slot &slot, const void *packed_hi, int prec_hi, const void *packed_lo, int recon,
                            const void *b64, double mass, int nshift, const double *shifts, double stop,
                            int maxiter, void *x64, char *ws, const MixedLayout &lay, stag_cg_info *info,
                            int *replacements, cudaStream_t st) {
    if (!cg_persistent_fits(ctx, STAG_F32)) return STAG_ERR_UNSUPPORTED;
    CgLayout cl;
    cg_workspace_layout(ctx, STAG_F32, nshift, &cl);
    char *cw = ws + lay.cg32;
    int base = 0;
    for (int i = 1; i < nshift; ++i)
        if (shifts[i] < shifts[base]) base = i;
    CgState *h = static_cast<CgState *>(slot.pinned_info);
    std::memset(h, 0, sizeof(*h));
    h->alpha_old = 1.0;
    h->c0 = mass * mass + shifts[base];
    h->stop = stop;
    for (int i = 0; i < nshift; ++i) {
        h->delta[i] = shifts[i] - shifts[base];
        h->zeta[i] = 1.0; h->theta[i] = 1.0; h->active[i] = 1; h->resid_shift[i] = 1.0;
    }
    h->nshift = nshift; h->base = base; h->maxiter = maxiter; h->freeze = ctx->opt.cg_freeze; h->fp32 = 1;
    STAG_CUDA_OK(cudaMemcpyAsync(cw + cl.state, h, sizeof(CgState), cudaMemcpyHostToDevice, st));
    MixedArgs a;
    std::memset(&a, 0, sizeof(a));
    a.W_lo = static_cast<const char *>(packed_lo);
    a.W_hi = static_cast<const char *>(packed_hi);
    a.b64 = static_cast<const char *>(b64);
    a.w32 = cw + cl.w; a.w64 = ws + lay.w64;
    a.r_g = cw + cl.r; a.q_g = cw + cl.q;
    a.p = cw + cl.p; a.p_stride = cl.vec_stride;
    a.x = static_cast<char *>(x64); a.x_stride = (size_t)ctx->g.Vh * vec_bytes_per_site(STAG_F64);
    a.state = reinterpret_cast<CgState *>(cw + cl.state);
    a.partials = reinterpret_cast<double *>(cw + cl.partials);
    a.ru_delta = 1.0 / (double)(ctx->opt.cg_mixed_delta_inv > 0 ? ctx->opt.cg_mixed_delta_inv : 10);
    const int nt = ctx->opt.cg_persistent_threads;
    int rc;
    if (prec_hi == STAG_F64_SPLIT)
        rc = recon == 18 ? (nt == 512 ? launch_mixed<18, 512, true>(ctx, a, st) : launch_mixed<18, 1024, true>(ctx, a, st))
                         : (nt == 512 ? launch_mixed<12, 512, true>(ctx, a, st) : launch_mixed<12, 1024, true>(ctx, a, st));
    else
        rc = recon == 18 ? (nt == 512 ? launch_mixed<18, 512, false>(ctx, a, st) : launch_mixed<18, 1024, false>(ctx, a, st))
                         : (nt == 512 ? launch_mixed<12, 512, false>(ctx, a, st) : launch_mixed<12, 1024, false>(ctx, a, st));
    if (rc) { cudaGetLastError(); return rc; }
    STAG_CUDA_OK(cudaMemcpyAsync(h, cw + cl.state, sizeof(CgState), cudaMemcpyDeviceToHost, st));
    STAG_CUDA_OK(cudaStreamSynchronize(st));
    std::memset(info, 0, sizeof(*info));
    info->iters = h->iter; info->converged = h->converged; info->breakdown = h->breakdown;
    info->stagnated = h->stagnated;
    info->bnorm2 = h->bb; info->rnorm2 = h->rr; info->kernel_launches = 1;
    for (int i = 0; i < nshift; ++i) {
        info->resid_iter[i] = h->bb > 0.0 ? h->resid_shift[i] : 0.0;
        info->iters_shift[i] = h->iters_shift[i];
    }
    *replacements = h->replacements;
    if (h->breakdown) return STAG_ERR_BREAKDOWN;
    return h->converged ? STAG_OK : STAG_ERR_NOTCONV;
}

}  // namespace stag

using namespace stag;

extern "C" int stag_vector_convert(const stag_ctx *ctx, const void *src, int src_prec, void *dst, int dst_prec,
                                   int nvec, void *stream) {
    if (!ctx || !src || !dst || !valid_prec(src_prec) || !valid_prec(dst_prec) || nvec < 1) return STAG_ERR_BADARG;
    const int sp = vec_prec(src_prec), dp = vec_prec(dst_prec);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const Geom &g = ctx->g;
    const size_t ss = (size_t)g.Vh * vec_bytes_per_site(sp), ds = (size_t)g.Vh * vec_bytes_per_site(dp);
    if (sp == dp) {
        if (src != dst) STAG_CUDA_OK(cudaMemcpyAsync(dst, src, ss * nvec, cudaMemcpyDeviceToDevice, st));
        return STAG_OK;
    }
    const dim3 grid((g.Vh + 255) / 256, nvec);
    if (dp == STAG_F32)
        vector_convert_kernel<true><<<grid, 256, 0, st>>>(g.Vh, static_cast<const char *>(src), static_cast<char *>(dst), ss, ds);
    else
        vector_convert_kernel<false><<<grid, 256, 0, st>>>(g.Vh, static_cast<const char *>(src), static_cast<char *>(dst), ss, ds);
    STAG_CUDA_OK(cudaGetLastError());
    return STAG_OK;
}

extern "C" size_t stag_cg_polish_workspace_bytes(const stag_ctx *ctx) {
    return ctx ? polish_layout(ctx).total : 0;
}

static int check_solve_args(const stag_ctx *ctx, const void *packed, int recon, const void *b, double mass,
                            int nshift, const double *shifts, double stop, int maxiter, const void *x,
                            const void *ws) {
    if (!ctx || !packed || !b || !shifts || !x || !ws) return STAG_ERR_BADARG;
    if (!valid_recon(recon)) return STAG_ERR_BADARG;
    if (nshift < 1 || nshift > STAG_MAX_SHIFTS || !(stop > 0.0) || maxiter < 0) return STAG_ERR_BADARG;
    for (int i = 0; i < nshift; ++i)
        if (!(shifts[i] >= 0.0) || !(mass * mass + shifts[i] > 0.0)) return STAG_ERR_BADARG;
    if (((uintptr_t)ws & 255) != 0) return STAG_ERR_BADARG;
    return STAG_OK;
}

extern "C" int stag_cg_polish(const stag_ctx *ctx, const void *packed, int prec, int recon, const void *b_even,
                              double mass, int nshift, const double *host_shifts, double stop, int maxiter,
                              void *x_even, void *workspace, stag_polish_info *info, void *stream) {
    const int bad = check_solve_args(ctx, packed, recon, b_even, mass, nshift, host_shifts, stop, maxiter, x_even, workspace);
    if (bad) return bad;
    if (prec != STAG_F64 && prec != STAG_F64_SPLIT) return STAG_ERR_BADARG;
    SlotLease lease(ctx);
    return polish(ctx, lease.slot(), packed, prec, recon, static_cast<const char *>(b_even), mass, nshift, host_shifts, stop,
                  maxiter, static_cast<char *>(x_even), static_cast<char *>(workspace), info,
                  static_cast<cudaStream_t>(stream));
}

extern "C" size_t stag_mshift_cg_mixed_workspace_bytes(const stag_ctx *ctx, int nshift) {
    if (!ctx || nshift < 1 || nshift > STAG_MAX_SHIFTS) return 0;
    return mixed_layout(ctx, nshift).total;
}

extern "C" int stag_mshift_cg_mixed(const stag_ctx *ctx, const void *packed_hi, int prec_hi, int recon_hi,
                                    const void *packed_lo, int recon_lo, const void *b_even, double mass,
                                    int nshift, const double *host_shifts, const double *host_residues,
                                    double residue0, double stop, double inner_stop, int maxiter, void *x_even,
                                    void *y_even, void *workspace, stag_mixed_info *info, void *stream) {
    const int bad = check_solve_args(ctx, packed_hi, recon_hi, b_even, mass, nshift, host_shifts, stop, maxiter, x_even, workspace);
    if (bad) return bad;
    if (!packed_lo || !valid_recon(recon_lo)) return STAG_ERR_BADARG;
    if (prec_hi != STAG_F64 && prec_hi != STAG_F64_SPLIT) return STAG_ERR_BADARG;
    if (y_even && !host_residues) return STAG_ERR_BADARG;
    if (!(inner_stop > 0.0)) inner_stop = 1e-5;
    if (inner_stop < stop) inner_stop = stop;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    char *ws = static_cast<char *>(workspace);
    const MixedLayout lay = mixed_layout(ctx, nshift);
    stag_mixed_info mi;
    std::memset(&mi, 0, sizeof(mi));
    SlotLease lease(ctx);
    Slot &slot = lease.slot();

    // Route (option "cg_mixed_fp64_from", default 3).  Measured at 32^3 x 8, stop 1e-10: one shift —
    // residual replacement wins (0.105 against 0.17 s); two — fp32 + polish (0.163 against 0.178 s); from three or
    // four shifts on the polish, which gives up the shared Krylov space (sum_i instead of max_i iterations), costs
    // more than fp32 saved: the fp64 multi-shift solve is the fastest way to the fp64 stop, which is the paper's own
    // conclusion for the Metropolis solves.  So from that many shifts on the call IS the fp64
    // multi-shift solve on packed_hi, followed by the same true-residual check (and, if ever needed, polish).
    const int fp64_from = ctx->opt.cg_mixed_fp64_from;
    if (fp64_from > 0 && nshift >= fp64_from && stop < 1e-6) {
        mi.route = 3;
        const int crc = mshift_cg_impl(ctx, slot, packed_hi, prec_hi, recon_hi, b_even, mass, nshift, host_shifts, nullptr, 0.0,
                                       stop, maxiter, x_even, nullptr, ws + lay.cg32, &mi.inner, st);
        if (crc != STAG_OK && crc != STAG_ERR_NOTCONV) {
            if (info) *info = mi;
            return crc;
        }
    } else {
    // inner stage, preferred form: one persistent kernel with residual replacement (fp32 matrices, fp64 x_i)
    int rc = STAG_ERR_UNSUPPORTED;
    // cg_mixed_reliable: 0 never | 1 (default) when it pays — a single shift, where nothing is left to polish
    // (32^3 x 8: 0.107 s against 0.169 s in fp64; with more shifts the shifted systems stop at the fp32
    // rounding of the matrices times ||x_i||/||b|| and the polish costs as much as after the plain fp32 run) | 2 always
    const bool want_ru = ctx->opt.cg_mixed_reliable == 2 || (ctx->opt.cg_mixed_reliable == 1 && nshift == 1);
    if (want_ru && ctx->opt.cg_persistent && recon_hi == recon_lo)
        rc = mixed_persistent(ctx, slot, packed_hi, prec_hi, packed_lo, recon_lo, b_even, mass, nshift, host_shifts, stop, maxiter,
                              x_even, ws, lay, &mi.inner, &mi.reliable_updates, st);
    if (rc != STAG_ERR_UNSUPPORTED) {
        mi.route = 1;
        if (rc != STAG_OK && rc != STAG_ERR_NOTCONV) {
            if (info) *info = mi;
            return rc;
        }
    } else {
    mi.route = 2;
    // plain fp32 stage: b -> fp32, multi-shift CG from zero, x -> fp64
    rc = stag_vector_convert(ctx, b_even, STAG_F64, ws + lay.b32, STAG_F32, 1, st);
    if (rc) return rc;
    rc = mshift_cg_impl(ctx, slot, packed_lo, STAG_F32, recon_lo, ws + lay.b32, mass, nshift, host_shifts, nullptr, 0.0,
                        inner_stop, maxiter, ws + lay.x32, nullptr, ws + lay.cg32, &mi.inner, st);
    if (rc != STAG_OK && rc != STAG_ERR_NOTCONV) {            // breakdown or a real error: nothing to polish
        if (info) *info = mi;
        return rc;
    }
    rc = stag_vector_convert(ctx, ws + lay.x32, STAG_F32, x_even, STAG_F64, nshift, st);
    if (rc) return rc;
    }
    }

    // fp64 stage: per-shift defect-correction polish
    const int prc = polish(ctx, slot, packed_hi, prec_hi, recon_hi, static_cast<const char *>(b_even), mass, nshift,
                           host_shifts, stop, maxiter, static_cast<char *>(x_even), ws + lay.polish, &mi.polish, st);
    if (prc != STAG_OK && prc != STAG_ERR_NOTCONV && prc != STAG_ERR_BREAKDOWN) return prc;

    if (y_even) {
        const Geom &g = ctx->g;
        const long nchunk = (long)g.Vh * 3;
        double *dres = reinterpret_cast<double *>(ws + lay.res);
        STAG_CUDA_OK(cudaMemcpyAsync(dres, host_residues, sizeof(double) * nshift, cudaMemcpyHostToDevice, st));
        const int grid = (int)((nchunk + 255) / 256 < (long)ctx->num_sms * 8 ? (nchunk + 255) / 256 : (long)ctx->num_sms * 8);
        partial_fraction64_kernel<<<grid, 256, 0, st>>>(nchunk, static_cast<const double2 *>(b_even),
                                                        static_cast<const double2 *>(x_even), (size_t)g.Vh * 3, nshift,
                                                        residue0, dres, static_cast<double2 *>(y_even));
        STAG_CUDA_OK(cudaGetLastError());
        STAG_CUDA_OK(cudaStreamSynchronize(st));
        mi.polish.kernel_launches += 1;
    }
    if (info) *info = mi;
    return prc;
}
