// stag_force.cu — N4: the first consumer of the multi-shift solutions, the fermion
// force of the rational pseudo-fermion action (PAPER.md:25 "fermion force", :93 "the inversions needed
// in the fermion force calculation"), one thread per link as in the paper's gauge update.
//
//   X_i = x_i on even sites, w_i = D_oe x_i on odd sites;  eps(z) = +1 even / -1 odd
//   M_mu(z) = eps(z) sum_i residues_i X_i(z+mu) X_i(z)^dag
//   F_mu(z) = 2 TA( W_mu(z) M_mu(z) ),  W_mu(z) = f U_mu(z) = the packed FORWARD hopping matrix of z
//   TA(G) = (G - G^dag)/2 - tr(G - G^dag)/6
// so that d/dt S[U_mu(z) -> exp(itT) U_mu(z)] = tr(i T F_mu(z))  (derivation: DESIGN.md "N4").
// The factor f = 1/2 eta s of the hop is already folded into the packed matrix, so the kernel reads
// exactly the buffers the solver used: no second copy of the gauge field.
#include "stag_dslash.cuh"

namespace stag {

struct ForceCoef { double a[STAG_MAX_SHIFTS]; };

// CTA = 32 consecutive sites of one parity x 4 directions; thread = one link (z, mu) with mu = the
// WARP index, so every 128-bit load instruction of a warp covers 32 consecutive sites (one 128-byte line per
// quarter-warp).  Two earlier mappings, both measured (profiles/README.md, N4): mu as the fastest LANE index
// made each gather of X_i(z+mu) touch 4 lines per quarter-warp and the kernel sat at 74 % of
// l1tex__data_pipe_lsu_wavefronts; one thread per site with all 4 directions needs 144 fp64 accumulators,
// leaves 8 warps per SM and is latency-bound (12 % warps active).  Here a thread keeps one 3x3 sum (36
// registers), which leaves room to unroll the shift loop (fp64: x2 at 16 warps per SM).  X_i(z) is requested by
// the 4 warps of a CTA (3 of the 4 hit L1).  fp32 runs with TWO links per thread (LPT below): its 36 float
// accumulators per link leave room for two, and X_i(z) is then loaded once for both.
// The CTA's 32 x 576 contiguous output bytes leave through shared memory as full sectors.
constexpr int kForceRow = 37;                          // 36 chunks of 16 B per site + 1 pad: conflict-free

// LPT = links per thread: 1 = direction mu is the warp index (4 warps per CTA); 2 = a thread owns the links (z, mu) and
// (z, mu + 2) and loads X_i(z) ONCE for both (2 warps per CTA): 9 instead of 12 vector loads per two links and shift.
// The kernel is bound by the SM's load/store pipe (L1 wavefronts), not by HBM or L2 bytes.
template <typename T, int RECON, int MINB, int UNR, bool SPLIT = false, int LPT = 1>
__global__ void __launch_bounds__(128 / LPT, MINB)
force_kernel(const Geom g, const char *__restrict__ W, const char *__restrict__ x_even,
             const char *__restrict__ w_odd, const size_t stride, const int nshift, const ForceCoef coef,
             double *__restrict__ force, const int accumulate) {
    __shared__ double2 stage[32 * kForceRow];          // [site][mu][9 complex] (+ pad)
    __shared__ int s_lex[32];
    const int wrp = threadIdx.x >> 5, ls = threadIdx.x & 31;
    // consecutive CTAs alternate parity over the same 32-site tile: the X_i one reads as X_i(z) the other reads
    // as X_i(z+mu) a moment later, out of L2 (measured: 316 -> 305 us per fp64 call)
    const int par = blockIdx.x & 1, tile = blockIdx.x >> 1;
    const int e = tile * 32 + ls;
    const int Vh = g.Vh;
    if (e < Vh) {
        const Site s = site_of(g, e, par);
        if (wrp == 0) s_lex[ls] = s.lex;
        const int x[4] = {s.x0, s.x1, s.x2, s.x3};
        // split-double links (N3, T = double): b planes in the fp32 layout, the c planes 16 sets further on
        const size_t set = SPLIT ? link_set_bytes<float, RECON>(Vh) : link_set_bytes<T, RECON>(Vh);
        int ef[LPT];
        T c3[LPT];
#pragma unroll
        for (int l = 0; l < LPT; ++l) {
            const int mu = wrp + l * (4 / LPT);
            int str = 1, phase_sum = 0;
            for (int nu = 0; nu < mu; ++nu) { str *= g.L[nu]; phase_sum += x[nu]; }
            const int Lmu = g.L[mu];
            ef[l] = (s.lex + str - (x[mu] == Lmu - 1 ? Lmu * str : 0)) >> 1;
            c3[l] = T(0);
            if (RECON == 12) {
                const T eta = (phase_sum & 1) ? T(-2) : T(2);
                c3[l] = (mu == 3 && x[3] == Lmu - 1) ? -eta : eta;
            }
            // the matrix is needed only after the shift loop: ask L2 for its lines now (no registers held), so the
            // load after the loop is an L2 hit instead of one more DRAM latency on every CTA's critical path
            const char *wl = W + (size_t)(par * 8 + 2 * mu) * set + (size_t)e * 16;
            constexpr int NCH = (RECON * (SPLIT ? 4 : (int)sizeof(T)) + 15) / 16;
#pragma unroll
            for (int k = 0; k < NCH; ++k) {
                asm volatile("prefetch.global.L2 [%0];" ::"l"(wl + (size_t)k * Vh * 16));
                if (SPLIT) asm volatile("prefetch.global.L2 [%0];" ::"l"(wl + 16 * set + (size_t)k * Vh * 16));
            }
        }
        const char *own = (par == 0 ? x_even : w_odd);     // X_i(z)
        const char *nbr = (par == 0 ? w_odd : x_even);     // X_i(z + mu)
        T m[LPT][18];
#pragma unroll
        for (int l = 0; l < LPT; ++l)
#pragma unroll
            for (int k = 0; k < 18; ++k) m[l][k] = T(0);
#pragma unroll UNR
        for (int i = 0; i < nshift; ++i) {
            T a[6], b[LPT][6];
            load_vec(own + (size_t)i * stride, Vh, e, a);
#pragma unroll
            for (int l = 0; l < LPT; ++l) load_vec(nbr + (size_t)i * stride, Vh, ef[l], b[l]);
            const T c = (T)coef.a[i];
#pragma unroll
            for (int l = 0; l < LPT; ++l)
#pragma unroll
                for (int r = 0; r < 3; ++r) {
                    const T br = c * b[l][2 * r], bi = c * b[l][2 * r + 1];
#pragma unroll
                    for (int q = 0; q < 3; ++q) {            // M[r][q] += c b_r conj(a_q)
                        m[l][6 * r + 2 * q] = fma(br, a[2 * q], fma(bi, a[2 * q + 1], m[l][6 * r + 2 * q]));
                        m[l][6 * r + 2 * q + 1] = fma(bi, a[2 * q], fma(-br, a[2 * q + 1], m[l][6 * r + 2 * q + 1]));
                    }
                }
        }
#pragma unroll
        for (int l = 0; l < LPT; ++l) {
            const int mu = wrp + l * (4 / LPT);
            T u[18];
            if constexpr (SPLIT) load_link_split<RECON>(W + (size_t)(par * 8 + 2 * mu) * set, 16 * set, Vh, e, u, c3[l], policy_evict_first());
            else load_link<RECON>(W + (size_t)(par * 8 + 2 * mu) * set, Vh, e, u, c3[l], policy_evict_first());
            // G = W M in fp64 (one 3x3 product per link: free next to the loads)
            double G[18];
#pragma unroll
            for (int r = 0; r < 3; ++r)
#pragma unroll
                for (int q = 0; q < 3; ++q) {
                    double re = 0.0, im = 0.0;
#pragma unroll
                    for (int k = 0; k < 3; ++k) {
                        const double ur = u[6 * r + 2 * k], ui = u[6 * r + 2 * k + 1];
                        const double mr = m[l][6 * k + 2 * q], mi = m[l][6 * k + 2 * q + 1];
                        re += ur * mr - ui * mi;
                        im += ur * mi + ui * mr;
                    }
                    G[6 * r + 2 * q] = re; G[6 * r + 2 * q + 1] = im;
                }
            const double eps2 = par ? -2.0 : 2.0;            // 2 eps(z)
            const double tr_im = (G[1] + G[9] + G[17]) * (2.0 / 6.0);     // tr(G - G^dag)/6 = i * 2 Im tr G / 6
            double2 *row = stage + ls * kForceRow + mu * 9;
#pragma unroll
            for (int r = 0; r < 3; ++r)
#pragma unroll
                for (int q = 0; q < 3; ++q) {
                    double re = 0.5 * (G[6 * r + 2 * q] - G[6 * q + 2 * r]);
                    double im = 0.5 * (G[6 * r + 2 * q + 1] + G[6 * q + 2 * r + 1]);
                    if (r == q) im -= tr_im;
                    row[3 * r + q] = make_double2(re * eps2, im * eps2);
                }
        }
    }
    __syncthreads();
    // 32 sites x 36 chunks of 16 bytes; consecutive threads write consecutive chunks of one site
    const int nsite = min(32, Vh - tile * 32);
    for (int k = threadIdx.x; k < nsite * 36; k += 128 / LPT) {
        const int site = k / 36, c = k - site * 36;
        double2 v = stage[site * kForceRow + c];
        double2 *out = reinterpret_cast<double2 *>(force + (size_t)s_lex[site] * 72) + c;
        if (accumulate) { const double2 o = *out; v.x += o.x; v.y += o.y; }
        *out = v;
    }
}

}  // namespace stag

using namespace stag;

extern "C" size_t stag_force_workspace_bytes(const stag_ctx *ctx, int prec, int nshift) {
    if (!ctx || !valid_prec(prec) || nshift < 1 || nshift > STAG_MAX_SHIFTS) return 0;
    return align256((size_t)nshift * ctx->g.Vh * vec_bytes_per_site(prec));
}

extern "C" int stag_fermion_force(const stag_ctx *ctx, const void *packed, int prec, int recon, int nshift,
                                  const double *host_residues, const void *x_even, double *dev_force,
                                  int accumulate, void *workspace, void *stream) {
    if (!ctx || !packed || !host_residues || !x_even || !dev_force || !workspace) return STAG_ERR_BADARG;
    if (!valid_prec(prec) || !valid_recon(recon)) return STAG_ERR_BADARG;
    if (nshift < 1 || nshift > STAG_MAX_SHIFTS) return STAG_ERR_BADARG;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const Geom &g = ctx->g;
    const size_t vbytes = (size_t)g.Vh * vec_bytes_per_site(prec);
    const char *x = static_cast<const char *>(x_even);
    char *w = static_cast<char *>(workspace);
    // w_i = D_oe x_i, STAG_MAX_RHS shifts per read of the links (N1 kernel); all groups of four in ONE launch of
    // the cp.async-ring kernel where it applies, so that the groups' fill / drain ramps overlap
    {
        const int rc = stag_dslash_block(ctx, packed, prec, recon, 1, nshift, x, w, st);
        if (rc) return rc;
    }
    ForceCoef coef;
    for (int i = 0; i < STAG_MAX_SHIFTS; ++i) coef.a[i] = i < nshift ? host_residues[i] : 0.0;
    const dim3 grid(2 * ((g.Vh + 31) / 32)), block(128);
    const char *W = static_cast<const char *>(packed);
    // occupancy / unroll measured at 32^3 x 8, 16 shifts (profiles/README.md "N4"): fp64 is fastest with one link per
    // thread, 128 registers (16 warps per SM) and the shift loop unrolled x2
#define STAG_FORCE(T, R, M, U) STAG_LAUNCH_K(ctx, (force_kernel<T, R, M, U>), grid, block, 0, st, g, W, x, w, vbytes, nshift, coef, dev_force, accumulate)
    if (prec == STAG_F64) { if (recon == 18) STAG_FORCE(double, 18, 4, 2); else STAG_FORCE(double, 12, 4, 2); }
    else if (prec == STAG_F64_SPLIT) {                    // N3: fp64 vectors, a = b + c rebuilt as the matrix is loaded
        if (recon == 18) STAG_LAUNCH_K(ctx, (force_kernel<double, 18, 4, 2, true>), grid, block, 0, st, g, W, x, w, vbytes, nshift, coef, dev_force, accumulate);
        else STAG_LAUNCH_K(ctx, (force_kernel<double, 12, 4, 2, true>), grid, block, 0, st, g, W, x, w, vbytes, nshift, coef, dev_force, accumulate);
    }
    else {
        // fp32: two links per thread ((z, mu) and (z, mu + 2): X_i(z) loaded once for both), 8 CTAs of 64 threads per SM,
        // shift loop unrolled x4 — the kernel is load/store-pipe-bound and this is 9 instead of 12 vector loads per two
        // links and shift: 119 -> 99 us at 32^3 x 8, 16 shifts.  (fp64: 72 accumulators per thread, measured slower.)
        const dim3 block2(64);
        if (recon == 18) STAG_LAUNCH_K(ctx, (force_kernel<float, 18, 8, 4, false, 2>), grid, block2, 0, st, g, W, x, w, vbytes, nshift, coef, dev_force, accumulate);
        else STAG_LAUNCH_K(ctx, (force_kernel<float, 12, 8, 4, false, 2>), grid, block2, 0, st, g, W, x, w, vbytes, nshift, coef, dev_force, accumulate);
    }
#undef STAG_FORCE
    STAG_CUDA_OK(cudaGetLastError());
    return STAG_OK;
}
