/* stag.h — C ABI of the B200-native staggered Dslash + multi-shift CG library.
 *
 * The data-parallel hot path of the RHMC of arxiv 1010.5433 ("Staggered fermions
 * simulations on GPUs", Bonati, Cossu, D'Elia, Di Giacomo): the even/odd-preconditioned
 * staggered hopping term D_eo / D_oe (PAPER.md:45 "even/odd preconditioning", :87 "Dirac
 * kernel") applied inside the multi-shift conjugate-gradient solve of
 *
 *        (m^2 - D_eo D_oe + sigma_i) x_i = b,     i = 0 .. nshift-1,
 *
 * the solve the rational approximation needs for MD forces and for the Metropolis step
 * (PAPER.md:43, :49).  The paper has no API (one monolithic program); the entry
 * points are the ones BASELINE.json:north_star names and their arguments are the paper's
 * statement of the problem: lattice extents, links, mass, shifts and residues, stopping
 * residual.  Definitions the paper leaves out (normalisation, phases, boundary condition)
 * are the readings A1-A5 in DESIGN.md.
 *
 * Operator (reading A1-A5).  Site x = (x0,x1,x2,x3), x3 = time, parity
 * (x0+x1+x2+x3) & 1 (0 = even), U_mu(x) in SU(3) the link from x to x+mu:
 *
 *   (D psi)(x) = 1/2 sum_mu eta_mu(x) [ s+ U_mu(x) psi(x+mu) - s- U_mu(x-mu)^dagger psi(x-mu) ]
 *   eta_0 = 1, eta_mu(x) = (-1)^(x0+...+x_{mu-1});   antiperiodic time: s+ = -1 iff mu = 3 and
 *   x3 = L3-1, s- = -1 iff mu = 3 and x3 = 0; periodic in 0,1,2.
 *   D_eo: even output from odd input.  D_oe: odd output from even input.
 *
 * CONVENTIONS
 *   Pointers   "host_*" arguments are host pointers, everything else named dev_* / packed /
 *              workspace / *_even / *_odd is a DEVICE pointer.  The caller owns every buffer
 *              (e.g. torch tensors' data_ptr()); the library allocates nothing per call.  A
 *              stag_ctx owns only the geometry and a few bytes of pinned host memory.
 *   stream     a cudaStream_t passed as void* (NULL = legacy default stream).
 *   Errors     every int-returning function returns STAG_OK (0) or a negative STAG_ERR_*;
 *              no exceptions, no exit().  Kernel launches are asynchronous: a launch error
 *              shows up as STAG_ERR_CUDA from the same or a later call.
 *   Aliasing   input and output buffers of one call must not overlap.
 *   Threads    a stag_ctx may be shared by host threads and by calls on different streams.  Every
 *              synchronising call (stag_mshift_cg*, stag_cg_polish, recon-12 stag_gauge_pack, the
 *              *_host calls) leases one of 4 host staging slots of the context for its duration, so
 *              up to 4 of them run concurrently — the paper's independent pseudo-fermion solves
 *               on separate streams — and a fifth waits for a free slot.  Calls that
 *              run concurrently must not share output buffers or workspaces.  stag_set_option is
 *              not synchronised with running calls.
 *
 * CANONICAL (interchange) FORMATS — always fp64
 *   site index   lex(x) = x0 + L0*(x1 + L1*(x2 + L2*x3));  one-parity index e = lex(x)/2
 *   links        double [V][4][3][3][2]   (site lex, direction mu, row, column, re/im), raw
 *                SU(3): no 1/2, no eta, no boundary sign — the library applies them.
 *   vector       double [Vh][3][2]        (e, colour, re/im) on one parity, Vh = V/2.
 *
 * DEVICE (compute) FORMATS — private to the library, sizes from the *_bytes() functions
 *   packed gauge "hopping matrices", per output parity p, direction d = 2*mu + (0 fwd | 1 bwd):
 *                W_d(x) = +1/2 eta s+ U_mu(x)  or  -1/2 eta s- U_mu(x-mu)^dagger,  indexed by
 *                the OUTPUT site e, stored as planes of 16-byte chunks [p][d][chunk][e] so that
 *                every load is a coalesced, aligned 128-bit access.  recon = 18 keeps all three
 *                rows, recon = 12 keeps rows 1-2 and rebuilds row 3.
 *   vector       colour planes of 16-byte chunks [chunk][e]: fp64 = 3 planes of one complex;
 *                fp32 = one plane of (c0,c1) + one 8-byte plane of c2.  Convert with
 *                stag_vector_pack / stag_vector_unpack.
 */
#ifndef STAG_H_
#define STAG_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define STAG_MAX_SHIFTS 32
#define STAG_MAX_RHS 4        /* sources per block solve (stag_mshift_cg_block) */

enum {
    STAG_OK = 0,
    STAG_ERR_BADARG = -1,       /* odd / too small extent, bad enum, null pointer, bad shift ... */
    STAG_ERR_UNSUPPORTED = -2,  /* valid request this build cannot serve (e.g. V >= 2^31)      */
    STAG_ERR_CUDA = -3,         /* a CUDA runtime call or kernel launch failed                  */
    STAG_ERR_NOT_SU3 = -4,      /* recon = 12 asked for links that are not SU(3) to 1e-12       */
    STAG_ERR_NOTCONV = -5,      /* maxiter reached (or fp32 stagnation); outputs still written  */
    STAG_ERR_BREAKDOWN = -6,    /* <p,Ap> <= 0 or NaN inside CG                                 */
    STAG_ERR_SCRATCH_LIMIT = -7 /* stag_fermion_force_static: needs more than STAG_FORCE_STATIC_BYTES */
};
/* STAG_F64_SPLIT (N3): fp64 vectors and arithmetic on links stored as TWO fp32
 * numbers per real, b = (float)a and c = (float)(a - (double)b); the kernels rebuild a' = b + c
 * (48 significant bits).  The first stag_gauge_packed_bytes(ctx, STAG_F32, recon) bytes of a split
 * buffer ARE the STAG_F32 packed format (the b planes), so the same resident buffer also serves
 * every prec = STAG_F32 call.  Wherever a `prec` sizes or converts a VECTOR, STAG_F64_SPLIT means
 * STAG_F64.  Accepted by every call that takes a `prec` (stag_dslash_block then always runs the register-staged
 * multi-source kernel: the cp.async ring has no split variant). */
enum { STAG_F64 = 0, STAG_F32 = 1, STAG_F64_SPLIT = 2 };
enum { STAG_RECON18 = 18, STAG_RECON12 = 12 };

typedef struct stag_ctx stag_ctx;

/* Result of one multi-shift solve (host struct, filled after the final stream sync). */
typedef struct stag_cg_info {
    int iters;                             /* iterations of the base (smallest-shift) system   */
    int converged;                         /* 1 iff ||r||/||b|| <= stop was reached            */
    int breakdown;                         /* 1 iff <p,Ap> <= 0 or NaN                         */
    int stagnated;                         /* fp32 only: stopped because ||r|| stopped falling */
    double bnorm2;                         /* <b,b>                                            */
    double rnorm2;                         /* iterated <r,r> of the base system at exit        */
    double resid_iter[STAG_MAX_SHIFTS];    /* iterated zeta_i*||r||/||b|| per shift at exit/freeze */
    int iters_shift[STAG_MAX_SHIFTS];      /* iteration at which shift i stopped being updated */
    int kernel_launches;                   /* kernels this call put on the stream (incl. no-op tail) */
} stag_cg_info;

/* ---- context --------------------------------------------------------------------------- */
/* L[mu] even and >= 2, time = L[3]; V = L0*L1*L2*L3 must be < 2^31.  Uses the current CUDA
 * device.  *out is set on success only. */
int stag_ctx_create(const int L[4], stag_ctx **out);
void stag_ctx_destroy(stag_ctx *ctx);
const char *stag_strerror(int err);
/* Tuning knobs (integers): "dslash_block" (threads per CTA: 64|128|256), "dslash_regs"
 * (register budget per thread: 0 auto | 64 | 128 | 255), "dslash_pipe" (1, default: stag_dslash_block
 * streams the matrices through a cp.async shared-memory ring where that is faster; 0: never),
 * "cg_check_every" (iterations between convergence polls), "cg_graph" (0|1: replay iterations as a CUDA
 * graph), "cg_freeze" (0|1: stop updating converged shifts, reading A10),
 * "cg_persistent" (1, default: lattices whose r, q, p_base slices fit in shared memory run the
 * whole solve as one cooperative kernel; 0: always the multi-kernel path),
 * "cg_persistent_threads" (0 auto | 256 | 512 | 1024 threads per CTA of that kernel),
 * "cg_mixed_fp64_from" (default 3; stag_mshift_cg_mixed runs the fp64 multi-shift solve from this many shifts on,
 * 0: never),
 * "cg_mixed_reliable" (stag_mshift_cg_mixed: run the inner stage as the persistent kernel with residual
 * replacement — 0 never | 1, default: single-shift solves | 2 always), "cg_mixed_delta_inv" (>= 2, default 10:
 * replace the residual whenever ||r|| has fallen by this factor),
 * "cg_resident_slices" (0..3, default 3: how many of r, q, p_base the persistent kernel may keep in shared
 * memory; fewer = the global-workspace path large lattices take),
 * "cg_l2_keep_mb" (default 64: the persistent kernel marks the x_i, p_i of the lightest shifts — the ones that stay
 * live longest — evict_last in L2, up to this many MB, and everything else that streams evict_first; 0: none),
 * "cg_fill" (1, default: the persistent kernel defers the shift updates of an iteration and works them off while
 * its CTAs wait at the sync points of the next; 0: all at once after the base shift),
 * "cg_nbflags" (1, default: after the two stencil phases a CTA of the persistent kernel waits only for the CTAs that
 * own its neighbouring sites; 0: for all of them),
 * "cg_single_reduction" (1, default: the single-source persistent kernel makes ONE grid-wide reduction per iteration —
 * <p,q>, <r,q>, <q,q> and <r,r> of the current r together, ||r - alpha q||^2 = rr - 2 alpha <r,q> + alpha^2 <q,q>,
 * rr recomputed from r every iteration; 0: two reductions, <p,q> then <r,r> of the updated r),
 * "cg_profile" (0, default; 1: see stag_cg_profile). */
int stag_set_option(stag_ctx *ctx, const char *key, int value);
int stag_get_option(const stag_ctx *ctx, const char *key, int *value);

/* ---- sizes (bytes) --------------------------------------------------------------------- */
size_t stag_gauge_canonical_bytes(const stag_ctx *ctx);              /* 4*V*18 doubles     */
size_t stag_gauge_packed_bytes(const stag_ctx *ctx, int prec, int recon);
size_t stag_vector_canonical_bytes(const stag_ctx *ctx);             /* Vh*6 doubles       */
size_t stag_vector_bytes(const stag_ctx *ctx, int prec);             /* device format      */
size_t stag_cg_workspace_bytes(const stag_ctx *ctx, int prec, int nshift);
size_t stag_host_scratch_bytes(const stag_ctx *ctx, int prec, int nshift); /* for *_host calls */

/* ---- a1: gauge load + pack (setup; "copy the starting gauge configuration on the
 *      device memory at the beginning", :109 12-real storage, :113 float cast, :119 layout) --- */
/* H->D copy of canonical links, asynchronous on stream (pin host_links for true overlap). */
int stag_gauge_load(const stag_ctx *ctx, const double *host_links,
                    double *dev_links_canonical, void *stream);
/* canonical device links -> packed hopping matrices.  prec = STAG_F32 rounds to nearest
 * (b = (float)a).  recon = 12 first checks max|U U^dag - 1| <= 1e-12 and
 * |det U - 1| <= 1e-12 on the device and returns STAG_ERR_NOT_SU3 otherwise (synchronises
 * the stream; recon = 18 does not synchronise). */
int stag_gauge_pack(const stag_ctx *ctx, const double *dev_links_canonical,
                    void *dev_packed, int prec, int recon, void *stream);

/* ---- vector format conversion (device to device, asynchronous) --------------------------- */
int stag_vector_pack(const stag_ctx *ctx, const double *dev_canonical, void *dev_vec,
                     int prec, void *stream);
int stag_vector_unpack(const stag_ctx *ctx, const void *dev_vec, int prec,
                       double *dev_canonical, void *stream);

/* ---- a2/a3: the hopping term (570 flop/site).  One kernel launch, no sync. ---- */
int stag_dslash_eo(const stag_ctx *ctx, const void *packed, int prec, int recon,
                   const void *in_odd, void *out_even, void *stream);
int stag_dslash_oe(const stag_ctx *ctx, const void *packed, int prec, int recon,
                   const void *in_even, void *out_odd, void *stream);

/* ---- a3-a7: multi-shift CG (ref [9]); start vector zero for every shift.
 *   b_even     source, device format
 *   shifts     host, nshift values sigma_i >= 0, any order; 1 <= nshift <= STAG_MAX_SHIFTS
 *   residues   host, nullable; with y_even != NULL:  y = residue0*b + sum_i residues[i]*x_i
 *   stop       on the iterated ||r||/||b|| of the smallest-shift system, tested every iteration
 *   x_even     out, nshift contiguous device-format vectors (x_i at byte offset
 *              i*stag_vector_bytes)
 *   workspace  stag_cg_workspace_bytes(ctx, prec, nshift) bytes, 256-byte aligned
 *   info       host, nullable
 * Vectors are prec; every reduction and scalar recurrence is fp64.  Synchronises the stream
 * before returning.  STAG_ERR_NOTCONV / STAG_ERR_BREAKDOWN still write x (and y) and info. */
int stag_mshift_cg(const stag_ctx *ctx, const void *packed, int prec, int recon,
                   const void *b_even, double mass, int nshift, const double *host_shifts,
                   const double *host_residues, double residue0, double stop, int maxiter,
                   void *x_even, void *y_even, void *workspace, stag_cg_info *info,
                   void *stream);

/* ---- N1: the hopping term on nrhs independent vectors, STAG_MAX_RHS of them per read of
 * the links.  in / out: nrhs (1 .. STAG_MAX_SHIFTS) contiguous device-format vectors (stride
 * stag_vector_bytes); out_parity 0 = D_eo (even output, odd input), 1 = D_oe.  nrhs <= STAG_MAX_RHS: one launch;
 * more: groups of STAG_MAX_RHS, in one launch where the cp.async-ring kernel applies.  No sync. */
int stag_dslash_block(const stag_ctx *ctx, const void *packed, int prec, int recon, int out_parity,
                      int nrhs, const void *in, void *out, void *stream);

/* ---- N1: block solve of nrhs INDEPENDENT sources — the paper's multiple
 * pseudo-fermions — with the same mass, shifts, residues and stop.  One persistent
 * kernel; each link is read once per Dslash for all nrhs sources (links are 92 % of the stencil's
 * bytes); every source keeps its own scalars, shift freezing and convergence latch, so each
 * result is what stag_mshift_cg returns for that source alone.
 *   nrhs       1 .. STAG_MAX_RHS
 *   b_even     nrhs contiguous device-format vectors (stride stag_vector_bytes)
 *   x_even     out, [nrhs][nshift] contiguous vectors: x of source s, shift i at byte offset
 *              (s*nshift + i) * stag_vector_bytes
 *   y_even     nullable, nrhs contiguous vectors
 *   workspace  stag_cg_block_workspace_bytes(ctx, prec, nshift, nrhs) bytes, 256-byte aligned
 *   info       host, nullable, nrhs structs (kernel_launches is counted in info[0])
 * Returns STAG_OK only if every source converged; else the worst of NOTCONV / BREAKDOWN. */
size_t stag_cg_block_workspace_bytes(const stag_ctx *ctx, int prec, int nshift, int nrhs);
int stag_mshift_cg_block(const stag_ctx *ctx, const void *packed, int prec, int recon, int nrhs,
                         const void *b_even, double mass, int nshift, const double *host_shifts,
                         const double *host_residues, double residue0, double stop, int maxiter,
                         void *x_even, void *y_even, void *workspace, stag_cg_info *info,
                         void *stream);

/* ---- N2: mixed precision the way the paper uses it (PAPER.md:93 fp32 for the
 * MD-force solves, fp64 for Metropolis; :127-129 a shifted solver cannot be restarted, but every
 * single system can): an fp32 multi-shift run followed by a per-shift fp64 DEFECT-CORRECTION POLISH —
 * ordinary CG with a non-zero start:  r_i = b - (A + sigma_i) x_i  in fp64,  (A + sigma_i) e_i = r_i
 * by CG from zero until ||r|| <= stop ||b||,  x_i += e_i;  then the true residual is recomputed and
 * the pass repeated (at most 3 passes) while it is above stop.  Up to STAG_MAX_RHS shifts are polished
 * together in one persistent launch with one read of the links per Dslash (the N1 kernel, one shift per
 * source).  Also the remedy for reading A8 (true residual slightly above stop after an fp64 multi-shift
 * run): shifts already at or below stop are left untouched (0 iterations). */
typedef struct stag_polish_info {
    int passes;                              /* defect-correction passes run (0 .. 3)                     */
    int iters[STAG_MAX_SHIFTS];              /* polish CG iterations of shift i, all passes               */
    double resid_before[STAG_MAX_SHIFTS];    /* TRUE ||b - (A+sigma_i) x_i|| / ||b|| on entry (fp64)      */
    double resid_after[STAG_MAX_SHIFTS];     /* ... on exit                                               */
    int kernel_launches;
} stag_polish_info;
typedef struct stag_mixed_info {
    stag_cg_info inner;                      /* the inner multi-shift run (fp32 matrices; route 3: fp64)  */
    stag_polish_info polish;
    int reliable_updates;                    /* residual replacements of the inner run (0: plain fp32 run) */
    int route;                               /* 1 residual replacement | 2 fp32 + polish | 3 fp64 multi-shift */
} stag_mixed_info;

/* dst = src converted between device vector formats (nvec contiguous vectors each side). */
int stag_vector_convert(const stag_ctx *ctx, const void *src, int src_prec, void *dst, int dst_prec,
                        int nvec, void *stream);

/* Polish x_i (in/out, nshift contiguous fp64 device-format vectors) of (A + sigma_i) x_i = b in place.
 * prec = STAG_F64 or STAG_F64_SPLIT (STAG_MAX_RHS shifts per persistent launch either way); vectors fp64.
 * Returns STAG_OK iff every resid_after <= stop, else STAG_ERR_NOTCONV (x still improved) /
 * STAG_ERR_BREAKDOWN.  Synchronises the stream.  workspace: stag_cg_polish_workspace_bytes, 256-aligned. */
size_t stag_cg_polish_workspace_bytes(const stag_ctx *ctx);
int stag_cg_polish(const stag_ctx *ctx, const void *packed, int prec, int recon, const void *b_even,
                   double mass, int nshift, const double *host_shifts, double stop, int maxiter,
                   void *x_even, void *workspace, stag_polish_info *info, void *stream);

/* Inner stage, then the polish, then y.  The call picks the fastest route to the fp64 stop for the number of
 * shifts (info->route; option "cg_mixed_fp64_from", default 3): from that many shifts on — where the per-shift polish
 * costs more than fp32 saved — it IS the fp64 multi-shift solve on packed_hi (the paper's own choice for the
 * Metropolis solves), followed by the same true-residual check; with stop >= 1e-6, which fp32 can
 * reach, always the fp32 routes.  Inner stage, single shift with recon_hi =
 * recon_lo (option "cg_mixed_reliable"): ONE persistent kernel with RESIDUAL REPLACEMENT (ref [7]):
 * fp32 matrices, r, q, p; x in fp64; whenever ||r|| has fallen tenfold, and again at stop, the true residual
 * b - (A + sigma) x is recomputed with the fp64 matrices and replaces the recursive one; convergence is declared
 * on that true residual, so the polish has nothing left to do.  Otherwise:
 * fp32 multi-shift CG to inner_stop (<= 0: default 1e-5) on packed_lo (STAG_F32 format — e.g. the first
 * half of a STAG_F64_SPLIT buffer), then the polish on packed_hi (prec_hi = STAG_F64 | STAG_F64_SPLIT) to
 * stop, then y.  b_even, x_even, y_even: fp64 device format.  The fp32 stage ending on stagnation or
 * maxiter is not an error: the polish finishes the job.  Returns as stag_cg_polish. */
size_t stag_mshift_cg_mixed_workspace_bytes(const stag_ctx *ctx, int nshift);
int stag_mshift_cg_mixed(const stag_ctx *ctx, const void *packed_hi, int prec_hi, int recon_hi,
                         const void *packed_lo, int recon_lo, const void *b_even, double mass, int nshift,
                         const double *host_shifts, const double *host_residues, double residue0,
                         double stop, double inner_stop, int maxiter, void *x_even, void *y_even,
                         void *workspace, stag_mixed_info *info, void *stream);

/* ---- N4: the first consumer of the x_i — the fermion force of the rational
 * pseudo-fermion action S[U] = b^dag (residue0 + sum_i residues_i (A + sigma_i)^-1) b,
 * one thread per link.  With X_i = x_i on even sites and D_oe x_i on odd sites,
 *   F_mu(z) = 2 TA( f U_mu(z) . eps(z) sum_i residues_i X_i(z+mu) X_i(z)^dag ),  f = 1/2 eta_mu(z) s_mu(z),
 *   eps = +1 / -1 on even / odd z,  TA(G) = (G - G^dag)/2 - tr(G - G^dag)/6,
 * i.e. d/dt S[U_mu(z) -> exp(itT) U_mu(z)] at t = 0 is tr(i T F_mu(z)) for Hermitian traceless T.
 *   x_even     nshift contiguous device-format vectors of `prec` (the output of stag_mshift_cg)
 *   dev_force  out, fp64 [V][4][3][3][2] (site lex, mu, row, column, re/im) — the canonical link layout;
 *              accumulate != 0 adds to it (several pseudo-fermions)
 *   workspace  stag_force_workspace_bytes (the nshift odd vectors D_oe x_i), 256-byte aligned
 * prec = STAG_F64 | STAG_F32 (the paper's choice for the force) | STAG_F64_SPLIT (fp64 vectors on a
 * split-double buffer); outer products in prec, the 3x3 product and projection in fp64.  Asynchronous: the D_oe x_i
 * launch(es), then the force kernel; no sync. */
size_t stag_force_workspace_bytes(const stag_ctx *ctx, int prec, int nshift);
int stag_fermion_force(const stag_ctx *ctx, const void *packed, int prec, int recon, int nshift,
                       const double *host_residues, const void *x_even, double *dev_force, int accumulate,
                       void *workspace, void *stream);

/* ---- the force for callers that cannot allocate device memory ------------------------------------------
 * stag_fermion_force wants a workspace, and a workspace has to come from somewhere.  A caller may have no way to
 * get one: a force routine plugged into another program's integrator receives the x_i and the force array and
 * nothing else; the host program may have handed every byte of device memory to its own pool when it started, so
 * that a cudaMalloc here fails or eats memory the host relies on; and cudaMalloc / cudaFree stall the whole device,
 * which an MD loop that evaluates the force thousands of times on busy streams cannot pay each time.
 * stag_fermion_force_static is stag_fermion_force without the workspace argument: same arguments otherwise, same
 * kernels, same result; the D_oe x_i go into a fixed array of STAG_FORCE_STATIC_BYTES that is part of the library's
 * device image.  The call itself allocates and frees nothing, on the host or on the device.
 *   Limit      stag_force_workspace_bytes(ctx, prec, nshift) <= STAG_FORCE_STATIC_BYTES (8 MiB: e.g. 16^3 x 4 with
 *              16 fp64 shifts = 6 MiB), else STAG_ERR_SCRATCH_LIMIT and nothing is launched.  Every GPU on which
 *              the process uses this library carries those 8 MiB until the process exits.
 *   Device     the context's GPU must be the current one (else STAG_ERR_BADARG): the array exists once per GPU.
 *   First call the first call on each GPU looks the array's device address up (cudaGetSymbolAddress, which also
 *              makes the runtime load the library's device code there) and caches it; make that call during
 *              start-up, before any stream capture begins.  Later calls only launch.
 *   Sharing    all calls on one GPU use the same array.  It keeps what the previous call wrote; nothing in it needs
 *              clearing, because each call overwrites every byte it later reads.  Two calls that can overlap on
 *              the GPU — other streams, host threads or contexts — race on it and both results are garbage:
 *              serialise them (one stream, or events).  Calls with a caller-owned workspace are not affected. */
#define STAG_FORCE_STATIC_BYTES (8u << 20)
size_t stag_fermion_force_static_max_bytes(void);                   /* = STAG_FORCE_STATIC_BYTES */
int stag_fermion_force_static(const stag_ctx *ctx, const void *packed, int prec, int recon, int nshift,
                              const double *host_residues, const void *x_even, double *dev_force,
                              int accumulate, void *stream);

/* ---- the same calls on HOST buffers in canonical fp64 format (copies inside) --------------
 * dev_scratch: stag_host_scratch_bytes(ctx, prec, nshift) bytes of device memory
 * (nshift = 0 for stag_dslash_host).  out_parity: 0 = D_eo, 1 = D_oe. */
int stag_dslash_host(const stag_ctx *ctx, const void *packed, int prec, int recon,
                     int out_parity, const double *host_in, double *host_out,
                     void *dev_scratch, void *stream);
int stag_mshift_cg_host(const stag_ctx *ctx, const void *packed, int prec, int recon,
                        const double *host_b, double mass, int nshift,
                        const double *host_shifts, const double *host_residues,
                        double residue0, double stop, int maxiter, double *host_x,
                        double *host_y, void *dev_scratch, stag_cg_info *info, void *stream);

/* ---- measurement aids (each roofline figure must name the kernel it is about) --------
 * stag_kernel_log: the demangled names of the distinct kernels the calls on ctx have launched since the last
 * stag_kernel_log_reset, one per line, into buf (host); returns their number, or STAG_ERR_BADARG if nbytes is
 * too small.  bench.py matches these names against the kernel names of the committed ncu captures.
 * stag_cg_profile: with option "cg_profile" = 1 the multi-kernel path of stag_mshift_cg runs without its CUDA
 * graph and brackets each of the four kernels of iterations 8 .. 39 with CUDA events on the caller's stream;
 * this returns the mean microseconds of a2 (D_oe), a3 (D_eo + <p,q>), a5 (r update) and a6 (shift update)
 * launches of the last such solve and how many iterations were averaged (0: none yet). */
int stag_kernel_log_reset(const stag_ctx *ctx);
int stag_kernel_log(const stag_ctx *ctx, char *host_buf, size_t nbytes);
int stag_cg_profile(const stag_ctx *ctx, double host_us_per_launch[4], int *host_iterations);

#ifdef __cplusplus
}
#endif
#endif /* STAG_H_ */
