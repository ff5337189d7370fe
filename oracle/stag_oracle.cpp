// ORACLE — TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, obviously-correct CPU implementation (fp64, one thread unless
// oracle_set_threads() is called) of what the hot path of arxiv 1010.5433
// computes: the even/odd staggered hopping term D_eo / D_oe and the multi-shift
// conjugate-gradient solve of (m^2 - D_eo D_oe + sigma_i) x_i = b.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
// reference legs may call this.  It shares no code with the CUDA path
// (paper_1010_5433_b200/csrc) and includes none of its headers.
//
// What follows which passage:
//   * oracle_dslash      — the DEFINITION of the operator.  The paper never writes it
//                          ("standard staggered fermions", "even/odd
//                          preconditioning"; "a thread per even site"); the
//                          formula is the reading A1-A5 of DESIGN.md / SURVEY.md §8(a):
//                          (D psi)(x) = 1/2 sum_mu eta_mu(x) [ s+ U_mu(x) psi(x+mu)
//                                                            - s- U_mu(x-mu)^dag psi(x-mu) ].
//                          Pinned by P1 (free spectrum), P2, P3, P5 (tests/test_oracle_pins.py).
//   * oracle_apply_A     — A v = m^2 v - D_eo D_oe v + sigma v  (north_star).
//   * oracle_mshift_cg   — the ALGORITHM (an iteration, so the oracle follows it step by
//                          step): CG for shifted systems (ref
//                          [9] = Jegerlehner hep-lat/9612014), zero start vector
//                          (PAPER.md:129); recurrences as in DESIGN.md reading C4, in that
//                          order and notation, zeta carried in ratio form (reading A15).
//                          Pinned by P7, P8.
//   * oracle_dense_*     — brute force for tiny lattices (north_star: "dense brute-force
//                          linear solves on 2^4 and 4^4 lattices for every shift").
//   * oracle_cg_polish   — N2: textbook CG for ONE shifted system from a non-zero
//                          start vector.  Pinned by P9 (dense solves; zero start = oracle_mshift_cg
//                          with one shift, iterate for iterate; exact start = 0 iterations).
//   * oracle_fermion_force — N4: derivative of the rational pseudo-fermion action on every link
//                          (outer products of x_i and D_oe x_i).  Pinned by P10: finite differences
//                          of the action computed from dense solves.
//   * oracle_partial_fraction — y = residue0*b + sum_i residues[i]*x_i.
//
// No blocking, fusion, tables or reordering: loops over sites, arithmetic neighbours.
// The threaded mode (oracle_set_threads(k > 1): OpenMP over sites, chunk-ordered deterministic
// reductions) is pinned by P11: bit-equal to one thread for k = 2, 5, 8.
// Every function here is pinned (no "parity unpinned" function); what is unpinned against
// the PAPER is only the particular equivalent eta / axis convention (readings A2, A4).

#include <cmath>
#include <complex>
#include <cstdlib>
#include <cstring>
#include <vector>

typedef std::complex<double> cd;

static int g_threads = 1;

static inline long lex_of(const int *L, int x0, int x1, int x2, int x3) {
    return x0 + (long)L[0] * (x1 + (long)L[1] * (x2 + (long)L[2] * x3));
}

static inline long vol(const int *L) { return (long)L[0] * L[1] * L[2] * L[3]; }

extern "C" {

void oracle_set_threads(int n) { g_threads = n < 1 ? 1 : n; }

// out(x) = (D in)(x) on the sites x of parity out_parity; `in` lives on the other parity.
// links: double[V][4][3][3][2] raw SU(3); in/out: double[Vh][3][2], index e = lex/2.
// out_parity = 0 is D_eo (even output, odd input); out_parity = 1 is D_oe.
int oracle_dslash(const int *L, const double *links, const double *in, double *out,
                  int out_parity) {
    for (int mu = 0; mu < 4; ++mu)
        if (L[mu] < 2 || (L[mu] & 1)) return -1;
    const cd *U = reinterpret_cast<const cd *>(links);
    const cd *psi = reinterpret_cast<const cd *>(in);
    cd *res = reinterpret_cast<cd *>(out);
#pragma omp parallel for collapse(2) num_threads(g_threads) schedule(static)
    for (int x3 = 0; x3 < L[3]; ++x3)
        for (int x2 = 0; x2 < L[2]; ++x2)
            for (int x1 = 0; x1 < L[1]; ++x1)
                for (int x0 = 0; x0 < L[0]; ++x0) {
                    if (((x0 + x1 + x2 + x3) & 1) != out_parity) continue;
                    const int x[4] = {x0, x1, x2, x3};
                    const long lx = lex_of(L, x0, x1, x2, x3);
                    cd acc[3] = {0.0, 0.0, 0.0};
                    int phase_sum = 0;  // x0 + ... + x_{mu-1}
                    for (int mu = 0; mu < 4; ++mu) {
                        const double eta = (phase_sum & 1) ? -1.0 : 1.0;
                        // forward hop: + s+ U_mu(x) psi(x+mu)
                        int xp[4] = {x0, x1, x2, x3};
                        xp[mu] = (x[mu] + 1) % L[mu];
                        const double sp = (mu == 3 && x[3] == L[3] - 1) ? -1.0 : 1.0;
                        const cd *Uf = U + (lx * 4 + mu) * 9;
                        const cd *pf = psi + (lex_of(L, xp[0], xp[1], xp[2], xp[3]) / 2) * 3;
                        for (int i = 0; i < 3; ++i) {
                            cd t = 0.0;
                            for (int j = 0; j < 3; ++j) t += Uf[i * 3 + j] * pf[j];
                            acc[i] += 0.5 * eta * sp * t;
                        }
                        // backward hop: - s- U_mu(x-mu)^dagger psi(x-mu)
                        int xm[4] = {x0, x1, x2, x3};
                        xm[mu] = (x[mu] - 1 + L[mu]) % L[mu];
                        const double sm = (mu == 3 && x[3] == 0) ? -1.0 : 1.0;
                        const long lm = lex_of(L, xm[0], xm[1], xm[2], xm[3]);
                        const cd *Ub = U + (lm * 4 + mu) * 9;
                        const cd *pb = psi + (lm / 2) * 3;
                        for (int i = 0; i < 3; ++i) {
                            cd t = 0.0;
                            for (int j = 0; j < 3; ++j) t += std::conj(Ub[j * 3 + i]) * pb[j];
                            acc[i] -= 0.5 * eta * sm * t;
                        }
                        phase_sum += x[mu];
                    }
                    for (int i = 0; i < 3; ++i) res[(lx / 2) * 3 + i] = acc[i];
                }
    return 0;
}

// out = (m^2 + sigma) in - D_eo (D_oe in), all on even sites.  tmp_odd: Vh*3 complex scratch.
int oracle_apply_A(const int *L, const double *links, double mass, double sigma,
                   const double *in_even, double *out_even, double *tmp_odd) {
    int rc = oracle_dslash(L, links, in_even, tmp_odd, 1);
    if (rc) return rc;
    rc = oracle_dslash(L, links, tmp_odd, out_even, 0);
    if (rc) return rc;
    const long n = vol(L) / 2 * 6;
    const double d = mass * mass + sigma;
    for (long k = 0; k < n; ++k) out_even[k] = d * in_even[k] - out_even[k];
    return 0;
}

}  // extern "C"

// <a,b> real part and norms with a long double accumulator (C6: the oracle's reductions are
// not the noisier side of a 1e-13 comparison).
static double re_dot(const double *a, const double *b, long n) {
    long double s = 0.0L;
    for (long k = 0; k < n; ++k) s += (long double)a[k] * (long double)b[k];
    return (double)s;
}

extern "C" {

double oracle_norm2(const double *a, long n) { return re_dot(a, a, n); }

// Multi-shift CG, reading C4 of DESIGN.md, step by step.
//   b:        double[Vh][3][2] even source
//   shifts:   nshift values sigma_i >= 0 (any order)
//   x:        double[nshift][Vh][3][2] out, started from zero
//   stop:     on the iterated ||r||/||b|| of the base (smallest-shift) system
//   zeta_out: nullable, nshift doubles: final zeta_i (residual of system i is zeta_i * r)
//   r_out:    nullable, Vh*6 doubles: final iterated base residual
//   rr_hist:  nullable, maxiter+1 doubles: rr after each iteration (rr_hist[0] = bb)
// returns 0 converged, -5 not converged in maxiter, -6 breakdown, -1 bad argument.
int oracle_mshift_cg(const int *L, const double *links, const double *b, double mass,
                     int nshift, const double *shifts, double stop, int maxiter, double *x,
                     int *iters_out, double *zeta_out, double *r_out, double *rr_hist) {
    if (nshift < 1 || stop <= 0.0 || maxiter < 0) return -1;
    const long n = vol(L) / 2 * 6;
    int base = 0;
    for (int i = 1; i < nshift; ++i)
        if (shifts[i] < shifts[base]) base = i;
    const double sigma0 = shifts[base];
    if (mass * mass + sigma0 <= 0.0) return -1;
    std::vector<double> delta(nshift);
    for (int i = 0; i < nshift; ++i) delta[i] = shifts[i] - sigma0;

    std::vector<double> r(b, b + n), q(n), tmp(n);
    std::vector<std::vector<double> > p(nshift, std::vector<double>(b, b + n));
    std::memset(x, 0, sizeof(double) * n * nshift);
    // theta_i = zeta_i / zetaold_i, carried as a state variable (reading A15): C4's
    //   zetanew_i = zeta_i zetaold_i alphaold / (alpha betaold (zetaold_i - zeta_i)
    //                                            + zetaold_i alphaold (1 + delta_i alpha))
    // divided through by zetaold_i alphaold is
    //   zetanew_i = zeta_i / ( (1 + delta_i alpha) + (alpha betaold / alphaold)(1 - theta_i) ),
    // the same number, but without the product zeta_i*zetaold_i that underflows (-> 0/0 = NaN)
    // for large shifts long before the base system converges.
    std::vector<double> zeta(nshift, 1.0), theta(nshift, 1.0), theta_new(nshift),
        alpha_i(nshift), beta_i(nshift);
    double alpha_old = 1.0, beta_old = 0.0;
    const double bb = re_dot(b, b, n);
    double rr = bb;
    int iters = 0, rc = -5;
    if (rr_hist) rr_hist[0] = bb;
    if (bb == 0.0) {
        rc = 0;
    } else {
        for (int it = 1; it <= maxiter; ++it) {
            // q = B p_base,  B = A + sigma0
            oracle_apply_A(L, links, mass, sigma0, p[base].data(), q.data(), tmp.data());
            const double pq = re_dot(p[base].data(), q.data(), n);
            const double alpha = rr / pq;
            if (!(pq > 0.0) || !std::isfinite(alpha)) { rc = -6; break; }
            for (int i = 0; i < nshift; ++i) {
                theta_new[i] = 1.0 / ((1.0 + delta[i] * alpha) +
                                      (alpha * beta_old / alpha_old) * (1.0 - theta[i]));
                alpha_i[i] = alpha * theta_new[i];          // alpha zetanew_i / zeta_i
            }
            for (int i = 0; i < nshift; ++i) {
                double *xi = x + (long)i * n;
                const double *pi = p[i].data();
                const double a = alpha_i[i];
#pragma omp parallel for num_threads(g_threads) schedule(static)
                for (long k = 0; k < n; ++k) xi[k] += a * pi[k];
            }
            for (long k = 0; k < n; ++k) r[k] -= alpha * q[k];
            const double rr_new = re_dot(r.data(), r.data(), n);
            const double beta = rr_new / rr;
            for (int i = 0; i < nshift; ++i) {
                beta_i[i] = beta * theta_new[i] * theta_new[i];   // beta (zetanew_i / zeta_i)^2
            }
            for (int i = 0; i < nshift; ++i) {
                double *pi = p[i].data();
                const double zn = zeta[i] * theta_new[i], bi = beta_i[i];   // zetanew_i
                const double *rp = r.data();
#pragma omp parallel for num_threads(g_threads) schedule(static)
                for (long k = 0; k < n; ++k) pi[k] = zn * rp[k] + bi * pi[k];
            }
            for (int i = 0; i < nshift; ++i) { zeta[i] *= theta_new[i]; theta[i] = theta_new[i]; }
            alpha_old = alpha; beta_old = beta; rr = rr_new;
            iters = it;
            if (rr_hist) rr_hist[it] = rr;
            if (std::sqrt(rr / bb) <= stop) { rc = 0; break; }
        }
    }
    if (iters_out) *iters_out = iters;
    if (zeta_out) for (int i = 0; i < nshift; ++i) zeta_out[i] = zeta[i];
    if (r_out) std::memcpy(r_out, r.data(), sizeof(double) * n);
    return rc;
}

// N2 polish: the shifted solver must start from zero, but ONE
// system (A + sigma) x = b may start anywhere — "ordinary CG with a non-zero start", the textbook
// algorithm written out:
//   r = b - (A + sigma) x ; p = r ; rr = <r,r>
//   while sqrt(rr / <b,b>) > stop:  q = (A + sigma) p ; alpha = rr / <p,q> ; x += alpha p ;
//                                   r -= alpha q ; beta = rr_new / rr ; p = r + beta p
// x: in = start vector, out = polished solution.  res0_out: true relative residual of the start.
// returns 0 converged (possibly after 0 iterations), -5 maxiter, -6 breakdown, -1 bad argument.
int oracle_cg_polish(const int *L, const double *links, const double *b, double mass, double sigma,
                     double stop, int maxiter, double *x, int *iters_out, double *res0_out) {
    if (stop <= 0.0 || maxiter < 0 || mass * mass + sigma <= 0.0) return -1;
    const long n = vol(L) / 2 * 6;
    std::vector<double> r(n), p(n), q(n), tmp(n);
    if (oracle_apply_A(L, links, mass, sigma, x, q.data(), tmp.data())) return -1;
    for (long k = 0; k < n; ++k) r[k] = b[k] - q[k];
    p = r;
    const double bb = re_dot(b, b, n);
    double rr = re_dot(r.data(), r.data(), n);
    if (res0_out) *res0_out = bb > 0.0 ? std::sqrt(rr / bb) : 0.0;
    int iters = 0, rc = -5;
    if (bb == 0.0 || std::sqrt(rr / bb) <= stop) rc = 0;
    else
        for (int it = 1; it <= maxiter; ++it) {
            oracle_apply_A(L, links, mass, sigma, p.data(), q.data(), tmp.data());
            const double pq = re_dot(p.data(), q.data(), n);
            const double alpha = rr / pq;
            if (!(pq > 0.0) || !std::isfinite(alpha)) { rc = -6; break; }
            for (long k = 0; k < n; ++k) x[k] += alpha * p[k];
            for (long k = 0; k < n; ++k) r[k] -= alpha * q[k];
            const double rr_new = re_dot(r.data(), r.data(), n);
            const double beta = rr_new / rr;
            for (long k = 0; k < n; ++k) p[k] = r[k] + beta * p[k];
            rr = rr_new;
            iters = it;
            if (std::sqrt(rr / bb) <= stop) { rc = 0; break; }
        }
    if (iters_out) *iters_out = iters;
    return rc;
}

// N4 (SURVEY.md §8(f); PAPER.md:25 "fermion force", :87 "a thread ... to every link", :93): the
// force of the rational pseudo-fermion action  S[U] = b^dag ( residue0 + sum_i residues_i (A+sigma_i)^-1 ) b
// on every link, given the solutions x_i = (A+sigma_i)^-1 b (even sites).  The paper prints no
// formula; this is the derivative of S written out (derivation in DESIGN.md "N4"):
//   X_i = x_i on even sites, D_oe x_i on odd sites;  eps(z) = +1 (z even) / -1 (z odd)
//   M_mu(z) = eps(z) sum_i residues_i X_i(z+mu) X_i(z)^dag                     (3x3 outer products)
//   F_mu(z) = 2 f_mu(z) TA( U_mu(z) M_mu(z) ),   f = 1/2 eta_mu(z) s_mu(z)  (the hop's own factor),
//   TA(G) = (G - G^dag)/2 - tr(G - G^dag)/6      (traceless anti-Hermitian part)
// so that  d/dt S[ U_mu(z) -> exp(i t T) U_mu(z) ] at t = 0  equals  tr( i T F_mu(z) )  for every
// Hermitian traceless T.  Pinned by exactly that statement with S from dense solves (P10).
// x: double[nshift][Vh][3][2]; force out: double[V][4][3][3][2] (site lex, mu, row, col, re/im).
int oracle_fermion_force(const int *L, const double *links, int nshift, const double *residues,
                         const double *x, double *force) {
    if (nshift < 1) return -1;
    for (int mu = 0; mu < 4; ++mu)
        if (L[mu] < 2 || (L[mu] & 1)) return -1;
    const long n = vol(L) / 2 * 6;
    std::vector<std::vector<double> > w(nshift, std::vector<double>(n));
    for (int i = 0; i < nshift; ++i)
        if (oracle_dslash(L, links, x + (long)i * n, w[i].data(), 1)) return -1;
    const cd *U = reinterpret_cast<const cd *>(links);
    cd *F = reinterpret_cast<cd *>(force);
    for (int x3 = 0; x3 < L[3]; ++x3)
        for (int x2 = 0; x2 < L[2]; ++x2)
            for (int x1 = 0; x1 < L[1]; ++x1)
                for (int x0 = 0; x0 < L[0]; ++x0) {
                    const int xx[4] = {x0, x1, x2, x3};
                    const long lz = lex_of(L, x0, x1, x2, x3);
                    const int par = (x0 + x1 + x2 + x3) & 1;
                    const double eps = par ? -1.0 : 1.0;
                    int phase_sum = 0;
                    for (int mu = 0; mu < 4; ++mu) {
                        const double eta = (phase_sum & 1) ? -1.0 : 1.0;
                        const double sgn = (mu == 3 && xx[3] == L[3] - 1) ? -1.0 : 1.0;
                        const double f = 0.5 * eta * sgn;
                        int xp[4] = {x0, x1, x2, x3};
                        xp[mu] = (xx[mu] + 1) % L[mu];
                        const long lzp = lex_of(L, xp[0], xp[1], xp[2], xp[3]);
                        cd M[9];
                        for (int k = 0; k < 9; ++k) M[k] = 0.0;
                        for (int i = 0; i < nshift; ++i) {
                            const cd *xe = reinterpret_cast<const cd *>(x + (long)i * n);
                            const cd *wo = reinterpret_cast<const cd *>(w[i].data());
                            const cd *Xz = (par == 0 ? xe : wo) + (lz / 2) * 3;
                            const cd *Xzp = (par == 0 ? wo : xe) + (lzp / 2) * 3;
                            for (int a = 0; a < 3; ++a)
                                for (int b = 0; b < 3; ++b)
                                    M[a * 3 + b] += eps * residues[i] * Xzp[a] * std::conj(Xz[b]);
                        }
                        const cd *Ul = U + (lz * 4 + mu) * 9;
                        cd G[9];
                        for (int a = 0; a < 3; ++a)
                            for (int b = 0; b < 3; ++b) {
                                cd t = 0.0;
                                for (int c = 0; c < 3; ++c) t += Ul[a * 3 + c] * M[c * 3 + b];
                                G[a * 3 + b] = t;
                            }
                        cd tr = 0.0;
                        for (int a = 0; a < 3; ++a) tr += G[a * 3 + a] - std::conj(G[a * 3 + a]);
                        cd *Fl = F + (lz * 4 + mu) * 9;
                        for (int a = 0; a < 3; ++a)
                            for (int b = 0; b < 3; ++b) {
                                cd t = 0.5 * (G[a * 3 + b] - std::conj(G[b * 3 + a]));
                                if (a == b) t -= tr / 6.0;
                                Fl[a * 3 + b] = 2.0 * f * t;
                            }
                        phase_sum += xx[mu];
                    }
                }
    return 0;
}

// y = residue0*b + sum_i residues[i]*x_i   (partial-fraction form of r(A) b)
void oracle_partial_fraction(long n, const double *b, int nshift, const double *residues,
                             double residue0, const double *x, double *y) {
    for (long k = 0; k < n; ++k) {
        long double s = (long double)residue0 * b[k];
        for (int i = 0; i < nshift; ++i) s += (long double)residues[i] * x[(long)i * n + k];
        y[k] = (double)s;
    }
}

// Dense A = m^2 - D_eo D_oe as an N x N complex matrix (row-major, N = 3*Vh), built column
// by column by applying the operator to unit vectors.  Tiny lattices only.
int oracle_dense_A(const int *L, const double *links, double mass, double *A_out) {
    const long N = vol(L) / 2 * 3;
    std::vector<double> e(2 * N, 0.0), col(2 * N), tmp(2 * N);
    cd *A = reinterpret_cast<cd *>(A_out);
    for (long k = 0; k < N; ++k) {
        e[2 * k] = 1.0;
        int rc = oracle_apply_A(L, links, mass, 0.0, e.data(), col.data(), tmp.data());
        if (rc) return rc;
        e[2 * k] = 0.0;
        for (long i = 0; i < N; ++i) A[i * N + k] = cd(col[2 * i], col[2 * i + 1]);
    }
    return 0;
}

// Solve (A + sigma) x = b by Gaussian elimination with partial pivoting in long double.
int oracle_dense_solve(long N, const double *A_in, double sigma, const double *b_in,
                       double *x_out) {
    typedef std::complex<long double> cl;
    std::vector<cl> M(N * (N + 1));
    const cd *A = reinterpret_cast<const cd *>(A_in);
    const cd *b = reinterpret_cast<const cd *>(b_in);
    for (long i = 0; i < N; ++i) {
        for (long j = 0; j < N; ++j) M[i * (N + 1) + j] = cl(A[i * N + j].real(), A[i * N + j].imag());
        M[i * (N + 1) + i] += cl(sigma, 0.0L);
        M[i * (N + 1) + N] = cl(b[i].real(), b[i].imag());
    }
    for (long c = 0; c < N; ++c) {
        long piv = c;
        long double best = std::abs(M[c * (N + 1) + c]);
        for (long i = c + 1; i < N; ++i) {
            const long double a = std::abs(M[i * (N + 1) + c]);
            if (a > best) { best = a; piv = i; }
        }
        if (best == 0.0L) return -6;
        if (piv != c)
            for (long j = c; j <= N; ++j) std::swap(M[c * (N + 1) + j], M[piv * (N + 1) + j]);
        const cl inv = cl(1.0L, 0.0L) / M[c * (N + 1) + c];
        for (long i = c + 1; i < N; ++i) {
            const cl f = M[i * (N + 1) + c] * inv;
            if (f == cl(0.0L, 0.0L)) continue;
            for (long j = c; j <= N; ++j) M[i * (N + 1) + j] -= f * M[c * (N + 1) + j];
        }
    }
    cd *x = reinterpret_cast<cd *>(x_out);
    std::vector<cl> xs(N);
    for (long i = N - 1; i >= 0; --i) {
        cl s = M[i * (N + 1) + N];
        for (long j = i + 1; j < N; ++j) s -= M[i * (N + 1) + j] * xs[j];
        xs[i] = s / M[i * (N + 1) + i];
        x[i] = cd((double)xs[i].real(), (double)xs[i].imag());
    }
    return 0;
}

}  // extern "C"
