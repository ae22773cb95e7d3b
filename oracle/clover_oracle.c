/*
 * oracle/clover_oracle.c  --  TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU statement of what the hot path of arXiv:1405.4524 computes:
 * the quenched Wilson-clover matrix D (the paper's "lattice fermion matrix computed in the
 * background of the gauge fields", sec. VII), its inverse applied to random
 * sources ("X is the solution vector and eta is the random source vector", PAPER.md L303,
 * eq. 7.3 at L300) with "clover fermions with tree-level improved clover coefficient"
 * (sec. VIII).  The paper never writes D down; the definition used here is the
 * textbook one fixed in SURVEY.md sec. 8(c) O1-O6 and listed as readings R1-R14 in DESIGN.md.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may load this file.  It shares no code, header, table or layout with the CUDA path under
 * paper_1405_4524_b200/csrc/.  No even-odd split, no spin projection, no 6x6 blocks, no
 * reordering: full 4x4 spin algebra, full 12x12 clover matrix, full-lattice operator.
 *
 * Canonical layouts (all complex numbers are (re,im) pairs of doubles, C order):
 *   links   U[mu][t][z][y][x][row][col]      U_mu(x) sits at x and points x -> x+mu
 *   spinor  psi[t][z][y][x][spin][colour]
 *   clover  A[t][z][y][x][12][12]            row/col index = 3*spin + colour
 *   Fhat    F[plane][t][z][y][x][3][3]       planes (mu,nu): 01 02 03 12 13 23
 * Directions mu = 0,1,2,3 = x,y,z,t; dims = {X,Y,Z,T}; bc[mu] = +1 or -1.
 *
 * Pins (tests/test_oracle_*.py): free-field closed form, gamma5-hermiticity, gauge
 * covariance, 2^4 dense inverse + estimator variance, abelian closed form of Fhat, tree-level
 * improvement inequality, block structure of A, SplitMix64 published vectors.
 * The BiCGStab *trajectory* (iteration count) is "parity unpinned" by design: only its
 * solution and true residual are pinned (against the dense inverse and the closed form).
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef double complex cplx;

/* ---- O1: gamma basis (Hermitian, Euclidean, chiral).  SURVEY 8(c) O1 / DESIGN R1 -------- */
static const cplx GAMMA[4][4][4] = {
    /* gamma_x */ {{0, 0, 0, -I}, {0, 0, -I, 0}, {0, I, 0, 0}, {I, 0, 0, 0}},
    /* gamma_y */ {{0, 0, 0, -1}, {0, 0, 1, 0}, {0, 1, 0, 0}, {-1, 0, 0, 0}},
    /* gamma_z */ {{0, 0, -I, 0}, {0, 0, 0, I}, {I, 0, 0, 0}, {0, -I, 0, 0}},
    /* gamma_t */ {{0, 0, 1, 0}, {0, 0, 0, 1}, {1, 0, 0, 0}, {0, 1, 0, 0}}};

/* sigma_{mu nu} = (i/2) [gamma_mu, gamma_nu] */
static void sigma_munu(int mu, int nu, cplx s[4][4])
{
    for (int a = 0; a < 4; a++)
        for (int b = 0; b < 4; b++) {
            cplx c = 0;
            for (int k = 0; k < 4; k++)
                c += GAMMA[mu][a][k] * GAMMA[nu][k][b] - GAMMA[nu][a][k] * GAMMA[mu][k][b];
            s[a][b] = 0.5 * I * c;
        }
}

/* ---- lattice geometry ------------------------------------------------------------------ */
static long volume(const int d[4]) { return (long)d[0] * d[1] * d[2] * d[3]; }

static long site_index(const int d[4], const int x[4])
{
    return (((long)x[3] * d[2] + x[2]) * d[1] + x[1]) * d[0] + x[0];
}

static void site_coords(const int d[4], long s, int x[4])
{
    x[0] = (int)(s % d[0]); s /= d[0];
    x[1] = (int)(s % d[1]); s /= d[1];
    x[2] = (int)(s % d[2]); s /= d[2];
    x[3] = (int)s;
}

/* index of the site x + step*mu_hat (step = +1 or -1), periodic wrap */
static long neighbour(const int d[4], const int x[4], int mu, int step)
{
    int y[4] = {x[0], x[1], x[2], x[3]};
    y[mu] = (x[mu] + step + d[mu]) % d[mu];
    return site_index(d, y);
}

static const cplx *link_at(const cplx *U, long V, int mu, long s) { return U + ((long)mu * V + s) * 9; }

/* ---- O2: hopping term -------------------------------------------------------------------
 * (H psi)(x) = sum_mu [ f_mu(x) (1 - gamma_mu) U_mu(x) psi(x+mu)
 *                     + g_mu(x) (1 + gamma_mu) U_mu(x-mu)^dagger psi(x-mu) ]
 * f_mu(x) = bc[mu] if x_mu = N_mu - 1 else 1;  g_mu(x) = bc[mu] if x_mu = 0 else 1.
 * SURVEY 8(c) O2 / DESIGN R1, R5.                                                         */
void oracle_hop(const double *U_, const int dims[4], const int bc[4], const double *in_, double *out_)
{
    const cplx *U = (const cplx *)U_, *in = (const cplx *)in_;
    cplx *out = (cplx *)out_;
    const long V = volume(dims);
#pragma omp parallel for schedule(static)
    for (long s = 0; s < V; s++) {
        int x[4];
        site_coords(dims, s, x);
        cplx acc[4][3];
        memset(acc, 0, sizeof acc);
        for (int mu = 0; mu < 4; mu++) {
            cplx chi[4][3];
            /* forward: (1 - gamma_mu) U_mu(x) psi(x+mu) */
            long sp = neighbour(dims, x, mu, +1);
            const cplx *u = link_at(U, V, mu, s);
            double f = (x[mu] == dims[mu] - 1) ? (double)bc[mu] : 1.0;
            for (int sp_ = 0; sp_ < 4; sp_++)
                for (int a = 0; a < 3; a++) {
                    cplx c = 0;
                    for (int b = 0; b < 3; b++) c += u[a * 3 + b] * in[(sp * 4 + sp_) * 3 + b];
                    chi[sp_][a] = c;
                }
            for (int a4 = 0; a4 < 4; a4++)
                for (int a = 0; a < 3; a++) {
                    cplx g = 0;
                    for (int b4 = 0; b4 < 4; b4++) g += GAMMA[mu][a4][b4] * chi[b4][a];
                    acc[a4][a] += f * (chi[a4][a] - g);
                }
            /* backward: (1 + gamma_mu) U_mu(x-mu)^dagger psi(x-mu) */
            long sm = neighbour(dims, x, mu, -1);
            u = link_at(U, V, mu, sm);
            double g_ = (x[mu] == 0) ? (double)bc[mu] : 1.0;
            for (int sp_ = 0; sp_ < 4; sp_++)
                for (int a = 0; a < 3; a++) {
                    cplx c = 0;
                    for (int b = 0; b < 3; b++) c += conj(u[b * 3 + a]) * in[(sm * 4 + sp_) * 3 + b];
                    chi[sp_][a] = c;
                }
            for (int a4 = 0; a4 < 4; a4++)
                for (int a = 0; a < 3; a++) {
                    cplx g = 0;
                    for (int b4 = 0; b4 < 4; b4++) g += GAMMA[mu][a4][b4] * chi[b4][a];
                    acc[a4][a] += g_ * (chi[a4][a] + g);
                }
        }
        for (int a4 = 0; a4 < 4; a4++)
            for (int a = 0; a < 3; a++) out[(s * 4 + a4) * 3 + a] = acc[a4][a];
    }
}

/* ---- O3: clover term --------------------------------------------------------------------
 * A path is a list of signed steps starting at x.  A forward step along mu multiplies by
 * U_mu(y) and moves y -> y+mu; a backward step multiplies by U_mu(y-mu)^dagger and moves
 * y -> y-mu.  The four leaves of the plane (mu,nu) all start and end at x and wind in the
 * same (mu -> nu) sense:
 *   L1 = (+mu,+nu,-mu,-nu)  L2 = (+nu,-mu,-nu,+mu)  L3 = (-mu,-nu,+mu,+nu)  L4 = (-nu,+mu,+nu,-mu)
 * Q = L1+L2+L3+L4,  Fhat = (Q - Q^dagger)/8  (anti-Hermitian, trace kept; DESIGN R2, R3).
 * Leaves use the raw links: each closed leaf crosses a boundary an even number of times.   */
static void mat_mul(const cplx a[9], const cplx b[9], cplx c[9])
{
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) {
            cplx s = 0;
            for (int k = 0; k < 3; k++) s += a[i * 3 + k] * b[k * 3 + j];
            c[i * 3 + j] = s;
        }
}

static void path_product(const cplx *U, const int dims[4], const int x0[4], int nsteps,
                         const int dir[], const int sgn[], cplx out[9])
{
    const long V = volume(dims);
    int y[4] = {x0[0], x0[1], x0[2], x0[3]};
    cplx acc[9] = {1, 0, 0, 0, 1, 0, 0, 0, 1}, tmp[9], m[9];
    for (int k = 0; k < nsteps; k++) {
        int mu = dir[k];
        if (sgn[k] > 0) {
            const cplx *u = link_at(U, V, mu, site_index(dims, y));
            for (int i = 0; i < 9; i++) m[i] = u[i];
            y[mu] = (y[mu] + 1) % dims[mu];
        } else {
            y[mu] = (y[mu] - 1 + dims[mu]) % dims[mu];
            const cplx *u = link_at(U, V, mu, site_index(dims, y));
            for (int i = 0; i < 3; i++)
                for (int j = 0; j < 3; j++) m[i * 3 + j] = conj(u[j * 3 + i]);
        }
        mat_mul(acc, m, tmp);
        for (int i = 0; i < 9; i++) acc[i] = tmp[i];
    }
    for (int i = 0; i < 9; i++) out[i] = acc[i];
}

static const int PLANE_MU[6] = {0, 0, 0, 1, 1, 2};
static const int PLANE_NU[6] = {1, 2, 3, 2, 3, 3};

static void fhat_site(const cplx *U, const int dims[4], const int x[4], int mu, int nu, cplx F[9])
{
    const int d1[4] = {mu, nu, mu, nu}, s1[4] = {+1, +1, -1, -1};
    const int d2[4] = {nu, mu, nu, mu}, s2[4] = {+1, -1, -1, +1};
    const int d3[4] = {mu, nu, mu, nu}, s3[4] = {-1, -1, +1, +1};
    const int d4[4] = {nu, mu, nu, mu}, s4[4] = {-1, +1, +1, -1};
    cplx Q[9] = {0}, L[9];
    path_product(U, dims, x, 4, d1, s1, L); for (int i = 0; i < 9; i++) Q[i] += L[i];
    path_product(U, dims, x, 4, d2, s2, L); for (int i = 0; i < 9; i++) Q[i] += L[i];
    path_product(U, dims, x, 4, d3, s3, L); for (int i = 0; i < 9; i++) Q[i] += L[i];
    path_product(U, dims, x, 4, d4, s4, L); for (int i = 0; i < 9; i++) Q[i] += L[i];
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) F[i * 3 + j] = (Q[i * 3 + j] - conj(Q[j * 3 + i])) / 8.0;
}

/* F[plane][site][3][3] */
void oracle_fhat(const double *U_, const int dims[4], double *F_)
{
    const cplx *U = (const cplx *)U_;
    cplx *F = (cplx *)F_;
    const long V = volume(dims);
#pragma omp parallel for schedule(static)
    for (long s = 0; s < V; s++) {
        int x[4];
        site_coords(dims, s, x);
        for (int pl = 0; pl < 6; pl++) fhat_site(U, dims, x, PLANE_MU[pl], PLANE_NU[pl], F + ((long)pl * V + s) * 9);
    }
}

/* A(x) = 1 + i c_sw kappa sum_{mu<nu} sigma_{mu nu} (x) Fhat_{mu nu}(x),  12x12, index 3*spin+colour */
void oracle_clover_matrix(const double *U_, const int dims[4], double kappa, double csw, double *A_)
{
    const cplx *U = (const cplx *)U_;
    cplx *A = (cplx *)A_;
    const long V = volume(dims);
    cplx sig[6][4][4];
    for (int pl = 0; pl < 6; pl++) sigma_munu(PLANE_MU[pl], PLANE_NU[pl], sig[pl]);
#pragma omp parallel for schedule(static)
    for (long s = 0; s < V; s++) {
        int x[4];
        site_coords(dims, s, x);
        cplx *a = A + s * 144;
        for (int i = 0; i < 144; i++) a[i] = 0;
        for (int i = 0; i < 12; i++) a[i * 12 + i] = 1;
        for (int pl = 0; pl < 6; pl++) {
            cplx F[9];
            fhat_site(U, dims, x, PLANE_MU[pl], PLANE_NU[pl], F);
            for (int s1 = 0; s1 < 4; s1++)
                for (int s2 = 0; s2 < 4; s2++)
                    for (int c1 = 0; c1 < 3; c1++)
                        for (int c2 = 0; c2 < 3; c2++)
                            a[(3 * s1 + c1) * 12 + 3 * s2 + c2] += I * csw * kappa * sig[pl][s1][s2] * F[c1 * 3 + c2];
        }
    }
}

/* out(x) = M(x) in(x), M a field of 12x12 matrices */
void oracle_site_matvec(const double *M_, long V, const double *in_, double *out_)
{
    const cplx *M = (const cplx *)M_, *in = (const cplx *)in_;
    cplx *out = (cplx *)out_;
#pragma omp parallel for schedule(static)
    for (long s = 0; s < V; s++)
        for (int i = 0; i < 12; i++) {
            cplx c = 0;
            for (int j = 0; j < 12; j++) c += M[s * 144 + i * 12 + j] * in[s * 12 + j];
            out[s * 12 + i] = c;
        }
}

/* Gauss-Jordan inverse with partial pivoting of an n x n complex matrix (row major).
 * Returns 0 on success, 1 if a pivot vanishes.  M is destroyed. */
static int gauss_jordan(cplx *M, int n, cplx *Minv)
{
    for (int i = 0; i < n; i++)
        for (int j = 0; j < n; j++) Minv[(long)i * n + j] = (i == j);
    for (int col = 0; col < n; col++) {
        int piv = col;
        double best = cabs(M[(long)col * n + col]);
        for (int r = col + 1; r < n; r++)
            if (cabs(M[(long)r * n + col]) > best) { best = cabs(M[(long)r * n + col]); piv = r; }
        if (best == 0.0) return 1;
        if (piv != col)
            for (int j = 0; j < n; j++) {
                cplx t = M[(long)col * n + j]; M[(long)col * n + j] = M[(long)piv * n + j]; M[(long)piv * n + j] = t;
                t = Minv[(long)col * n + j]; Minv[(long)col * n + j] = Minv[(long)piv * n + j]; Minv[(long)piv * n + j] = t;
            }
        cplx d = 1.0 / M[(long)col * n + col];
        for (int j = 0; j < n; j++) { M[(long)col * n + j] *= d; Minv[(long)col * n + j] *= d; }
        for (int r = 0; r < n; r++) {
            if (r == col) continue;
            cplx f = M[(long)r * n + col];
            if (f == 0) continue;
            for (int j = 0; j < n; j++) {
                M[(long)r * n + j] -= f * M[(long)col * n + j];
                Minv[(long)r * n + j] -= f * Minv[(long)col * n + j];
            }
        }
    }
    return 0;
}

int oracle_dense_inverse(const double *M_, int n, double *Minv_)
{
    cplx *W = (cplx *)malloc(sizeof(cplx) * (size_t)n * n);
    memcpy(W, M_, sizeof(cplx) * (size_t)n * n);
    int rc = gauss_jordan(W, n, (cplx *)Minv_);
    free(W);
    return rc;
}

/* Ainv(x) = A(x)^{-1}, site by site (12x12 Gauss-Jordan). Returns number of singular sites. */
int oracle_clover_inverse(const double *A_, long V, double *Ainv_)
{
    int bad = 0;
#pragma omp parallel for schedule(static) reduction(+ : bad)
    for (long s = 0; s < V; s++) {
        cplx W[144];
        memcpy(W, (const cplx *)A_ + s * 144, sizeof W);
        bad += gauss_jordan(W, 12, (cplx *)Ainv_ + s * 144);
    }
    return bad;
}

/* ---- O4: D = A - kappa H  (kappa normalisation; DESIGN R4) ------------------------------- */
void oracle_D(const double *U, const double *A, const int dims[4], const int bc[4], double kappa,
              const double *in, double *out)
{
    const long V = volume(dims), n = V * 12;
    double *h = (double *)malloc(sizeof(double) * 2 * n);
    oracle_hop(U, dims, bc, in, h);
    oracle_site_matvec(A, V, in, out);
#pragma omp parallel for schedule(static)
    for (long i = 0; i < 2 * n; i++) out[i] -= kappa * h[i];
    free(h);
}

/* dense matrix of D, built column by column: M[i][j] = (D e_j)_i, n = 12 V */
void oracle_dense_D(const double *U, const double *A, const int dims[4], const int bc[4], double kappa, double *M_)
{
    const long n = volume(dims) * 12;
    cplx *M = (cplx *)M_;
    cplx *e = (cplx *)calloc((size_t)n, sizeof(cplx)), *col = (cplx *)malloc(sizeof(cplx) * (size_t)n);
    for (long j = 0; j < n; j++) {
        e[j] = 1;
        oracle_D(U, A, dims, bc, kappa, (double *)e, (double *)col);
        e[j] = 0;
        for (long i = 0; i < n; i++) M[i * n + j] = col[i];
    }
    free(e);
    free(col);
}

/* ---- O6: textbook BiCGStab on D psi = eta, fp64, psi0 = 0, r~ = r0 = eta -----------------
 * <a,b> = sum conj(a) b.  Returns 0 converged, 1 max_iter, 2 repeated breakdown.
 * Breakdown (<r~,v> or rho numerically zero, e.g. a point source on unit links) restarts the
 * recurrence with r~ = p = r (SURVEY 8(c) O6 / DESIGN R11); psi and r are kept.
 * iters_out = number of iterations, resid_out = recomputed true ||eta - D psi|| / ||eta||. */
static cplx cdot(const cplx *a, const cplx *b, long n)
{
    double re = 0, im = 0;
#pragma omp parallel for schedule(static) reduction(+ : re, im)
    for (long i = 0; i < n; i++) {
        cplx c = conj(a[i]) * b[i];
        re += creal(c);
        im += cimag(c);
    }
    return re + I * im;
}

int oracle_bicgstab(const double *U, const double *A, const int dims[4], const int bc[4], double kappa,
                    const double *eta_, double *psi_, double tol, int max_iter, int *iters_out, double *resid_out)
{
    const long n = volume(dims) * 12;
    const cplx *eta = (const cplx *)eta_;
    cplx *psi = (cplx *)psi_;
    cplx *r = malloc(sizeof(cplx) * n), *rt = malloc(sizeof(cplx) * n), *p = malloc(sizeof(cplx) * n);
    cplx *v = malloc(sizeof(cplx) * n), *s = malloc(sizeof(cplx) * n), *t = malloc(sizeof(cplx) * n);
    int status = 1, it = 0, restart = 0, nrestart = 0;
    const double BREAKDOWN = 1e-14; /* |<r~,v>| or |rho| below this fraction of the Cauchy-Schwarz bound */
    const double eta_norm = sqrt(creal(cdot(eta, eta, n)));
    for (long i = 0; i < n; i++) { psi[i] = 0; r[i] = rt[i] = p[i] = eta[i]; }
    cplx rho = cdot(rt, r, n);
    if (eta_norm == 0.0) { status = 0; goto done; }
    for (it = 1; it <= max_iter; it++) {
        if (restart) { /* breakdown: restart the recurrence from the current residual, r~ = p = r */
            for (long i = 0; i < n; i++) rt[i] = p[i] = r[i];
            rho = cdot(rt, r, n);
            restart = 0;
            nrestart++;
            if (nrestart > 20) { status = 2; break; }
        }
        oracle_D(U, A, dims, bc, kappa, (double *)p, (double *)v);
        cplx rtv = cdot(rt, v, n);
        const double rtn = sqrt(creal(cdot(rt, rt, n)));
        if (!(cabs(rtv) > BREAKDOWN * rtn * sqrt(creal(cdot(v, v, n))))) { restart = 1; continue; }
        cplx alpha = rho / rtv;
        for (long i = 0; i < n; i++) s[i] = r[i] - alpha * v[i];
        oracle_D(U, A, dims, bc, kappa, (double *)s, (double *)t);
        double tt = creal(cdot(t, t, n));
        if (!(tt > 0.0)) { /* s = 0: exact solution reached */
            for (long i = 0; i < n; i++) { psi[i] += alpha * p[i]; r[i] = s[i]; }
            status = 0; break;
        }
        cplx omega = cdot(t, s, n) / tt;
        for (long i = 0; i < n; i++) { psi[i] += alpha * p[i] + omega * s[i]; r[i] = s[i] - omega * t[i]; }
        const double rn = sqrt(creal(cdot(r, r, n)));
        if (rn / eta_norm < tol) { status = 0; break; }
        cplx rho1 = cdot(rt, r, n);
        if (!(cabs(omega) > 0.0) || !(cabs(rho1) > BREAKDOWN * rtn * rn)) { restart = 1; continue; }
        cplx beta = (rho1 / rho) * (alpha / omega);
        for (long i = 0; i < n; i++) p[i] = r[i] + beta * (p[i] - omega * v[i]);
        rho = rho1;
    }
    if (it > max_iter) it = max_iter;
done:
    /* true residual, recomputed from scratch */
    oracle_D(U, A, dims, bc, kappa, (double *)psi, (double *)v);
    for (long i = 0; i < n; i++) v[i] = eta[i] - v[i];
    if (resid_out) *resid_out = (eta_norm > 0) ? sqrt(creal(cdot(v, v, n))) / eta_norm : 0.0;
    if (iters_out) *iters_out = it;
    free(r); free(rt); free(p); free(v); free(s); free(t);
    return status;
}

/* ---- O5: Z4 noise (docs/NOISE.md).  eta_r(x,s,c) = scale * z4[k], k = top two bits of the
 * SplitMix64 output function at state  seed + GOLDEN*(ctr+1),  ctr = r*12V + n,
 * n = (((t*Z+z)*Y+y)*X+x)*12 + 3*s + c.  Values come from a table so zeros are +0.0.
 * Time dilution ("the ith random source is located on the timeslice t"):
 * eta_r is kept only on t == r mod T, same counters.  r = rhs_offset + local index.        */
uint64_t oracle_splitmix64(uint64_t seed, uint64_t ctr)
{
    uint64_t z = seed + 0x9E3779B97F4A7C15ULL * (ctr + 1ULL);
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}

/* dilution (bit 0 = time, bit 1 = spin-colour; docs/NOISE.md): source r lives on timeslice t_r = r mod T (time bit) and on the
 * single spin-colour component sc_r = (r / T) mod 12 (both bits) or r mod 12 (spin-colour only), sc = 3*spin + colour. */
static int oracle_noise_keep(int dilution, uint64_t r, int t, int sc, int T)
{
    if ((dilution & 1) && t != (int)(r % (uint64_t)T)) return 0;
    if (dilution & 2) {
        const uint64_t q = (dilution & 1) ? r / (uint64_t)T : r;
        if (sc != (int)(q % 12ULL)) return 0;
    }
    return 1;
}

void oracle_noise_fill(double *out, const int dims[4], uint64_t seed, int n_rhs, int rhs_offset,
                       int time_dilution, double scale)
{
    const long V = volume(dims);
    const double tab[4][2] = {{scale, 0.0}, {0.0, scale}, {-scale, 0.0}, {0.0, -scale}};
    for (int j = 0; j < n_rhs; j++) {
        const uint64_t r = (uint64_t)(rhs_offset + j);
        double *o = out + (size_t)j * V * 24;
#pragma omp parallel for schedule(static)
        for (long n = 0; n < V * 12; n++) {
            int t = (int)((n / 12) / ((long)dims[0] * dims[1] * dims[2]));
            int k = (int)(oracle_splitmix64(seed, r * 12ULL * (uint64_t)V + (uint64_t)n) >> 62);
            if (!oracle_noise_keep(time_dilution, r, t, (int)(n % 12), dims[3])) { o[2 * n] = 0.0; o[2 * n + 1] = 0.0; }
            else { o[2 * n] = tab[k][0]; o[2 * n + 1] = tab[k][1]; }
        }
    }
}

void oracle_noise_fill_f32(float *out, const int dims[4], uint64_t seed, int n_rhs, int rhs_offset,
                           int time_dilution, float scale)
{
    const long V = volume(dims);
    const float tab[4][2] = {{scale, 0.0f}, {0.0f, scale}, {-scale, 0.0f}, {0.0f, -scale}};
    for (int j = 0; j < n_rhs; j++) {
        const uint64_t r = (uint64_t)(rhs_offset + j);
        float *o = out + (size_t)j * V * 24;
#pragma omp parallel for schedule(static)
        for (long n = 0; n < V * 12; n++) {
            int t = (int)((n / 12) / ((long)dims[0] * dims[1] * dims[2]));
            int k = (int)(oracle_splitmix64(seed, r * 12ULL * (uint64_t)V + (uint64_t)n) >> 62);
            if (!oracle_noise_keep(time_dilution, r, t, (int)(n % 12), dims[3])) { o[2 * n] = 0.0f; o[2 * n + 1] = 0.0f; }
            else { o[2 * n] = tab[k][0]; o[2 * n + 1] = tab[k][1]; }
        }
    }
}
