/*
 * oci_oracle.c -- CPU fp64 ORACLE for the one-cell-inversion (OCI) iteration and the source-iteration (SI)
 * comparator of arXiv 2503.00264 (time-dependent 1-D slab multigroup S_N, simple corner balance in space,
 * multiple balance in time).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT. Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call it. It shares no code, header, table or
 * helper with paper_2503_00264_b200/ (the CUDA path) and neither includes the other.
 *
 * It is deliberately plain: dense row-major matrices, textbook Gaussian elimination with partial pivoting
 * (own code, no LAPACK/BLAS), loops in the paper's order and notation, `#pragma omp parallel for` over the
 * one axis the method itself declares parallel (cells for OCI; angle x group for SI,
 * PAPER.md:25, 638). No blocking, fusion or re-ordering. Build with -ffp-contract=off (oracle/__init__.py).
 *
 * Citations are PAPER.md:<line> (+ equation). Readings of garbled / silent passages are the ones listed in
 * SURVEY.md section 8(c) (A1..A22) and DESIGN.md "Readings of the paper".
 *
 * Pins (tests/test_oracle_*.py): brute-force global solve assembled independently from Eq. 3 (a), OCI = SI
 * fixed points (b), infinite-medium closed forms (c, c'), particle balance (d), Fourier spectral radii
 * (e, e'), numpy.linalg.solve for the Gaussian elimination, Eq. 41 occupancy for the matrix structure.
 * Parity unpinned: the ABSOLUTE spectral radii printed in Table 1 and the 0.4831 of PAPER.md:479 at the
 * stated tau -- they are not reproduced by the paper's own equations; used as trend pins only.
 *
 * Layouts (Eq. 11a-b, 40c-d): row/column index inside a cell r = (g*N + m)*4 + p with
 * p = 0:(k,L) 1:(k,R) 2:(k+1/2,L) 3:(k+1/2,R); Psi[J][n], n = 4*N*G; phi[J][G][4]; q[J][G][4];
 * psi_prev[J][G][N][2] = psi_{k-1/2} at (L,R); transfer[J][G_to][G_from]; inc_*[G][N][2] (levels k, k+1/2).
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define BC_VACUUM 0
#define BC_REFLECTIVE 1
#define BC_PRESCRIBED 2

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------------------------------------
 * Eq. 8b, PAPER.md:132 -- the 4x4 within-cell block L_{c,j,g,m} (valid for either sign of mu; it is what
 * Eq. 3a-d + closures 4a-b, 5a-b give once the upstream edge flux is moved to the right-hand side).
 * ---------------------------------------------------------------------------------------------- */
static void lc_block(double dx, double sig, double v, double dt, double mu, double Lc[4][4])
{
    double a = (fabs(mu) + dx * sig) / 2.0; /* (|mu_m| + dx_j Sigma_{j,g}) / 2 */
    double gam = dx / (v * dt);             /* dx_j / (v_g dt) */
    double h = mu / 2.0;
    Lc[0][0] = a;    Lc[0][1] = h;    Lc[0][2] = gam / 2.0; Lc[0][3] = 0.0;
    Lc[1][0] = -h;   Lc[1][1] = a;    Lc[1][2] = 0.0;       Lc[1][3] = gam / 2.0;
    Lc[2][0] = -gam; Lc[2][1] = 0.0;  Lc[2][2] = gam + a;   Lc[2][3] = h;
    Lc[3][0] = 0.0;  Lc[3][1] = -gam; Lc[3][2] = -h;        Lc[3][3] = gam + a;
}

/* ------------------------------------------------------------------------------------------------
 * Eq. 40b: A_j = [delta_{gg'} L_{c,j,g} - S_{g'->g,j}], with L_c block-diagonal in m
 * (Eq. 8a) and S from Eq. 10 / 39 read as:
 *   [S_{g'->g}]_{(m,p),(m',p')} = delta_{pp'} (dx_j Sigma_{s,g'->g,j} / 4) w_{m'}
 * i.e. the term (dx/2)(1/2) Sigma_s sum_n w_n psi_n of Eq. 3a-d.
 * sig_t[G], K[G][G] = transfer[g_to][g_from] of this cell. A is n x n row-major.
 * ---------------------------------------------------------------------------------------------- */
void orc_assemble_cell(int N, int G, double dx, const double *sig_t, const double *K, const double *v,
                       const double *mu, const double *w, double dt, double *A)
{
    int n = 4 * N * G;
    memset(A, 0, sizeof(double) * (size_t)n * n);
    for (int g = 0; g < G; ++g)
        for (int m = 0; m < N; ++m) {
            double Lc[4][4];
            lc_block(dx, sig_t[g], v[g], dt, mu[m], Lc);
            int r0 = (g * N + m) * 4;
            for (int p = 0; p < 4; ++p)
                for (int pp = 0; pp < 4; ++pp)
                    A[(size_t)(r0 + p) * n + (r0 + pp)] += Lc[p][pp];
            for (int gp = 0; gp < G; ++gp)
                for (int mp = 0; mp < N; ++mp) {
                    double s = dx * K[g * G + gp] / 4.0 * w[mp];
                    int c0 = (gp * N + mp) * 4;
                    for (int p = 0; p < 4; ++p)
                        A[(size_t)(r0 + p) * n + (c0 + p)] -= s;
                }
        }
}

/* ------------------------------------------------------------------------------------------------
 * Gaussian elimination with partial pivoting (what `_gesv` does): in place, row-major,
 * P A = L U with unit-diagonal L below the diagonal and U on/above it. piv[k] = row exchanged with row k at
 * step k (first row of maximal |entry|). Returns 0, or k+1 if the k-th pivot is zero / NaN.
 * ---------------------------------------------------------------------------------------------- */
int orc_gepp_factor(int n, double *A, int *piv)
{
    for (int k = 0; k < n; ++k) {
        int p = k;
        double best = fabs(A[(size_t)k * n + k]);
        for (int i = k + 1; i < n; ++i) {
            double a = fabs(A[(size_t)i * n + k]);
            if (a > best) { best = a; p = i; }
        }
        piv[k] = p;
        if (!(best > 0.0)) return k + 1;
        if (p != k)
            for (int c = 0; c < n; ++c) {
                double t = A[(size_t)k * n + c];
                A[(size_t)k * n + c] = A[(size_t)p * n + c];
                A[(size_t)p * n + c] = t;
            }
        double d = A[(size_t)k * n + k];
        for (int i = k + 1; i < n; ++i) {
            double l = A[(size_t)i * n + k] / d;
            A[(size_t)i * n + k] = l;
            for (int c = k + 1; c < n; ++c)
                A[(size_t)i * n + c] -= l * A[(size_t)k * n + c];
        }
    }
    return 0;
}

/* `_getrs` (Alg. 2): apply the row exchanges, forward substitution with
 * unit L, back substitution with U. b is overwritten by the solution. */
void orc_gepp_solve(int n, const double *LU, const int *piv, double *b)
{
    for (int k = 0; k < n; ++k)
        if (piv[k] != k) { double t = b[k]; b[k] = b[piv[k]]; b[piv[k]] = t; }
    for (int i = 1; i < n; ++i) {
        double s = b[i];
        for (int c = 0; c < i; ++c) s -= LU[(size_t)i * n + c] * b[c];
        b[i] = s;
    }
    for (int i = n - 1; i >= 0; --i) {
        double s = b[i];
        for (int c = i + 1; c < n; ++c) s -= LU[(size_t)i * n + c] * b[c];
        b[i] = s / LU[(size_t)i * n + i];
    }
}

/* Assemble and factor every cell (Alg. 2: the first `_gesv` leaves L+U in A).
 * LU[J][n][n], piv[J][n]. Returns 0 or the 1-based index of the first singular cell. */
int orc_factor_all(int J, int N, int G, const double *dx, const double *sigma_t, const double *transfer,
                   const double *v, const double *mu, const double *w, double dt, double *LU, int *piv)
{
    int n = 4 * N * G;
    int bad = 0;
#pragma omp parallel for schedule(static)
    for (int j = 0; j < J; ++j) {
        double *A = LU + (size_t)j * n * n;
        orc_assemble_cell(N, G, dx[j], sigma_t + (size_t)j * G, transfer + (size_t)j * G * G, v, mu, w, dt, A);
        if (orc_gepp_factor(n, A, piv + (size_t)j * n)) {
#pragma omp critical
            if (bad == 0 || j + 1 < bad) bad = j + 1;
        }
    }
    return bad;
}

/* ------------------------------------------------------------------------------------------------
 * Constant part of b_j (Alg. 2), Eq. 9c-d PAPER.md:145-150 without the incident terms:
 *   rows (k,L),(k,R):        dx_j/4 Q_{k,j,L/R} + dx_j/(2 v_g dt) psi_{m,k-1/2,j,L/R}
 *   rows (k+1/2,L),(k+1/2,R): dx_j/4 Q_{k+1/2,j,L/R}            (4th row of 9c restored)
 * ---------------------------------------------------------------------------------------------- */
void orc_const_rhs(int J, int N, int G, const double *dx, const double *v, double dt, const double *q,
                   const double *psi_prev, double *c)
{
    int n = 4 * N * G;
    for (int j = 0; j < J; ++j)
        for (int g = 0; g < G; ++g)
            for (int m = 0; m < N; ++m) {
                double *cj = c + (size_t)j * n + (size_t)(g * N + m) * 4;
                const double *qj = q + ((size_t)j * G + g) * 4;
                const double *pp = psi_prev + (((size_t)j * G + g) * N + m) * 2;
                double half_gam = dx[j] / (2.0 * v[g] * dt);
                cj[0] = dx[j] / 4.0 * qj[0] + half_gam * pp[0];
                cj[1] = dx[j] / 4.0 * qj[1] + half_gam * pp[1];
                cj[2] = dx[j] / 4.0 * qj[2];
                cj[3] = dx[j] / 4.0 * qj[3];
            }
}

/* Incident angular flux on cell j for ordinate (g,m) at time level lev (0: k, 1: k+1/2), taken from the
 * iterate Psi_src of the PREVIOUS iteration ("prior iteration values are employed for all
 * information incident on cell j"); upstream closure Eq. 5a-b. Boundary cells use the
 * boundary condition; reflective ends use the mirror ordinate N-1-m of the same cell,
 * also from the previous iteration. */
static double incident(int J, int N, int G, int bc_left, int bc_right, const double *inc_left,
                       const double *inc_right, const double *Psi_src, int j, int g, int m, int lev, double mu_m)
{
    int n = 4 * N * G;
    if (mu_m > 0.0) {
        if (j > 0) return Psi_src[(size_t)(j - 1) * n + (size_t)(g * N + m) * 4 + 2 * lev + 1]; /* (j-1,R) */
        if (bc_left == BC_REFLECTIVE) return Psi_src[(size_t)(g * N + (N - 1 - m)) * 4 + 2 * lev + 0];
        if (bc_left == BC_PRESCRIBED) return inc_left[((size_t)g * N + m) * 2 + lev];
        return 0.0;
    } else {
        if (j < J - 1) return Psi_src[(size_t)(j + 1) * n + (size_t)(g * N + m) * 4 + 2 * lev + 0]; /* (j+1,L) */
        if (bc_right == BC_REFLECTIVE)
            return Psi_src[(size_t)(J - 1) * n + (size_t)(g * N + (N - 1 - m)) * 4 + 2 * lev + 1];
        if (bc_right == BC_PRESCRIBED) return inc_right[((size_t)g * N + m) * 2 + lev];
        return 0.0;
    }
}

/* ------------------------------------------------------------------------------------------------
 * One OCI (cell-wise block-Jacobi) iteration, Eq. 7, Alg. 2 PAPER.md:427-436:
 *   b_j = c_j + incident(Psi^(l))   (Eq. 9c: rows (k,L),(k+1/2,L) get +mu psi_{j-1,R} for mu>0;
 *                                    Eq. 9d: rows (k,R),(k+1/2,R) get -mu psi_{j+1,L} for mu<0)
 *   Psi_j^(l+1) = A_j^{-1} b_j      (stored LU, `_getrs`)
 * Only psi_old is read (Jacobi). psi_new must not alias psi_old.
 * ---------------------------------------------------------------------------------------------- */
void orc_oci_iterate(int J, int N, int G, const double *mu, int bc_left, int bc_right, const double *inc_left,
                     const double *inc_right, const double *LU, const int *piv, const double *c,
                     const double *psi_old, double *psi_new)
{
    int n = 4 * N * G;
#pragma omp parallel for schedule(static)
    for (int j = 0; j < J; ++j) {
        double *b = psi_new + (size_t)j * n;
        memcpy(b, c + (size_t)j * n, sizeof(double) * n);
        for (int g = 0; g < G; ++g)
            for (int m = 0; m < N; ++m) {
                int r0 = (g * N + m) * 4;
                for (int lev = 0; lev < 2; ++lev) {
                    double in = incident(J, N, G, bc_left, bc_right, inc_left, inc_right, psi_old, j, g, m, lev, mu[m]);
                    if (mu[m] > 0.0) b[r0 + 2 * lev + 0] += mu[m] * in;  /* L rows */
                    else             b[r0 + 2 * lev + 1] += -mu[m] * in; /* R rows */
                }
            }
        orc_gepp_solve(n, LU + (size_t)j * n * n, piv + (size_t)j * n, b);
    }
}

/* ------------------------------------------------------------------------------------------------
 * Red-black ordering of the same cell solves (block Gauss-Seidel variant the paper names, PAPER.md:29, 550;
 * SURVEY 8f row f4): first every even cell, then every odd cell, each from the CURRENT values of its two
 * neighbours (which have the other colour), in place. Within one colour the cells are independent. A
 * reflective end reads the mirror ordinate of the same cell before that cell is overwritten, i.e. its
 * value from the previous iteration, as in orc_oci_iterate. scratch: n doubles per thread.
 * ---------------------------------------------------------------------------------------------- */
void orc_oci_iterate_redblack(int J, int N, int G, const double *mu, int bc_left, int bc_right,
                              const double *inc_left, const double *inc_right, const double *LU, const int *piv,
                              const double *c, double *psi)
{
    int n = 4 * N * G;
    for (int colour = 0; colour < 2; ++colour) {
#pragma omp parallel
        {
            double *b = (double *)malloc(sizeof(double) * n);
#pragma omp for schedule(static)
            for (int j = colour; j < J; j += 2) {
                memcpy(b, c + (size_t)j * n, sizeof(double) * n);
                for (int g = 0; g < G; ++g)
                    for (int m = 0; m < N; ++m) {
                        int r0 = (g * N + m) * 4;
                        for (int lev = 0; lev < 2; ++lev) {
                            double in = incident(J, N, G, bc_left, bc_right, inc_left, inc_right, psi, j, g, m, lev, mu[m]);
                            if (mu[m] > 0.0) b[r0 + 2 * lev + 0] += mu[m] * in;  /* L rows */
                            else             b[r0 + 2 * lev + 1] += -mu[m] * in; /* R rows */
                        }
                    }
                orc_gepp_solve(n, LU + (size_t)j * n * n, piv + (size_t)j * n, b);
                memcpy(psi + (size_t)j * n, b, sizeof(double) * n);
            }
            free(b);
        }
    }
}

/* Eq. 44: phi_{g,j,p} = sum_n w_n psi_{n,g,j,p}. */
void orc_scalar_flux(int J, int N, int G, const double *w, const double *psi, double *phi)
{
    for (int j = 0; j < J; ++j)
        for (int g = 0; g < G; ++g)
            for (int p = 0; p < 4; ++p) {
                double s = 0.0;
                for (int m = 0; m < N; ++m) s += w[m] * psi[((size_t)j * G * N + (size_t)g * N + m) * 4 + p];
                phi[((size_t)j * G + g) * 4 + p] = s;
            }
}

double orc_max_abs_diff(long len, const double *a, const double *b)
{
    double r = 0.0;
    for (long i = 0; i < len; ++i) { double d = fabs(a[i] - b[i]); if (d > r || d != d) r = d; }
    return r;
}

double orc_l2_diff(long len, const double *a, const double *b)
{
    double s = 0.0;
    for (long i = 0; i < len; ++i) { double d = a[i] - b[i]; s += d * d; }
    return sqrt(s);
}

/* ------------------------------------------------------------------------------------------------
 * One source iteration, Appendix A: for every group g and ordinate m (parallel, "Jacobi" in
 * groups) sweep the cells in the direction of mu_m, solving the 4x4 system Eq. 42 with L_{c,j,g,m} of Eq. 8b
 * and d of Eq. 43b-c, where the scattering (+fission) source is lagged:
 *   s_{j,g,p} = sum_{g'} transfer_j[g][g'] phi^(l)_{j,g',p}     (all groups from iteration l)
 * and the upstream flux is the one just computed in THIS sweep (l+1/2). Reflective ends take the mirror
 * ordinate from iteration l (psi_old), because both directions are swept in unison.
 * Then phi^(l+1) by Eq. 44.
 * ---------------------------------------------------------------------------------------------- */
void orc_si_iterate(int J, int N, int G, const double *dx, const double *sigma_t, const double *transfer,
                    const double *v, const double *mu, const double *w, double dt, int bc_left, int bc_right,
                    const double *inc_left, const double *inc_right, const double *q, const double *psi_prev,
                    const double *phi_old, const double *psi_old, double *psi_new, double *phi_new)
{
    int n = 4 * N * G;
#pragma omp parallel for schedule(static)
    for (int gm = 0; gm < G * N; ++gm) {
        int g = gm / N, m = gm % N;
        int fwd = mu[m] > 0.0;
        double in[2];
        for (int lev = 0; lev < 2; ++lev) {
            if (fwd) {
                in[lev] = bc_left == BC_REFLECTIVE ? psi_old[(size_t)(g * N + (N - 1 - m)) * 4 + 2 * lev + 0]
                        : bc_left == BC_PRESCRIBED ? inc_left[((size_t)g * N + m) * 2 + lev] : 0.0;
            } else {
                in[lev] = bc_right == BC_REFLECTIVE
                              ? psi_old[(size_t)(J - 1) * n + (size_t)(g * N + (N - 1 - m)) * 4 + 2 * lev + 1]
                        : bc_right == BC_PRESCRIBED ? inc_right[((size_t)g * N + m) * 2 + lev] : 0.0;
            }
        }
        for (int jj = 0; jj < J; ++jj) {
            int j = fwd ? jj : J - 1 - jj;
            double Lc[4][4], A[16], d[4];
            int piv[4];
            lc_block(dx[j], sigma_t[(size_t)j * G + g], v[g], dt, mu[m], Lc);
            for (int p = 0; p < 4; ++p)
                for (int pp = 0; pp < 4; ++pp) A[p * 4 + pp] = Lc[p][pp];
            const double *Kj = transfer + (size_t)j * G * G + (size_t)g * G;
            const double *pp_ = psi_prev + (((size_t)j * G + g) * N + m) * 2;
            double half_gam = dx[j] / (2.0 * v[g] * dt);
            for (int p = 0; p < 4; ++p) {
                double s = 0.0;
                for (int gp = 0; gp < G; ++gp) s += Kj[gp] * phi_old[((size_t)j * G + gp) * 4 + p];
                d[p] = dx[j] / 4.0 * (s + q[((size_t)j * G + g) * 4 + p]);
            }
            d[0] += half_gam * pp_[0];
            d[1] += half_gam * pp_[1];
            if (fwd) { d[0] += mu[m] * in[0];  d[2] += mu[m] * in[1]; }
            else     { d[1] += -mu[m] * in[0]; d[3] += -mu[m] * in[1]; }
            orc_gepp_factor(4, A, piv);
            orc_gepp_solve(4, A, piv, d);
            double *out = psi_new + (size_t)j * n + (size_t)(g * N + m) * 4;
            for (int p = 0; p < 4; ++p) out[p] = d[p];
            if (fwd) { in[0] = d[1]; in[1] = d[3]; } /* outgoing (j,R) at k and k+1/2, Eq. 5a-b */
            else     { in[0] = d[0]; in[1] = d[2]; } /* outgoing (j,L) */
        }
    }
    orc_scalar_flux(J, N, G, w, psi_new, phi_new);
}

/* ------------------------------------------------------------------------------------------------
 * Convergence loops of one time step (Alg. 2 PAPER.md:417-453 and Alg. 1).
 * rule 0: stop when max_{j,g,p} |phi^(l+1) - phi^(l)| < tol (BASELINE.json configs).
 * rule 1: the paper's Eq. 12-13 PAPER.md:166-171 (OCI: L2 norm of Psi^(l+1) - Psi^(l); SI: Eq. 46 with phi):
 *         e < tol (1 - rho_e), rho_e = e_l / e_{l-1}, tested from the second iteration on (Alg. 2 computes e
 *         only in the else-branch).
 * psi, phi: in = iterate (l = 0), out = converged iterate. work: 1 x J*n (OCI), J*n + J*G*4 (SI) doubles.
 * resid[max_iters] receives the tested quantity of every iteration. Returns the number of iterations done
 * (== max_iters if not converged).
 * ---------------------------------------------------------------------------------------------- */
int orc_oci_converge(int J, int N, int G, const double *mu, const double *w, int bc_left, int bc_right,
                     const double *inc_left, const double *inc_right, const double *LU, const int *piv,
                     const double *c, double tol, int max_iters, int rule, double *psi, double *phi,
                     double *work, double *resid)
{
    int n = 4 * N * G;
    size_t len = (size_t)J * n;
    double *psi_new = work;
    double *phi_new = (double *)malloc(sizeof(double) * (size_t)J * G * 4);
    double e_prev = 0.0;
    int it = 0;
    while (it < max_iters) {
        orc_oci_iterate(J, N, G, mu, bc_left, bc_right, inc_left, inc_right, LU, piv, c, psi, psi_new);
        orc_scalar_flux(J, N, G, w, psi_new, phi_new);
        int done;
        double e;
        if (rule == 0) {
            e = orc_max_abs_diff((long)J * G * 4, phi_new, phi);
            done = e < tol;
        } else {
            e = orc_l2_diff((long)len, psi_new, psi);
            done = it >= 1 && e < tol * (1.0 - e / e_prev);
            e_prev = e;
        }
        memcpy(psi, psi_new, sizeof(double) * len);
        memcpy(phi, phi_new, sizeof(double) * (size_t)J * G * 4);
        resid[it++] = e;
        if (done) break;
    }
    free(phi_new);
    return it;
}

/* As orc_oci_converge with the red-black ordering of the cell solves (one iteration = both colours). */
int orc_oci_converge_redblack(int J, int N, int G, const double *mu, const double *w, int bc_left, int bc_right,
                              const double *inc_left, const double *inc_right, const double *LU, const int *piv,
                              const double *c, double tol, int max_iters, int rule, double *psi, double *phi,
                              double *work, double *resid)
{
    int n = 4 * N * G;
    size_t len = (size_t)J * n;
    double *psi_old = work;
    double *phi_new = (double *)malloc(sizeof(double) * (size_t)J * G * 4);
    double e_prev = 0.0;
    int it = 0;
    while (it < max_iters) {
        memcpy(psi_old, psi, sizeof(double) * len);
        orc_oci_iterate_redblack(J, N, G, mu, bc_left, bc_right, inc_left, inc_right, LU, piv, c, psi);
        orc_scalar_flux(J, N, G, w, psi, phi_new);
        int done;
        double e;
        if (rule == 0) {
            e = orc_max_abs_diff((long)J * G * 4, phi_new, phi);
            done = e < tol;
        } else {
            e = orc_l2_diff((long)len, psi, psi_old);
            done = it >= 1 && e < tol * (1.0 - e / e_prev);
            e_prev = e;
        }
        memcpy(phi, phi_new, sizeof(double) * (size_t)J * G * 4);
        resid[it++] = e;
        if (done) break;
    }
    free(phi_new);
    return it;
}

int orc_si_converge(int J, int N, int G, const double *dx, const double *sigma_t, const double *transfer,
                    const double *v, const double *mu, const double *w, double dt, int bc_left, int bc_right,
                    const double *inc_left, const double *inc_right, const double *q, const double *psi_prev,
                    double tol, int max_iters, int rule, double *psi, double *phi, double *work, double *resid)
{
    int n = 4 * N * G;
    size_t len = (size_t)J * n, lphi = (size_t)J * G * 4;
    double *psi_new = work, *phi_new = work + len;
    double e_prev = 0.0;
    int it = 0;
    while (it < max_iters) {
        orc_si_iterate(J, N, G, dx, sigma_t, transfer, v, mu, w, dt, bc_left, bc_right, inc_left, inc_right, q,
                       psi_prev, phi, psi, psi_new, phi_new);
        int done;
        double e;
        if (rule == 0) {
            e = orc_max_abs_diff((long)lphi, phi_new, phi);
            done = e < tol;
        } else {
            e = orc_l2_diff((long)lphi, phi_new, phi);
            done = it >= 1 && e < tol * (1.0 - e / e_prev);
            e_prev = e;
        }
        memcpy(psi, psi_new, sizeof(double) * len);
        memcpy(phi, phi_new, sizeof(double) * lphi);
        resid[it++] = e;
        if (done) break;
    }
    return it;
}
