/*
 * chefsi_next_oracle.c -- CPU ORACLE for the SURVEY.md section 8(f) "next" rows.  TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 *   NEXT-3  gradient (first-derivative) finite-difference stencil, the projector contraction chi^T X and the nonlocal
 *           Hellmann-Feynman force assembled from them
 *   NEXT-1  the N_s x N_s generalized symmetric eigenproblem  H~ Z~ = M~ Z~ D~  of the subspace step
 *           (Algorithm 1 "Subspace diagonalization", 148-154 section II.C eq. 9)
 *   NEXT-4  the complex (k-point) Hamiltonian with Bloch phases and the Hermitian subspace products
 *
 *
 * Plain, slow, obviously-correct restatements written from the paper and the readings R21-R27 of DESIGN.md section 3.
 * Same rules as chefsi_oracle.c: only tests/, smoke() and bench.py's cpu_baseline / --impl reference legs may call
 * this; it shares no code, header, table or constant with the CUDA path (and none with chefsi_oracle.c either: the
 * struct below is restated so that this file stands alone).  Sums are accumulated in acc_t = long double
 * (-DORACLE_ACC_DOUBLE: double, the timed CPU baseline).
 *
 * Pins (tests/test_oracle_next_pins.py, -m "not gpu"): exact rational first-derivative weights, odd-moment conditions,
 * the symbol sum_p 2 w_p sin(p k h) / h on plane waves, antisymmetry <x, D y> = -<D x, y>, polynomial exactness,
 * Dirichlet = restricted zero-padded periodic, dense brute-force force; residual / M-orthonormality / ordering /
 * closed forms / LAPACK eigenvalues for the eigensolver; Hermiticity, the Gamma-point limit, Bloch plane waves and a dense
 * brute-force H(k) for the complex operator.  No function here is "parity unpinned".
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifdef ORACLE_ACC_DOUBLE
typedef double acc_t;
typedef double complex cacc_t;
#else
typedef long double acc_t;
typedef long double complex cacc_t;
#endif

#define ORACLE_MAX_RADIUS 6

/* H = -1/2 Laplacian + Veff + V_nl; plain host pointers owned by the caller (oracle only). */
typedef struct {
    int32_t n[3];
    double h[3];
    int32_t bc[3];            /* 0 periodic, 1 Dirichlet (zero outside [0, n-1]) (reading R9) */
    int32_t radius;           /* n0 / 2 */
    int32_t n_atoms;
    const int64_t *supp_ptr;  /* [n_atoms+1] */
    const int32_t *supp_idx;  /* grid indices of each atom's projector support */
    const int32_t *n_proj;    /* [n_atoms] */
    const int64_t *chi_ptr;   /* [n_atoms+1] offsets into chi */
    const double *chi;        /* per atom n_J x P_J column-major */
    const double *gamma;      /* concatenated P_J per atom */
    const double *veff;       /* [Nd] */
} oracle_ham;

int oracle_next_acc_bits(void) { return (int)(8 * sizeof(acc_t)); }

static inline int nbr_coord(int c, int p, int n, int bc)
{
    int q = c + p;
    if (bc == 0) { q %= n; if (q < 0) q += n; return q; }
    return (q < 0 || q >= n) ? -1 : q;
}

/* =================================================================================================================
 * NEXT-3.  Gradient stencil, projector contraction, nonlocal force.
 * ================================================================================================================= */

/* G1.  Central finite-difference weights of the FIRST derivative, radius n (order 2n), reading R21:
 *   w_p = (-1)^{p+1} (n!)^2 / (p (n-p)! (n+p)!),  p = 1..n;  w_{-p} = -w_p;  w_0 = 0.
 * The paper names only "the application of the gradient operator on the Kohn-Sham orbitals" on the same
 * finite-difference grid of order n0: the standard central weights of that order. */
void oracle_fd1_weights(int radius, double *w)
{
    w[0] = 0.0;
    for (int p = 1; p <= radius; ++p) {
        long double ratio = 1.0L;                          /* (n!)^2 / ((n-p)! (n+p)!) = prod_j (n-p+j)/(n+j) */
        for (int j = 1; j <= p; ++j) ratio *= (long double)(radius - p + j) / (long double)(radius + j);
        long double sign = (p % 2 == 1) ? 1.0L : -1.0L;
        w[p] = (double)(sign * ratio / (long double)p);
    }
}

/* G2.  (D_axis psi)(i) = sum_{p=1..n} w_p / h_axis * (psi(i + p e_axis) - psi(i - p e_axis)); neighbours outside a
 * Dirichlet face contribute 0, periodic axes wrap (reading R9). */
void oracle_gradient(const oracle_ham *H, int axis, const double *X, int64_t ldx, double *Y, int64_t ldy, int64_t ncols)
{
    double w[ORACLE_MAX_RADIUS + 1];
    oracle_fd1_weights(H->radius, w);
    const int nx = H->n[0], ny = H->n[1], nz = H->n[2], r = H->radius;
    const double ih = 1.0 / H->h[axis];
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t j = 0; j < ncols; ++j) {
        const double *psi = X + j * ldx;
        double *out = Y + j * ldy;
        for (int z = 0; z < nz; ++z)
            for (int y = 0; y < ny; ++y)
                for (int x = 0; x < nx; ++x) {
                    acc_t s = 0;
                    for (int p = 1; p <= r; ++p)
                        for (int sg = -1; sg <= 1; sg += 2) {
                            int cx = x, cy = y, cz = z;
                            int q;
                            if (axis == 0) { q = nbr_coord(x, sg * p, nx, H->bc[0]); cx = q; }
                            else if (axis == 1) { q = nbr_coord(y, sg * p, ny, H->bc[1]); cy = q; }
                            else { q = nbr_coord(z, sg * p, nz, H->bc[2]); cz = q; }
                            if (q >= 0) s += (acc_t)(sg * w[p]) * (acc_t)psi[cx + (int64_t)nx * (cy + (int64_t)ny * cz)];
                        }
                    out[x + (int64_t)nx * (y + (int64_t)ny * z)] = (double)(s * (acc_t)ih);
                }
    }
}

/* G3.  Projector contraction W = chi^T X ("nonlocal projector multiplication"):
 *   W[po_J + q, col] = sum_t chi_J[t, q] X[idx_J[t], col],  W is n_proj_total x ncols column-major (ld = n_proj_total),
 *   po_J = sum_{I<J} P_I.  No gamma, no volume factor (readings R6, R7). */
void oracle_nl_project(const oracle_ham *H, const double *X, int64_t ldx, int64_t ncols, double *W)
{
    int64_t ptot = 0;
    for (int J = 0; J < H->n_atoms; ++J) ptot += H->n_proj[J];
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t j = 0; j < ncols; ++j) {
        const double *psi = X + j * ldx;
        int64_t po = 0;
        for (int J = 0; J < H->n_atoms; ++J) {
            const int64_t s0 = H->supp_ptr[J], nJ = H->supp_ptr[J + 1] - s0;
            const double *chi = H->chi + H->chi_ptr[J];
            for (int q = 0; q < H->n_proj[J]; ++q) {
                acc_t s = 0;
                for (int64_t t = 0; t < nJ; ++t) s += (acc_t)chi[t + q * nJ] * (acc_t)psi[H->supp_idx[s0 + t]];
                W[po + q + j * ptot] = (double)s;
            }
            po += H->n_proj[J];
        }
    }
}

/* G4.  Nonlocal Hellmann-Feynman force (reading R22; the paper gives the two kernels, and refers to
 * [34, 47, 63] for the expression): with E_nl = sum_n g_n psi_n^T V_nl psi_n, V_nl = sum_J chi_J Gamma_J chi_J^T and
 * projectors that move rigidly with their atom, d chi_J / d R_J = -grad chi_J, and after one summation by parts on the grid
 *   F[J, a] = -dE_nl/dR_{J,a} = -2 sum_n g_n sum_q gamma_{Jq} (chi_Jq^T psi_n) (chi_Jq^T D_a psi_n),
 * g_n = occupation (times spin degeneracy) of orbital n, D_a the FD gradient of G2.  F is n_atoms x 3, row-major
 * (F[3 J + a]).  Any volume element is folded into gamma by the caller (reading R6).  scratch: Nd x ns doubles. */
void oracle_nonlocal_force(const oracle_ham *H, const double *Psi, int64_t ld, int64_t ns, const double *occ, double *F,
                           double *scratch)
{
    const int64_t nd = (int64_t)H->n[0] * H->n[1] * H->n[2];
    int64_t ptot = 0;
    for (int J = 0; J < H->n_atoms; ++J) ptot += H->n_proj[J];
    double *W = (double *)malloc(sizeof(double) * (size_t)(ptot > 0 ? ptot : 1) * (size_t)(ns > 0 ? ns : 1));
    double *G = (double *)malloc(sizeof(double) * (size_t)(ptot > 0 ? ptot : 1) * (size_t)(ns > 0 ? ns : 1));
    oracle_nl_project(H, Psi, ld, ns, W);
    for (int a = 0; a < 3; ++a) {
        oracle_gradient(H, a, Psi, ld, scratch, nd, ns);
        oracle_nl_project(H, scratch, nd, ns, G);
        int64_t po = 0;
        for (int J = 0; J < H->n_atoms; ++J) {
            acc_t s = 0;
            for (int64_t n = 0; n < ns; ++n)
                for (int q = 0; q < H->n_proj[J]; ++q)
                    s += (acc_t)occ[n] * (acc_t)H->gamma[po + q] * (acc_t)W[po + q + n * ptot] * (acc_t)G[po + q + n * ptot];
            F[3 * J + a] = (double)(-2 * s);
            po += H->n_proj[J];
        }
    }
    free(W);
    free(G);
}

/* =================================================================================================================
 * NEXT-1.  Generalized symmetric-definite eigenproblem  Hs Z = Ms Z D  (Algorithm 1, eq. 9 at 152;
 * the paper calls cusolverDnDsygvd).  Hs symmetric, Ms symmetric positive definite, n x n column-major
 * (ld = n).  The result the method needs is fixed up to the sign of each eigenvector (and rotations inside degenerate
 * eigenspaces): eigenvalues D ascending, Z^T Ms Z = I, Hs Z = Ms Z D (reading R23).  Steps, all in acc_t:
 *   E1  Cholesky  Ms = L L^T                          (textbook, column by column)
 *   E2  A = L^-1 Hs L^-T                              (two triangular solves per column; A symmetrised)
 *   E3  cyclic Jacobi on A: rotations (p, q) that annihilate A_pq, rows/columns updated in place, V accumulated,
 *       swept until off(A)^2 <= (eps ||A||_F)^2       (classical Jacobi eigenvalue method)
 *   E4  sort the eigenpairs ascending (stable), Z = L^-T V  (back substitution)
 * Returns 0, or 1 if Ms is not positive definite, 2 if Jacobi did not converge in 60 sweeps.
 * ================================================================================================================= */
int oracle_sygv(int64_t n, const double *Hs, const double *Ms, double *Z, double *D)
{
    if (n <= 0) return 0;
    acc_t *L = (acc_t *)calloc((size_t)(n * n), sizeof(acc_t));
    acc_t *A = (acc_t *)calloc((size_t)(n * n), sizeof(acc_t));
    acc_t *V = (acc_t *)calloc((size_t)(n * n), sizeof(acc_t));
    int rc = 0;
#define LL(i, j) L[(i) + (j) * n]
#define AA(i, j) A[(i) + (j) * n]
#define VV(i, j) V[(i) + (j) * n]
    /* E1 */
    for (int64_t j = 0; j < n && !rc; ++j) {
        acc_t d = (acc_t)Ms[j + j * n];
        for (int64_t k = 0; k < j; ++k) d -= LL(j, k) * LL(j, k);
        if (!(d > 0)) { rc = 1; break; }
        LL(j, j) = sqrtl((long double)d);
        for (int64_t i = j + 1; i < n; ++i) {
            acc_t s = (acc_t)Ms[i + j * n];
            for (int64_t k = 0; k < j; ++k) s -= LL(i, k) * LL(j, k);
            LL(i, j) = s / LL(j, j);
        }
    }
    if (!rc) {
        /* E2: column c of Y = L^-1 Hs by forward substitution; then row r of A = Y L^-T, i.e. A^T = L^-1 Y^T */
        for (int64_t c = 0; c < n; ++c)
            for (int64_t i = 0; i < n; ++i) {
                acc_t s = (acc_t)Hs[i + c * n];
                for (int64_t k = 0; k < i; ++k) s -= LL(i, k) * AA(k, c);
                AA(i, c) = s / LL(i, i);
            }
        /* now A holds Y; solve X L^T = Y row by row:  X[r, j] = (Y[r, j] - sum_{k<j} X[r, k] L[j, k]) / L[j, j] */
        for (int64_t r = 0; r < n; ++r)
            for (int64_t j = 0; j < n; ++j) {
                acc_t s = AA(r, j);
                for (int64_t k = 0; k < j; ++k) s -= AA(r, k) * LL(j, k);
                AA(r, j) = s / LL(j, j);
            }
        for (int64_t j = 0; j < n; ++j)
            for (int64_t i = j + 1; i < n; ++i) { acc_t m = (AA(i, j) + AA(j, i)) / 2; AA(i, j) = AA(j, i) = m; }
        /* E3 */
        for (int64_t i = 0; i < n; ++i) VV(i, i) = 1;
        acc_t fro2 = 0;
        for (int64_t k = 0; k < n * n; ++k) fro2 += A[k] * A[k];
        /* rounding floor of the rotations: a few units of the working precision per row */
        const acc_t eps = (sizeof(acc_t) > 8 ? (acc_t)1.1e-19L : (acc_t)2.3e-16L) * (acc_t)(4 + n);
        int sweep = 0;
        for (; sweep < 60; ++sweep) {
            acc_t off2 = 0;
            for (int64_t j = 0; j < n; ++j)
                for (int64_t i = 0; i < n; ++i)
                    if (i != j) off2 += AA(i, j) * AA(i, j);
            if (off2 <= eps * eps * fro2) break;
            for (int64_t p = 0; p < n - 1; ++p)
                for (int64_t q = p + 1; q < n; ++q) {
                    const acc_t apq = AA(p, q);
                    if (apq == 0) continue;
                    const acc_t theta = (AA(q, q) - AA(p, p)) / (2 * apq);
                    const acc_t t = (theta >= 0 ? 1 : -1) / (fabsl((long double)theta) + sqrtl((long double)(theta * theta + 1)));
                    const acc_t cs = 1 / sqrtl((long double)(t * t + 1)), sn = t * cs;
                    for (int64_t k = 0; k < n; ++k) {            /* columns p, q:  A <- A J */
                        const acc_t akp = AA(k, p), akq = AA(k, q);
                        AA(k, p) = cs * akp - sn * akq;
                        AA(k, q) = sn * akp + cs * akq;
                    }
                    for (int64_t k = 0; k < n; ++k) {            /* rows p, q:  A <- J^T A */
                        const acc_t apk = AA(p, k), aqk = AA(q, k);
                        AA(p, k) = cs * apk - sn * aqk;
                        AA(q, k) = sn * apk + cs * aqk;
                    }
                    for (int64_t k = 0; k < n; ++k) {            /* V <- V J */
                        const acc_t vkp = VV(k, p), vkq = VV(k, q);
                        VV(k, p) = cs * vkp - sn * vkq;
                        VV(k, q) = sn * vkp + cs * vkq;
                    }
                }
        }
        if (sweep == 60) rc = 2;
        /* E4: stable ascending order, then Z = L^-T V by back substitution */
        int64_t *ord = (int64_t *)malloc(sizeof(int64_t) * (size_t)n);
        for (int64_t i = 0; i < n; ++i) ord[i] = i;
        for (int64_t i = 1; i < n; ++i) {                        /* insertion sort */
            const int64_t o = ord[i];
            int64_t k = i;
            while (k > 0 && AA(ord[k - 1], ord[k - 1]) > AA(o, o)) { ord[k] = ord[k - 1]; --k; }
            ord[k] = o;
        }
        for (int64_t c = 0; c < n; ++c) {
            const int64_t o = ord[c];
            D[c] = (double)AA(o, o);
            for (int64_t i = n - 1; i >= 0; --i) {
                acc_t s = VV(i, o);
                for (int64_t k = i + 1; k < n; ++k) s -= LL(k, i) * (acc_t)Z[k + c * n];
                Z[i + c * n] = (double)(s / LL(i, i));
            }
        }
        free(ord);
    }
#undef LL
#undef AA
#undef VV
    free(L); free(A); free(V);
    return rc;
}

/* =================================================================================================================
 * NEXT-4.  Complex (k-point) variant ("complex-valued ... Bloch wavevectors", 126 / 146 / 166 the Zgemm
 * forms, 176 Monkhorst-Pack grids).  Readings R24-R27: orbitals are the cell-periodic-times-phase Bloch functions sampled
 * on the cell's grid, psi(r + L_a e_a) = exp(i theta_a) psi(r), theta_a = k_a L_a on a periodic axis; a stencil tap that
 * wraps across the face of axis a therefore picks up exp(+i theta_a) (leaving through the upper face) or exp(-i theta_a)
 * (lower face); Dirichlet axes have no phase.  Projector values chi are real; a support point that was folded into the
 * cell by w_a cells along axis a (image shift, w_a in {-1, 0, +1}, supplied per support row) contributes with the factor
 * exp(i sum_a w_a theta_a): chi~_J[t, q] = chi_J[t, q] exp(-i phi_t) acts as  V_nl = sum_J chi~_J Gamma_J chi~_J^H  with
 * phi_t = sum_a w_a[t] theta_a.  Complex numbers are interleaved (re, im) doubles; X is Nd x ncols complex column-major.
 * ================================================================================================================= */
typedef struct {
    oracle_ham base;
    double theta[3];          /* Bloch phase per axis (0 on Dirichlet axes) */
    const int8_t *shift;      /* [supp_total][3] image shift of each support row, or NULL (all zero) */
} oracle_ham_k;

static inline cacc_t cexp_i(acc_t t) { return (cacc_t)(cosl((long double)t) + I * sinl((long double)t)); }

/* K1.  Y = H(k) X = -1/2 L(k) X + Veff X + V_nl(k) X  on complex columns. */
void oracle_h_apply_k(const oracle_ham_k *Hk, const double *Xri, int64_t ldx, double *Yri, int64_t ldy, int64_t ncols)
{
    const oracle_ham *H = &Hk->base;
    const int nx = H->n[0], ny = H->n[1], nz = H->n[2], r = H->radius;
    const int64_t nd = (int64_t)nx * ny * nz;
    /* second-derivative weights restated (standard central weights, reading R1) */
    long double w[ORACLE_MAX_RADIUS + 1];
    w[0] = 0;
    for (int p = 1; p <= r; ++p) {
        long double ratio = 1.0L;
        for (int j = 1; j <= p; ++j) ratio *= (long double)(r - p + j) / (long double)(r + j);
        w[p] = 2.0L * ((p % 2) ? 1.0L : -1.0L) / ((long double)p * p) * ratio;
        w[0] -= 2.0L / ((long double)p * p);
    }
    const double complex *X = (const double complex *)Xri;
    double complex *Y = (double complex *)Yri;
    const int nn[3] = {nx, ny, nz};
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t j = 0; j < ncols; ++j) {
        const double complex *psi = X + j * ldx;
        double complex *out = Y + j * ldy;
        for (int z = 0; z < nz; ++z)
            for (int y = 0; y < ny; ++y)
                for (int x = 0; x < nx; ++x) {
                    const int c[3] = {x, y, z};
                    cacc_t lap = 0;
                    for (int a = 0; a < 3; ++a) {
                        cacc_t s = 0;
                        for (int p = -r; p <= r; ++p) {
                            int q = c[a] + p, wraps = 0;
                            if (H->bc[a] == 0) {
                                while (q < 0) { q += nn[a]; --wraps; }
                                while (q >= nn[a]) { q -= nn[a]; ++wraps; }
                            } else if (q < 0 || q >= nn[a]) continue;
                            int cc[3] = {x, y, z};
                            cc[a] = q;
                            const cacc_t v = (cacc_t)psi[cc[0] + (int64_t)nx * (cc[1] + (int64_t)ny * cc[2])];
                            s += (acc_t)w[p < 0 ? -p : p] * v * cexp_i((acc_t)wraps * (acc_t)Hk->theta[a]);
                        }
                        lap += s / ((acc_t)H->h[a] * (acc_t)H->h[a]);
                    }
                    const int64_t i = x + (int64_t)nx * (y + (int64_t)ny * z);
                    out[i] = (double complex)(-lap / 2 + (acc_t)H->veff[i] * (cacc_t)psi[i]);
                }
        /* nonlocal part */
        int64_t g0 = 0;
        for (int J = 0; J < H->n_atoms; ++J) {
            const int64_t s0 = H->supp_ptr[J], nJ = H->supp_ptr[J + 1] - s0;
            const double *chi = H->chi + H->chi_ptr[J];
            const int P = H->n_proj[J];
            for (int q = 0; q < P; ++q) {
                cacc_t cq = 0;                     /* chi~^H psi = sum_t chi[t, q] exp(+i phi_t) psi[idx_t] */
                for (int64_t t = 0; t < nJ; ++t) {
                    acc_t phi = 0;
                    if (Hk->shift) for (int a = 0; a < 3; ++a) phi += (acc_t)Hk->shift[3 * (s0 + t) + a] * (acc_t)Hk->theta[a];
                    cq += (acc_t)chi[t + q * nJ] * cexp_i(phi) * (cacc_t)psi[H->supp_idx[s0 + t]];
                }
                cq *= (acc_t)H->gamma[g0 + q];
                for (int64_t t = 0; t < nJ; ++t) {
                    acc_t phi = 0;
                    if (Hk->shift) for (int a = 0; a < 3; ++a) phi += (acc_t)Hk->shift[3 * (s0 + t) + a] * (acc_t)Hk->theta[a];
                    out[H->supp_idx[s0 + t]] += (double complex)((acc_t)chi[t + q * nJ] * cexp_i(-phi) * cq);
                }
            }
            g0 += P;
        }
    }
    (void)nd;
}

/* K2.  Scaled Chebyshev filter with H(k): the recurrence of chefsi_oracle.c's O6 (R3) on complex columns. */
int oracle_chebyshev_filter_k(const oracle_ham_k *Hk, double *Xri, int64_t ldx, int64_t ncols, int degree, double a,
                              double b, double a0)
{
    if (degree < 0 || !(a0 < a && a < b)) return 1;
    if (degree == 0 || ncols == 0) return 0;
    const oracle_ham *H = &Hk->base;
    const int64_t nd = (int64_t)H->n[0] * H->n[1] * H->n[2];
    const acc_t e = ((acc_t)b - (acc_t)a) / 2, c = ((acc_t)b + (acc_t)a) / 2;
    const acc_t sigma1 = e / ((acc_t)a0 - c), tau = 2 / sigma1;
    double complex *Xc = (double complex *)Xri;
    double complex *Y = (double complex *)malloc(sizeof(double complex) * (size_t)nd);
    double complex *Yn = (double complex *)malloc(sizeof(double complex) * (size_t)nd);
    double complex *HY = (double complex *)malloc(sizeof(double complex) * (size_t)nd);
    for (int64_t j = 0; j < ncols; ++j) {
        double complex *X = Xc + j * ldx;
        oracle_h_apply_k(Hk, (const double *)X, nd, (double *)HY, nd, 1);
        for (int64_t i = 0; i < nd; ++i) Y[i] = (double complex)((sigma1 / e) * ((cacc_t)HY[i] - c * (cacc_t)X[i]));
        acc_t sigma = sigma1;
        for (int k = 2; k <= degree; ++k) {
            const acc_t sigma2 = 1 / (tau - sigma);
            oracle_h_apply_k(Hk, (const double *)Y, nd, (double *)HY, nd, 1);
            for (int64_t i = 0; i < nd; ++i)
                Yn[i] = (double complex)((2 * sigma2 / e) * ((cacc_t)HY[i] - c * (cacc_t)Y[i]) - (sigma * sigma2) * (cacc_t)X[i]);
            memcpy(X, Y, sizeof(double complex) * (size_t)nd);
            memcpy(Y, Yn, sizeof(double complex) * (size_t)nd);
            sigma = sigma2;
        }
        memcpy(X, Y, sizeof(double complex) * (size_t)nd);
    }
    free(Y); free(Yn); free(HY);
    return 0;
}

/* K3.  Hermitian Gram contraction  out[i, j] = sum_r conj(A[r, i]) B[r, j]  (Hs = Psi^H H Psi, Ms = Psi^H Psi; the
 * Zgemm of PAPER.md:146 with the conjugate transpose), out nI x nJ complex column-major. */
void oracle_gram_k(const double *Ari, int64_t lda, const double *Bri, int64_t ldb, int64_t nd, int64_t nI, int64_t nJ,
                   double *outri)
{
    const double complex *A = (const double complex *)Ari, *B = (const double complex *)Bri;
    double complex *out = (double complex *)outri;
#pragma omp parallel for collapse(2) schedule(static)
    for (int64_t j = 0; j < nJ; ++j)
        for (int64_t i = 0; i < nI; ++i) {
            cacc_t s = 0;
            for (int64_t r = 0; r < nd; ++r) s += conjl((cacc_t)A[r + i * lda]) * (cacc_t)B[r + j * ldb];
            out[i + j * nI] = (double complex)s;
        }
}

/* K4.  Complex rotation  out[r, j] = sum_i Psi[r, i] Q[i, j]  (PAPER.md:166 Zgemm), Q ns x ns complex. */
void oracle_rotate_k(const double *Psiri, int64_t ld, int64_t nrows, int64_t ns, const double *Qri, double *outri)
{
    const double complex *Psi = (const double complex *)Psiri, *Q = (const double complex *)Qri;
    double complex *out = (double complex *)outri;
#pragma omp parallel for schedule(static)
    for (int64_t j = 0; j < ns; ++j)
        for (int64_t r = 0; r < nrows; ++r) {
            cacc_t s = 0;
            for (int64_t i = 0; i < ns; ++i) s += (cacc_t)Psi[r + i * ld] * (cacc_t)Q[i + j * ns];
            out[r + j * nrows] = (double complex)s;
        }
}
