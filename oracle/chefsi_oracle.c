/*
 * chefsi_oracle.c -- CPU ORACLE for the CheFSI hot path.  TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * Plain, slow, obviously-correct restatement of what the hot path computes, written from the
 * paper (arxiv 2302.09708, /root/reference/PAPER.md) and the readings listed in DESIGN.md
 * section 3 (which restate SURVEY.md section 8(c)).  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may call this.  It shares no code, header,
 * table or constant with the CUDA path under paper_2302_09708_b200/csrc/.
 *
 * Every operator is an exact linear-algebra definition, so the oracle is that definition written
 * out.  Arithmetic: IEEE double for data; every stencil sum and inner product is accumulated in
 * `acc_t` = long double (x87 80-bit) so the oracle's own rounding (~1e-19 per term) sits far
 * below the 1e-10 / 1e-11 parity gates.  Building with -DORACLE_ACC_DOUBLE makes acc_t = double:
 * that build is the "plain FP64" CPU baseline bench.py times.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): P1 exact rational weights and moment
 * conditions; P2 closed-form FD symbol on plane waves; P3 polynomial exactness; P4 Dirichlet =
 * restricted zero-padded periodic; P5 dense brute-force H and eigen-decomposition filter on a tiny
 * anisotropic mixed-BC grid; P6 symmetry; P7 T_m scaling of plane-wave eigenvectors and the
 * single-atom orthogonal-projector eigen relation; P8 small degrees; P9 column-block independence;
 * P10 Gram / rotation invariants.  No function here is "parity unpinned".
 *
 * Layout conventions (PAPER.md:102, 124, 126 -- "each column of X", cuBLAS column-major):
 *   grid linear index i = x + nx*(y + ny*z);  X is Nd x ncols column-major with leading dim ld.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifdef ORACLE_ACC_DOUBLE
typedef double acc_t;
#else
typedef long double acc_t;
#endif

#define ORACLE_MAX_RADIUS 6

/* Description of H = -1/2 Laplacian + Veff + V_nl (section II.A).  Plain host pointers,
 * all owned by the caller.  This struct belongs to the oracle only. */
typedef struct {
    int32_t n[3];             /* nx, ny, nz                                                    */
    double h[3];              /* grid spacing per axis                                         */
    int32_t bc[3];            /* 0 periodic, 1 Dirichlet (zero outside [0, n-1]) (reading R9)  */
    int32_t radius;           /* n0/2, n0 = finite-difference order             */
    int32_t n_atoms;
    const int64_t *supp_ptr;  /* [n_atoms+1]                                                   */
    const int32_t *supp_idx;  /* grid indices of each atom's projector support                 */
    const int32_t *n_proj;    /* [n_atoms]                                                     */
    const int64_t *chi_ptr;   /* [n_atoms+1] offsets into chi                                  */
    const double *chi;        /* per atom n_J x P_J column-major                               */
    const double *gamma;      /* concatenated P_J per atom                                     */
    const double *veff;       /* [Nd]                                                          */
} oracle_ham;

int oracle_acc_bits(void) { return (int)(8 * sizeof(acc_t)); }

/* ---------------------------------------------------------------------------------------------
 * O1.  Central finite-difference weights of the second derivative, radius n (order n0 = 2n).
 *   w_0 = -sum_{q=1..n} 2/q^2
 *   w_p = 2 (-1)^{p+1} / p^2 * (n!)^2 / ((n-p)! (n+p)!),  p = 1..n;  w_{-p} = w_p.
 * (The paper says only "finite-difference order n0" and "3 n0 + 1 computations", PAPER.md:124;
 *  reading R1: the standard central weights.)  Evaluated in long double regardless of acc_t.
 * ------------------------------------------------------------------------------------------- */
void oracle_fd_weights(int radius, double *w)
{
    long double w0 = 0.0L;
    for (int p = 1; p <= radius; ++p) {
        /* (n!)^2 / ((n-p)! (n+p)!) = prod_{j=1..p} (n-p+j) / (n+j) */
        long double ratio = 1.0L;
        for (int j = 1; j <= p; ++j) ratio *= (long double)(radius - p + j) / (long double)(radius + j);
        long double sign = (p % 2 == 1) ? 1.0L : -1.0L;
        w[p] = (double)(2.0L * sign / ((long double)p * (long double)p) * ratio);
        w0 -= 2.0L / ((long double)p * (long double)p);
    }
    w[0] = (double)w0;
}

/* neighbour coordinate along one axis: mod n on a periodic axis, -1 (contributes 0) outside a
 * Dirichlet axis (reading R9: all n planes are unknowns, psi = 0 at index -1, -2, ... and n, n+1, ...) */
static inline int nbr_coord(int c, int p, int n, int bc)
{
    int q = c + p;
    if (bc == 0) { q %= n; if (q < 0) q += n; return q; }
    return (q < 0 || q >= n) ? -1 : q;
}

/* ---------------------------------------------------------------------------------------------
 * O2.  Laplacian of one column:  (L psi)(x,y,z) = sum_axis sum_{p=-n..n} w_p / h_axis^2 * psi(.. + p ..)
 * 3 n0 + 1 taps, no cross terms.
 * ------------------------------------------------------------------------------------------- */
static void laplacian_column(const oracle_ham *H, const double *w, const double *psi, double *out)
{
    const int nx = H->n[0], ny = H->n[1], nz = H->n[2], r = H->radius;
    const double ihx = 1.0 / (H->h[0] * H->h[0]);
    const double ihy = 1.0 / (H->h[1] * H->h[1]);
    const double ihz = 1.0 / (H->h[2] * H->h[2]);
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                acc_t sx = 0, sy = 0, sz = 0;
                for (int p = -r; p <= r; ++p) {
                    const double wp = w[p < 0 ? -p : p];
                    int q = nbr_coord(x, p, nx, H->bc[0]);
                    if (q >= 0) sx += (acc_t)wp * (acc_t)psi[q + (int64_t)nx * (y + (int64_t)ny * z)];
                    q = nbr_coord(y, p, ny, H->bc[1]);
                    if (q >= 0) sy += (acc_t)wp * (acc_t)psi[x + (int64_t)nx * (q + (int64_t)ny * z)];
                    q = nbr_coord(z, p, nz, H->bc[2]);
                    if (q >= 0) sz += (acc_t)wp * (acc_t)psi[x + (int64_t)nx * (y + (int64_t)ny * q)];
                }
                out[x + (int64_t)nx * (y + (int64_t)ny * z)] =
                    (double)(sx * (acc_t)ihx + sy * (acc_t)ihy + sz * (acc_t)ihz);
            }
}

void oracle_laplacian(const oracle_ham *H, const double *X, int64_t ldx, double *Y, int64_t ldy,
                      int64_t ncols)
{
    double w[ORACLE_MAX_RADIUS + 1];
    oracle_fd_weights(H->radius, w);
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t j = 0; j < ncols; ++j) laplacian_column(H, w, X + j * ldx, Y + j * ldy);
}

/* ---------------------------------------------------------------------------------------------
 * O4.  Nonlocal Kleinman-Bylander term on one column, ADDED to out:
 *   for each atom J, projector q:  c_q = sum_t chi_J[t,q] psi[idx_J[t]]
 *   out[idx_J[t]] += sum_q chi_J[t,q] gamma_J[q] c_q
 * Gamma diagonal (reading R7), no volume factor (reading R6).
 * ------------------------------------------------------------------------------------------- */
static void vnl_add_column(const oracle_ham *H, const double *psi, double *out)
{
    int64_t g0 = 0;
    for (int J = 0; J < H->n_atoms; ++J) {
        const int64_t s0 = H->supp_ptr[J], nJ = H->supp_ptr[J + 1] - s0;
        const int P = H->n_proj[J];
        const int32_t *idx = H->supp_idx + s0;
        const double *chi = H->chi + H->chi_ptr[J];
        acc_t c[64];
        for (int q = 0; q < P; ++q) {
            acc_t s = 0;
            for (int64_t t = 0; t < nJ; ++t) s += (acc_t)chi[t + q * nJ] * (acc_t)psi[idx[t]];
            c[q] = (acc_t)H->gamma[g0 + q] * s;
        }
        for (int64_t t = 0; t < nJ; ++t) {
            acc_t s = 0;
            for (int q = 0; q < P; ++q) s += (acc_t)chi[t + q * nJ] * c[q];
            out[idx[t]] = (double)((acc_t)out[idx[t]] + s);
        }
        g0 += P;
    }
}

void oracle_vnl_apply(const oracle_ham *H, const double *X, int64_t ldx, double *Y, int64_t ldy,
                      int64_t ncols)
{
    const int64_t nd = (int64_t)H->n[0] * H->n[1] * H->n[2];
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t j = 0; j < ncols; ++j) {
        memset(Y + j * ldy, 0, sizeof(double) * (size_t)nd);
        vnl_add_column(H, X + j * ldx, Y + j * ldy);
    }
}

/* ---------------------------------------------------------------------------------------------
 * O3 + O5.  y = H psi = -1/2 L psi + Veff .* psi + V_nl psi   (Hartree units, reading R2)
 * `work` holds Nd doubles.
 * ------------------------------------------------------------------------------------------- */
static void h_apply_column(const oracle_ham *H, const double *w, const double *psi, double *y)
{
    const int64_t nd = (int64_t)H->n[0] * H->n[1] * H->n[2];
    laplacian_column(H, w, psi, y);
    for (int64_t i = 0; i < nd; ++i)
        y[i] = (double)((acc_t)(-0.5) * (acc_t)y[i] + (acc_t)H->veff[i] * (acc_t)psi[i]);
    vnl_add_column(H, psi, y);
}

void oracle_h_apply(const oracle_ham *H, const double *X, int64_t ldx, double *Y, int64_t ldy,
                    int64_t ncols)
{
    double w[ORACLE_MAX_RADIUS + 1];
    oracle_fd_weights(H->radius, w);
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t j = 0; j < ncols; ++j) h_apply_column(H, w, X + j * ldx, Y + j * ldy);
}

/* ---------------------------------------------------------------------------------------------
 * O6.  Scaled Chebyshev filter (three-term scaled recurrence of refs [61, 62], PAPER.md:31, 51-53,
 * 281-282; reading R3: b = lambda_Nd upper bound, a = lambda_c cutoff, a0 = lower bound):
 *   e = (b - a)/2;  c = (b + a)/2;  sigma = sigma_1 = e / (a0 - c);  tau = 2 / sigma_1
 *   Y = (sigma_1 / e) (H X - c X)
 *   for k = 2..m:  sigma' = 1 / (tau - sigma);  Y' = (2 sigma' / e)(H Y - c Y) - (sigma sigma') X;
 *                  X <- Y;  Y <- Y';  sigma <- sigma'
 *   return Y (m >= 1) or X (m = 0).            In place on X, column by column (eq. 4).
 * Equals T_m((H - cI)/e) X / T_m((a0 - c)/e).  Returns 0, or -1 on bad arguments (R4, R5).
 * ------------------------------------------------------------------------------------------- */
int oracle_chebyshev_filter(const oracle_ham *H, double *X, int64_t ldx, int64_t ncols, int degree,
                            double a, double b, double a0)
{
    if (degree < 0 || !(a0 < a && a < b)) return -1;
    if (degree == 0) return 0;
    const int64_t nd = (int64_t)H->n[0] * H->n[1] * H->n[2];
    double w[ORACLE_MAX_RADIUS + 1];
    oracle_fd_weights(H->radius, w);
    const double e = 0.5 * (b - a), c = 0.5 * (b + a);
    const double sigma1 = e / (a0 - c), tau = 2.0 / sigma1;
    int fail = 0;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t j = 0; j < ncols; ++j) {
        double *x = (double *)malloc(sizeof(double) * (size_t)nd);
        double *y = (double *)malloc(sizeof(double) * (size_t)nd);
        double *t = (double *)malloc(sizeof(double) * (size_t)nd);
        if (!x || !y || !t) { fail = 1; free(x); free(y); free(t); continue; }
        memcpy(x, X + j * ldx, sizeof(double) * (size_t)nd);
        h_apply_column(H, w, x, t);
        for (int64_t i = 0; i < nd; ++i)
            y[i] = (double)((acc_t)(sigma1 / e) * ((acc_t)t[i] - (acc_t)c * (acc_t)x[i]));
        double sigma = sigma1;
        for (int k = 2; k <= degree; ++k) {
            const double sigma2 = 1.0 / (tau - sigma);
            h_apply_column(H, w, y, t);
            for (int64_t i = 0; i < nd; ++i) {
                acc_t v = (acc_t)(2.0 * sigma2 / e) * ((acc_t)t[i] - (acc_t)c * (acc_t)y[i])
                          - (acc_t)(sigma * sigma2) * (acc_t)x[i];
                x[i] = y[i];
                y[i] = (double)v;
            }
            sigma = sigma2;
        }
        memcpy(X + j * ldx, y, sizeof(double) * (size_t)nd);
        free(x); free(y); free(t);
    }
    return fail ? -2 : 0;
}

/* ---------------------------------------------------------------------------------------------
 * O7.  Gram-type contraction over the Nd rows:
 *   out[i, j] = sum_r A[r, I[i]] * B[r, J[j]],  out is nI x nJ column-major (ld = nI).
 * I, J may be NULL (identity 0..nI-1 / 0..nJ-1).  Hs = gram(Psi, H Psi), Ms = gram(Psi, Psi);
 * index lists give the sampled-entry oracle of pin P11.
 * ------------------------------------------------------------------------------------------- */
void oracle_gram(const double *A, int64_t lda, const double *B, int64_t ldb, int64_t nd,
                 const int64_t *I, int64_t nI, const int64_t *J, int64_t nJ, double *out)
{
#pragma omp parallel for collapse(2) schedule(static)
    for (int64_t j = 0; j < nJ; ++j)
        for (int64_t i = 0; i < nI; ++i) {
            const double *a = A + (I ? I[i] : i) * lda;
            const double *bcol = B + (J ? J[j] : j) * ldb;
            acc_t s = 0;
            for (int64_t r = 0; r < nd; ++r) s += (acc_t)a[r] * (acc_t)bcol[r];
            out[i + j * nI] = (double)s;
        }
}

/* O7 as one call: Y = H Psi (O5), Hs = Psi^T Y, Ms = Psi^T Psi (reading R11). Y is caller scratch. */
void oracle_project(const oracle_ham *H, const double *Psi, int64_t ld, int64_t ns, double *Y,
                    double *Hs, double *Ms)
{
    const int64_t nd = (int64_t)H->n[0] * H->n[1] * H->n[2];
    oracle_h_apply(H, Psi, ld, Y, nd, ns);
    oracle_gram(Psi, ld, Y, nd, nd, NULL, ns, NULL, ns, Hs);
    oracle_gram(Psi, ld, Psi, ld, nd, NULL, ns, NULL, ns, Ms);
}

/* ---------------------------------------------------------------------------------------------
 * O8.  Rotation:  out[k, j] = sum_i Psi[rows[k], i] * Q[i, j]
 * out is nrows x ns column-major (ld = nrows); rows may be NULL (0..nrows-1). Q is ns x ns, ld = ns.
 * ------------------------------------------------------------------------------------------- */
void oracle_rotate(const double *Psi, int64_t ld, int64_t ns, const double *Q, const int64_t *rows,
                   int64_t nrows, double *out)
{
#pragma omp parallel for schedule(static)
    for (int64_t j = 0; j < ns; ++j)
        for (int64_t k = 0; k < nrows; ++k) {
            const int64_t r = rows ? rows[k] : k;
            acc_t s = 0;
            for (int64_t i = 0; i < ns; ++i) s += (acc_t)Psi[r + i * ld] * (acc_t)Q[i + j * ns];
            out[k + j * nrows] = (double)s;
        }
}
