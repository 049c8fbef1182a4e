/*
 * oracle_next.c -- TEST INFRASTRUCTURE ONLY (same rules as oracle.c: only tests/, smoke() and bench.py's
 * cpu_baseline leg may call it; it shares nothing with the CUDA library).  Plain CPU statements of the
 * operations that sit right after / beside H psi in the paper's loop (SURVEY.md section 8(f) "next" rows):
 *
 *   f1  block operations between orbitals: "copies, linear combinations, and dot products ... implemented
 *       ... using the block-of-orbitals approach"                                PAPER.md:260-266 (sec. VIII);
 *       RMM-DIIS works on residuals H psi - eps psi                               PAPER.md:65-69 (sec. III).
 *         dot_j      = sum_p conj(a_j(p)) b_j(p)            (plain sums, no h^3 factor: reading S11)
 *         axpy       : y_j(p) += alpha_j x_j(p)
 *         residual   : r_j(p) = (H psi)_j(p) - eps_j psi_j(p),  eps_j real
 *   f2  overlap / subspace matrices        S_jk = <phi_j|phi_k> (eq. 5),  h_jk = <phi_j|H|phi_k> (eq. 7):
 *         M_jk = sum_p conj(a_j(p)) b_k(p)    with b = phi (eq. 5) or b = H phi (eq. 7)
 *                                                                   PAPER.md:203-215, :225-235 (sec. VI).
 *   f3  non-local potential, eq. (4)                                 PAPER.md:173-197 (sec. V.C, eq. 4 :181):
 *         (V_nl phi)(r) = sum_A sum_lm gamma^A_lm(r - R_A) * Integral_{r' in sphere A} gamma^A_lm(r' - R_A) phi(r') dr'
 *       first "the integrals over r' ... store the results", then "multiply the stored integrals by the radial
 *       functions and sum over angular-momentum components".  Readings: the integral
 *       is the lattice sum times h^3; the sphere is the closed ball |r - R_A| <= r_c restricted to the mesh; eq. 4 as
 *       printed carries no extra coefficient; projector values are real INPUTS (synthetic stand-ins for pseudopotentials).
 *
 * Layout here: one orbital after another, psi[ist][np] in canonical point order, `lanes` = 1 (real) or 2
 * (complex, interleaved re, im).  Every loop is the definition written out; one accumulator per result, points
 * visited in ascending order.  Pins: tests/test_oracle_next_pins.py.
 */
#include <stddef.h>
#include <stdint.h>

/* f1: out[j] (lanes doubles each) = sum_p conj(a[j][p]) * b[j][p]                                             */
void orc_block_dot(const double *a, const double *b, int64_t np, int nst, int lanes, double *out)
{
    for (int j = 0; j < nst; ++j) {
        double re = 0.0, im = 0.0;
        for (int64_t p = 0; p < np; ++p) {
            const size_t q = ((size_t)j * np + p) * lanes;
            if (lanes == 1) {
                re += a[q] * b[q];
            } else { /* conj(a) b = (ar - i ai)(br + i bi) */
                re += a[q] * b[q] + a[q + 1] * b[q + 1];
                im += a[q] * b[q + 1] - a[q + 1] * b[q];
            }
        }
        out[(size_t)j * lanes] = re;
        if (lanes == 2) out[(size_t)j * lanes + 1] = im;
    }
}

/* f1: y[j][p] += alpha[j] * x[j][p]; alpha has `lanes` doubles per orbital (complex alpha for complex data)     */
void orc_block_axpy(const double *alpha, const double *x, double *y, int64_t np, int nst, int lanes)
{
    for (int j = 0; j < nst; ++j)
        for (int64_t p = 0; p < np; ++p) {
            const size_t q = ((size_t)j * np + p) * lanes;
            if (lanes == 1) {
                y[q] += alpha[j] * x[q];
            } else {
                const double ar = alpha[2 * j], ai = alpha[2 * j + 1];
                y[q] += ar * x[q] - ai * x[q + 1];
                y[q + 1] += ar * x[q + 1] + ai * x[q];
            }
        }
}

/* f1: r[j][p] = hpsi[j][p] - eps[j] * psi[j][p], eps real (an eigenvalue estimate)                              */
void orc_block_residual(const double *hpsi, const double *psi, const double *eps, int64_t np, int nst, int lanes,
                        double *r)
{
    for (int j = 0; j < nst; ++j)
        for (int64_t p = 0; p < np; ++p)
            for (int l = 0; l < lanes; ++l) {
                const size_t q = ((size_t)j * np + p) * lanes + l;
                r[q] = hpsi[q] - eps[j] * psi[q];
            }
}

/* f2: M[j][k] (lanes doubles each, row-major [nsa][nsb]) = sum_p conj(a[j][p]) * b[k][p]     (eqs. 5, 7)        */
void orc_overlap(const double *a, int nsa, const double *b, int nsb, int64_t np, int lanes, double *M)
{
    for (int j = 0; j < nsa; ++j)
        for (int k = 0; k < nsb; ++k) {
            double re = 0.0, im = 0.0;
            for (int64_t p = 0; p < np; ++p) {
                const size_t qa = ((size_t)j * np + p) * lanes, qb = ((size_t)k * np + p) * lanes;
                if (lanes == 1) {
                    re += a[qa] * b[qb];
                } else {
                    re += a[qa] * b[qb] + a[qa + 1] * b[qb + 1];
                    im += a[qa] * b[qb + 1] - a[qa + 1] * b[qb];
                }
            }
            M[((size_t)j * nsb + k) * lanes] = re;
            if (lanes == 2) M[((size_t)j * nsb + k) * lanes + 1] = im;
        }
}

/* f3: membership of the projector spheres.  For atom A: the canonical indices of the mesh points with
 * |h (i,j,k) - R_A|^2 <= rc^2 (closed ball, fp64, same convention as the mesh itself, reading S4).
 * ijk: [np][3] lattice indices of the canonical points.  Pass idx = NULL to count only.  Returns the count.    */
int64_t orc_sphere_points(const int32_t *ijk, int64_t np, double h, const double *center, double rc, int64_t *idx)
{
    int64_t cnt = 0;
    const double rc2 = rc * rc;
    for (int64_t p = 0; p < np; ++p) {
        const double dx = (double)ijk[3 * p] * h - center[0];
        const double dy = (double)ijk[3 * p + 1] * h - center[1];
        const double dz = (double)ijk[3 * p + 2] * h - center[2];
        if (dx * dx + dy * dy + dz * dz <= rc2) {
            if (idx) idx[cnt] = p;
            ++cnt;
        }
    }
    return cnt;
}

/* f3: out[j] += V_nl psi[j] (eq. 4).  Atom A owns npts[A] sphere points: canonical indices idx[off[A] ..] and
 * projector values gamma[(off[A] + q) * nlm + lm] (real).  Part 1: P = h3 * sum_q gamma psi (the stored integral);
 * part 2: out(point q) += gamma * P, summed over lm, atom after atom.                                         */
void orc_nonlocal(int natoms, const int64_t *off, const int64_t *npts, const int64_t *idx, const double *gamma, int nlm,
                  double h3, const double *psi, double *out, int64_t np, int nst, int lanes)
{
    for (int j = 0; j < nst; ++j)
        for (int A = 0; A < natoms; ++A)
            for (int lm = 0; lm < nlm; ++lm)
                for (int l = 0; l < lanes; ++l) {
                    double P = 0.0;
                    for (int64_t q = 0; q < npts[A]; ++q)
                        P += gamma[(size_t)(off[A] + q) * nlm + lm] * psi[((size_t)j * np + idx[off[A] + q]) * lanes + l];
                    P *= h3;
                    for (int64_t q = 0; q < npts[A]; ++q)
                        out[((size_t)j * np + idx[off[A] + q]) * lanes + l] += gamma[(size_t)(off[A] + q) * nlm + lm] * P;
                }
}
