/*
 * ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, serial, fp64 CPU statement of what the hot path of arXiv 1810.12742 computes:
 * the per-cell Hines solve (Listing 2) and, for unbranched cables, the
 * Thomas algorithm (Listing 1).  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference leg may call this.  It shares no code, header,
 * table or constant with paper_1810_12742_b200/ and neither side includes the other.
 *
 * Compile WITHOUT -ffast-math and WITH -ffp-contract=off (oracle/build.py does) so the
 * arithmetic is exactly the one written here: one rounding per operation, in the listing's order.
 *
 * Readings of the paper taken here (each listed in DESIGN.md "Readings"):
 *   G1  Listing 2's backward sweep prints u[p[i]]; read u[i]
 *       (u[i] = A[i,p[i]], "u also stores the coupling entries to the parent of a
 *       compartment").  With u[p[i]] a compartment with two children could hold
 *       only one coupling value.
 *   G2  Listing 1 mixes u[i-1] (backward) and u[i] (forward) (PAPER.md:58-62 vs :72); read
 *       u[i] = coupling of i with i-1 in both sweeps = Listing 2 with p[i] = i-1.
 *   S1  p[root] = -1, the root is local index 0 ("root A_{0,0}"); the loops stop
 *       at i = 1 so p[0] and u[0] are never read.
 *   S3  batch = concatenated cells + cell_offsets; parent[] holds cell-local indices.
 *
 * Pins (tests/test_oracle_*.py, all -m "not gpu"): dense LAPACK solve on every tree with
 * n <= 7 and on random trees; scipy banded solver and the constant-coefficient closed form on
 * cables; star-tree closed form; residual; x = 1 for b = A 1; M-matrix invariants; oracle_rel_err
 * against a numpy per-cell max-norm (NaN at the first / middle / last element of a cell, zero
 * reference); oracle_hines_solve_range bit-equal to oracle_hines_solve over splits of the cells and
 * against dense solves; oracle_pivots against Schur complements from dense inverses.
 */
#include <stdint.h>
#include <stddef.h>
#include <math.h>
#include <stdlib.h>

/* Listing 2 for one cell of n unknowns.
 * d, u, b are not written; dw (n doubles of scratch) holds the working diagonal,
 * x receives the working right-hand side and finally the solution. */
void oracle_hines_cell(int64_t n, const int32_t* p, const double* d, const double* u,
                       const double* b, double* x, double* dw)
{
    for (int64_t i = 0; i < n; ++i) { dw[i] = d[i]; x[i] = b[i]; }
    /* backward substitution (read per G1) */
    for (int64_t i = n - 1; i >= 1; --i) {
        double f = u[i] / dw[i];
        dw[p[i]] = dw[p[i]] - f * u[i];
        x[p[i]]  = x[p[i]]  - f * x[i];
    }
    /* solve root */
    x[0] = x[0] / dw[0];
    /* forward substitution */
    for (int64_t i = 1; i < n; ++i)
        x[i] = (x[i] - u[i] * x[p[i]]) / dw[i];
}

/* The batch: every cell independently ("each Hines matrix can be solved
 * independently").  dw: N doubles of scratch.  Returns 0. */
int oracle_hines_solve(int64_t ncells, const int64_t* cell_offsets, const int32_t* parent,
                       const double* d, const double* u, const double* b, double* x, double* dw)
{
    for (int64_t c = 0; c < ncells; ++c) {
        int64_t o = cell_offsets[c], n = cell_offsets[c + 1] - o;
        oracle_hines_cell(n, parent + o, d + o, u + o, b + o, x + o, dw + o);
    }
    return 0;
}

/* Same routine on a contiguous range of cells [c0, c1): lets a caller (bench.py's CPU
 * baseline) run a plain parallel-for over cells with one call per thread. */
int oracle_hines_solve_range(int64_t c0, int64_t c1, const int64_t* cell_offsets,
                             const int32_t* parent, const double* d, const double* u,
                             const double* b, double* x, double* dw)
{
    for (int64_t c = c0; c < c1; ++c) {
        int64_t o = cell_offsets[c], n = cell_offsets[c + 1] - o;
        oracle_hines_cell(n, parent + o, d + o, u + o, b + o, x + o, dw + o);
    }
    return 0;
}

/* Listing 1 (read per G2): Thomas on one tridiagonal system where
 * u[i] couples i with i-1 (u[0] unused). */
void oracle_thomas(int64_t n, const double* d, const double* u, const double* b,
                   double* x, double* dw)
{
    for (int64_t i = 0; i < n; ++i) { dw[i] = d[i]; x[i] = b[i]; }
    for (int64_t i = n - 1; i >= 1; --i) {
        double f = u[i] / dw[i];
        dw[i - 1] = dw[i - 1] - f * u[i];
        x[i - 1]  = x[i - 1]  - f * x[i];
    }
    x[0] = x[0] / dw[0];
    for (int64_t i = 1; i < n; ++i)
        x[i] = (x[i] - u[i] * x[i - 1]) / dw[i];
}

/* y = A x for the batch, straight from (d, u, p) without forming A:
 * A[i,i] = d[i], A[i,p[i]] = A[p[i],i] = u[i]. */
void oracle_matvec(int64_t ncells, const int64_t* cell_offsets, const int32_t* parent,
                   const double* d, const double* u, const double* x, double* y)
{
    for (int64_t c = 0; c < ncells; ++c) {
        int64_t o = cell_offsets[c], n = cell_offsets[c + 1] - o;
        for (int64_t i = 0; i < n; ++i) y[o + i] = d[o + i] * x[o + i];
        for (int64_t i = 1; i < n; ++i) {
            int64_t pi = parent[o + i];
            y[o + i]  += u[o + i] * x[o + pi];
            y[o + pi] += u[o + i] * x[o + i];
        }
    }
}

/* per cell: res[c] = ||A x - b||_inf / ||b||_inf  (S15-style per-cell norm). */
void oracle_residual(int64_t ncells, const int64_t* cell_offsets, const int32_t* parent,
                     const double* d, const double* u, const double* b, const double* x,
                     double* y /* N scratch */, double* res /* ncells */)
{
    oracle_matvec(ncells, cell_offsets, parent, d, u, x, y);
    for (int64_t c = 0; c < ncells; ++c) {
        double r = 0.0, nb = 0.0;
        for (int64_t i = cell_offsets[c]; i < cell_offsets[c + 1]; ++i) {
            double e = fabs(y[i] - b[i]); if (e > r) r = e;
            double a = fabs(b[i]);        if (a > nb) nb = a;
        }
        res[c] = (nb > 0.0) ? r / nb : r;
    }
}

/* The working diagonal after the backward sweep (the pivots d'), for the invariants
 * I1 (d'[i] > 0 and bounded below) and I2 (|f| < 1): PAPER.md:36. */
void oracle_pivots(int64_t ncells, const int64_t* cell_offsets, const int32_t* parent,
                   const double* d, const double* u, double* dw)
{
    for (int64_t c = 0; c < ncells; ++c) {
        int64_t o = cell_offsets[c], n = cell_offsets[c + 1] - o;
        for (int64_t i = 0; i < n; ++i) dw[o + i] = d[o + i];
        for (int64_t i = n - 1; i >= 1; --i) {
            double f = u[o + i] / dw[o + i];
            dw[o + parent[o + i]] -= f * u[o + i];
        }
    }
}

/* per cell relative max-norm error  ||xa - xb||_inf / ||xb||_inf  (reading S15); the absolute error
 * where xb is identically zero.  A NaN anywhere in a cell's xa (or xb) makes that cell's error NaN, and
 * only that cell's.  Pinned by tests/test_oracle_solve.py against numpy, cell by cell. */
void oracle_rel_err(int64_t ncells, const int64_t* cell_offsets, const double* xa,
                    const double* xb, double* err)
{
    for (int64_t c = 0; c < ncells; ++c) {
        double e = 0.0, nrm = 0.0;
        for (int64_t i = cell_offsets[c]; i < cell_offsets[c + 1]; ++i) {
            double t = fabs(xa[i] - xb[i]);
            if (t != t || (e == e && t > e)) e = t;   /* NaN-sticky max: once NaN, stays NaN */
            double a = fabs(xb[i]); if (a > nrm) nrm = a;
        }
        err[c] = (nrm > 0.0) ? e / nrm : e;
    }
}

/* ---- f3: factor once, solve many (with a fixed time step the matrix does not change between steps,
 * only the right-hand side does).  Listing 2 (reading G1) split in two: the part that touches only
 * d and u, and the part that touches b.  Same operations in the same order as oracle_hines_cell, so the two
 * together give bit-identical x (pinned in tests/test_oracle_solve.py). */

/* dw[i] = the pivots d' after the backward sweep, f[i] = u[i] / dw[i] (f[0] unused, set to 0). */
void oracle_hines_factor_cell(int64_t n, const int32_t* p, const double* d, const double* u,
                              double* dw, double* f)
{
    for (int64_t i = 0; i < n; ++i) dw[i] = d[i];
    f[0] = 0.0;
    for (int64_t i = n - 1; i >= 1; --i) {
        f[i] = u[i] / dw[i];
        dw[p[i]] = dw[p[i]] - f[i] * u[i];
    }
}

/* x = A^-1 b from the factors: backward x[p[i]] -= f[i] x[i]; root x[0] /= dw[0]; forward
 * x[i] = (x[i] - u[i] x[p[i]]) / dw[i]. */
void oracle_hines_solve_rhs_cell(int64_t n, const int32_t* p, const double* dw, const double* f,
                                 const double* u, const double* b, double* x)
{
    for (int64_t i = 0; i < n; ++i) x[i] = b[i];
    for (int64_t i = n - 1; i >= 1; --i) x[p[i]] = x[p[i]] - f[i] * x[i];
    x[0] = x[0] / dw[0];
    for (int64_t i = 1; i < n; ++i) x[i] = (x[i] - u[i] * x[p[i]]) / dw[i];
}

int oracle_hines_factor(int64_t ncells, const int64_t* cell_offsets, const int32_t* parent,
                        const double* d, const double* u, double* dw, double* f)
{
    for (int64_t c = 0; c < ncells; ++c) {
        int64_t o = cell_offsets[c], n = cell_offsets[c + 1] - o;
        oracle_hines_factor_cell(n, parent + o, d + o, u + o, dw + o, f + o);
    }
    return 0;
}

int oracle_hines_solve_rhs(int64_t ncells, const int64_t* cell_offsets, const int32_t* parent,
                           const double* dw, const double* f, const double* u, const double* b, double* x)
{
    for (int64_t c = 0; c < ncells; ++c) {
        int64_t o = cell_offsets[c], n = cell_offsets[c + 1] - o;
        oracle_hines_solve_rhs_cell(n, parent + o, dw + o, f + o, u + o, b + o, x + o);
    }
    return 0;
}
