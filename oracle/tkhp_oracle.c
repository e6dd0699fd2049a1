/*
 * tkhp_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, obviously-correct FP64 CPU oracle for the real-space AMOEBA
 * polarization hot path of arXiv 2011.01207 (Tinker-HP on GPUs).  It shares no
 * code, header, table or constant with the CUDA library under
 * paper_2011_01207_b200/csrc/ and must never be imported by it.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may load it.
 *
 * What the paper gives: the organisation of the real-space kernels (pair loop
 * with a cutoff test, Listing 1; "compute unscaled, then a
 * separate scaling-correction pass", L98-129 Listing 2; PCG with a diagonal
 * preconditioner and one polarization matrix-vector product per iteration,
 * L160 and L437; 32-atom groups and group-pair list, L296-366).  It prints NO
 * interaction formula (refs only, L734, L760-764), so the arithmetic below is
 * the standard AMOEBA real-space Ewald field with Thole damping as written out
 * in SURVEY.md section 8(c) (equations F1-F4, T1-T2, S, U, N and readings
 * Q1-Q18, restated in DESIGN.md "Readings").
 *
 * Method: the block list only prunes pairs beyond the cutoff, so the result has
 * a plain definition -- a double loop over ALL ordered pairs i != j with the
 * minimum image and an R^2 <= rc^2 test.  That definition is what is coded
 * here: O(N^2), no lists, no blocks, no use of pair symmetry (each ordered
 * pair is evaluated on its own, so symmetry of T is a non-trivial check).
 * OpenMP parallelises over the rows i only.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): SURVEY 8(c) P1-P13 -- closed-form
 * radial values (tests/golden/), finite-difference gradient of an independently
 * written scalar potential, point-charge-cluster limit of the dipole and
 * quadrupole terms, two-site analytic solve, dense Cholesky vs PCG,
 * T symmetry, translation / image / permutation invariance, mask cases,
 * energy = minimum of the quadratic functional.
 * No function here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define SQRT_PI 1.7724538509055160272981674833411451827975

/* ---------- radial functions (SURVEY 8(c) "Radial functions") ------------ */

/* Ewald: bn0 = erfc(beta R)/R ; bn_k = [(2k-1) bn_{k-1} + (2 beta^2)^k/(beta sqrt(pi)) exp(-beta^2 R^2)] / R^2.
 * beta == 0 (test mode): bn_k = rr_k exactly = 1/R, 1/R^3, 3/R^5, 15/R^7. */
void oracle_ewald_bn(double beta, double R, double bn[4])
{
    double R2 = R * R;
    if (beta == 0.0) {
        bn[0] = 1.0 / R;
        bn[1] = bn[0] / R2;
        bn[2] = 3.0 * bn[1] / R2;
        bn[3] = 5.0 * bn[2] / R2;
        return;
    }
    double ex = exp(-beta * beta * R2);
    double pref = 1.0 / (beta * SQRT_PI);
    double tb2 = 2.0 * beta * beta;
    double p = 1.0;
    bn[0] = erfc(beta * R) / R;
    for (int k = 1; k <= 3; ++k) {
        p *= tb2;
        bn[k] = ((2.0 * k - 1.0) * bn[k - 1] + p * pref * ex) / R2;
    }
}

/* Thole (AMOEBA exponential form): u = R/(alpha_i alpha_j)^(1/6), x = a u^3,
 * lam3 = 1-e^-x, lam5 = 1-(1+x)e^-x, lam7 = 1-(1+x+(3/5)x^2)e^-x. */
void oracle_thole_lambda(double a, double alpha_i, double alpha_j, double R, double lam[3])
{
    double u = R / pow(alpha_i * alpha_j, 1.0 / 6.0);
    double x = a * u * u * u;
    double e = exp(-x);
    lam[0] = 1.0 - e;
    lam[1] = 1.0 - (1.0 + x) * e;
    lam[2] = 1.0 - (1.0 + x + 0.6 * x * x) * e;
}

/* (F1) G_k = bn_k - (1 - s lam_{2k+1}) rr_k, k=1..3 ; s = 0 for a masked pair */
void oracle_pair_G(double beta, double a, double alpha_i, double alpha_j, double s,
                   double R, double G[3])
{
    double bn[4], lam[3];
    oracle_ewald_bn(beta, R, bn);
    oracle_thole_lambda(a, alpha_i, alpha_j, R, lam);
    double R2 = R * R;
    double rr1 = 1.0 / (R2 * R);
    double rr2 = 3.0 * rr1 / R2;
    double rr3 = 5.0 * rr2 / R2;
    G[0] = bn[1] - (1.0 - s * lam[0]) * rr1;
    G[1] = bn[2] - (1.0 - s * lam[1]) * rr2;
    G[2] = bn[3] - (1.0 - s * lam[2]) * rr3;
}

static inline void min_image(double d[3], double box)
{
    if (box > 0.0) {
        for (int c = 0; c < 3; ++c)
            d[c] -= box * nearbyint(d[c] / box);
    }
}

static inline double self_coeff(double beta)
{
    /* (F3)/(Q8): 4 beta^3 / (3 sqrt(pi)) ; zero in the beta = 0 test mode */
    return 4.0 * beta * beta * beta / (3.0 * SQRT_PI);
}

/* field at atom i (F1-F3), one row of the definition */
static void field_row(int64_t i, int64_t n, const double *pos, const double *q,
                      const double *dip, const double *quad, const double *alpha,
                      const int32_t *grp, double box, double rc, double beta,
                      double a, double Ei[3])
{
    double ex = 0.0, ey = 0.0, ez = 0.0;
    double rc2 = rc * rc;
    for (int64_t j = 0; j < n; ++j) {
        if (j == i) continue;
        double R[3] = { pos[3 * i] - pos[3 * j], pos[3 * i + 1] - pos[3 * j + 1],
                        pos[3 * i + 2] - pos[3 * j + 2] };
        min_image(R, box);
        double R2 = R[0] * R[0] + R[1] * R[1] + R[2] * R[2];
        if (R2 > rc2) continue;                      /* (Q7) include iff R^2 <= rc^2 */
        double s = (grp[i] == grp[j]) ? 0.0 : 1.0;   /* (Q3,Q4) one mask */
        double G[3];
        oracle_pair_G(beta, a, alpha[i], alpha[j], s, sqrt(R2), G);
        const double *d = dip + 3 * j;
        const double *t = quad + 6 * j;              /* xx xy xz yy yz zz */
        double dR = d[0] * R[0] + d[1] * R[1] + d[2] * R[2];
        double TR[3] = { t[0] * R[0] + t[1] * R[1] + t[2] * R[2],
                         t[1] * R[0] + t[3] * R[1] + t[4] * R[2],
                         t[2] * R[0] + t[4] * R[1] + t[5] * R[2] };
        double RTR = R[0] * TR[0] + R[1] * TR[1] + R[2] * TR[2];
        /* (F2) */
        double radial = q[j] * G[0] + G[1] * dR + (G[2] / 3.0) * RTR;
        ex += radial * R[0] - G[0] * d[0] - (2.0 / 3.0) * G[1] * TR[0];
        ey += radial * R[1] - G[0] * d[1] - (2.0 / 3.0) * G[1] * TR[1];
        ez += radial * R[2] - G[0] * d[2] - (2.0 / 3.0) * G[1] * TR[2];
    }
    double sc = self_coeff(beta);                    /* (F3) */
    Ei[0] = ex + sc * dip[3 * i];
    Ei[1] = ey + sc * dip[3 * i + 1];
    Ei[2] = ez + sc * dip[3 * i + 2];
}

/* (T1,T2) one row of T mu, incl. the Ewald self term on mu_i (Q8) */
static void tmu_row(int64_t i, int64_t n, const double *pos, const double *alpha,
                    const double *mu, double box, double rc, double beta, double a,
                    double out[3])
{
    double ox = 0.0, oy = 0.0, oz = 0.0;
    double rc2 = rc * rc;
    for (int64_t j = 0; j < n; ++j) {
        if (j == i) continue;
        double R[3] = { pos[3 * i] - pos[3 * j], pos[3 * i + 1] - pos[3 * j + 1],
                        pos[3 * i + 2] - pos[3 * j + 2] };
        min_image(R, box);
        double R2 = R[0] * R[0] + R[1] * R[1] + R[2] * R[2];
        if (R2 > rc2) continue;
        double Rn = sqrt(R2);
        double bn[4], lam[3];
        oracle_ewald_bn(beta, Rn, bn);
        oracle_thole_lambda(a, alpha[i], alpha[j], Rn, lam);
        double m1 = bn[1] - (1.0 - lam[0]) / (R2 * Rn);             /* (T1) */
        double m2 = bn[2] - 3.0 * (1.0 - lam[1]) / (R2 * R2 * Rn);  /* (T2) */
        const double *m = mu + 3 * j;
        double mR = m[0] * R[0] + m[1] * R[1] + m[2] * R[2];
        ox += -m1 * m[0] + m2 * mR * R[0];
        oy += -m1 * m[1] + m2 * mR * R[1];
        oz += -m1 * m[2] + m2 * mR * R[2];
    }
    double sc = self_coeff(beta);
    out[0] = ox + sc * mu[3 * i];
    out[1] = oy + sc * mu[3 * i + 1];
    out[2] = oz + sc * mu[3 * i + 2];
}

/* F: permanent field, all rows.  E is N*3. */
int oracle_perm_field(int64_t n, const double *pos, const double *q, const double *dip,
                      const double *quad, const double *alpha, const int32_t *grp,
                      double box, double rc, double beta, double a, double *E)
{
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t i = 0; i < n; ++i)
        field_row(i, n, pos, q, dip, quad, alpha, grp, box, rc, beta, a, E + 3 * i);
    return 0;
}

/* F on selected rows only (sampled parity at full sizes). E is n_rows*3. */
int oracle_perm_field_rows(int64_t n, const double *pos, const double *q, const double *dip,
                           const double *quad, const double *alpha, const int32_t *grp,
                           double box, double rc, double beta, double a,
                           int64_t n_rows, const int64_t *rows, double *E)
{
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t k = 0; k < n_rows; ++k)
        field_row(rows[k], n, pos, q, dip, quad, alpha, grp, box, rc, beta, a, E + 3 * k);
    return 0;
}

/* T: out = T_real mu + self mu, all rows. */
int oracle_tmatvec(int64_t n, const double *pos, const double *alpha, const double *mu,
                   double box, double rc, double beta, double a, double *out)
{
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t i = 0; i < n; ++i)
        tmu_row(i, n, pos, alpha, mu, box, rc, beta, a, out + 3 * i);
    return 0;
}

int oracle_tmatvec_rows(int64_t n, const double *pos, const double *alpha, const double *mu,
                        double box, double rc, double beta, double a,
                        int64_t n_rows, const int64_t *rows, double *out)
{
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t k = 0; k < n_rows; ++k)
        tmu_row(rows[k], n, pos, alpha, mu, box, rc, beta, a, out + 3 * k);
    return 0;
}

/* Dense T (3N x 3N, row-major), incl. the self term on the diagonal.  Small N only. */
int oracle_dense_T(int64_t n, const double *pos, const double *alpha, double box, double rc,
                   double beta, double a, double *T)
{
    int64_t m = 3 * n;
    memset(T, 0, sizeof(double) * (size_t)m * (size_t)m);
    double rc2 = rc * rc;
    double sc = self_coeff(beta);
    for (int64_t i = 0; i < n; ++i) {
        for (int c = 0; c < 3; ++c) T[(3 * i + c) * m + 3 * i + c] = sc;
        for (int64_t j = 0; j < n; ++j) {
            if (j == i) continue;
            double R[3] = { pos[3 * i] - pos[3 * j], pos[3 * i + 1] - pos[3 * j + 1],
                            pos[3 * i + 2] - pos[3 * j + 2] };
            min_image(R, box);
            double R2 = R[0] * R[0] + R[1] * R[1] + R[2] * R[2];
            if (R2 > rc2) continue;
            double Rn = sqrt(R2);
            double bn[4], lam[3];
            oracle_ewald_bn(beta, Rn, bn);
            oracle_thole_lambda(a, alpha[i], alpha[j], Rn, lam);
            double m1 = bn[1] - (1.0 - lam[0]) / (R2 * Rn);
            double m2 = bn[2] - 3.0 * (1.0 - lam[1]) / (R2 * R2 * Rn);
            for (int c = 0; c < 3; ++c)
                for (int e = 0; e < 3; ++e)
                    T[(3 * i + c) * m + 3 * j + e] = m2 * R[c] * R[e] - (c == e ? m1 : 0.0);
        }
    }
    return 0;
}

/* number of unordered pairs {i,j}, i != j, R^2 <= rc^2 (the "useful pair" count N_pair) */
int64_t oracle_count_pairs(int64_t n, const double *pos, double box, double rc)
{
    int64_t total = 0;
    double rc2 = rc * rc;
#pragma omp parallel for schedule(dynamic, 16) reduction(+ : total)
    for (int64_t i = 0; i < n; ++i) {
        for (int64_t j = i + 1; j < n; ++j) {
            double R[3] = { pos[3 * i] - pos[3 * j], pos[3 * i + 1] - pos[3 * j + 1],
                            pos[3 * i + 2] - pos[3 * j + 2] };
            min_image(R, box);
            if (R[0] * R[0] + R[1] * R[1] + R[2] * R[2] <= rc2) ++total;
        }
    }
    return total;
}

/* pairs counted from selected rows only: sum_k #{j != rows[k] : R <= rc} (ordered) */
int64_t oracle_count_pairs_rows(int64_t n, const double *pos, double box, double rc,
                                int64_t n_rows, const int64_t *rows)
{
    int64_t total = 0;
    double rc2 = rc * rc;
#pragma omp parallel for schedule(dynamic, 4) reduction(+ : total)
    for (int64_t k = 0; k < n_rows; ++k) {
        int64_t i = rows[k];
        for (int64_t j = 0; j < n; ++j) {
            if (j == i) continue;
            double R[3] = { pos[3 * i] - pos[3 * j], pos[3 * i + 1] - pos[3 * j + 1],
                            pos[3 * i + 2] - pos[3 * j + 2] };
            min_image(R, box);
            if (R[0] * R[0] + R[1] * R[1] + R[2] * R[2] <= rc2) ++total;
        }
    }
    return total;
}

/* ------------------------- N: neighbour list ----------------------------- *
 * (Q16) FP64 throughout, no FMA contraction (this file is compiled with
 * -ffp-contract=off): wrapped coordinate w = x - L floor(x/L) (clamped into
 * [0,L)); per block of 32 consecutive entries of perm (entries < 0 are
 * phantoms and are skipped) lo/hi = exact min/max of w; c = 0.5 (lo+hi),
 * h = 0.5 (hi-lo); per axis D = |c_I - c_J|, D = min(D, L - D) when periodic,
 * gap = max(0, D - (h_I + h_J)); d2 = (gap_x^2 + gap_y^2) + gap_z^2;
 * keep (I,J), I <= J, iff d2 <= (rc+skin)^2 (right side passed in).          */

double oracle_wrap(double x, double box)
{
    if (box <= 0.0) return x;
    double w = x - box * floor(x / box);
    if (w >= box) w -= box;
    if (w < 0.0) w = 0.0;
    return w;
}

int oracle_block_boxes(int64_t n_blocks, const int32_t *perm, const double *pos, double box,
                       double *centre /* n_blocks*3 */, double *half /* n_blocks*3 */)
{
    for (int64_t b = 0; b < n_blocks; ++b) {
        double lo[3] = { INFINITY, INFINITY, INFINITY };
        double hi[3] = { -INFINITY, -INFINITY, -INFINITY };
        for (int k = 0; k < 32; ++k) {
            int32_t a = perm[32 * b + k];
            if (a < 0) continue;
            for (int c = 0; c < 3; ++c) {
                double w = oracle_wrap(pos[3 * (int64_t)a + c], box);
                if (w < lo[c]) lo[c] = w;
                if (w > hi[c]) hi[c] = w;
            }
        }
        for (int c = 0; c < 3; ++c) {
            centre[3 * b + c] = 0.5 * (lo[c] + hi[c]);
            half[3 * b + c] = 0.5 * (hi[c] - lo[c]);
        }
    }
    return 0;
}

/* one box-box test, exactly as specified above */
static int boxes_within(const double *centre, const double *half, int64_t I, int64_t J,
                        double box, double reach2)
{
    double g2[3];
    for (int c = 0; c < 3; ++c) {
        double D = fabs(centre[3 * I + c] - centre[3 * J + c]);
        if (box > 0.0) {
            double D2 = box - D;
            if (D2 < D) D = D2;
        }
        double gap = D - (half[3 * I + c] + half[3 * J + c]);
        if (gap < 0.0) gap = 0.0;
        g2[c] = gap * gap;
    }
    double d2 = (g2[0] + g2[1]) + g2[2];
    return d2 <= reach2;
}

/* brute force over all I <= J; writes pairs (I,J) in lexicographic order.
 * Returns the number of kept pairs; if it exceeds capacity nothing is written. */
int64_t oracle_block_pairs(int64_t n_blocks, const double *centre, const double *half,
                           double box, double reach2, int32_t *pairs, int64_t capacity)
{
    int64_t *start = (int64_t *)calloc((size_t)n_blocks + 1, sizeof(int64_t));
    if (!start) return -1;
#pragma omp parallel for schedule(dynamic, 8)
    for (int64_t I = 0; I < n_blocks; ++I) {
        int64_t cnt = 0;
        for (int64_t J = I; J < n_blocks; ++J)
            cnt += boxes_within(centre, half, I, J, box, reach2);
        start[I + 1] = cnt;
    }
    for (int64_t I = 0; I < n_blocks; ++I) start[I + 1] += start[I];
    int64_t total = start[n_blocks];
    if (total <= capacity) {
#pragma omp parallel for schedule(dynamic, 8)
        for (int64_t I = 0; I < n_blocks; ++I) {
            int64_t w = start[I];
            for (int64_t J = I; J < n_blocks; ++J) {
                if (boxes_within(centre, half, I, J, box, reach2)) {
                    pairs[2 * w] = (int32_t)I;
                    pairs[2 * w + 1] = (int32_t)J;
                    ++w;
                }
            }
        }
    }
    free(start);
    return total;
}
