/*
 * qmmm_oracle.c -- CPU ORACLE (test infrastructure, NOT part of the product).
 *
 * Plain, slow, obviously-correct FP64 evaluation of the electrostatic potential and
 * field that fixed point charges produce at a set of evaluation points:
 *
 *     V(r_i) = sum_j q_j / |r_i - R_j|                    (Eq. 4)
 *     E(r_i) = -grad V(r_i) = sum_j q_j (r_i - R_j) / |r_i - R_j|^3
 *
 * Eq. 4 of the paper is U_ES(r) = sum_m rho(r_m)/|r - r_m| - sum_b Z_b/|r - R_b|,
 * the potential ENERGY of an electron (charge -1).  With cell charges
 * q_m = -rho(r_m) (x cell volume, reading 1 in DESIGN.md) and nuclear charges +Z_b
 * the quantity computed here is the electrostatic potential of a +1 test charge,
 * V = -U_ES (reading 2).  E is not in the paper; it is the term-by-term
 * negative gradient of the same expression (north_star extension).
 *
 * The paper's Eq. 5-8 only regroup the terms of
 * Eq. 4 for parallel execution, so the oracle is the definition itself: a double
 * loop in array order (grid sources first, then nuclei), every accumulator with
 * its own Kahan compensation, IEEE sqrt and divide, no FMA contraction
 * (compile with -ffp-contract=off -fno-fast-math), no blocking, no reordering.
 * OpenMP runs over evaluation points only, so the result does not depend on the
 * thread count.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / reference
 * legs may call this.  It shares no code, header, table or constant with the
 * CUDA path (paper_1011_4687_b200/csrc).
 *
 * Pins (tests/test_oracle_pins.py): single term, uniform shell by product
 * quadrature, ring / cube symmetric cases, Gaussian cloud vs erf closed form,
 * math.fsum of the terms, mpmath 50-digit brute force, scipy cdist restatement,
 * superposition, power-of-two scaling (bitwise), permutation, dyadic-lattice
 * translation (bitwise), 90-degree rotation, E = -grad V by central differences,
 * mean-value property and Gauss's law; the absolute sums absV, absE (condition
 * numbers) against |q|/d, |q|/d^2, math.fsum of numpy-formed terms and mpmath.
 * Nothing here is "parity unpinned".
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct { double s, c; } kahan_t;

/* Kahan (compensated) addition: s += x with running compensation c. */
static inline void kahan_add(kahan_t *k, double x)
{
    double y = x - k->c;
    double t = k->s + y;
    k->c = (t - k->s) - y;
    k->s = t;
}

/* One list of point charges (positions xyz[n][3], charges q[n]) added, in array
 * order, into the seven running sums of evaluation point r. */
static void accumulate_list(const double *xyz, const double *q, int64_t n,
                            const double r[3],
                            kahan_t *V, kahan_t E[3], kahan_t *absV, kahan_t *absE)
{
    for (int64_t j = 0; j < n; ++j) {
        double dx = r[0] - xyz[3 * j + 0];
        double dy = r[1] - xyz[3 * j + 1];
        double dz = r[2] - xyz[3 * j + 2];
        double r2 = dx * dx + dy * dy + dz * dz;
        double rr = sqrt(r2);
        double t  = q[j] / rr;          /* q_j / |r_i - R_j|            */
        double g  = t / r2;             /* q_j / |r_i - R_j|^3          */
        kahan_add(V, t);
        kahan_add(&E[0], g * dx);
        kahan_add(&E[1], g * dy);
        kahan_add(&E[2], g * dz);
        kahan_add(absV, fabs(t));       /* sum |q_j|/r   (condition number kappa_V) */
        kahan_add(absE, fabs(t) / rr);  /* sum |q_j|/r^2 (condition number kappa_E) */
    }
}

/*
 * qmmm_oracle_field: V[P], E[P][3] (E may be NULL), and optionally the absolute
 * sums absV[P] = sum_j |q_j|/r_ij, absE[P] = sum_j |q_j|/r_ij^2 (either may be
 * NULL) used for the condition numbers kappa_V, kappa_E of DESIGN.md.
 * All pointers are host pointers, arrays C-contiguous FP64.
 * nthreads <= 0: use the OpenMP default.  Returns the thread count used.
 */
int qmmm_oracle_field(const double *src_xyz, const double *src_q, int64_t M,
                      const double *nuc_xyz, const double *nuc_Z, int64_t K,
                      const double *elec_xyz, int64_t P,
                      double *V, double *E, double *absV, double *absE,
                      int nthreads)
{
    int used = 1;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
    used = omp_get_max_threads();
#endif
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t i = 0; i < P; ++i) {
        kahan_t v = {0.0, 0.0}, e[3] = {{0.0, 0.0}, {0.0, 0.0}, {0.0, 0.0}};
        kahan_t av = {0.0, 0.0}, ae = {0.0, 0.0};
        const double *r = elec_xyz + 3 * i;
        accumulate_list(src_xyz, src_q, M, r, &v, e, &av, &ae);   /* cells  */
        accumulate_list(nuc_xyz, nuc_Z, K, r, &v, e, &av, &ae);   /* nuclei */
        V[i] = v.s;
        if (E) { E[3 * i] = e[0].s; E[3 * i + 1] = e[1].s; E[3 * i + 2] = e[2].s; }
        if (absV) absV[i] = av.s;
        if (absE) absE[i] = ae.s;
    }
    return used;
}

/*
 * qmmm_oracle_terms: the individual potential terms t_j = q_j/|r - R_j| of ONE
 * evaluation point, in array order (cells then nuclei), for the math.fsum pin of
 * the summation.  terms has room for M + K doubles.
 */
void qmmm_oracle_terms(const double *src_xyz, const double *src_q, int64_t M,
                       const double *nuc_xyz, const double *nuc_Z, int64_t K,
                       const double r[3], double *terms)
{
    for (int64_t j = 0; j < M + K; ++j) {
        const double *p = (j < M) ? src_xyz + 3 * j : nuc_xyz + 3 * (j - M);
        double q = (j < M) ? src_q[j] : nuc_Z[j - M];
        double dx = r[0] - p[0], dy = r[1] - p[1], dz = r[2] - p[2];
        terms[j] = q / sqrt(dx * dx + dy * dy + dz * dz);
    }
}
