/*
 * polar_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU direct summation of the thin-disk potential on a
 * log-polar grid.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call this file.
 * It shares no code, header, table or constant with the CUDA path under
 * paper_2409_02294_b200/csrc/, and neither includes the other.
 *
 * What it computes (BASELINE.json north_star; conventions = the readings
 * A1..A8 listed in SURVEY.md section 8(c) and DESIGN.md section 3, because
 * PAPER.md prints no formula -- PAPER.md:267 only names "the convolution
 * method for solving potential fields"):
 *
 *   edges    re_i = r_in * (r_out/r_in)^(i/N_r),  i = 0..N_r            (A1)
 *   centres  r_i  = sqrt(re_i * re_{i+1})          (geometric centre)   (A1)
 *            phi_j = (j + 1/2) * dphi,  dphi = 2 pi / N_phi             (A6)
 *   area     dA_i = (re_{i+1}^2 - re_i^2)/2 * dphi (exact sector)       (A2)
 *   size     h_i  = sqrt(dA_i)
 *   soften   e2(i,i') = eps^2 * h_i * h_i'                              (A3)
 *   dist^2   d2 = (r_i - r_i')^2 + 4 r_i r_i' sin^2((phi_j - phi_j')/2) + e2
 *   result   Phi_ij = -G * sum_{i'j'} Sigma_{i'j'} dA_{i'} / sqrt(d2),
 *            G = 1, self term (i'=i, j'=j) included                     (A4, A5)
 *
 * Two implementations of that same sum:
 *   O0  po_potential_o0_*  the definition, four nested loops from the
 *       coordinates, Neumaier-compensated accumulation.
 *   O1  po_potential_o1_*  ring-pair form: for a ring pair (i,i') the pair
 *       kernel depends on j-j' only (uniform phi grid, exact rotational
 *       symmetry), so g_l = 1/sqrt(d2(l)) is evaluated once per l and reused
 *       for all N_phi targets of the ring; two-level accumulation (A8).
 *       No FFT, no index-difference trick in r.
 *
 * Pins (tests/test_oracle_pins.py): elliptic-integral ring closed form,
 * 50-digit brute force on tiny grids, single-cell response, far-field
 * monopole + quadrupole, phi-independence, linearity, roll, reciprocity,
 * scale covariance, total area.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define PO_OK 0
#define PO_EINVAL (-1)
#define PO_ENOMEM (-2)

static const double PO_TWO_PI = 6.283185307179586476925286766559;

int po_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* Grid tables from the edge definition (A1, A2).  Any output may be NULL. */
int po_grid(int n_r, int n_phi, double r_in, double r_out,
            double *r, double *phi, double *area, double *edges)
{
    if (n_r < 1 || n_phi < 1 || !(r_in > 0.0) || !(r_out > r_in)) return PO_EINVAL;
    const double dphi = PO_TWO_PI / (double)n_phi;
    const double ratio = r_out / r_in;
    double lo = r_in;
    for (int i = 0; i < n_r; ++i) {
        double hi = (i + 1 == n_r) ? r_out : r_in * pow(ratio, (double)(i + 1) / (double)n_r);
        if (edges) { edges[i] = lo; edges[i + 1] = hi; }
        if (r) r[i] = sqrt(lo * hi);
        if (area) area[i] = 0.5 * (hi - lo) * (hi + lo) * dphi;
        lo = hi;
    }
    if (phi) for (int j = 0; j < n_phi; ++j) phi[j] = ((double)j + 0.5) * dphi;
    return PO_OK;
}

/* Neumaier compensated accumulation: (s, c) += x */
static inline void neumaier_add(double *s, double *c, double x)
{
    double t = *s + x;
    if (fabs(*s) >= fabs(x)) *c += (*s - t) + x;
    else                     *c += (x - t) + *s;
    *s = t;
}

/* O0: the definition, evaluated for a list of targets (flat index i*n_phi+j).
 * sigma: [n_r][n_phi]; out: [n_targets]. */
int po_potential_o0_targets(int n_r, int n_phi, double r_in, double r_out, double eps,
                            const double *sigma, const long *targets, long n_targets,
                            double *out)
{
    if (!sigma || !targets || !out || !(eps > 0.0)) return PO_EINVAL;
    double *r = (double *)malloc(sizeof(double) * n_r);
    double *phi = (double *)malloc(sizeof(double) * n_phi);
    double *dA = (double *)malloc(sizeof(double) * n_r);
    if (!r || !phi || !dA) { free(r); free(phi); free(dA); return PO_ENOMEM; }
    int st = po_grid(n_r, n_phi, r_in, r_out, r, phi, dA, NULL);
    if (st != PO_OK) { free(r); free(phi); free(dA); return st; }

#pragma omp parallel for schedule(dynamic, 1)
    for (long t = 0; t < n_targets; ++t) {
        const int i = (int)(targets[t] / n_phi), j = (int)(targets[t] % n_phi);
        const double hi = sqrt(dA[i]);
        double s = 0.0, c = 0.0;
        for (int ip = 0; ip < n_r; ++ip) {
            const double dr = r[i] - r[ip];
            const double e2 = eps * eps * hi * sqrt(dA[ip]);
            const double rr4 = 4.0 * r[i] * r[ip];
            for (int jp = 0; jp < n_phi; ++jp) {
                const double sh = sin(0.5 * (phi[j] - phi[jp]));
                const double d2 = dr * dr + rr4 * sh * sh + e2;
                neumaier_add(&s, &c, sigma[(long)ip * n_phi + jp] * dA[ip] / sqrt(d2));
            }
        }
        out[t] = -(s + c);
    }
    free(r); free(phi); free(dA);
    return PO_OK;
}

/* O0 on the whole grid. out: [n_r][n_phi]. */
int po_potential_o0_full(int n_r, int n_phi, double r_in, double r_out, double eps,
                         const double *sigma, double *out)
{
    const long n = (long)n_r * n_phi;
    long *tg = (long *)malloc(sizeof(long) * n);
    if (!tg) return PO_ENOMEM;
    for (long t = 0; t < n; ++t) tg[t] = t;
    int st = po_potential_o0_targets(n_r, n_phi, r_in, r_out, eps, sigma, tg, n, out);
    free(tg);
    return st;
}

/* O1: ring-pair form for a list of target rings.  out: [n_rings][n_phi]. */
int po_potential_o1_rings(int n_r, int n_phi, double r_in, double r_out, double eps,
                          const double *sigma, const int *rings, int n_rings, double *out)
{
    if (!sigma || !rings || !out || !(eps > 0.0)) return PO_EINVAL;
    double *r = (double *)malloc(sizeof(double) * n_r);
    double *phi = (double *)malloc(sizeof(double) * n_phi);
    double *dA = (double *)malloc(sizeof(double) * n_r);
    double *s2 = (double *)malloc(sizeof(double) * n_phi);
    if (!r || !phi || !dA || !s2) { free(r); free(phi); free(dA); free(s2); return PO_ENOMEM; }
    int st = po_grid(n_r, n_phi, r_in, r_out, r, phi, dA, NULL);
    if (st != PO_OK) { free(r); free(phi); free(dA); free(s2); return st; }
    for (int i = 0; i < n_rings; ++i)
        if (rings[i] < 0 || rings[i] >= n_r) { free(r); free(phi); free(dA); free(s2); return PO_EINVAL; }
    /* sin^2 of half the azimuthal separation of cells l apart, from the coordinates */
    for (int l = 0; l < n_phi; ++l) {
        const double sh = sin(0.5 * (phi[l] - phi[0]));
        s2[l] = sh * sh;
    }
    int err = 0;
#pragma omp parallel
    {
        /* grev[q] = g[(n_phi - q) mod n_phi] on a doubled array, so that
         * sum_{j'} w[j'] * g[(j - j') mod n] = sum_{j'} w[j'] * grev[j' - j + n]  (contiguous) */
        double *grev = (double *)malloc(sizeof(double) * 2 * (size_t)n_phi);
        double *acc = (double *)malloc(sizeof(double) * (size_t)n_phi);
        if (!grev || !acc) {
#pragma omp atomic write
            err = 1;
        }
#pragma omp barrier
        if (!err) {
#pragma omp for schedule(dynamic, 1)
            for (int t = 0; t < n_rings; ++t) {
                const int i = rings[t];
                const double hi = sqrt(dA[i]);
                for (int j = 0; j < n_phi; ++j) acc[j] = 0.0;
                for (int ip = 0; ip < n_r; ++ip) {
                    const double dr = r[i] - r[ip];
                    const double base = dr * dr + eps * eps * hi * sqrt(dA[ip]);
                    const double rr4 = 4.0 * r[i] * r[ip];
                    for (int q = 0; q < 2 * n_phi; ++q) {
                        const int l = (2 * n_phi - q) % n_phi;
                        grev[q] = 1.0 / sqrt(base + rr4 * s2[l]);
                    }
                    const double *w = sigma + (long)ip * n_phi;
                    const double a = dA[ip];
                    for (int j = 0; j < n_phi; ++j) {
                        const double *g = grev + (n_phi - j);
                        double ring = 0.0;                 /* level 1: within the source ring */
#pragma omp simd reduction(+ : ring)
                        for (int jp = 0; jp < n_phi; ++jp) ring += w[jp] * g[jp];
                        acc[j] += a * ring;                /* level 2: over source rings */
                    }
                }
                for (int j = 0; j < n_phi; ++j) out[(long)t * n_phi + j] = -acc[j];
            }
        }
        free(grev); free(acc);
    }
    free(r); free(phi); free(dA); free(s2);
    return err ? PO_ENOMEM : PO_OK;
}

/* O1 on the whole grid. out: [n_r][n_phi]. */
int po_potential_o1_full(int n_r, int n_phi, double r_in, double r_out, double eps,
                         const double *sigma, double *out)
{
    int *rg = (int *)malloc(sizeof(int) * n_r);
    if (!rg) return PO_ENOMEM;
    for (int i = 0; i < n_r; ++i) rg[i] = i;
    int st = po_potential_o1_rings(n_r, n_phi, r_in, r_out, eps, sigma, rg, n_r, out);
    free(rg);
    return st;
}
