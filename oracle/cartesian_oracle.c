/*
 * cartesian_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Oracle for row NEXT-2 of SURVEY.md section 8(f): the paper's own per-GPU workload, "the convolution method for
 * solving potential fields on nested grids in three dimensions" (section 3) on ONE uniform Cartesian
 * mesh level of N^3 cells, N = 64 or 128 in the paper's runs.  The numerical method itself is in the
 * paper's ref. [13], which is not available here, and PAPER.md prints no formula; the definition
 * below is the plain Newtonian sum with the readings C1-C4 of DESIGN.md section 3:
 *
 *   C1  cell-centred uniform mesh, N x N x N cells of size h = box / N; array order [z][y][x], x fastest.
 *   C2  Phi_c = -G h^3 sum_{c'} rho_{c'} g(c - c'),   g(d) = 1 / (h |d|) for d != 0   (cells as point masses), G = 1.
 *   C3  self term: g(0) = S / h with S = integral over the unit cube of 1/|x| = 3 ln(2 + sqrt 3) - pi/2
 *       (= 2.38007...: the potential at the centre of a homogeneous cube), so that a cell's own mass is spread over
 *       its volume instead of sitting on the field point.
 *   C4  isolated (vacuum) boundary: the sum runs over the N^3 cells of the mesh only, no periodic images -- what the
 *       zero padding of the convolution method achieves.
 *
 * Plain triple loops from the cell indices, Neumaier-compensated; shares nothing with paper_2409_02294_b200/csrc/.
 * Pins: tests/test_oracle3d_pins.py (S by quadrature, 50-digit brute force, single cell, cube symmetries, shifts,
 * far field).
 */
#include <math.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define PO_OK 0
#define PO_EINVAL (-1)

/* C3: integral of 1/|x| over the unit cube centred on the origin */
double po3_self_constant(void) { return 3.0 * log(2.0 + sqrt(3.0)) - 2.0 * atan(1.0); }

static inline void nadd3(double *s, double *c, double x)
{
    double t = *s + x;
    if (fabs(*s) >= fabs(x)) *c += (*s - t) + x;
    else                     *c += (x - t) + *s;
    *s = t;
}

/* Potential at listed target cells (flat index (z*N + y)*N + x). rho: [N][N][N]. */
int po3_potential_targets(int n, double box, const double *rho, const long *targets, long n_targets, double *out)
{
    if (n < 1 || !(box > 0.0) || !rho || !targets || !out) return PO_EINVAL;
    const double h = box / (double)n;
    const double self = po3_self_constant();
#pragma omp parallel for schedule(dynamic, 1)
    for (long t = 0; t < n_targets; ++t) {
        const int x = (int)(targets[t] % n), y = (int)((targets[t] / n) % n), z = (int)(targets[t] / ((long)n * n));
        double s = 0.0, c = 0.0;
        for (int zp = 0; zp < n; ++zp)
            for (int yp = 0; yp < n; ++yp)
                for (int xp = 0; xp < n; ++xp) {
                    const double dx = x - xp, dy = y - yp, dz = z - zp;
                    const double d2 = dx * dx + dy * dy + dz * dz;
                    const double g = d2 > 0.0 ? 1.0 / sqrt(d2) : self;
                    nadd3(&s, &c, rho[((long)zp * n + yp) * n + xp] * g);
                }
        out[t] = -(s + c) * h * h;          /* h^3 * (1/h) */
    }
    return PO_OK;
}

int po3_potential_full(int n, double box, const double *rho, double *out)
{
    const long m = (long)n * n * n;
    long *tg = (long *)malloc(sizeof(long) * m);
    if (!tg) return -2;
    for (long t = 0; t < m; ++t) tg[t] = t;
    int st = po3_potential_targets(n, box, rho, tg, m, out);
    free(tg);
    return st;
}
