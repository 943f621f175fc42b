/*
 * polar_oracle_ext.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Oracle for the variants of the thin-disk path that SURVEY.md section 8(f) lists as NEXT-4 ("variants of this
 * path: unsymmetric softening, ..., fused -grad Phi output"; not in the paper -- PAPER.md:267 only names the
 * convolution method).  Same rules as polar_oracle.c: plain fp64 direct summation from the coordinates, no
 * FFT, no index-difference trick in r, nothing shared with paper_2409_02294_b200/csrc/.  The grid conventions
 * (A1, A2, A6) are those of polar_oracle.c, whose po_grid this file calls.
 *
 * Readings (N1 and N2):
 *
 *   N1  softening of a pair (field ring i, source ring i'), eps dimensionless, h = sqrt(cell area):
 *         soft = 0   e2 = eps^2 h_i h_i'     symmetric (reading A3, what polar_oracle.c computes)
 *         soft = 1   e2 = eps^2 h_i^2        softening length of the FIELD cell
 *         soft = 2   e2 = eps^2 h_i'^2       softening length of the SOURCE cell
 *       Phi_ij = - sum_{i'j'} Sigma_{i'j'} dA_{i'} / sqrt(d2),
 *       d2 = (r_i - r_i')^2 + 4 r_i r_i' sin^2((phi_j - phi_j')/2) + e2,   self term included.
 *
 *   N2  acceleration = the Plummer-softened pair force summed over the sources, the softening length of each
 *       pair held fixed, in the polar basis of the field point (x = field point, x' = source):
 *         a(x) = - sum Sigma' dA' (x - x') / (|x - x'|^2 + e2)^(3/2)
 *         a_r   = - sum Sigma' dA' (r - r' cos(dphi)) / d2^(3/2),   r - r' cos(dphi) = (r - r') + 2 r' sin^2(dphi/2)
 *         a_phi = - sum Sigma' dA'  r' sin(dphi)      / d2^(3/2),   dphi = phi_j - phi_j'
 *       (the self term contributes nothing).  For soft = 2 the softening length depends on the source only,
 *       so a = -grad Phi exactly; for soft = 0, 1 it is the force law hydro codes apply, not the gradient of
 *       the Phi above with respect to a field point that carries its own softening length.
 *
 * O0-style functions evaluate listed targets with Neumaier-compensated sums; O1-style functions evaluate whole
 * target rings with one kernel evaluation per (ring pair, azimuthal lag), two-level accumulation.
 */
#include <math.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define PO_OK 0
#define PO_EINVAL (-1)
#define PO_ENOMEM (-2)

int po_grid(int n_r, int n_phi, double r_in, double r_out, double *r, double *phi, double *area, double *edges);

static inline void nadd(double *s, double *c, double x)
{
    double t = *s + x;
    if (fabs(*s) >= fabs(x)) *c += (*s - t) + x;
    else                     *c += (x - t) + *s;
    *s = t;
}

/* N1: squared softening length of the pair (field ring area a_i, source ring area a_ip) */
static inline double soft2(int soft, double eps, double a_i, double a_ip)
{
    if (soft == 1) return eps * eps * a_i;
    if (soft == 2) return eps * eps * a_ip;
    return eps * eps * sqrt(a_i) * sqrt(a_ip);
}

typedef struct { double *r, *phi, *dA; } tables;

static int make_tables(tables *t, int n_r, int n_phi, double r_in, double r_out)
{
    t->r = (double *)malloc(sizeof(double) * n_r);
    t->phi = (double *)malloc(sizeof(double) * n_phi);
    t->dA = (double *)malloc(sizeof(double) * n_r);
    if (!t->r || !t->phi || !t->dA) return PO_ENOMEM;
    return po_grid(n_r, n_phi, r_in, r_out, t->r, t->phi, t->dA, NULL);
}
static void free_tables(tables *t) { free(t->r); free(t->phi); free(t->dA); }

/* Potential (N1) and acceleration (N2) at listed targets (flat index i*n_phi+j), the definition written out.
 * Any of out_phi / out_ar / out_aphi may be NULL. */
int po_ext_o0_targets(int n_r, int n_phi, double r_in, double r_out, double eps, int soft, const double *sigma,
                      const long *targets, long n_targets, double *out_phi, double *out_ar, double *out_aphi)
{
    if (!sigma || !targets || !(eps > 0.0) || soft < 0 || soft > 2) return PO_EINVAL;
    tables g;
    int st = make_tables(&g, n_r, n_phi, r_in, r_out);
    if (st != PO_OK) { free_tables(&g); return st; }
#pragma omp parallel for schedule(dynamic, 1)
    for (long t = 0; t < n_targets; ++t) {
        const int i = (int)(targets[t] / n_phi), j = (int)(targets[t] % n_phi);
        double sp = 0, cp = 0, sr = 0, cr = 0, sa = 0, ca = 0;
        for (int ip = 0; ip < n_r; ++ip) {
            const double dr = g.r[i] - g.r[ip];
            const double e2 = soft2(soft, eps, g.dA[i], g.dA[ip]);
            for (int jp = 0; jp < n_phi; ++jp) {
                const double dphi = g.phi[j] - g.phi[jp];
                const double sh = sin(0.5 * dphi);
                const double d2 = dr * dr + 4.0 * g.r[i] * g.r[ip] * sh * sh + e2;
                const double m = sigma[(long)ip * n_phi + jp] * g.dA[ip];
                const double inv = 1.0 / sqrt(d2);
                nadd(&sp, &cp, m * inv);
                const double inv3 = inv / d2;
                nadd(&sr, &cr, m * (dr + 2.0 * g.r[ip] * sh * sh) * inv3);
                nadd(&sa, &ca, m * g.r[ip] * sin(dphi) * inv3);
            }
        }
        if (out_phi) out_phi[t] = -(sp + cp);
        if (out_ar) out_ar[t] = -(sr + cr);
        if (out_aphi) out_aphi[t] = -(sa + ca);
    }
    free_tables(&g);
    return PO_OK;
}

/* Ring-pair form for whole target rings: the pair kernels depend on the azimuthal lag only.
 * out_*: [n_rings][n_phi]; any may be NULL. */
int po_ext_o1_rings(int n_r, int n_phi, double r_in, double r_out, double eps, int soft, const double *sigma,
                    const int *rings, int n_rings, double *out_phi, double *out_ar, double *out_aphi)
{
    if (!sigma || !rings || !(eps > 0.0) || soft < 0 || soft > 2) return PO_EINVAL;
    for (int t = 0; t < n_rings; ++t) if (rings[t] < 0 || rings[t] >= n_r) return PO_EINVAL;
    tables g;
    int st = make_tables(&g, n_r, n_phi, r_in, r_out);
    if (st != PO_OK) { free_tables(&g); return st; }
    int err = 0;
#pragma omp parallel
    {
        /* kernels by azimuthal lag l = (j - j') mod n_phi, from the coordinates of cells l apart */
        double *kp = (double *)malloc(sizeof(double) * n_phi), *kr = (double *)malloc(sizeof(double) * n_phi),
               *ka = (double *)malloc(sizeof(double) * n_phi);
        double *ap = (double *)malloc(sizeof(double) * n_phi), *ar = (double *)malloc(sizeof(double) * n_phi),
               *aa = (double *)malloc(sizeof(double) * n_phi);
        if (!kp || !kr || !ka || !ap || !ar || !aa) {
#pragma omp atomic write
            err = 1;
        }
#pragma omp barrier
        if (!err) {
#pragma omp for schedule(dynamic, 1)
            for (int t = 0; t < n_rings; ++t) {
                const int i = rings[t];
                for (int j = 0; j < n_phi; ++j) ap[j] = ar[j] = aa[j] = 0.0;
                for (int ip = 0; ip < n_r; ++ip) {
                    const double dr = g.r[i] - g.r[ip];
                    const double e2 = soft2(soft, eps, g.dA[i], g.dA[ip]);
                    for (int l = 0; l < n_phi; ++l) {
                        const double dphi = g.phi[l] - g.phi[0];
                        const double sh = sin(0.5 * dphi);
                        const double d2 = dr * dr + 4.0 * g.r[i] * g.r[ip] * sh * sh + e2;
                        const double inv = 1.0 / sqrt(d2), inv3 = inv / d2;
                        kp[l] = inv;
                        kr[l] = (dr + 2.0 * g.r[ip] * sh * sh) * inv3;
                        ka[l] = g.r[ip] * sin(dphi) * inv3;
                    }
                    const double *w = sigma + (long)ip * n_phi;
                    for (int j = 0; j < n_phi; ++j) {
                        double s0 = 0.0, s1 = 0.0, s2 = 0.0;   /* level 1: within the source ring */
                        for (int jp = 0; jp < n_phi; ++jp) {
                            int l = j - jp; if (l < 0) l += n_phi;
                            s0 += w[jp] * kp[l]; s1 += w[jp] * kr[l]; s2 += w[jp] * ka[l];
                        }
                        ap[j] += g.dA[ip] * s0; ar[j] += g.dA[ip] * s1; aa[j] += g.dA[ip] * s2;   /* level 2 */
                    }
                }
                for (int j = 0; j < n_phi; ++j) {
                    if (out_phi) out_phi[(long)t * n_phi + j] = -ap[j];
                    if (out_ar) out_ar[(long)t * n_phi + j] = -ar[j];
                    if (out_aphi) out_aphi[(long)t * n_phi + j] = -aa[j];
                }
            }
        }
        free(kp); free(kr); free(ka); free(ap); free(ar); free(aa);
    }
    free_tables(&g);
    return err ? PO_ENOMEM : PO_OK;
}
