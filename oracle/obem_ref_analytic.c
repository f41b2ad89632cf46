/*
 * obem_ref_analytic.c -- fp64 CPU ORACLE for the EXACT cell integrals of Eq (2.13)/(2.14) over flat triangles
 * (near-field-accurate panels).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules as obem_ref.c): only tests/, smoke() and bench.py's
 * cpu_baseline leg may build, load or call it; it shares nothing with paper_2110_09214_b200/csrc/.
 *
 * What it computes.  PAPER.md:141-147, section 2.2:
 *     V(r) = sum_i sigma_i/(4 pi eps0) Int_{C_i} 1/||r - r'|| d2r'                                  (2.13)
 *     E(r) = sum_i sigma_i/(4 pi eps0) Int_{C_i} (r - r')/||r - r'||^3 d2r'                         (2.14)
 * "the corresponding integrals are calculated analytically"; the paper does not print its
 * formulae (reading A1).  Here the two integrals over a flat triangle are the classical closed forms for a
 * uniformly charged planar polygon (the edge-wise decomposition used throughout the BEM literature, e.g. Wilton
 * et al., IEEE Trans. AP-32 (1984) 276; restated below in this file's own notation).  With
 *     n  = unit normal of the triangle (v1 - v0) x (v2 - v0) / ||.||,      d = n . (r - v0)   (signed height)
 *     rho = r - d n   (projection of r on the plane)
 * and, for edge i from a = v_i to b = v_{i+1}:
 *     l = (b - a)/||b - a||,  u = l x n  (in-plane outward normal),   P0 = (a - rho) . u,
 *     lm = (a - rho) . l,  lp = (b - rho) . l,   R0^2 = P0^2 + d^2,  Rm = ||r - a||,  Rp = ||r - b||,
 *     f    = ln((Rp + lp)/(Rm + lm))                      [ = Int_edge dl / R ]
 *     beta = atan(P0 lp/(R0^2 + |d| Rp)) - atan(P0 lm/(R0^2 + |d| Rm)),
 * the integrals are
 *     I_phi = Int dS/R           = sum_i ( P0_i f_i - |d| beta_i )
 *     I_E   = Int (r - r')/R^3 dS = sum_i u_i f_i  +  n sgn(d) sum_i beta_i
 * (sum_i beta_i is the solid angle the triangle subtends at r; the in-plane part is the surface-gradient theorem
 * Int grad'_s (1/R) dS = closed-loop Int u/R dl).  On the plane itself (d = 0) the normal component is 0 (the
 * principal value: the +-sigma/2eps0 jump of Eq 2.7/2.8 is not modelled, reading A8).  A point exactly on an edge
 * line with d = 0 makes that edge's f singular (the physical log singularity at the rim of a charged sheet): such
 * an edge contributes 0, like reading A4.
 *
 * Pins (tests/test_oracle_next3_pins.py; none re-types these formulas): on-axis closed form of a uniformly charged
 * rectangle down to h = 0.01 cell (P7 at small h), in-plane vertex potential k_e sigma h (asinh tan b1 + asinh tan
 * b2) (P8), the van Oosterom-Strackee solid-angle formula for the normal component, brute-force subdivided
 * quadrature (4^6 sub-triangles, 7-point rule each), E = -grad phi by central differences, Gauss flux, agreement
 * with the 7-point oracle in the far field with the (h/r)^6 slope.
 */
#include <math.h>
#include <stdint.h>
#include <stddef.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ANA_EPS0 8.8541878128e-12
#define ANA_PI   3.14159265358979323846

static double ana_dot(const double a[3], const double b[3]) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }
static void ana_cross(const double a[3], const double b[3], double c[3])
{
    c[0] = a[1] * b[2] - a[2] * b[1];
    c[1] = a[2] * b[0] - a[0] * b[2];
    c[2] = a[0] * b[1] - a[1] * b[0];
}

/* f = Int_{lm}^{lp} dl / sqrt(l^2 + R0^2) = ln((Rp + lp)/(Rm + lm)), written so that neither the numerator nor
 * the denominator cancels: (R + l)(R - l) = R0^2. */
static double ana_edge_log(double lm, double lp, double Rm, double Rp, double R02, int* singular)
{
    *singular = 0;
    if (lm >= 0.0) {
        if (Rm + lm <= 0.0) { *singular = 1; return 0.0; }       /* r is the vertex a itself */
        return log((Rp + lp) / (Rm + lm));
    }
    if (lp <= 0.0) {
        if (Rp - lp <= 0.0) { *singular = 1; return 0.0; }       /* r is the vertex b itself */
        return log((Rm - lm) / (Rp - lp));
    }
    if (R02 <= 0.0) { *singular = 1; return 0.0; }               /* r lies on the open edge */
    return log((Rp + lp) * (Rm - lm) / R02);
}

/* I_phi and I_E of ONE flat triangle (v0, v1, v2) at r.  Degenerate (zero-area) triangle: both 0. */
void obem_ref_tri_integrals(const double v0[3], const double v1[3], const double v2[3], const double r[3],
                            double* I_phi, double I_E[3])
{
    const double* V[3];
    double e1[3], e2[3], n[3], nn, d, rho[3], rel[3];
    double sum_beta = 0.0, phi = 0.0, Ein[3] = {0.0, 0.0, 0.0};
    int i, k;
    V[0] = v0; V[1] = v1; V[2] = v2;
    *I_phi = 0.0;
    I_E[0] = I_E[1] = I_E[2] = 0.0;
    for (k = 0; k < 3; ++k) { e1[k] = v1[k] - v0[k]; e2[k] = v2[k] - v0[k]; }
    ana_cross(e1, e2, n);
    nn = sqrt(ana_dot(n, n));
    if (!(nn > 0.0)) return;
    for (k = 0; k < 3; ++k) n[k] /= nn;
    for (k = 0; k < 3; ++k) rel[k] = r[k] - v0[k];
    d = ana_dot(n, rel);
    for (k = 0; k < 3; ++k) rho[k] = r[k] - d * n[k];
    for (i = 0; i < 3; ++i) {
        const double* a = V[i];
        const double* b = V[(i + 1) % 3];
        double l[3], u[3], am[3], bm[3], ra[3], rb[3], len, P0, lm, lp, R02, Rm, Rp, f, beta;
        int sing;
        for (k = 0; k < 3; ++k) l[k] = b[k] - a[k];
        len = sqrt(ana_dot(l, l));
        if (!(len > 0.0)) continue;
        for (k = 0; k < 3; ++k) l[k] /= len;
        ana_cross(l, n, u);
        for (k = 0; k < 3; ++k) { am[k] = a[k] - rho[k]; bm[k] = b[k] - rho[k]; ra[k] = r[k] - a[k]; rb[k] = r[k] - b[k]; }
        P0 = ana_dot(am, u);
        lm = ana_dot(am, l);
        lp = ana_dot(bm, l);
        R02 = P0 * P0 + d * d;
        Rm = sqrt(ana_dot(ra, ra));
        Rp = sqrt(ana_dot(rb, rb));
        f = ana_edge_log(lm, lp, Rm, Rp, R02, &sing);
        if (sing) continue;
        beta = 0.0;
        if (P0 != 0.0) {
            const double ad = fabs(d);
            beta = atan(P0 * lp / (R02 + ad * Rp)) - atan(P0 * lm / (R02 + ad * Rm));
        }
        phi += P0 * f - fabs(d) * beta;
        sum_beta += beta;
        for (k = 0; k < 3; ++k) Ein[k] += u[k] * f;
    }
    *I_phi = phi;
    {
        const double sg = (d > 0.0) ? 1.0 : ((d < 0.0) ? -1.0 : 0.0);
        for (k = 0; k < 3; ++k) I_E[k] = Ein[k] + n[k] * sg * sum_beta;
    }
}

/* Eq (2.13)/(2.14) with the exact cell integrals: out[t] = k_e sum_p sigma_p (I_E, I_phi)(panel p, target t).
 * verts [np][3][3] fp32, sigma [np] fp32, targets [nt][4] fp32 (4th lane ignored) -- the arrays the GPU gets,
 * promoted to double; out [nt][4] double = Ex, Ey, Ez, phi.  Plain summation in panel order. */
int obem_ref_eval_panels_analytic(const float* verts, const float* sigma, int64_t np, const float* targets,
                                  int64_t nt, double* out, int n_threads)
{
    const double ke = 1.0 / (4.0 * ANA_PI * ANA_EPS0);
    int64_t t;
    if (np < 0 || nt < 0 || (np > 0 && (!verts || !sigma)) || (nt > 0 && (!targets || !out))) return -1;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#else
    (void)n_threads;
#endif
#pragma omp parallel for schedule(dynamic, 4)
    for (t = 0; t < nt; ++t) {
        double r[3], acc[4] = {0.0, 0.0, 0.0, 0.0};
        int64_t p;
        int k, j;
        for (k = 0; k < 3; ++k) r[k] = (double)targets[t * 4 + k];
        for (p = 0; p < np; ++p) {
            double v[3][3], Iphi, IE[3];
            const double s = (double)sigma[p];
            for (j = 0; j < 3; ++j)
                for (k = 0; k < 3; ++k) v[j][k] = (double)verts[(p * 3 + j) * 3 + k];
            obem_ref_tri_integrals(v[0], v[1], v[2], r, &Iphi, IE);
            acc[0] += s * IE[0];
            acc[1] += s * IE[1];
            acc[2] += s * IE[2];
            acc[3] += s * Iphi;
        }
        for (k = 0; k < 4; ++k) out[t * 4 + k] = ke * acc[k];
    }
    return 0;
}
