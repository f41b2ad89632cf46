/*
 * obem_ref.c -- fp64 CPU ORACLE for the OuroborosBEM field-evaluation hot path (arXiv 2110.09214).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may build, load or call it.  It shares no code,
 * header, table or constant generator with the CUDA path under paper_2110_09214_b200/csrc/.
 *
 * What it computes (plain definition, written out; no blocking, fusion or reordering):
 *
 *   N-body part  -- PAPER.md:272-277, section 3.2.4, Eq (3.8):
 *       E_Nbody(r_p') = 1/(4 pi eps0) * sum_{p != p'} q_p (r_p' - r_p) / ||r_p' - r_p||^3
 *     with the Plummer softening BASELINE.json adds (reading A2):
 *       r2 = ||d||^2 + eps_pp^2,  E += q d / r2^(3/2),  phi += q / r2^(1/2);   eps_pp = 0 is Eq (3.8).
 *     The self term is excluded BY INDEX (reading A3), never by position.
 *
 *   Panel part   -- PAPER.md:141-147, section 2.2, Eq (2.13) and (2.14):
 *       V(r) = sum_i sigma_i/(4 pi eps0) * Int_{C_i} 1/||r - r'|| d2r'
 *       E(r) = sum_i sigma_i/(4 pi eps0) * Int_{C_i} (r - r')/||r - r'||^3 d2r'
 *     sigma_i constant over the flat cell C_i.  The surface integral over each flat
 *     triangle is taken with the 7-point degree-5 rule BASELINE.json fixes for the synthetic configs
 *     (reading A1: the paper's analytic integrals are not published).
 *
 *   Both sums follow the sign convention (r - r') of the paper: E points away from positive charge.
 *   A source at exactly zero (softened) distance contributes 0 (reading A4).
 *   The two parts are returned separately (superposition) so each is checked alone.
 *
 * Inputs are the same fp32 arrays the GPU path gets, promoted to double; all arithmetic is double,
 * plain left-to-right summation in source order.
 *
 * Pins (tests/test_oracle_pins.py, none of them re-types these loops): point-charge closed form,
 * hand-computed 2- and 3-body values, Newton's third law, Gauss flux through a sphere (charges and
 * panels), monomial exactness of the 7-point rule up to degree 5 and its failure at degree 6, far
 * field of a charged triangle -> k_e Q / r^2 with (h/r)^2 slope, on-axis field of a uniformly charged
 * rectangle (closed form), parallel plates sigma/eps0, rotation / translation / scaling invariance,
 * linearity, neutral-pair force.  Every function here is pinned; none is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stddef.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* reading A7: e and eps0 are CODATA 2018; k_e = 1/(4 pi eps0). */
#define OBEM_REF_EPS0 8.8541878128e-12
#define OBEM_REF_PI   3.14159265358979323846

#define OBEM_REF_NBODY  1u
#define OBEM_REF_PANELS 2u

static double ref_ke(void) { return 1.0 / (4.0 * OBEM_REF_PI * OBEM_REF_EPS0); }

/* 7-point degree-5 rule on a triangle (Radon 1948; tabulated e.g. in Strang & Fix): barycentric
 * coordinates l[k][0..2] and weights w[k], sum w = 1 (multiply by the triangle's area).
 * SURVEY.md section 8(c) table.  Filled at run time from the closed-form surds. */
void obem_ref_quad_rule(double l[7][3], double w[7])
{
    const double s15 = sqrt(15.0);
    const double b1 = (6.0 - s15) / 21.0, a1 = 1.0 - 2.0 * b1, w1 = (155.0 - s15) / 1200.0;
    const double b2 = (6.0 + s15) / 21.0, a2 = 1.0 - 2.0 * b2, w2 = (155.0 + s15) / 1200.0;
    int k, j;
    l[0][0] = l[0][1] = l[0][2] = 1.0 / 3.0;
    w[0] = 9.0 / 40.0;
    for (k = 0; k < 3; ++k) {
        for (j = 0; j < 3; ++j) {
            l[1 + k][j] = (j == k) ? a1 : b1;
            l[4 + k][j] = (j == k) ? a2 : b2;
        }
        w[1 + k] = w1;
        w[4 + k] = w2;
    }
}

/* Area of the flat triangle (v0, v1, v2): A = 1/2 ||(v1 - v0) x (v2 - v0)||. */
static double ref_tri_area(const double v0[3], const double v1[3], const double v2[3])
{
    double a[3], b[3], c[3];
    int d;
    for (d = 0; d < 3; ++d) { a[d] = v1[d] - v0[d]; b[d] = v2[d] - v0[d]; }
    c[0] = a[1] * b[2] - a[2] * b[1];
    c[1] = a[2] * b[0] - a[0] * b[2];
    c[2] = a[0] * b[1] - a[1] * b[0];
    return 0.5 * sqrt(c[0] * c[0] + c[1] * c[1] + c[2] * c[2]);
}

/* Quadrature sources of every panel, for inspection by the tests:
 * out[(p*7+k)*4 + 0..2] = x_pk = sum_j l_kj v_j,  out[..+3] = sigma_p * A_p * w_k  (units C). */
int obem_ref_panel_sources(const float* verts /*[np][3][3]*/, const float* sigma /*[np]*/,
                           int64_t np, double* out /*[np*7][4]*/)
{
    double l[7][3], w[7];
    int64_t p;
    if (np < 0 || (np > 0 && (!verts || !sigma || !out))) return -1;
    obem_ref_quad_rule(l, w);
    for (p = 0; p < np; ++p) {
        double v[3][3];
        int j, d, k;
        double A;
        for (j = 0; j < 3; ++j) for (d = 0; d < 3; ++d) v[j][d] = (double)verts[(p * 3 + j) * 3 + d];
        A = ref_tri_area(v[0], v[1], v[2]);
        for (k = 0; k < 7; ++k) {
            for (d = 0; d < 3; ++d)
                out[(p * 7 + k) * 4 + d] = l[k][0] * v[0][d] + l[k][1] * v[1][d] + l[k][2] * v[2][d];
            out[(p * 7 + k) * 4 + 3] = (double)sigma[p] * A * w[k];
        }
    }
    return 0;
}

/*
 * The oracle proper.  Host pointers only.
 *   xyzq      [n][4]  fp32 (x, y, z [m], q [C])                 charges (sources of the N-body part)
 *   verts     [np][3][3] fp32 [m], sigma [np] fp32 [C/m^2]       panels
 *   targets   [nt][4] fp32, 4th lane ignored
 *   self_index[nt]    index into xyzq of the charge the target IS (excluded from its own sum),
 *                     or -1 for a free point; may be NULL (= all -1)
 *   flags     OBEM_REF_NBODY | OBEM_REF_PANELS
 *   out_nbody [nt][4], out_panel [nt][4]  double (Ex, Ey, Ez [V/m], phi [V]); a part whose flag is
 *                     clear is written as zeros; either pointer may be NULL if its flag is clear
 *   n_threads OpenMP threads over targets (<= 0: library default).  Threads split TARGETS only; the
 *             sum for one target is always one thread, in source order.
 * Returns 0, or -1 on a bad argument.
 */
int obem_ref_eval(const float* xyzq, int64_t n, const float* verts, const float* sigma, int64_t np,
                  double eps_pp, double eps_panel, const float* targets, const int64_t* self_index,
                  int64_t nt, unsigned flags, double* out_nbody, double* out_panel, int n_threads)
{
    double l[7][3], w[7];
    const double ke = ref_ke();
    int64_t t;
    if (n < 0 || np < 0 || nt < 0) return -1;
    if (nt > 0 && !targets) return -1;
    if ((flags & OBEM_REF_NBODY) && ((n > 0 && !xyzq) || (nt > 0 && !out_nbody))) return -1;
    if ((flags & OBEM_REF_PANELS) && ((np > 0 && (!verts || !sigma)) || (nt > 0 && !out_panel))) return -1;
    obem_ref_quad_rule(l, w);
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#else
    (void)n_threads;
#endif

#pragma omp parallel for schedule(dynamic, 16)
    for (t = 0; t < nt; ++t) {
        const double rx = (double)targets[t * 4 + 0];
        const double ry = (double)targets[t * 4 + 1];
        const double rz = (double)targets[t * 4 + 2];
        const int64_t self = self_index ? self_index[t] : -1;

        if (out_nbody) {
            double ex = 0.0, ey = 0.0, ez = 0.0, ph = 0.0;
            if (flags & OBEM_REF_NBODY) {
                int64_t j;
                for (j = 0; j < n; ++j) {                       /* Eq (3.8): sum over p != p' */
                    double dx, dy, dz, r2, inv, q;
                    if (j == self) continue;
                    dx = rx - (double)xyzq[j * 4 + 0];          /* r_p' - r_p */
                    dy = ry - (double)xyzq[j * 4 + 1];
                    dz = rz - (double)xyzq[j * 4 + 2];
                    r2 = dx * dx + dy * dy + dz * dz + eps_pp * eps_pp;
                    if (r2 == 0.0) continue;                    /* reading A4 */
                    inv = 1.0 / sqrt(r2);
                    q = (double)xyzq[j * 4 + 3];
                    ph += q * inv;
                    ex += q * inv * inv * inv * dx;
                    ey += q * inv * inv * inv * dy;
                    ez += q * inv * inv * inv * dz;
                }
            }
            out_nbody[t * 4 + 0] = ke * ex;
            out_nbody[t * 4 + 1] = ke * ey;
            out_nbody[t * 4 + 2] = ke * ez;
            out_nbody[t * 4 + 3] = ke * ph;
        }

        if (out_panel) {
            double ex = 0.0, ey = 0.0, ez = 0.0, ph = 0.0;
            if (flags & OBEM_REF_PANELS) {
                int64_t p;
                for (p = 0; p < np; ++p) {                      /* Eq (2.13)/(2.14): sum over cells */
                    double v[3][3], A;
                    int j, d, k;
                    for (j = 0; j < 3; ++j)
                        for (d = 0; d < 3; ++d) v[j][d] = (double)verts[(p * 3 + j) * 3 + d];
                    A = ref_tri_area(v[0], v[1], v[2]);
                    for (k = 0; k < 7; ++k) {                   /* 7-point rule for Int_{C_i} ... d2r' */
                        const double x = l[k][0] * v[0][0] + l[k][1] * v[1][0] + l[k][2] * v[2][0];
                        const double y = l[k][0] * v[0][1] + l[k][1] * v[1][1] + l[k][2] * v[2][1];
                        const double z = l[k][0] * v[0][2] + l[k][1] * v[1][2] + l[k][2] * v[2][2];
                        const double dx = rx - x, dy = ry - y, dz = rz - z;   /* r - r' */
                        const double r2 = dx * dx + dy * dy + dz * dz + eps_panel * eps_panel;
                        double inv, wq;
                        if (r2 == 0.0) continue;                /* reading A4 */
                        inv = 1.0 / sqrt(r2);
                        wq = (double)sigma[p] * A * w[k];       /* sigma_i * (area element) */
                        ph += wq * inv;
                        ex += wq * inv * inv * inv * dx;
                        ey += wq * inv * inv * inv * dy;
                        ez += wq * inv * inv * inv * dz;
                    }
                }
            }
            out_panel[t * 4 + 0] = ke * ex;
            out_panel[t * 4 + 1] = ke * ey;
            out_panel[t * 4 + 2] = ke * ez;
            out_panel[t * 4 + 3] = ke * ph;
        }
    }
    return 0;
}

/* Number of OpenMP threads a call with n_threads <= 0 would use (for the bench's "cores" field). */
int obem_ref_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
