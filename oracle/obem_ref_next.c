/*
 * obem_ref_next.c -- fp64 CPU ORACLE for the steps adjacent to the field-evaluation hot path
 * of the OuroborosBEM method (arXiv 2110.09214).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules as obem_ref.c): only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may build, load or call
 * it; it shares no code, header, table or constant generator with paper_2110_09214_b200/csrc/.
 *
 * NEXT-1  influence of the particles on the cells, section 3.2.2:
 *   obem_ref_influence   Eq (3.3), (3.4): area-averaged potential and field of all particles over cell C_i
 *   obem_ref_rhs         Eq (3.5), (3.6): left-hand sides V_i - Vbar_i (ed cells), sigma_F,i - (eps2-eps1) Ebar_i.n_i
 *   obem_ref_matvec      sigma = M^-1 b with the stored inverse
 *
 * All arithmetic is double, plain loops in the order the equations are written.  The surface average
 * (1/A_i) Int_{C_i} f d2r is taken with the same 7-point degree-5 rule as the panel sums (DESIGN.md
 * reading A1): sum_k w_k f(x_ik), weights summing to 1; the rule itself is obem_ref_quad_rule (obem_ref.c).
 *
 * Pins (tests/test_oracle_next_pins.py; none re-types these loops): Green reciprocity against the
 * separately pinned panel oracle (sum_i sigma_i A_i Vbar_i = sum_p q_p phi_panels(r_p) and the momentum
 * version for E), flux of a point charge through a meshed rectangle against the solid-angle closed form,
 * far-charge limit k_e q / R, hand values for the right-hand side, numpy's matmul and the identity /
 * permutation special cases for the mat-vec.
 */
#include <math.h>
#include <stdint.h>
#include <stddef.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define NEXT_EPS0 8.8541878128e-12
#define NEXT_PI   3.14159265358979323846

void obem_ref_quad_rule(double l[7][3], double w[7]); /* obem_ref.c */

static double next_ke(void) { return 1.0 / (4.0 * NEXT_PI * NEXT_EPS0); }

/* Unit normal of the flat triangle, n = (v1 - v0) x (v2 - v0) / ||.|| (orientation = vertex order, DESIGN.md
 * reading A16), and its area.  A degenerate triangle gets n = 0, A = 0. */
static void next_normal_area(const double v[3][3], double nrm[3], double* area)
{
    double a[3], b[3], c[3], len;
    int d;
    for (d = 0; d < 3; ++d) { a[d] = v[1][d] - v[0][d]; b[d] = v[2][d] - v[0][d]; }
    c[0] = a[1] * b[2] - a[2] * b[1];
    c[1] = a[2] * b[0] - a[0] * b[2];
    c[2] = a[0] * b[1] - a[1] * b[0];
    len = sqrt(c[0] * c[0] + c[1] * c[1] + c[2] * c[2]);
    *area = 0.5 * len;
    for (d = 0; d < 3; ++d) nrm[d] = (len > 0.0) ? c[d] / len : 0.0;
}

/*
 * Eq (3.3) and (3.4), PAPER.md:245-249:
 *   Vbar_i = 1/(4 pi eps0) sum_p q_p / A_i  Int_{C_i} 1/||r - r_p|| d2r
 *   Ebar_i = 1/(4 pi eps0) sum_p q_p / A_i  Int_{C_i} (r - r_p)/||r - r_p||^3 d2r
 * with (1/A_i) Int_{C_i} f d2r = sum_k w_k f(x_ik).  eps: softening of the cell-particle distance (same
 * role as eps_panel in the panel sums; 0 = the equations as printed); zero distance contributes 0 (A4).
 *   out    [np][4] = (Ebar_x, Ebar_y, Ebar_z [V/m], Vbar [V])
 *   out_en [np]    = Ebar_i . n_i (the quantity Eq (3.6) needs), may be NULL
 *   out_na [np][4] = (n_x, n_y, n_z, A_i), may be NULL
 */
int obem_ref_influence(const float* xyzq, int64_t n, const float* verts, int64_t np, double eps,
                       double* out, double* out_en, double* out_na, int n_threads)
{
    double l[7][3], w[7];
    const double ke = next_ke();
    int64_t i;
    if (n < 0 || np < 0 || (n > 0 && !xyzq) || (np > 0 && (!verts || !out))) return -1;
    obem_ref_quad_rule(l, w);
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#else
    (void)n_threads;
#endif
#pragma omp parallel for schedule(dynamic, 4)
    for (i = 0; i < np; ++i) {
        double v[3][3], nrm[3], A;
        double ex = 0.0, ey = 0.0, ez = 0.0, vb = 0.0;
        int j, d, k;
        int64_t p;
        for (j = 0; j < 3; ++j) for (d = 0; d < 3; ++d) v[j][d] = (double)verts[(i * 3 + j) * 3 + d];
        next_normal_area(v, nrm, &A);
        for (p = 0; p < n; ++p) {                              /* sum over the particles */
            const double px = (double)xyzq[p * 4 + 0], py = (double)xyzq[p * 4 + 1], pz = (double)xyzq[p * 4 + 2];
            const double q = (double)xyzq[p * 4 + 3];
            for (k = 0; k < 7; ++k) {                          /* (1/A_i) Int_{C_i} ... d2r */
                const double x = l[k][0] * v[0][0] + l[k][1] * v[1][0] + l[k][2] * v[2][0];
                const double y = l[k][0] * v[0][1] + l[k][1] * v[1][1] + l[k][2] * v[2][1];
                const double z = l[k][0] * v[0][2] + l[k][1] * v[1][2] + l[k][2] * v[2][2];
                const double dx = x - px, dy = y - py, dz = z - pz;     /* r - r_p */
                const double r2 = dx * dx + dy * dy + dz * dz + eps * eps;
                double inv;
                if (r2 == 0.0) continue;
                inv = 1.0 / sqrt(r2);
                vb += q * w[k] * inv;
                ex += q * w[k] * inv * inv * inv * dx;
                ey += q * w[k] * inv * inv * inv * dy;
                ez += q * w[k] * inv * inv * inv * dz;
            }
        }
        out[i * 4 + 0] = ke * ex;
        out[i * 4 + 1] = ke * ey;
        out[i * 4 + 2] = ke * ez;
        out[i * 4 + 3] = ke * vb;
        if (out_en) out_en[i] = ke * (ex * nrm[0] + ey * nrm[1] + ez * nrm[2]);
        if (out_na) { out_na[i * 4 + 0] = nrm[0]; out_na[i * 4 + 1] = nrm[1]; out_na[i * 4 + 2] = nrm[2]; out_na[i * 4 + 3] = A; }
    }
    return 0;
}

/*
 * Eq (3.5) and (3.6): the modified left-hand sides of the BEM system,
 *   kind[i] == 0 (ed cell, electrode):       b_i = V_i - Vbar_i
 *   kind[i] == 1 (dd cell, dielectric face): b_i = sigma_F,i - (eps2 - eps1)_i * (Ebar_i . n_i)
 * bc[i] is V_i [V] or sigma_F,i [C/m^2]; deps[i] = eps2 - eps1 [F/m] (unused for ed cells);
 * infl [np][4] and en [np] as returned by obem_ref_influence.
 */
int obem_ref_rhs(const int32_t* kind, const float* bc, const float* deps, const double* infl, const double* en,
                 int64_t np, double* b)
{
    int64_t i;
    if (np < 0 || (np > 0 && (!kind || !bc || !deps || !infl || !en || !b))) return -1;
    for (i = 0; i < np; ++i) {
        if (kind[i] == 0) b[i] = (double)bc[i] - infl[i * 4 + 3];
        else if (kind[i] == 1) b[i] = (double)bc[i] - (double)deps[i] * en[i];
        else return -1;
    }
    return 0;
}

/* sigma = M^-1 b (the inverse is computed once and stored; every new right-hand side is a
 * matrix-vector product).  minv [n][ld] row-major fp32 (ld >= n), b [n] fp32, sigma [n] double. */
int obem_ref_matvec(const float* minv, int64_t n, int64_t ld, const float* b, double* sigma, int n_threads)
{
    int64_t i;
    if (n < 0 || ld < n || (n > 0 && (!minv || !b || !sigma))) return -1;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#else
    (void)n_threads;
#endif
#pragma omp parallel for schedule(static)
    for (i = 0; i < n; ++i) {
        double s = 0.0;
        int64_t j;
        for (j = 0; j < n; ++j) s += (double)minv[i * ld + j] * (double)b[j];
        sigma[i] = s;
    }
    return 0;
}

/*
 * NEXT-2  electron-ion recombination, PAPER.md:341-355 (section 3.3.3): "taken into account microscopically for
 * any electron and ion using the distances obtained during the N-body calculation process".  For every charge i
 * the nearest charge of OPPOSITE sign: its true (unsoftened) distance d_i and its index j_i (ties: the smallest
 * index; -1 and d = +infinity if there is no opposite charge).  Charges with q = 0 have no partner and are nobody's
 * partner.
 */
int obem_ref_nearest_opposite_subset(const float* xyzq, int64_t n, const int64_t* idx, int64_t nidx, double* out_d,
                                     int64_t* out_j, int n_threads);

int obem_ref_nearest_opposite(const float* xyzq, int64_t n, double* out_d, int64_t* out_j, int n_threads)
{
    return obem_ref_nearest_opposite_subset(xyzq, n, NULL, n, out_d, out_j, n_threads);
}

/* Same for the charges idx[0..nidx) only (idx == NULL: charge t itself, nidx = n); out_d, out_j have nidx entries.
 * The candidates are always ALL n charges. */
int obem_ref_nearest_opposite_subset(const float* xyzq, int64_t n, const int64_t* idx, int64_t nidx, double* out_d,
                                     int64_t* out_j, int n_threads)
{
    int64_t t;
    if (n < 0 || nidx < 0 || (nidx > 0 && (!xyzq || !out_d || !out_j))) return -1;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#else
    (void)n_threads;
#endif
#pragma omp parallel for schedule(dynamic, 16)
    for (t = 0; t < nidx; ++t) {
        const int64_t i = idx ? idx[t] : t;
        const double x = (double)xyzq[i * 4 + 0], y = (double)xyzq[i * 4 + 1], z = (double)xyzq[i * 4 + 2];
        const double q = (double)xyzq[i * 4 + 3];
        double best = INFINITY;
        int64_t bj = -1, j;
        for (j = 0; j < n; ++j) {
            double dx, dy, dz, r2;
            if (j == i) continue;
            if (!(q * (double)xyzq[j * 4 + 3] < 0.0)) continue;       /* opposite polarity only */
            dx = x - (double)xyzq[j * 4 + 0];
            dy = y - (double)xyzq[j * 4 + 1];
            dz = z - (double)xyzq[j * 4 + 2];
            r2 = dx * dx + dy * dy + dz * dz;
            if (r2 < best) { best = r2; bj = j; }
        }
        out_d[t] = (bj >= 0) ? sqrt(best) : INFINITY;
        out_j[t] = bj;
    }
    return 0;
}

/* Eq (3.12): a pair recombines when d <= 1/(4 pi eps0) * e / (2 E_ioni), E_ioni the ionisation
 * energy.  With E_ioni given in eV (= volts times e) the right-hand side is k_e * e / (2 E_ioni[V]) metres. */
double obem_ref_recombination_radius(double e_ioni_ev)
{
    const double e = 1.602176634e-19;
    return next_ke() * e / (2.0 * e_ioni_ev);
}
