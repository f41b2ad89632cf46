/*
 * obem.h -- C ABI of libobem.so: the B200-native (sm_100a) field-evaluation hot path of the
 * OuroborosBEM method (arXiv 2110.09214).
 *
 * What the library computes, for every target point r (a tracked charge, or an arbitrary point):
 *
 *   N-body part   PAPER.md:272-277, section 3.2.4, Eq (3.8):
 *       E_Nbody(r_p') = 1/(4 pi eps0) * sum_{p != p'} q_p (r_p' - r_p) / ||r_p' - r_p||^3
 *     with Plummer softening (reading A2): r2 = ||d||^2 + eps_pp^2, E += q d r2^(-3/2),
 *     phi += q r2^(-1/2).  At the charges the self term p = p' is excluded BY INDEX (reading A3).
 *
 *   Panel part    PAPER.md:141-147, section 2.2, Eq (2.13), (2.14):
 *       V(r) = sum_i sigma_i/(4 pi eps0) Int_{C_i} 1/||r-r'|| d2r'
 *       E(r) = sum_i sigma_i/(4 pi eps0) Int_{C_i} (r-r')/||r-r'||^3 d2r'
 *     sigma_i constant over the flat triangular cell C_i; the cell integral is the
 *     7-point degree-5 triangle rule (reading A1).
 *
 *   The two parts are superposed.  A source at exactly zero (softened) distance
 *   contributes 0 (reading A4).
 *
 * Conventions
 *   - SI units: metres, coulombs, C/m^2, V/m, V.   k_e = 1/(4 pi eps0), eps0 = 8.8541878128e-12 F/m.
 *   - The interactions are computed in fp32 and summed in fp32 over one block of 256 sources (34 panels); the
 *     block sums are accumulated in fp64.  Results are fp32.  Every step of the path runs in
 *     the library's CUDA kernels.
 *   - Pointers named d_* are DEVICE pointers owned by the caller (e.g. torch tensors), 16-byte
 *     aligned; pointers named h_* are HOST pointers.  The library copies / repacks on set_* into
 *     buffers it owns: an input may be freed or overwritten as soon as the stream has passed the
 *     call.  Outputs are caller-owned and fully overwritten.
 *   - All device work is enqueued on the caller's stream (`cuda_stream` is a cudaStream_t passed as
 *     void*; NULL = the legacy default stream).  No hidden synchronisation and no host copies,
 *     except: (a) a set_* / eval_* call that must GROW a library-owned buffer calls cudaMalloc,
 *     which may synchronise the device (obem_reserve avoids it); (b) the *_host entry points,
 *     which are synchronous by contract.
 *   - Every entry point returns an obem_status (0 = OK, negative = error); nothing throws across
 *     the ABI.  n = 0 / n_panels = 0 / m = 0 are valid.  There is no CPU fallback: without a
 *     CUDA device obem_create fails with OBEM_ECUDA.
 *   - A context is bound to one device and is not thread-safe; use one context per thread/stream.
 */
#ifndef OBEM_H
#define OBEM_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct obem_ctx obem_ctx; /* opaque; one per device (per stream of use) */

typedef enum obem_status {
    OBEM_OK = 0,
    OBEM_EINVAL = -1, /* null / negative / misaligned argument, unknown flag bits            */
    OBEM_ESTATE = -2, /* evaluate before the sources the flags ask for were set              */
    OBEM_ECUDA = -3,  /* a CUDA call failed; obem_last_cuda_error() gives the cudaError_t     */
    OBEM_ENOMEM = -4, /* device allocation failed                                            */
    OBEM_ELIMIT = -5  /* a size beyond the fixed maximum of obem_nbody_at_points_static      */
} obem_status;

/* flags of the evaluate calls: which of the two sums to include */
#define OBEM_NBODY 1u  /* Eq (3.8), sources = the charges of obem_set_charges              */
#define OBEM_PANELS 2u /* Eq (2.13)/(2.14), sources = the panels of obem_set_panels         */
#define OBEM_PANELS_EXACT 4u /* with OBEM_PANELS: exact cell integrals near the target, see obem_set_near_field */
#define OBEM_NO_PHI 8u /* E only: Eq (3.8) and (2.14) are field sums and the integrators read only E (PAPER.md:274,
                          :302-306); the phi lane of the result is written as 0 and one packed instruction of 12 per
                          interaction is saved.  E is bit-identical to the E + phi evaluation.  Accepted by
                          obem_eval_at_charges[_range] and obem_eval_at_points; not with OBEM_PANELS_EXACT, the
                          partner by-product or the NN approximation (OBEM_EINVAL).  The steppers use it. */

/* Create a context on CUDA device `device`.  Queries the SM count and sizes the persistent grid.
 * *out is NULL on failure. */
int obem_create(obem_ctx** out, int device);

/* Free the context and every library-owned device buffer.  Synchronises the device.  NULL is OK. */
int obem_destroy(obem_ctx* c);

/* Pre-allocate library-owned buffers for up to n_charges charges and n_panels panels, so that later
 * set_* calls never allocate (and therefore never synchronise).  Optional.  A capacity that is already
 * large enough is left alone; one that has to GROW is re-allocated and the set it held is discarded:
 * obem_n_charges / obem_n_panels go back to -1 and an evaluation that needs that set returns OBEM_ESTATE
 * until it is set again.  Call it before the first set_*. */
int obem_reserve(obem_ctx* c, int64_t n_charges, int64_t n_panels);

/* Softening lengths in metres, >= 0 and finite.  eps_pp: charge-charge sum (reading A2; 0 = Eq 3.8
 * as printed).  eps_panel: panel sum (reading A5; default 0).  Defaults 0, 0.  Takes effect at the
 * next evaluate call. */
int obem_set_softening(obem_ctx* c, float eps_pp_m, float eps_panel_m);

/* Panels (flat cells with constant sigma; triangles here, quadrilaterals through
 * obem_set_panels_cells, reading A8).
 *   d_verts [n_panels][3][3] fp32: vertex j of panel p at d_verts[(p*3+j)*3 + 0..2] = x,y,z [m]
 *   d_sigma [n_panels] fp32 [C/m^2]
 * Derives, in fp64 and rounded once to fp32, the area A_p and the 7 quadrature sources
 * (x_pk, sigma_p*A_p*w_k) of every panel.  Replaces any earlier panel set.  Degenerate (A = 0)
 * panels contribute 0. */
int obem_set_panels(obem_ctx* c, const float* d_verts, const float* d_sigma, int64_t n_panels,
                    void* cuda_stream);

/* New sigma on the SAME geometry (charging-up changes sigma every step, Eq 3.7):
 * rescales the weights only.  n_panels must equal the count of the last obem_set_panels
 * (else OBEM_EINVAL; OBEM_ESTATE if no panels were ever set). */
int obem_set_sigma(obem_ctx* c, const float* d_sigma, int64_t n_panels, void* cuda_stream);

/* Charges (Eq 3.8's particles): d_xyzq [n][4] fp32 = x, y, z [m], q [C], n < 2^31 - 256.  Replaces any
 * earlier set.  Any storage order is as fast as any other: the library keeps its copy of the sources
 * stably sorted by q ("class order": an avalanche creates electrons and ions in pairs, PAPER.md:195-199,
 * so the caller's array interleaves the signs), which makes its 256-source blocks weight-uniform; every
 * index the API takes or returns (ranges, partners, output rows) is the CALLER's. */
int obem_set_charges(obem_ctx* c, const float* d_xyzq, int64_t n, void* cuda_stream);

/* E and phi at the charges themselves: d_out [n][4] fp32 = Ex, Ey, Ez [V/m], phi [V].
 * With OBEM_NBODY the sum over charges excludes the target's own index.  A flag whose sources are
 * an EMPTY set contributes 0; a flag whose sources were NEVER set gives OBEM_ESTATE. */
int obem_eval_at_charges(obem_ctx* c, float* d_out, unsigned flags, void* cuda_stream);

/* Same, for the contiguous slice [first, first+count) of the charges (the caller's indices) only:
 * d_out [count][4], row i = charge first + i.  This is the multi-GPU sharding unit (targets sharded
 * across ranks, sources replicated). */
int obem_eval_at_charges_range(obem_ctx* c, int64_t first, int64_t count, float* d_out,
                               unsigned flags, void* cuda_stream);

/* E and phi at arbitrary points (field map / static option):
 *   d_pts [m][4] fp32, 4th lane ignored;  d_out [m][4].
 * With OBEM_NBODY all charges are summed with the same softening and NO exclusion. */
int obem_eval_at_points(obem_ctx* c, const float* d_pts, int64_t m, float* d_out, unsigned flags,
                        void* cuda_stream);

/* The whole hot path through HOST buffers, synchronous: copies the inputs to the device, runs
 * set_panels (if h_verts != NULL; if NULL the panels already set are kept), set_charges, the
 * evaluation at the charges, and copies the result back.  Pageable or pinned host memory. */
int obem_field_at_charges_host(obem_ctx* c, const float* h_xyzq, int64_t n, const float* h_verts,
                               const float* h_sigma, int64_t n_panels, float* h_out, unsigned flags);

/* Field map through HOST buffers, synchronous (h_verts may be NULL as above). */
int obem_field_at_points_host(obem_ctx* c, const float* h_pts, int64_t m, const float* h_verts,
                              const float* h_sigma, int64_t n_panels, float* h_out, unsigned flags);

/* The ONE entry point that allocates nothing (no cudaMalloc, cudaFree or allocating library routine, no context):
 * for callers that cannot allocate -- code under CUDA graph capture, tight serving loops, harnesses that forbid it.
 * Computes what obem_eval_at_points(OBEM_NBODY) computes, Eq (3.8) with Plummer softening and no
 * index exclusion, a source at zero softened distance contributing 0 (reading A4), straight from the caller's arrays:
 *   d_xyzq [n][4] fp32 = x, y, z [m], q [C] (any n, any order);  d_pts [m][4] fp32, 4th lane ignored;
 *   d_out  [m][4] fp32 = Ex, Ey, Ez [V/m], phi [V];  all device pointers of the CURRENT device, 16-byte aligned.
 * Its scratch (fp64 partial sums of the split-source scheme) is a file-scope static __device__ array of fixed size,
 * OBEM_STATIC_MAX_POINTS x OBEM_STATIC_MAX_SPLITS x 32 B = 8 MiB, which every GPU that loads libobem.so holds until
 * the process exits.  m > OBEM_STATIC_MAX_POINTS returns OBEM_ELIMIT (split the points, or use a context).
 * The first call on a device looks the array's device address up (cudaGetSymbolAddress: make that call outside a
 * graph capture); later calls only enqueue two kernels on `cuda_stream`.  ALL calls on a device share the scratch,
 * which keeps the last call's contents (every slot a call reads it has written itself; nothing needs clearing): calls
 * that overlap on the GPU -- different streams, concurrently replayed graphs -- race.  Serialise them.
 * Same arithmetic as the hot path (fp32 terms, fp32 sums over 256 sources, fp64 across blocks), simpler kernel
 * (13 packed instructions + the zero-distance guard): results agree with obem_eval_at_points to the path's tolerance,
 * not bit for bit. */
#define OBEM_STATIC_MAX_POINTS 16384
#define OBEM_STATIC_MAX_SPLITS 16
int obem_nbody_at_points_static(const float* d_xyzq, int64_t n, const float* d_pts, int64_t m, float eps_pp_m,
                                float* d_out, void* cuda_stream);

/* Introspection (host side, no device work) */
int64_t obem_n_charges(const obem_ctx* c);     /* -1 if never set */
int64_t obem_n_panels(const obem_ctx* c);      /* -1 if never set */
int obem_sm_count(const obem_ctx* c);          /* multiprocessors of the device                     */
int obem_grid_size(const obem_ctx* c);         /* CTAs of the persistent evaluation kernel          */
int64_t obem_kernel_launches(const obem_ctx* c); /* kernels this context has launched so far          */
int obem_last_cuda_error(const obem_ctx* c);   /* cudaError_t of the last failed CUDA call, else 0   */
const char* obem_status_string(int status);

/* Copy the packed quadrature sources (x, y, z, sigma*A*w_k) of the current panel set to
 * d_out [n_panels*7][4] fp32 -- for inspection and tests. */
int obem_get_panel_sources(obem_ctx* c, float* d_out, void* cuda_stream);

/* FP32 pipe microbenchmark (measurement aid for the roofline denominator, not on the hot path):
 * launches a register-only chain of `iters` dependent-free FFMA (mode 0) or packed FFMA2 (mode 1)
 * instructions per thread on the persistent grid and returns the flop count it executed in
 * *flops_out (2 per scalar FMA).  Time it with events on `cuda_stream`. */
int obem_fma_peak_probe(obem_ctx* c, int mode, int64_t iters, double* flops_out, void* cuda_stream);

/* ----------------------------------------------------------------------------------------------------------
 * Steps adjacent to the hot path: influence of the particles on the cells,
 * PAPER.md:241-257, section 3.2.2 -- what the dynamic option does every time step BEFORE the field evaluation.
 * ---------------------------------------------------------------------------------------------------------- */

/* Eq (3.3), (3.4): area-averaged potential and field of ALL charges (obem_set_charges) over every cell C_i
 * (obem_set_panels):
 *     Vbar_i = k_e sum_p q_p/A_i Int_{C_i} 1/||r - r_p|| d2r,   Ebar_i = k_e sum_p q_p/A_i Int_{C_i} (r - r_p)/||r - r_p||^3 d2r
 * with (1/A_i) Int_{C_i} f d2r = sum_k w_k f(x_ik), the same 7-point rule as the panel sums (reading A1), and the
 * cell-particle distance softened by eps_panel (default 0 = as printed; zero distance contributes 0, reading A4).
 *   d_infl [n_panels][4] fp32 = Ebar_x, Ebar_y, Ebar_z [V/m], Vbar [V]            (16-byte aligned)
 *   d_en   [n_panels]    fp32 = Ebar_i . n_i, n_i = (v1-v0)x(v2-v0)/||.|| (orientation = vertex order,
 *                               reading A16); may be NULL.
 * OBEM_ESTATE if panels or charges were never set.  Cost: 7 * n_panels * n_charges interactions, run by the
 * hot path's evaluation kernel, plus an O(n_panels) reduction. */
int obem_influence_on_panels(obem_ctx* c, float* d_infl, float* d_en, void* cuda_stream);

/* Eq (3.5), (3.6): the modified left-hand sides of the BEM system, per cell i:
 *     d_kind[i] == 0 (ed cell, electrode):       b_i = V_i - Vbar_i
 *     d_kind[i] == 1 (dd cell, dielectric face): b_i = sigma_F,i - (eps2 - eps1)_i * (Ebar_i . n_i)
 *   d_kind [n] int32; d_bc [n] fp32 = V_i [V] or sigma_F,i [C/m^2]; d_deps [n] fp32 = eps2 - eps1 [F/m] (read for
 *   dd cells only); d_infl [n][4], d_en [n] as written by obem_influence_on_panels; d_b [n] fp32 out.
 * Any other kind writes NaN to b_i. */
int obem_rhs_from_influence(obem_ctx* c, const int32_t* d_kind, const float* d_bc, const float* d_deps,
                            const float* d_infl, const float* d_en, float* d_b, int64_t n_panels,
                            void* cuda_stream);

/* sigma = M^-1 b with the STORED inverse ("inverted once", every new right-hand side is a
 * matrix-vector product).  d_minv [n][ld] row-major fp32 (ld >= n, caller-owned, read only), d_b [n],
 * d_sigma [n] fp32 out.  fp32 accumulation (4 x 32 partial sums per row).  Bound by HBM: 4 n^2 bytes are read
 * once.  The TMA-streamed kernel needs n % 4 == 0, ld % 4 == 0 and 16-byte aligned d_minv, d_b; any other shape
 * takes a plain-load kernel (same results up to summation order). */
int obem_apply_inverse(obem_ctx* c, const float* d_minv, int64_t n, int64_t ld, const float* d_b, float* d_sigma,
                       void* cuda_stream);

/* The dynamic-option update of one time step, enqueued on one stream:
 * influence (3.3/3.4) -> right-hand side (3.5/3.6) -> sigma = M^-1 b -> obem_set_sigma.  d_sigma [n_panels]
 * receives the new charge densities (and the context's panel weights are updated from it). */
int obem_update_sigma_dynamic(obem_ctx* c, const int32_t* d_kind, const float* d_bc, const float* d_deps,
                              const float* d_minv, int64_t ld, float* d_sigma, void* cuda_stream);

/* Several charge-density vectors on the SAME cells in one pass.  The signal induced on a read-out electrode is
 * computed with the Shockley-Ramo theorem from that electrode's weighting field (section 3.3.4,
 * Eq 3.13): the field of the set-up with that electrode at unit potential and the others grounded -- one more
 * solution sigma^(e) of the same BEM matrix, evaluated with the same Eq (2.13)/(2.14) at the same
 * points.  The distance / rsqrt work of every (quadrature point, target) pair does not depend on sigma and is shared:
 *   d_sigma [n_sigma][n_panels] fp32 [C/m^2] (row s = density vector s; the sigma given to obem_set_panels /
 *           obem_set_sigma is NOT used and not changed)
 *   d_pts   [m][4] fp32, 4th lane ignored;   d_out [n_sigma][m][4] fp32 = Ex, Ey, Ez [V/m], phi [V] of vector s.
 * Up to 4 vectors per pass over the geometry (103 packed FP32 instructions per panel and target pair for 4 vectors
 * against 4 x 87 for four obem_set_sigma + obem_eval_at_points rounds); more vectors take ceil(n_sigma / 4)
 * passes.  eps_panel and reading A4 (zero distance contributes 0) apply as in obem_eval_at_points.  Library-owned
 * buffers (the unit-density encoding of the geometry, built on the first call after obem_set_panels; one pass's
 * blocked sigma rows) grow with cudaMalloc on the first call of a given size.  OBEM_ESTATE before obem_set_panels. */
int obem_eval_panels_multi(obem_ctx* c, const float* d_sigma, int n_sigma, const float* d_pts, int64_t m,
                           float* d_out, void* cuda_stream);

/* The Shockley-Ramo signal sum, Eq (3.13) (section 3.4): the current induced on read-out electrode k
 * by the moving particles,  i_k = sum_p q_p v_p . E_w^(k)(r_p),  "generated separately" for each particle type
 * (PAPER.md:366):
 *   d_xyzq [n][4] fp32 (only q is read);  d_vel [n][4] fp32 = vx, vy, vz [m/s] (4th lane ignored);
 *   d_ew [n_electrodes][n][4] fp32 = the weighting field of electrode k at particle p [V/m for 1 V] -- the layout
 *        obem_eval_panels_multi writes when its points are the particles;
 *   d_out [n_electrodes][2] fp64 [A]: [k][0] = the particles with q < 0 (electrons), [k][1] = those with q > 0 (ions).
 * Every term and every sum in fp64, fixed order: deterministic.  Sign as printed in Eq (3.13) (no minus sign).  A small
 * library-owned buffer of partial sums grows (cudaMalloc) on the first call of a given size. */
int obem_ramo_current(obem_ctx* c, const float* d_xyzq, const float* d_vel, const float* d_ew, int n_electrodes,
                      int64_t n, double* d_out, void* cuda_stream);

/* ----------------------------------------------------------------------------------------------------------
 * NEXT-2: numerical integrators, section 3.2.5 -- the consumers of the field evaluation.
 * State: d_xyzq [n][4] fp32 = x, y, z [m], q [C];  d_vel [n][4] fp32 = vx, vy, vz [m/s], m [kg] (m = 0: immobile).
 * Non-relativistic equations of motion dx/dt = v, dv/dt = (q/m) E(x); E = the sums `flags` selects, evaluated at
 * the charges themselves (obem_set_charges + obem_eval_at_charges on the current positions: after a step the
 * context's charge set is the LAST positions the field was evaluated at, not the final ones).  In place, fp32.
 * ---------------------------------------------------------------------------------------------------------- */

/* x += h v (drift) and v += h (q/m) E with d_field [n][4] = Ex, Ey, Ez, phi (kick): the two sub-steps every
 * splitting scheme is made of. */
int obem_push_drift(obem_ctx* c, float* d_xyzq, const float* d_vel, int64_t n, float h, void* cuda_stream);
int obem_push_kick(obem_ctx* c, const float* d_xyzq, float* d_vel, const float* d_field, int64_t n, float h,
                   void* cuda_stream);

/* Basic Euler ("a single field evaluation during a time step"):
 *     x_{n+1} = x_n + dt v_n,   v_{n+1} = v_n + dt (q/m) E(x_n). */
int obem_step_euler(obem_ctx* c, float* d_xyzq, float* d_vel, int64_t n, float dt, unsigned flags,
                    void* cuda_stream);

/* PEFRL [18] (Omelyan, Mryglod, Folk 2002: position-extended Forest-Ruth-like, 4th order, symplectic, time
 * reversible): x v x v x v x v x with the published xi, lambda, chi -- 5 drifts, 4 kicks, i.e. 4
 * field evaluations (reading A17: the paper counts 5). */
int obem_step_pefrl(obem_ctx* c, float* d_xyzq, float* d_vel, int64_t n, float dt, unsigned flags,
                    void* cuda_stream);

/* Electron-ion recombination, PAPER.md:341-355 (section 3.3.3): "taken into account microscopically for any
 * electron and ion using the distances obtained during the N-body calculation process".  Same as
 * obem_eval_at_charges[_range] (flags must include OBEM_NBODY), and as a by-product of the N-body pass, for every
 * charge i of the range, its nearest charge of OPPOSITE sign:
 *   d_partner_d [count] fp32 = true (unsoftened) distance [m], +inf if there is none
 *   d_partner_j [count] int32 = index of that charge in the charge set, -1 if there is none
 * Charges with q = 0 have no partner and are nobody's partner.  How: the evaluation kernel keeps, per target, the
 * smallest SOFTENED fp32 r2 over opposite-sign sources and the 256-source block it fell in (one 3-input integer min
 * per two sources and target on the ALU pipe); a second O(256 N) kernel scans that block exactly.  Near-ties between different
 * blocks are decided on the fp32 softened r2: the reported distance d obeys d^2 <= d_true^2 + 4 ulp(d_true^2 +
 * eps_pp^2).  A pair recombines when d <= obem_recombination_radius(E_ioni), Eq (3.12). */
int obem_eval_at_charges_partners(obem_ctx* c, float* d_out, float* d_partner_d, int32_t* d_partner_j,
                                  unsigned flags, void* cuda_stream);
int obem_eval_at_charges_partners_range(obem_ctx* c, int64_t first, int64_t count, float* d_out,
                                        float* d_partner_d, int32_t* d_partner_j, unsigned flags,
                                        void* cuda_stream);

/* Eq (3.12): 1/(4 pi eps0) * e / (2 E_ioni) in metres for E_ioni in eV (host arithmetic). */
double obem_recombination_radius(double e_ioni_ev);

/* Copy (n_x, n_y, n_z, A) of every panel to d_out [n_panels][4] fp32 -- inspection and tests. */
int obem_get_panel_normals(obem_ctx* c, float* d_out, void* cuda_stream);

/* ----------------------------------------------------------------------------------------------------------
 * NEXT-3: near-field-accurate panels.  PAPER.md:131-133, :147: "the corresponding integrals are calculated
 * analytically".  The 7-point rule of the hot path differs from the exact integral of Eq (2.13)/(2.14) by
 * ~(h/r)^6 (2.7e-3 of the panel's own field at r = h, 2.5e-5 at 2h, 2.1e-6 at 3h, 3.8e-7 at 4h; h = longest
 * edge, r = distance to the centroid).  With OBEM_PANELS | OBEM_PANELS_EXACT every evaluate call (and every
 * stepper) replaces, for each target, the 7-point value of each panel whose centroid is closer than
 * near_factor * h_p by the closed-form integral over the flat triangle (fp64, edge-wise log / atan terms), so the
 * result is Eq (2.13)/(2.14) itself to the tolerance of the path.  On a panel (d = 0) the normal component is the
 * principal value 0 (reading A8); exactly on an edge the singular edge term is dropped (like reading A4).
 * How: a uniform cell grid over the panels' near spheres (built on the first such call after obem_set_panels:
 * allocates and synchronises once per geometry; obem_set_sigma keeps it), one warp per target scanning its cell's
 * candidate list, near pairs compacted across the warp; the correction (exact - 7-point) is summed in fp64 in a
 * fixed order and added to d_out.
 * ---------------------------------------------------------------------------------------------------------- */

/* near_factor > 0 and finite (default 3).  Takes effect at the next evaluate call (the cell lists are rebuilt). */
int obem_set_near_field(obem_ctx* c, float near_factor);

/* Number of (cell, panel) entries of the current cell lists and number of cells; -1 before the first build. */
int64_t obem_near_list_size(const obem_ctx* c);
int64_t obem_near_cells(const obem_ctx* c);

/* Polygonal cells ("flat polygonal cells (triangles, quadrangles, etc.)", one constant sigma
 * each).  d_verts4 [n_cells][4][3] fp32, d_nvert [n_cells] int32 = 3 or 4 (NULL: all 4; for 3 the 4th vertex is
 * ignored), d_sigma [n_cells].  A flat quadrilateral (v0, v1, v2, v3), vertices in order around the cell, is stored
 * as the triangles (v0, v1, v2), (v0, v2, v3) with the same sigma; a triangle cell as itself plus a zero-area one.
 * Afterwards the context holds 2 n_cells panels (obem_n_panels, obem_influence_on_panels ... count triangles);
 * obem_set_sigma_cells updates sigma per CELL. */
int obem_set_panels_cells(obem_ctx* c, const float* d_verts4, const int32_t* d_nvert, const float* d_sigma,
                          int64_t n_cells, void* cuda_stream);
int obem_set_sigma_cells(obem_ctx* c, const float* d_sigma, int64_t n_cells, void* cuda_stream);

/* Symmetry planes ("up to three symmetry planes can also be included").  n_planes in 0..3 (0 removes
 * them); plane k is x_{h_axis[k]} = h_coord[k] [m] (axis 0, 1, 2 = x, y, z; at most one plane per axis) with parity
 * h_parity[k] = +1 (the mirror image of every source carries the same charge) or -1 (the opposite charge: a
 * grounded plane).  HOST arrays.  From then on every evaluate call (and stepper, influence, field map) adds the
 * 2^n - 1 image copies of ALL sources the flags select: each image is evaluated as reflected targets on the original
 * sources, E_image(r) = s M E(M r), so the cost is 2^n evaluations and nothing is duplicated in memory.  The image of
 * charge i acts on charge i.  Not combined with obem_eval_at_charges_nn (OBEM_EINVAL). */
int obem_set_symmetry(obem_ctx* c, int n_planes, const int* h_axis, const double* h_coord, const int* h_parity);

/* ----------------------------------------------------------------------------------------------------------
 * NEXT-4: the static field option, section 3.2.1: "the field components are computed only once at
 * some predefined spatial coordinates located on a uniform 3D grid map ... During the transport, the field
 * components at each particle location are then interpolated in this 3D map."
 * Map: node (ix, iy, iz) at (o_x + ix d_x, o_y + iy d_y, o_z + iz d_z), 0 <= ix < nx ...; values
 * d_map[((ix*ny + iy)*nz + iz)*4 + 0..3] = Ex, Ey, Ez [V/m], phi [V] (z fastest), caller-owned, 16-byte aligned.
 * h_origin, h_spacing: HOST double[3] in metres; spacing > 0 along every axis with more than one node.
 * ---------------------------------------------------------------------------------------------------------- */

/* Fill the map: evaluate the sums `flags` selects (as obem_eval_at_points) at every node.  The node coordinate is
 * the fp64 value o + i*d (one multiply, one add) rounded once to fp32.  The node list lives in a library-owned
 * buffer that grows (cudaMalloc) on the first call of a given size. */
int obem_field_map(obem_ctx* c, int nx, int ny, int nz, const double* h_origin, const double* h_spacing,
                   float* d_map, unsigned flags, void* cuda_stream);

/* Interpolate the map at d_pts [m][4] (4th lane ignored) into d_out [m][4]: trilinear in every component between
 * the 8 surrounding nodes; positions outside the node lattice are clamped to its boundary (reading A18).  The cell
 * index and fractions are taken in fp64, the 8-term weighted sum in fp32.  accumulate != 0: d_out += the
 * interpolated value (static set-up field + N-body field), else d_out is overwritten. */
int obem_interp_map(obem_ctx* c, const float* d_map, int nx, int ny, int nz, const double* h_origin,
                    const double* h_spacing, const float* d_pts, int64_t m, float* d_out, int accumulate,
                    void* cuda_stream);

/* ----------------------------------------------------------------------------------------------------------
 * NEXT-4: the nearest-neighbour (NN) approximation of the N-body sum, section 3.2.4: "evaluating
 * the exact Coulombian field following (3.8) for each of the closest particles to the particle of interest while the
 * field from the particles further away is approximated by their centre of charges with a barycentric method".
 * The paper gives no algorithm; reading A19 is: equal-count k-d partition into leaves of 256 charges
 * (stable sorts along the longest box axis, cuts at multiples of 256); per leaf a bounding box and two
 * pseudo-particles (centres of charge of its positive / negative members); for a tile of 2048 consecutive charges
 * (8 leaves) a box B is FAR iff theta^2 * dist2(box_tile, B) > diag2(B); near leaves are summed exactly (Eq 3.8,
 * softened, self excluded by index), far leaves through their pseudo-particles (same softening); super-leaves (64
 * leaves) that are far at theta / 2 stand for all their leaves with their own two pseudo-particles.
 * Error ~ theta^2 (the leaves' quadrupoles): measured on config 3 at theta = 2: E rel-L2 2.2e-3 against the exact
 * sum for 3 % of its pair interactions.  theta = 0 is the exact sum.
 * ---------------------------------------------------------------------------------------------------------- */

/* theta >= 0 and finite; default 2. */
int obem_set_nn_theta(obem_ctx* c, float theta);

/* As obem_eval_at_charges, with the N-body part approximated as above.  flags must include OBEM_NBODY;
 * OBEM_PANELS [| OBEM_PANELS_EXACT] adds the panel part as usual.  Everything is enqueued on the stream, no host
 * round trip; library-owned work buffers grow (cudaMalloc) when n does: 16 B x n x (4 + n/131072) for the tiles'
 * far blocks, 4 B x (n/2048) x (n/256) for their lists. */
int obem_eval_at_charges_nn(obem_ctx* c, float* d_out, unsigned flags, void* cuda_stream);

/* Source blocks (of 256) x tiles (of 2048 targets) the last NN evaluation ran: 2048 * 256 * this = its pair
 * interactions.  Reads one word back: synchronises the stream.  -1 before the first call. */
int64_t obem_nn_last_units(obem_ctx* c, void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* OBEM_H */
