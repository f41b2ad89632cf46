/*
 * obem_internal.cuh -- pieces shared by the translation units of libobem.so (obem.cu: the hot path;
 * obem_next.cu: the adjacent steps of SURVEY.md section 8(f)).  Internal: not part of the C ABI (include/obem.h),
 * not shared with oracle/.
 */
#ifndef OBEM_INTERNAL_CUH
#define OBEM_INTERNAL_CUH

#include <cuda_runtime.h>
#include <stdint.h>
#include <math.h>

#include "obem.h"

namespace {

typedef unsigned long long u64;

/* ------------------------------------------------------------------------------------------- */
/* packed f32x2 helpers (PTX ISA: add/sub/mul/fma .f32x2, sm_100+).  A u64 holds {lo, hi}.       */
/* ------------------------------------------------------------------------------------------- */
__device__ __forceinline__ u64 pk(float lo, float hi)
{
    u64 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
/* same, but opaque to the optimiser: the pair is built once and kept (used for loop-invariant targets,
 * which the compiler would otherwise re-pack from their float4 registers inside the hot loop) */
__device__ __forceinline__ u64 pk_keep(float lo, float hi)
{
    u64 r;
    asm volatile("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void upk(u64 v, float& lo, float& hi)
{
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c)
{
    u64 r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}
__device__ __forceinline__ u64 add2(u64 a, u64 b)
{
    u64 r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ u64 sub2(u64 a, u64 b)
{
    u64 r;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ u64 mul2(u64 a, u64 b)
{
    u64 r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ float rsqrt_approx(float x)
{
    float r;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); /* one MUFU.RSQ */
    return r;
}

/* ------------------------------------------------------------------------------------------- */
/* mbarrier + 1-D TMA bulk copy (global -> shared)                                              */
/* ------------------------------------------------------------------------------------------- */
__device__ __forceinline__ uint32_t smem_u32(const void* p)
{
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(u64* bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(u64* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(u64* bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void tma_load_1d(void* dst_smem, const void* src_gmem, uint32_t bytes, u64* bar)
{
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
            smem_u32(dst_smem)),
        "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
        : "memory");
}


inline long long ceil_div(long long a, long long b) { return (a + b - 1) / b; }

/* ------------------------------------------------------------------------------------------- */
/* blocked panel buffer (obem.cu: the panel launch; obem_multi.cu: the multi-sigma launch)       */
/* ------------------------------------------------------------------------------------------- */
/* Panel blocks: PPB panels x (1 origin + 7 x 2) float4 = 510 of 512 slots, + header. */
constexpr int PPB = 34;
constexpr int PANEL_SLOTS = 15;
constexpr int SBH_P = 512 + 1;
constexpr int PANELS_PER_BLOCK = PPB;

/* first float4 (the frame origin) of panel p inside the blocked panel buffer */
__device__ __forceinline__ long long panel_entry(long long p)
{
    return (p / PPB) * SBH_P + 1 + (p % PPB) * PANEL_SLOTS;
}

/* The two float4 of one quadrature source (see panel_loop): weight w [C], offset (sx, sy, sz) from the frame
 * origin, all in double; rounded once.  a is rounded first and b, c_phi are derived from the ROUNDED a, so that
 * fma(T, a, b) = a (T - s) up to one rounding of b. */
__device__ __forceinline__ void panel_encode(double w, double sx, double sy, double sz, float4& A, float4& B)
{
    if (w == 0.0 || !isfinite(w)) {
        A = make_float4(0.f, 1.0e17f, 1.0e17f, 1.0e17f);
        B = make_float4(0.f, 0.f, 0.f, 0.f);
        return;
    }
    const float a = (float)((w > 0.0 ? 1.0 : -1.0) / sqrt(fabs(w)));
    const double ad = (double)a;
    A = make_float4(a, (float)(-ad * sx), (float)(-ad * sy), (float)(-ad * sz));
    B = make_float4((float)(w * fabs(ad)), (float)(ad * ad), (float)w, 0.f);
}

} /* namespace */

/* obem_nn.cu: buffers of the NN approximation (all library-owned, grown on demand) */
struct obem_nn_state {
    float theta = 2.0f;
    int* perm[2] = {nullptr, nullptr};
    unsigned long long* key[2] = {nullptr, nullptr};
    size_t perm_cap[2] = {0, 0}, key_cap[2] = {0, 0};
    unsigned* seg = nullptr;         /* [2][n_leaf][3] ordered min / max coordinates of the segments of a level */
    float4* sorted = nullptr;        /* [n_leaf * 256] the charges in k-d order (padded): the targets           */
    float4* pool = nullptr;          /* [(n_leaf + n_group * far_cap)][OBEM_SBH] leaf blocks, then far blocks */
    float* leafbox = nullptr;        /* [n_leaf][6] */
    float4* pseudo = nullptr;        /* [n_leaf][2] centre of charge of the positive / negative members         */
    double* leafmom = nullptr;       /* [n_leaf][8] Q+, Q+ R+, Q-, Q- R- in fp64 (for the super-leaves)          */
    float* superbox = nullptr;       /* [n_super][6] */
    float4* superpseudo = nullptr;   /* [n_super][2] */
    size_t leafmom_cap = 0, superbox_cap = 0, superpseudo_cap = 0;
    long long* cnt = nullptr;        /* [n_group] units of each tile */
    long long* tile_ptr = nullptr;   /* [n_group + 1] + the unit count U */
    int* list = nullptr;
    float4* out_sorted = nullptr;
    void* tmp = nullptr;             /* radix-sort workspace */
    float4* pan = nullptr;           /* panel part when the flags ask for it */
    size_t seg_cap = 0, sorted_cap = 0, pool_cap = 0, leafbox_cap = 0, pseudo_cap = 0, cnt_cap = 0, tile_ptr_cap = 0,
           list_cap = 0, out_sorted_cap = 0, tmp_cap = 0, pan_cap = 0;
    long long last_n = 0;
};

struct obem_ctx {
    int device = 0;
    int sm_count = 0;
    int grid = 0;
    float eps_pp = 0.f, eps_panel = 0.f;
    /* charges */
    float4* d_chg = nullptr;     /* plain copy [n]: the targets of eval_at_charges                */
    float4* d_chg_blk = nullptr; /* blocked copy with headers [nblk][SBH]: the sources, in CLASS ORDER */
    long long chg_cap = 0;       /* capacity in charges (a multiple of SB)                        */
    long long n_chg = -1;
    /* class order: the charges stably sorted by q (set_charges), so that the 256-source blocks are weight-uniform
     * whatever order the caller stores electrons and ions in */
    float4* d_chg_sorted = nullptr; /* [chg_cap] plain copy in class order: the targets of eval_at_charges          */
    int* d_perm = nullptr;          /* [chg_cap] class-order position -> input index                                */
    int* d_inv = nullptr;           /* [chg_cap] input index -> class-order position                                */
    unsigned* d_skey[2] = {nullptr, nullptr}; /* [chg_cap] sort keys (ordered bit pattern of q), in / out           */
    int* d_sval = nullptr;          /* [chg_cap] 0, 1, 2, ...: the values the sort permutes                         */
    void* d_sort_tmp = nullptr;     /* CUB workspace (radix sort, select)                                           */
    size_t sort_tmp_cap = 0;
    /* evaluation at a sub-range [first, first + count) of the charges: its members in class order */
    int* d_rng_spos = nullptr;      /* [chg_cap] their class-order positions, ascending                             */
    int* d_rng_idx = nullptr;       /* [chg_cap] their output slots (input index - first)                           */
    float4* d_rng_tgt = nullptr;    /* [chg_cap] their coordinates                                                  */
    int* d_rng_num = nullptr;       /* [1] how many the select wrote (== count)                                     */
    /* panels */
    float4* d_psrc = nullptr;
    double* d_area = nullptr;
    float4* d_qpts = nullptr;     /* [np*7] quadrature points in global coordinates, .w = rule weight w_k */
    float4* d_qrel = nullptr;     /* [np*7] quadrature offsets from the panel's frame origin, .w = w_k A      */
    float4* d_nrm = nullptr;      /* [np] unit normal (vertex-order orientation) and area                 */
    float4* d_infl_tmp = nullptr; /* [np*7] field of the charges at the quadrature points (influence pass) */
    long long pan_cap = 0; /* capacity in panels */
    long long n_pan = -1;
    /* split-tile workspace [grid][2][TT] */
    float2* d_trk = nullptr;     /* [chg_cap] (min softened r2 to an opposite charge, its source block) per charge */
    float2* d_trk_ws = nullptr;  /* [grid][2][TT] the same for split tiles                                        */
    double* d_ws = nullptr;      /* [grid][2][TT_MAX][4] fp64 partial sums of split tiles */
    float* d_sink = nullptr;
    unsigned* d_bad_count = nullptr;
    long long* d_bad_list = nullptr;
    /* staging for the *_host entry points */
    cudaStream_t hstream = nullptr;
    void* d_stage[4] = {nullptr, nullptr, nullptr, nullptr};
    size_t stage_cap[4] = {0, 0, 0, 0};
    long long launches = 0;
    int last_cuda = 0;
    /* obem_next.cu */
    void* d_next_scratch = nullptr; /* [np][6] floats: influence, E.n and right-hand side of the dynamic update */
    size_t next_scratch_cap = 0;
    int gemv_attr_set = 0;
    float4* d_step_field = nullptr; /* [n] E, phi at the charges: scratch of the steppers */
    long long step_field_cap = 0;
    /* obem_near.cu: exact near-field panel integrals (NEXT-3) */
    float* d_pverts = nullptr;   /* [np][3][3] copy of the vertices given to obem_set_panels            */
    float* d_psigma = nullptr;   /* [np] copy of the current sigma                                       */
    float4* d_porg = nullptr;    /* [np] frame origin of every panel (what the evaluation kernel shifts by) */
    float4* d_pcr = nullptr;     /* [np] centroid and near radius R_p = near_factor * longest edge        */
    long long near_cap = 0;      /* capacity of the four arrays above, in panels                         */
    int* d_cell_start = nullptr; /* [ncells + 1] CSR offsets of the per-cell candidate lists             */
    int* d_cell_fill = nullptr;  /* [ncells] fill cursors (build only)                                   */
    int* d_cell_list = nullptr;  /* panels whose near sphere overlaps the cell, ascending                */
    long long cell_cap = 0, list_cap = 0;
    double* d_near_red = nullptr; /* [8] bounding box of the near spheres, sum and count of R (build only) */
    void* d_scan_tmp = nullptr;
    size_t scan_tmp_cap = 0;
    double near_lo[3] = {0, 0, 0}, near_s = 0; /* grid origin and cell edge [m]                          */
    int near_n[3] = {0, 0, 0};                 /* cells per axis; 0 = no cell (no panel has R > 0)       */
    float near_factor = 3.0f;
    int near_valid = 0; /* the grid matches the current panels and near_factor */
    int* d_redo_list = nullptr;       /* targets too close to a quadrature source: recomputed in fp64 */
    unsigned* d_redo_count = nullptr;
    long long redo_cap = 0;
    float4* d_exact_tmp = nullptr;    /* [nt] panel part of an N-body + exact-panels evaluation */
    long long exact_tmp_cap = 0;
    long long near_entries = -1; /* (cell, panel) entries of the current lists; -1 before the first build */
    /* the targets of one evaluation grouped by cell (near_tcount / near_tfill) */
    int* d_near_tcell = nullptr;  /* [nt] cell of every target, -1 = none */
    int* d_near_tlist = nullptr;  /* [nt] targets in cell order */
    int* d_near_tcount = nullptr; /* [ncells + 1] targets per cell; then the fill cursor */
    int* d_near_tstart = nullptr; /* [ncells + 1] its exclusive scan; [ncells] = targets that have a cell */
    long long near_t_cap = 0, near_c_cap = 0;
    obem_nn_state nn;
    /* obem_geom.cu: symmetry planes and polygonal cells */
    int sym_n = 0, sym_axis[3] = {0, 0, 0}, sym_sign[3] = {1, 1, 1};
    double sym_coord[3] = {0, 0, 0};
    int sym_busy = 0;             /* inside obem_eval_symmetric: its own calls evaluate plainly */
    float4* d_sym_pts = nullptr;  /* reflected targets of one image */
    float4* d_sym_out = nullptr;  /* that image's field */
    size_t sym_pts_cap = 0, sym_out_cap = 0;
    float* d_cell_tri = nullptr;  /* [2 n_cells][3][3] triangles of the polygonal cells */
    float* d_cell_sig = nullptr;  /* [2 n_cells] */
    size_t cell_tri_cap = 0, cell_sig_cap = 0;
    /* obem_multi.cu: multi-sigma panel evaluation */
    long long geom_version = 0;  /* incremented by every obem_set_panels */
    float4* d_munit = nullptr;   /* blocked panel buffer encoded with sigma = 1 (bare weights A_p w_k) */
    float* d_msig = nullptr;     /* one pass's density vectors, blocked */
    size_t munit_cap = 0, msig_cap = 0;
    long long munit_geom = -1;   /* geom_version d_munit was built for */
    double* d_ramo = nullptr;    /* [K][blocks][2] partial sums of obem_ramo_current */
    size_t ramo_cap = 0;
    /* obem_map.cu */
    float4* d_map_pts = nullptr; /* node coordinates of the last obem_field_map */
    size_t map_pts_cap = 0;      /* bytes */
};

namespace {

struct DeviceGuard {
    int prev = -1;
    bool ok = true;
    explicit DeviceGuard(int dev)
    {
        if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
        if (prev != dev) ok = (cudaSetDevice(dev) == cudaSuccess);
    }
    ~DeviceGuard()
    {
        if (prev >= 0) cudaSetDevice(prev);
    }
};

int cuda_fail(obem_ctx* c, cudaError_t e)
{
    if (c) c->last_cuda = (int)e;
    cudaGetLastError(); /* clear the sticky-less error state */
    return (e == cudaErrorMemoryAllocation) ? OBEM_ENOMEM : OBEM_ECUDA;
}

#define OBEM_CUDA(c, call)                                 \
    do {                                                   \
        cudaError_t e__ = (call);                          \
        if (e__ != cudaSuccess) return cuda_fail((c), e__); \
    } while (0)

bool aligned16(const void* p) { return (((uintptr_t)p) & 15u) == 0; }
bool aligned4(const void* p) { return (((uintptr_t)p) & 3u) == 0; }

} /* namespace */

/* The evaluation proper (obem.cu): targets tgt[0..nt) -> out[0..nt) on stream st.  self_first >= 0: target i IS
 * charge self_first + i and is excluded from its own N-body sum by index.  eps_nbody: softening of the N-body
 * section for this call (eval_at_*: eps_pp; influence on the cells: eps_panel).  trk_out != NULL (targets must be
 * charges): also record, per target, the source block of its nearest opposite-sign charge (recombination). */
int obem_eval_internal(obem_ctx* c, const float4* tgt, long long nt, float4* out, unsigned flags, long long self_first,
                       float eps_nbody, cudaStream_t st, float2* trk_out = nullptr);

/* obem.cu: LIST-mode evaluation kernel launch (see there).  Block layout of `pool`: OBEM_SBH float4 per block = one
 * header (x = the weight all 256 sources share, or NaN) + 256 sources (x, y, z, w). */
#define OBEM_SB 256
#define OBEM_SBH 257
#define OBEM_TT 2048
int obem_eval_list(obem_ctx* c, const float4* tgt, long long nt, float4* out, const float4* pool,
                   const long long* tile_ptr, const int* list, const long long* U_dev, long long self_blocks, float eps,
                   cudaStream_t st);

/* obem.cu: copy the frame origin of every panel (what panel_loop shifts the targets by) to out[0..n_pan). */
int obem_panel_origins(obem_ctx* c, float4* out, cudaStream_t st);

/* obem_near.cu.  Called by obem_set_panels / obem_set_sigma: keep a copy of the geometry and of sigma for the exact
 * near-field integrals.  obem_near_correct: out[t] += k_e sum over panels p near target t of sigma_p (exact cell
 * integral - the 7-point value the evaluation kernel already added); builds the cell lists first if they are stale
 * (allocates and synchronises: once per geometry).  obem_near_free: release everything (obem_destroy). */
int obem_near_store_panels(obem_ctx* c, const float* d_verts, const float* d_sigma, long long np, cudaStream_t st);
int obem_near_store_sigma(obem_ctx* c, const float* d_sigma, long long np, cudaStream_t st);
int obem_near_correct(obem_ctx* c, const float4* tgt, long long nt, float4* out, cudaStream_t st);
/* the evaluation with OBEM_PANELS_EXACT: N-body part (if asked) into out, panel part + correction into scratch, sum */
int obem_eval_exact(obem_ctx* c, const float4* tgt, long long nt, float4* out, unsigned flags, long long self_first,
                    float eps_nbody, cudaStream_t st, float2* trk_out);
void obem_near_free(obem_ctx* c);

void obem_nn_free(obem_ctx* c);
void obem_multi_free(obem_ctx* c);
/* obem_geom.cu */
int obem_eval_symmetric(obem_ctx* c, const float4* tgt, long long nt, float4* out, unsigned flags, long long self_first,
                        float eps_nbody, cudaStream_t st, float2* trk_out);
void obem_geom_free(obem_ctx* c);

#endif /* OBEM_INTERNAL_CUH */
