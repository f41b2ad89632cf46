/*
 * obem_next.cu -- libobem.so, the steps adjacent to the field-evaluation hot path:
 *
 *   NEXT-1  influence of the particles on the cells, PAPER.md:241-257 (section 3.2.2):
 *     obem_influence_on_panels   Eq (3.3)/(3.4): area-averaged V and E of all charges over every cell.  With
 *                                the 7-point rule this is the adjoint of the panel->point sum: the field of the
 *                                charges at the 7*Np quadrature points (the hot path's evaluation kernel,
 *                                unchanged) followed by a 7-way weighted sum per cell (influence_reduce_kernel).
 *     obem_rhs_from_influence    Eq (3.5)/(3.6): modified left-hand sides of the BEM system.
 *     obem_apply_inverse         sigma = M^-1 b with the stored inverse: an HBM-bound fp32
 *                                GEMV streamed through a TMA ring (gemv_tma_kernel).
 *     obem_update_sigma_dynamic  the chain influence -> rhs -> M^-1 b -> set_sigma of the dynamic option
 *                                (PAPER.md:237, :257), enqueued on one stream.
 *
 * This file shares no code, header, table or constant with oracle/.
 */
#include "obem_internal.cuh"

namespace {

/* ------------------------------------------------------------------------------------------- */
/* Eq (3.3)/(3.4): 7-way weighted sum per cell                                                  */
/* ------------------------------------------------------------------------------------------- */
/* tmp [np*7] = k_e * (E, phi) of all charges at quadrature point k of cell i (from obem_eval_kernel);
 * qpts[..].w = rule weight w_k (sum 1), so (1/A_i) Int_{C_i} f d2r = sum_k w_k f(x_ik).  fp64 sum of 7. */
__global__ void influence_reduce_kernel(const float4* __restrict__ tmp, const float4* __restrict__ qpts,
                                        const float4* __restrict__ nrm, float4* __restrict__ infl,
                                        float* __restrict__ en, long long np)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= np) return;
    double ex = 0.0, ey = 0.0, ez = 0.0, vb = 0.0;
#pragma unroll
    for (int k = 0; k < 7; ++k) {
        const float4 f = tmp[i * 7 + k];
        const double w = (double)qpts[i * 7 + k].w;
        ex += w * (double)f.x;
        ey += w * (double)f.y;
        ez += w * (double)f.z;
        vb += w * (double)f.w;
    }
    infl[i] = make_float4((float)ex, (float)ey, (float)ez, (float)vb);
    if (en) {
        const float4 n = nrm[i];
        en[i] = (float)(ex * (double)n.x + ey * (double)n.y + ez * (double)n.z);
    }
}

/* Eq (3.5): b_i = V_i - Vbar_i (ed cells, kind 0); Eq (3.6): b_i = sigma_F,i - (eps2-eps1)_i Ebar_i.n_i (dd, kind 1).
 * An unknown kind writes NaN (the host cannot see device data without a copy). */
__global__ void rhs_kernel(const int* __restrict__ kind, const float* __restrict__ bc, const float* __restrict__ deps,
                           const float4* __restrict__ infl, const float* __restrict__ en, float* __restrict__ b,
                           long long np)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= np) return;
    const int k = kind[i];
    float r;
    if (k == 0) r = bc[i] - infl[i].w;
    else if (k == 1) r = fmaf(-deps[i], en[i], bc[i]);
    else r = __int_as_float(0x7fc00000);
    b[i] = r;
}

/* ------------------------------------------------------------------------------------------- */
/* sigma = M^-1 b : fp32 GEMV, bound by HBM (4 n^2 bytes read once)                             */
/* ------------------------------------------------------------------------------------------- */
constexpr int GV_THREADS = 256;           /* 8 warps                                                    */
constexpr int GV_ROWS = 16;               /* rows per tile: 2 per warp                                  */
constexpr int GV_COLS = 1024;             /* columns per tile: 4 KiB per row segment                    */
constexpr int GV_STAGES = 3;
constexpr int GV_STAGE_FLOATS = (GV_ROWS + 1) * GV_COLS; /* 16 row segments + the b segment            */
constexpr size_t GV_SMEM = (size_t)GV_STAGES * GV_STAGE_FLOATS * sizeof(float) + 64;

/*
 * Persistent CTAs; CTA c owns the row groups g = c, c + G, ... (16 rows each) and walks the columns of each in
 * chunks of 1024.  Thread 0 keeps a 3-stage ring of (16 row segments + b segment) full with 1-D TMA bulk copies
 * (17 x 4 KiB per stage, ~136 KiB in flight per SM: more than HBM latency x per-SM bandwidth); warp w reads rows
 * 2w, 2w+1 of the stage with conflict-free LDS.128, 4 fp32 partial sums per lane and row, reduced by shuffles at
 * the end of the row group.  Requires n % 4 == 0, ld % 4 == 0 and 16-byte aligned pointers (TMA granularity).
 */
__global__ void __launch_bounds__(GV_THREADS, 1) gemv_tma_kernel(const float* __restrict__ m, long long n, long long ld,
                                                                  const float* __restrict__ b, float* __restrict__ out)
{
    extern __shared__ __align__(128) unsigned char gv_smem[];
    float* ring = (float*)gv_smem;
    u64* full = (u64*)(gv_smem + (size_t)GV_STAGES * GV_STAGE_FLOATS * sizeof(float));

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const long long G = gridDim.x;
    const long long ngroups = (n + GV_ROWS - 1) / GV_ROWS;
    const long long nchunks = (n + GV_COLS - 1) / GV_COLS;
    const long long mygroups = (ngroups > blockIdx.x) ? (ngroups - blockIdx.x + G - 1) / G : 0;
    const long long items = mygroups * nchunks;
    if (items == 0) return;

    if (tid == 0) {
        for (int s = 0; s < GV_STAGES; ++s) mbar_init(&full[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    auto issue = [&](long long item) {
        const int s = (int)(item % GV_STAGES);
        const long long g = blockIdx.x + (item / nchunks) * G, ch = item % nchunks;
        const long long c0 = ch * GV_COLS, r0 = g * GV_ROWS;
        const unsigned cols = (unsigned)min((long long)GV_COLS, n - c0);
        const int rows = (int)min((long long)GV_ROWS, n - r0);
        float* st = ring + (size_t)s * GV_STAGE_FLOATS;
        mbar_expect_tx(&full[s], (unsigned)(rows + 1) * cols * 4u);
        tma_load_1d(st + GV_ROWS * GV_COLS, b + c0, cols * 4u, &full[s]);
        for (int r = 0; r < rows; ++r) tma_load_1d(st + r * GV_COLS, m + (r0 + r) * ld + c0, cols * 4u, &full[s]);
    };

    if (tid == 0)
        for (long long it = 0; it < GV_STAGES - 1 && it < items; ++it) issue(it);

    float4 acc0 = make_float4(0.f, 0.f, 0.f, 0.f), acc1 = acc0;
    for (long long it = 0; it < items; ++it) {
        __syncthreads(); /* everyone is done with the stage consumed in the previous iteration */
        if (tid == 0 && it + GV_STAGES - 1 < items) issue(it + GV_STAGES - 1);
        const int s = (int)(it % GV_STAGES);
        mbar_wait(&full[s], (unsigned)((it / GV_STAGES) & 1));

        const long long g = blockIdx.x + (it / nchunks) * G, ch = it % nchunks;
        const long long c0 = ch * GV_COLS, r0 = g * GV_ROWS;
        const int cols4 = (int)(min((long long)GV_COLS, n - c0) >> 2);
        const float4* st = (const float4*)(ring + (size_t)s * GV_STAGE_FLOATS);
        const float4* bs = st + GV_ROWS * (GV_COLS / 4);
        const float4* ra = st + (2 * warp) * (GV_COLS / 4);
        const float4* rb = ra + (GV_COLS / 4);
        const bool va = r0 + 2 * warp < n, vb = r0 + 2 * warp + 1 < n;
        if (va) {
#pragma unroll 4
            for (int j = lane; j < cols4; j += 32) {
                const float4 x = bs[j];
                const float4 a = ra[j];
                acc0.x = fmaf(a.x, x.x, acc0.x);
                acc0.y = fmaf(a.y, x.y, acc0.y);
                acc0.z = fmaf(a.z, x.z, acc0.z);
                acc0.w = fmaf(a.w, x.w, acc0.w);
                if (vb) {
                    const float4 c = rb[j];
                    acc1.x = fmaf(c.x, x.x, acc1.x);
                    acc1.y = fmaf(c.y, x.y, acc1.y);
                    acc1.z = fmaf(c.z, x.z, acc1.z);
                    acc1.w = fmaf(c.w, x.w, acc1.w);
                }
            }
        }
        if (ch == nchunks - 1) { /* row group finished: reduce and write its two rows */
            float s0 = (acc0.x + acc0.y) + (acc0.z + acc0.w), s1 = (acc1.x + acc1.y) + (acc1.z + acc1.w);
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                s0 += __shfl_xor_sync(0xffffffffu, s0, o);
                s1 += __shfl_xor_sync(0xffffffffu, s1, o);
            }
            if (lane == 0) {
                if (va) out[r0 + 2 * warp] = s0;
                if (vb) out[r0 + 2 * warp + 1] = s1;
            }
            acc0 = acc1 = make_float4(0.f, 0.f, 0.f, 0.f);
        }
    }
}

/* Any n / ld / alignment: one warp per row, scalar coalesced loads.  Same summation shape per lane. */
__global__ void __launch_bounds__(256) gemv_plain_kernel(const float* __restrict__ m, long long n, long long ld,
                                                          const float* __restrict__ b, float* __restrict__ out)
{
    const int lane = threadIdx.x & 31;
    const long long wpg = (long long)gridDim.x * (blockDim.x >> 5);
    for (long long r = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); r < n; r += wpg) {
        const float* row = m + r * ld;
        float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f;
        long long j = lane;
        for (; j + 96 < n; j += 128) {
            a0 = fmaf(__ldg(row + j), __ldg(b + j), a0);
            a1 = fmaf(__ldg(row + j + 32), __ldg(b + j + 32), a1);
            a2 = fmaf(__ldg(row + j + 64), __ldg(b + j + 64), a2);
            a3 = fmaf(__ldg(row + j + 96), __ldg(b + j + 96), a3);
        }
        for (; j < n; j += 32) a0 = fmaf(__ldg(row + j), __ldg(b + j), a0);
        float s = (a0 + a1) + (a2 + a3);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
        if (lane == 0) out[r] = s;
    }
}

/* ------------------------------------------------------------------------------------------- */
/* NEXT-2: numerical integrators, PAPER.md:300-306 (section 3.2.5)                              */
/* ------------------------------------------------------------------------------------------- */
/* state: xyzq [n] = (x, y, z [m], q [C]), vel [n] = (vx, vy, vz [m/s], m [kg]); dx/dt = v, dv/dt = (q/m) E(x).
 * m = 0 marks an immobile charge (q/m taken as 0). */
__device__ __forceinline__ float q_over_m(float q, float m) { return (m != 0.f) ? q / m : 0.f; }

/* drift: x += h v */
__global__ void drift_kernel(float4* __restrict__ xyzq, const float4* __restrict__ vel, float h, long long n)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float4 x = xyzq[i];
    const float4 v = vel[i];
    x.x = fmaf(h, v.x, x.x);
    x.y = fmaf(h, v.y, x.y);
    x.z = fmaf(h, v.z, x.z);
    xyzq[i] = x;
}

/* kick: v += h (q/m) E */
__global__ void kick_kernel(const float4* __restrict__ xyzq, float4* __restrict__ vel, const float4* __restrict__ field,
                            float h, long long n)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float4 v = vel[i];
    const float4 e = field[i];
    const float a = h * q_over_m(xyzq[i].w, v.w);
    v.x = fmaf(a, e.x, v.x);
    v.y = fmaf(a, e.y, v.y);
    v.z = fmaf(a, e.z, v.z);
    vel[i] = v;
}

/* basic Euler: x_{n+1} = x_n + h v_n, v_{n+1} = v_n + h (q/m) E(x_n) -- both from the state at the start */
__global__ void euler_kernel(float4* __restrict__ xyzq, float4* __restrict__ vel, const float4* __restrict__ field,
                             float h, long long n)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float4 x = xyzq[i];
    float4 v = vel[i];
    const float4 e = field[i];
    x.x = fmaf(h, v.x, x.x);
    x.y = fmaf(h, v.y, x.y);
    x.z = fmaf(h, v.z, x.z);
    const float a = h * q_over_m(x.w, v.w);
    v.x = fmaf(a, e.x, v.x);
    v.y = fmaf(a, e.y, v.y);
    v.z = fmaf(a, e.z, v.z);
    xyzq[i] = x;
    vel[i] = v;
}

int grow_step_field(obem_ctx* c, long long n)
{
    if (n <= c->step_field_cap) return OBEM_OK;
    float4* p = nullptr;
    OBEM_CUDA(c, cudaMalloc(&p, (size_t)n * sizeof(float4)));
    if (c->d_step_field) cudaFree(c->d_step_field);
    c->d_step_field = p;
    c->step_field_cap = n;
    return OBEM_OK;
}

/* field at the current positions: set_charges(x) + eval_at_charges -> c->d_step_field */
int field_at_state(obem_ctx* c, const float* d_xyzq, long long n, unsigned flags, void* stream)
{
    int rc = obem_set_charges(c, d_xyzq, n, stream);
    if (rc != OBEM_OK) return rc;
    /* the kicks read only E: the E-only instantiations of the evaluation kernels */
    return obem_eval_at_charges(c, (float*)c->d_step_field, flags | OBEM_NO_PHI, stream);
}

int step_args_ok(obem_ctx* c, const float* d_xyzq, const float* d_vel, int64_t n, unsigned flags)
{
    if (!c || n < 0) return OBEM_EINVAL;
    if (flags & ~(OBEM_NBODY | OBEM_PANELS)) return OBEM_EINVAL;
    if (n > 0 && (!d_xyzq || !d_vel || !aligned16(d_xyzq) || !aligned16(d_vel))) return OBEM_EINVAL;
    if ((flags & OBEM_PANELS) && c->n_pan < 0) return OBEM_ESTATE;
    return OBEM_OK;
}

int grow_scratch(obem_ctx* c, long long np)
{
    const size_t need = (size_t)(np > 0 ? np : 1) * 6 * sizeof(float);
    if (need <= c->next_scratch_cap) return OBEM_OK;
    void* p = nullptr;
    OBEM_CUDA(c, cudaMalloc(&p, need));
    if (c->d_next_scratch) cudaFree(c->d_next_scratch);
    c->d_next_scratch = p;
    c->next_scratch_cap = need;
    return OBEM_OK;
}

} /* namespace */

extern "C" {

int obem_influence_on_panels(obem_ctx* c, float* d_infl, float* d_en, void* cuda_stream)
{
    if (!c) return OBEM_EINVAL;
    if (c->n_pan < 0 || c->n_chg < 0) return OBEM_ESTATE;
    const long long np = c->n_pan;
    if (np == 0) return OBEM_OK;
    if (!d_infl || !aligned16(d_infl) || (d_en && !aligned4(d_en))) return OBEM_EINVAL;
    DeviceGuard g(c->device);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    /* field of all charges at the 7 np quadrature points, softened like the panel sums (the adjoint of a4) */
    int rc = obem_eval_internal(c, c->d_qpts, np * 7, c->d_infl_tmp, OBEM_NBODY, -1, c->eps_panel, st);
    if (rc != OBEM_OK) return rc;
    influence_reduce_kernel<<<(unsigned)ceil_div(np, 128), 128, 0, st>>>(c->d_infl_tmp, c->d_qpts, c->d_nrm,
                                                                         (float4*)d_infl, d_en, np);
    OBEM_CUDA(c, cudaGetLastError());
    c->launches += 1;
    return OBEM_OK;
}

int obem_rhs_from_influence(obem_ctx* c, const int32_t* d_kind, const float* d_bc, const float* d_deps,
                            const float* d_infl, const float* d_en, float* d_b, int64_t n_panels, void* cuda_stream)
{
    if (!c || n_panels < 0) return OBEM_EINVAL;
    if (n_panels == 0) return OBEM_OK;
    if (!d_kind || !d_bc || !d_deps || !d_infl || !d_en || !d_b || !aligned16(d_infl) || !aligned4(d_kind) ||
        !aligned4(d_bc) || !aligned4(d_deps) || !aligned4(d_en) || !aligned4(d_b))
        return OBEM_EINVAL;
    DeviceGuard g(c->device);
    rhs_kernel<<<(unsigned)ceil_div(n_panels, 256), 256, 0, (cudaStream_t)cuda_stream>>>(
        d_kind, d_bc, d_deps, (const float4*)d_infl, d_en, d_b, n_panels);
    OBEM_CUDA(c, cudaGetLastError());
    c->launches += 1;
    return OBEM_OK;
}

int obem_apply_inverse(obem_ctx* c, const float* d_minv, int64_t n, int64_t ld, const float* d_b, float* d_sigma,
                       void* cuda_stream)
{
    if (!c || n < 0 || ld < n) return OBEM_EINVAL;
    if (n == 0) return OBEM_OK;
    if (!d_minv || !d_b || !d_sigma || !aligned4(d_minv) || !aligned4(d_b) || !aligned4(d_sigma)) return OBEM_EINVAL;
    DeviceGuard g(c->device);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const bool tma_ok = (n % 4 == 0) && (ld % 4 == 0) && aligned16(d_minv) && aligned16(d_b);
    if (tma_ok) {
        if (!c->gemv_attr_set) {
            OBEM_CUDA(c, cudaFuncSetAttribute(gemv_tma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                              (int)GV_SMEM));
            c->gemv_attr_set = 1;
        }
        const long long ngroups = ceil_div(n, GV_ROWS);
        const unsigned grid = (unsigned)(ngroups < c->sm_count ? ngroups : c->sm_count);
        gemv_tma_kernel<<<grid, GV_THREADS, GV_SMEM, st>>>(d_minv, n, ld, d_b, d_sigma);
    } else {
        const long long want = ceil_div(n, 8);
        const unsigned grid = (unsigned)(want < 8LL * c->sm_count ? want : 8LL * c->sm_count);
        gemv_plain_kernel<<<grid, 256, 0, st>>>(d_minv, n, ld, d_b, d_sigma);
    }
    OBEM_CUDA(c, cudaGetLastError());
    c->launches += 1;
    return OBEM_OK;
}

int obem_update_sigma_dynamic(obem_ctx* c, const int32_t* d_kind, const float* d_bc, const float* d_deps,
                              const float* d_minv, int64_t ld, float* d_sigma, void* cuda_stream)
{
    if (!c) return OBEM_EINVAL;
    if (c->n_pan < 0 || c->n_chg < 0) return OBEM_ESTATE;
    const long long np = c->n_pan;
    if (np == 0) return OBEM_OK;
    if (!d_sigma || !aligned4(d_sigma)) return OBEM_EINVAL;
    int rc;
    {
        DeviceGuard g(c->device);
        rc = grow_scratch(c, np);
    }
    if (rc != OBEM_OK) return rc;
    float* infl = (float*)c->d_next_scratch; /* [np][4] */
    float* en = infl + 4 * np;               /* [np]    */
    float* b = en + np;                      /* [np]    */
    rc = obem_influence_on_panels(c, infl, en, cuda_stream);
    if (rc == OBEM_OK) rc = obem_rhs_from_influence(c, d_kind, d_bc, d_deps, infl, en, b, np, cuda_stream);
    if (rc == OBEM_OK) rc = obem_apply_inverse(c, d_minv, np, ld, b, d_sigma, cuda_stream);
    if (rc == OBEM_OK) rc = obem_set_sigma(c, d_sigma, np, cuda_stream);
    return rc;
}

int obem_push_drift(obem_ctx* c, float* d_xyzq, const float* d_vel, int64_t n, float h, void* cuda_stream)
{
    if (!c || n < 0 || !isfinite(h)) return OBEM_EINVAL;
    if (n == 0) return OBEM_OK;
    if (!d_xyzq || !d_vel || !aligned16(d_xyzq) || !aligned16(d_vel)) return OBEM_EINVAL;
    DeviceGuard g(c->device);
    drift_kernel<<<(unsigned)ceil_div(n, 256), 256, 0, (cudaStream_t)cuda_stream>>>((float4*)d_xyzq,
                                                                                    (const float4*)d_vel, h, n);
    OBEM_CUDA(c, cudaGetLastError());
    c->launches += 1;
    return OBEM_OK;
}

int obem_push_kick(obem_ctx* c, const float* d_xyzq, float* d_vel, const float* d_field, int64_t n, float h,
                   void* cuda_stream)
{
    if (!c || n < 0 || !isfinite(h)) return OBEM_EINVAL;
    if (n == 0) return OBEM_OK;
    if (!d_xyzq || !d_vel || !d_field || !aligned16(d_xyzq) || !aligned16(d_vel) || !aligned16(d_field))
        return OBEM_EINVAL;
    DeviceGuard g(c->device);
    kick_kernel<<<(unsigned)ceil_div(n, 256), 256, 0, (cudaStream_t)cuda_stream>>>(
        (const float4*)d_xyzq, (float4*)d_vel, (const float4*)d_field, h, n);
    OBEM_CUDA(c, cudaGetLastError());
    c->launches += 1;
    return OBEM_OK;
}

int obem_step_euler(obem_ctx* c, float* d_xyzq, float* d_vel, int64_t n, float dt, unsigned flags, void* cuda_stream)
{
    int rc = step_args_ok(c, d_xyzq, d_vel, n, flags);
    if (rc != OBEM_OK || !isfinite(dt)) return rc != OBEM_OK ? rc : OBEM_EINVAL;
    DeviceGuard g(c->device);
    rc = grow_step_field(c, n);
    if (rc != OBEM_OK) return rc;
    rc = field_at_state(c, d_xyzq, n, flags, cuda_stream);
    if (rc != OBEM_OK || n == 0) return rc;
    euler_kernel<<<(unsigned)ceil_div(n, 256), 256, 0, (cudaStream_t)cuda_stream>>>(
        (float4*)d_xyzq, (float4*)d_vel, c->d_step_field, dt, n);
    OBEM_CUDA(c, cudaGetLastError());
    c->launches += 1;
    return OBEM_OK;
}

int obem_step_pefrl(obem_ctx* c, float* d_xyzq, float* d_vel, int64_t n, float dt, unsigned flags, void* cuda_stream)
{
    int rc = step_args_ok(c, d_xyzq, d_vel, n, flags);
    if (rc != OBEM_OK || !isfinite(dt)) return rc != OBEM_OK ? rc : OBEM_EINVAL;
    DeviceGuard g(c->device);
    rc = grow_step_field(c, n);
    if (rc != OBEM_OK) return rc;
    /* Omelyan, Mryglod, Folk, Comput. Phys. Commun. 146 (2002) 188: position-extended Forest-Ruth-like scheme */
    const double xi = 0.1786178958448091, lam = -0.2123418310626054, chi = -0.6626458266981849e-1;
    const double h = (double)dt;
    const float drift[5] = {(float)(xi * h), (float)(chi * h), (float)((1.0 - 2.0 * (chi + xi)) * h), (float)(chi * h),
                            (float)(xi * h)};
    const float kick[4] = {(float)((1.0 - 2.0 * lam) * 0.5 * h), (float)(lam * h), (float)(lam * h),
                           (float)((1.0 - 2.0 * lam) * 0.5 * h)};
    for (int s = 0; s < 5; ++s) {
        rc = obem_push_drift(c, d_xyzq, d_vel, n, drift[s], cuda_stream);
        if (rc != OBEM_OK) return rc;
        if (s == 4) break;
        rc = field_at_state(c, d_xyzq, n, flags, cuda_stream);
        if (rc == OBEM_OK) rc = obem_push_kick(c, d_xyzq, d_vel, (const float*)c->d_step_field, n, kick[s], cuda_stream);
        if (rc != OBEM_OK) return rc;
    }
    return OBEM_OK;
}

int obem_get_panel_normals(obem_ctx* c, float* d_out, void* cuda_stream)
{
    if (!c) return OBEM_EINVAL;
    if (c->n_pan < 0) return OBEM_ESTATE;
    if (c->n_pan == 0) return OBEM_OK;
    if (!d_out || !aligned16(d_out)) return OBEM_EINVAL;
    DeviceGuard g(c->device);
    OBEM_CUDA(c, cudaMemcpyAsync(d_out, c->d_nrm, (size_t)c->n_pan * sizeof(float4), cudaMemcpyDeviceToDevice,
                                 (cudaStream_t)cuda_stream));
    return OBEM_OK;
}

} /* extern "C" */
