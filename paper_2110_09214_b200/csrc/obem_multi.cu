/*
 * obem_multi.cu -- the panel sums Eq (2.13)/(2.14) for SEVERAL charge-density vectors on one
 * geometry in one pass ("multi-sigma evaluation").
 *
 * Why the method needs it: the induced signal on read-out electrode e is computed with the Shockley-Ramo theorem from
 * that electrode's WEIGHTING field (section 3.3.4, Eq 3.13) -- the field of the set-up with electrode
 * e at unit potential and all others grounded, i.e. one more solution sigma^(e) of the same BEM matrix (PAPER.md:
 * 137-139: "inverted once").  A detector with K read-out electrodes therefore evaluates K + 1 panel sums on the same
 * cells at the same points; the geometry part of every (quadrature point, target) interaction -- distance, rsqrt,
 * u^3 d -- does not depend on sigma.
 *
 * How: the hot path's panel launch folds sigma_p A_p w_k into the encoded geometry (panel_encode), which is exactly
 * what ties it to one sigma.  Here the encoded weight is the BARE quadrature weight A_p w_k (> 0, sigma = 1), the
 * 7 sources of a panel are summed into the panel's unit-density integrals G_p = sum_k A w_k u^3 d, H_p = sum_k A w_k u
 * (same 12 packed FP32 instructions per source and target pair as the hot path), and each of the KS density vectors
 * of the pass then costs 4 packed FMAs per PANEL and pair: E^(s) += sigma^(s)_p G_p, phi^(s) += sigma^(s)_p H_p.
 * Packed instructions per panel and target pair: 3 (frame shift) + 7 x 12 + 4 KS = 103 for KS = 4 against 4 x 87 for
 * four single-sigma launches.  K > 4 runs ceil(K / 4) passes.
 *
 * Launch shape: persistent grid, one CTA per SM, tiles of 1024 targets (256 threads x 4) taken round-robin -- a tile
 * is never split, so there is no workspace and no fix-up; panel blocks (and the pass's sigma rows, re-blocked to
 * 36 x 4 floats per block: the four densities of a panel side by side) stream through the same 4-stage TMA ring as the hot path; block sums in fp32, the
 * running sums in fp64 in shared memory (4 KS doubles per target).  A target at zero distance from a quadrature
 * point (reading A4) poisons its sums with inf/NaN; that is detected when the tile is written and the owning thread
 * recomputes that target in fp64 with the guard (rare: a measure-zero event).
 *
 * Part of libobem.so; shares nothing with oracle/.
 */
#include "obem_internal.cuh"

namespace {

constexpr int M_THREADS = 256;
constexpr int M_NP = 2;                      /* target pairs per thread                         */
constexpr int M_TT = M_THREADS * 2 * M_NP;   /* targets per tile                                */
constexpr int M_STAGES = 4;
constexpr int M_KS = 4;                      /* density vectors per pass                        */
static_assert(M_KS == 4, "the kernel reads the densities of a panel as one float4");
constexpr int M_SROW = 36;                   /* floats per (block, vector) sigma row: PPB = 34 padded to 144 B */
#ifndef OBEM_M_DEPTH
#define OBEM_M_DEPTH 4
#endif
constexpr int M_DEPTH = OBEM_M_DEPTH;        /* software-pipeline distance of the source loop   */
constexpr double M_KE = 1.0 / (4.0 * 3.14159265358979323846 * 8.8541878128e-12); /* reading A7 */

struct MultiParams {
    const float4* unit;   /* blocked panel buffer encoded with the bare weights A_p w_k (sigma = 1)      */
    const float* sig;     /* [nblk][M_SROW][M_KS] the pass's density vectors, blocked                      */
    const float4* qrel;   /* [np*7] plain offsets from the frame origin, .w = A_p w_k (repair)            */
    const float* sigma;   /* [K][np] the caller's vectors (repair)                                       */
    long long np, nblk;
    const float4* tgt;
    long long nt, ntiles;
    float4* out;          /* [K][nt]                                                                     */
    int k0, ks;           /* this pass computes vectors k0 .. k0 + ks - 1                                 */
    float eps2;
};

/* unit-density encoding of every quadrature source: weight = A_p w_k, which pack_panels_kernel left in qrel.w */
__global__ void __launch_bounds__(128) multi_unit_kernel(const float4* __restrict__ psrc, const float4* __restrict__ qrel,
                                                         float4* __restrict__ unit, long long np, long long np_pad)
{
    const long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= np_pad) return;
    const long long e = panel_entry(p);
    if (p % PPB == 0) {
        unit[e - 1] = make_float4(0.f, 0.f, 0.f, 0.f);
        unit[e - 1 + SBH_P - 2] = make_float4(0.f, 0.f, 0.f, 0.f);
        unit[e - 1 + SBH_P - 1] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    unit[e] = (p < np) ? psrc[e] : make_float4(0.f, 0.f, 0.f, 0.f); /* the frame origin */
#pragma unroll
    for (int k = 0; k < 7; ++k) {
        if (p < np) {
            const float4 r = qrel[p * 7 + k];
            panel_encode((double)r.w, (double)r.x, (double)r.y, (double)r.z, unit[e + 1 + 2 * k], unit[e + 2 + 2 * k]);
        } else {
            panel_encode(0.0, 0.0, 0.0, 0.0, unit[e + 1 + 2 * k], unit[e + 2 + 2 * k]);
        }
    }
}

/* sigma[k0 + s][p] -> sig[(block b, slot j, vector s of M_KS)]: the up to 4 densities of a panel side by side, so
 * that the kernel reads them with ONE LDS.128; zero beyond np, in the two pad slots and for vectors >= ks */
__global__ void __launch_bounds__(256) multi_sigma_kernel(const float* __restrict__ sigma, float* __restrict__ sig,
                                                          long long np, long long nblk, int k0, int ks)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nblk * M_KS * M_SROW) return;
    const int s = (int)(i % M_KS);
    const long long r = i / M_KS;
    const int j = (int)(r % M_SROW);
    const long long b = r / M_SROW, p = b * PPB + j;
    sig[i] = (s < ks && j < PPB && p < np) ? sigma[(long long)(k0 + s) * np + p] : 0.f;
}

/* guarded fp64 recomputation of one target for one density vector (the rare zero-distance case, reading A4) */
__device__ float4 multi_repair(const MultiParams& P, const float4 t, const int k)
{
    double ex = 0.0, ey = 0.0, ez = 0.0, ph = 0.0;
    const double e2 = (double)P.eps2;
    for (long long p = 0; p < P.np; ++p) {
        const double sg = (double)P.sigma[(long long)k * P.np + p];
        if (sg == 0.0) continue;
        const float4 o = P.unit[panel_entry(p)];
        double gx = 0.0, gy = 0.0, gz = 0.0, gh = 0.0;
        for (int q = 0; q < 7; ++q) {
            const float4 r = P.qrel[p * 7 + q];
            if (r.w == 0.f) continue;
            /* shift into the frame in fp32 like the hot loop, then subtract the plain offset */
            const double dx = (double)(t.x - o.x) - r.x, dy = (double)(t.y - o.y) - r.y, dz = (double)(t.z - o.z) - r.z;
            const double r2 = dx * dx + dy * dy + dz * dz + e2;
            if (!(r2 > 0.0)) continue;
            const double u = rsqrt(r2), wu = (double)r.w * u, s3 = wu * u * u;
            gh += wu;
            gx += s3 * dx;
            gy += s3 * dy;
            gz += s3 * dz;
        }
        ex += sg * gx;
        ey += sg * gy;
        ez += sg * gz;
        ph += sg * gh;
    }
    return make_float4((float)(M_KE * ex), (float)(M_KE * ey), (float)(M_KE * ez), (float)(M_KE * ph));
}

template <int KS, bool HAS_EPS>
__global__ void __launch_bounds__(M_THREADS, 1) panels_multi_kernel(const MultiParams P)
{
    extern __shared__ __align__(16) double macc_dyn[]; /* [4 KS x 2 M_NP][M_THREADS] running sums, fp64 */
    __shared__ __align__(128) float4 ring[M_STAGES][SBH_P];
    __shared__ __align__(16) float sring[M_STAGES][M_KS * M_SROW];
    __shared__ __align__(8) u64 full[M_STAGES];

    const int tid = threadIdx.x;
    double* const acc = macc_dyn + tid;
    const long long G = gridDim.x, c = blockIdx.x;
    if (c >= P.ntiles) return;
    const long long my_tiles = (P.ntiles - c + G - 1) / G;
    const long long units = my_tiles * P.nblk;
    if (tid == 0) {
        for (int s = 0; s < M_STAGES; ++s) mbar_init(&full[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const unsigned bytes_p = (unsigned)(SBH_P * sizeof(float4)), bytes_s = (unsigned)(M_KS * M_SROW * sizeof(float));
    long long pu = 0, pblk = 0; /* producer (thread 0): next unit and its block */
    auto produce = [&](int stage) {
        mbar_expect_tx(&full[stage], bytes_p + bytes_s);
        tma_load_1d(&ring[stage][0], P.unit + pblk * SBH_P, bytes_p, &full[stage]);
        tma_load_1d(&sring[stage][0], P.sig + pblk * (M_KS * M_SROW), bytes_s, &full[stage]);
        ++pu;
        if (++pblk == P.nblk) pblk = 0;
    };
    if (tid == 0)
        for (int s = 0; s < M_STAGES - 1 && pu < units; ++s) produce(s);

    unsigned it = 0;
    for (long long tile = c; tile < P.ntiles; tile += G) {
        const long long tbase = tile * (long long)M_TT + tid;
        u64 X[M_NP], Y[M_NP], Z[M_NP];
#pragma unroll
        for (int p = 0; p < M_NP; ++p) {
            const long long i0 = tbase + (2 * p) * M_THREADS, i1 = i0 + M_THREADS;
            const float* ta = (const float*)(P.tgt + i0);
            const float* tb = (const float*)(P.tgt + i1);
            const bool va = i0 < P.nt, vb = i1 < P.nt;
            X[p] = pk_keep(va ? __ldg(ta + 0) : 0.f, vb ? __ldg(tb + 0) : 0.f);
            Y[p] = pk_keep(va ? __ldg(ta + 1) : 0.f, vb ? __ldg(tb + 1) : 0.f);
            Z[p] = pk_keep(va ? __ldg(ta + 2) : 0.f, vb ? __ldg(tb + 2) : 0.f);
        }
#pragma unroll
        for (int v = 0; v < 8 * KS * M_NP; ++v) acc[v * M_THREADS] = 0.0;

        for (long long blk = 0; blk < P.nblk; ++blk, ++it) {
            __syncthreads(); /* everyone is done with the stage consumed in the previous iteration */
            if (tid == 0 && pu < units) produce((it + M_STAGES - 1) % M_STAGES);
            const int st = it % M_STAGES;
            mbar_wait(&full[st], (it / M_STAGES) & 1u);
            const float4* sblk = &ring[st][1];
            const float* ssig = &sring[st][0];

            u64 aX[KS][M_NP], aY[KS][M_NP], aZ[KS][M_NP], aP[KS][M_NP];
#pragma unroll
            for (int s = 0; s < KS; ++s)
#pragma unroll
                for (int p = 0; p < M_NP; ++p) aX[s][p] = aY[s][p] = aZ[s][p] = aP[s][p] = 0ull;

#pragma unroll 1
            for (int pp = 0; pp < PPB; ++pp) {
                const float4* ps = sblk + pp * PANEL_SLOTS;
                const float4 o = ps[0];
                u64 TX[M_NP], TY[M_NP], TZ[M_NP];
#pragma unroll
                for (int p = 0; p < M_NP; ++p) {
                    TX[p] = sub2(X[p], pk(o.x, o.x));
                    TY[p] = sub2(Y[p], pk(o.y, o.y));
                    TZ[p] = sub2(Z[p], pk(o.z, o.z));
                }
                float4 qa[7];
                float2 qb[7];
#pragma unroll
                for (int j = 0; j < 7; ++j) {
                    qa[j] = ps[1 + 2 * j];
                    qb[j] = *reinterpret_cast<const float2*>(ps + 2 + 2 * j);
                }
                /* the panel's unit-density integrals for this thread's targets */
                u64 gX[M_NP], gY[M_NP], gZ[M_NP], gH[M_NP];
#pragma unroll
                for (int p = 0; p < M_NP; ++p) gX[p] = gY[p] = gZ[p] = gH[p] = 0ull;
                constexpr int K = 7 * M_NP;
                u64 dX[K], dY[K], dZ[K], U[K];
#pragma unroll
                for (int k = 0; k < K + M_DEPTH; ++k) {
                    if (k < K) {
                        const int j = k / M_NP, p = k % M_NP;
                        const u64 a2 = pk(qa[j].x, qa[j].x);
                        dX[k] = fma2(TX[p], a2, pk(qa[j].y, qa[j].y));
                        dY[k] = fma2(TY[p], a2, pk(qa[j].z, qa[j].z));
                        dZ[k] = fma2(TZ[p], a2, pk(qa[j].w, qa[j].w));
                        u64 r2;
                        if (HAS_EPS) {
                            const float e = qb[j].y * P.eps2;
                            r2 = fma2(dX[k], dX[k], pk(e, e));
                        } else {
                            r2 = mul2(dX[k], dX[k]);
                        }
                        r2 = fma2(dY[k], dY[k], r2);
                        r2 = fma2(dZ[k], dZ[k], r2);
                        float r2l, r2h;
                        upk(r2, r2l, r2h);
                        U[k] = pk(rsqrt_approx(r2l), rsqrt_approx(r2h));
                    }
                    if (k >= M_DEPTH) {
                        const int kk = k - M_DEPTH, j = kk / M_NP, p = kk % M_NP;
                        gH[p] = fma2(U[kk], pk(qb[j].x, qb[j].x), gH[p]);
                        const u64 u2 = mul2(U[kk], U[kk]);
                        const u64 u3 = mul2(u2, U[kk]);
                        gX[p] = fma2(u3, dX[kk], gX[p]);
                        gY[p] = fma2(u3, dY[kk], gY[p]);
                        gZ[p] = fma2(u3, dZ[kk], gZ[p]);
                    }
                }
                /* 4 packed FMAs per density vector, panel and pair */
                const float4 sg4 = *reinterpret_cast<const float4*>(ssig + pp * M_KS); /* one broadcast LDS.128 */
                const float sgv[4] = {sg4.x, sg4.y, sg4.z, sg4.w};
#pragma unroll
                for (int s = 0; s < KS; ++s) {
                    const float sg = sgv[s];
                    const u64 sg2 = pk(sg, sg);
#pragma unroll
                    for (int p = 0; p < M_NP; ++p) {
                        aX[s][p] = fma2(gX[p], sg2, aX[s][p]);
                        aY[s][p] = fma2(gY[p], sg2, aY[s][p]);
                        aZ[s][p] = fma2(gZ[p], sg2, aZ[s][p]);
                        aP[s][p] = fma2(gH[p], sg2, aP[s][p]);
                    }
                }
            }
            /* second accumulation level: fp64 in shared memory, acc[((s * 2 M_NP + slot) * 4 + comp) * THREADS] */
#pragma unroll
            for (int s = 0; s < KS; ++s)
#pragma unroll
                for (int p = 0; p < M_NP; ++p) {
                    double* a = acc + (size_t)((s * 2 * M_NP + 2 * p) * 4) * M_THREADS;
                    float l, h;
                    upk(aX[s][p], l, h);
                    a[0 * M_THREADS] += (double)l;
                    a[4 * M_THREADS] += (double)h;
                    upk(aY[s][p], l, h);
                    a[1 * M_THREADS] += (double)l;
                    a[5 * M_THREADS] += (double)h;
                    upk(aZ[s][p], l, h);
                    a[2 * M_THREADS] += (double)l;
                    a[6 * M_THREADS] += (double)h;
                    upk(aP[s][p], l, h);
                    a[3 * M_THREADS] += (double)l;
                    a[7 * M_THREADS] += (double)h;
                }
        }

#pragma unroll
        for (int s = 0; s < KS; ++s)
#pragma unroll
            for (int k = 0; k < 2 * M_NP; ++k) {
                const long long i = tbase + (long long)k * M_THREADS;
                if (i >= P.nt) continue;
                const double* a = acc + (size_t)((s * 2 * M_NP + k) * 4) * M_THREADS;
                float4 o = make_float4((float)(M_KE * a[0]), (float)(M_KE * a[M_THREADS]), (float)(M_KE * a[2 * M_THREADS]),
                                       (float)(M_KE * a[3 * M_THREADS]));
                if (!(isfinite(o.x) && isfinite(o.y) && isfinite(o.z) && isfinite(o.w))) o = multi_repair(P, P.tgt[i], P.k0 + s);
                P.out[(long long)(P.k0 + s) * P.nt + i] = o;
            }
    }
}

/*
 * The Shockley-Ramo signal sum, Eq (3.13): i_k = sum_p q_p v_p . E_w^(k)(r_p), separately for the
 * particles with q < 0 and with q > 0 ("the signals created by each type are generated separately").
 * ew [K][n] is what obem_eval_panels_multi writes for K weighting-field density vectors at the charges.  fp32 inputs,
 * every term and every sum in fp64, fixed summation order (strided per thread, tree per block; the blocks' partials
 * the same way in a second launch): the result is deterministic.  Bound: HBM (16 B of E_w per particle and electrode; q and v come from L2 after the first
 * electrode).  Grid: (blocks, K).
 */
constexpr int R_THREADS = 256;
__global__ void __launch_bounds__(R_THREADS) ramo_partial_kernel(const float4* __restrict__ xyzq, const float4* __restrict__ vel,
                                                                 const float4* __restrict__ ew, long long n, long long chunk,
                                                                 double* __restrict__ part)
{
    __shared__ double red[2][R_THREADS];
    const int tid = threadIdx.x, k = blockIdx.y;
    const long long i0 = (long long)blockIdx.x * chunk, i1 = (i0 + chunk < n) ? i0 + chunk : n;
    double neg = 0.0, pos = 0.0;
#pragma unroll 4
    for (long long i = i0 + tid; i < i1; i += R_THREADS) {
        const float q = xyzq[i].w;
        const float4 v = vel[i], e = ew[(long long)k * n + i];
        const double term = (double)q * ((double)v.x * (double)e.x + (double)v.y * (double)e.y + (double)v.z * (double)e.z);
        if (q < 0.f) neg += term;
        else if (q > 0.f) pos += term;
    }
    red[0][tid] = neg, red[1][tid] = pos;
    __syncthreads();
    for (int h = R_THREADS / 2; h > 0; h >>= 1) {
        if (tid < h) red[0][tid] += red[0][tid + h], red[1][tid] += red[1][tid + h];
        __syncthreads();
    }
    if (tid == 0) {
        part[((size_t)k * gridDim.x + blockIdx.x) * 2 + 0] = red[0][0];
        part[((size_t)k * gridDim.x + blockIdx.x) * 2 + 1] = red[1][0];
    }
}
/* one CTA per electrode: thread t sums the partials t, t + 256, ... in ascending order, then the same fixed tree */
__global__ void __launch_bounds__(R_THREADS) ramo_final_kernel(const double* __restrict__ part, int blocks, int K,
                                                               double* __restrict__ out)
{
    __shared__ double red[2][R_THREADS];
    const int tid = threadIdx.x, k = blockIdx.x;
    double neg = 0.0, pos = 0.0;
    for (int b = tid; b < blocks; b += R_THREADS) {
        neg += part[((size_t)k * blocks + b) * 2];
        pos += part[((size_t)k * blocks + b) * 2 + 1];
    }
    red[0][tid] = neg, red[1][tid] = pos;
    __syncthreads();
    for (int h = R_THREADS / 2; h > 0; h >>= 1) {
        if (tid < h) red[0][tid] += red[0][tid + h], red[1][tid] += red[1][tid + h];
        __syncthreads();
    }
    if (tid == 0) out[2 * k] = red[0][0], out[2 * k + 1] = red[1][0];
}

template <int KS>
cudaError_t launch_pass(obem_ctx* c, const MultiParams& P, cudaStream_t st)
{
    const size_t dyn = (size_t)8 * KS * M_NP * M_THREADS * sizeof(double);
    cudaError_t e;
    if (P.eps2 != 0.f) {
        e = cudaFuncSetAttribute(panels_multi_kernel<KS, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn);
        if (e != cudaSuccess) return e;
        panels_multi_kernel<KS, true><<<c->sm_count, M_THREADS, dyn, st>>>(P);
    } else {
        e = cudaFuncSetAttribute(panels_multi_kernel<KS, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn);
        if (e != cudaSuccess) return e;
        panels_multi_kernel<KS, false><<<c->sm_count, M_THREADS, dyn, st>>>(P);
    }
    return cudaGetLastError();
}

} /* namespace */

void obem_multi_free(obem_ctx* c)
{
    if (c->d_munit) cudaFree(c->d_munit);
    if (c->d_msig) cudaFree(c->d_msig);
    if (c->d_ramo) cudaFree(c->d_ramo);
    c->d_ramo = nullptr;
    c->ramo_cap = 0;
    c->d_munit = nullptr;
    c->d_msig = nullptr;
    c->munit_cap = c->msig_cap = 0;
}

extern "C" int obem_eval_panels_multi(obem_ctx* c, const float* d_sigma, int n_sigma, const float* d_pts, int64_t m,
                                      float* d_out, void* cuda_stream)
{
    if (!c || n_sigma < 0 || m < 0) return OBEM_EINVAL;
    if (c->n_pan < 0) return OBEM_ESTATE;
    if (n_sigma == 0 || m == 0) return OBEM_OK;
    if (!d_pts || !d_out || !aligned16(d_pts) || !aligned16(d_out)) return OBEM_EINVAL;
    if (c->n_pan > 0 && (!d_sigma || !aligned4(d_sigma))) return OBEM_EINVAL;
    DeviceGuard g(c->device);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const long long np = c->n_pan;
    if (np == 0) {
        OBEM_CUDA(c, cudaMemsetAsync(d_out, 0, (size_t)n_sigma * (size_t)m * sizeof(float4), st));
        return OBEM_OK;
    }
    const long long nblk = ceil_div(np, PPB), np_pad = nblk * PPB;
    /* the unit-density encoding of the geometry: once per obem_set_panels */
    const size_t unit_need = (size_t)nblk * SBH_P;
    if (unit_need > c->munit_cap) {
        float4* p = nullptr;
        OBEM_CUDA(c, cudaMalloc(&p, unit_need * sizeof(float4)));
        if (c->d_munit) cudaFree(c->d_munit);
        c->d_munit = p;
        c->munit_cap = unit_need;
        c->munit_geom = -1;
    }
    if (c->munit_geom != c->geom_version) {
        multi_unit_kernel<<<(unsigned)ceil_div(np_pad, 128), 128, 0, st>>>(c->d_psrc, c->d_qrel, c->d_munit, np, np_pad);
        OBEM_CUDA(c, cudaGetLastError());
        c->launches += 1;
        c->munit_geom = c->geom_version;
    }
    const size_t sig_need = (size_t)nblk * M_KS * M_SROW;
    if (sig_need > c->msig_cap) {
        float* p = nullptr;
        OBEM_CUDA(c, cudaMalloc(&p, sig_need * sizeof(float)));
        if (c->d_msig) cudaFree(c->d_msig);
        c->d_msig = p;
        c->msig_cap = sig_need;
    }
    MultiParams P;
    P.unit = c->d_munit;
    P.sig = c->d_msig;
    P.qrel = c->d_qrel;
    P.sigma = d_sigma;
    P.np = np;
    P.nblk = nblk;
    P.tgt = (const float4*)d_pts;
    P.nt = m;
    P.ntiles = ceil_div(m, M_TT);
    P.out = (float4*)d_out;
    P.eps2 = c->eps_panel * c->eps_panel;
    for (int k0 = 0; k0 < n_sigma; k0 += M_KS) {
        const int ks = (n_sigma - k0 < M_KS) ? n_sigma - k0 : M_KS;
        P.k0 = k0;
        P.ks = ks;
        const long long cells = nblk * M_KS * M_SROW;
        multi_sigma_kernel<<<(unsigned)ceil_div(cells, 256), 256, 0, st>>>(d_sigma, c->d_msig, np, nblk, k0, ks);
        OBEM_CUDA(c, cudaGetLastError());
        cudaError_t e = cudaSuccess;
        switch (ks) {
        case 1: e = launch_pass<1>(c, P, st); break;
        case 2: e = launch_pass<2>(c, P, st); break;
        case 3: e = launch_pass<3>(c, P, st); break;
        default: e = launch_pass<4>(c, P, st); break;
        }
        OBEM_CUDA(c, e);
        c->launches += 2;
    }
    return OBEM_OK;
}

extern "C" int obem_ramo_current(obem_ctx* c, const float* d_xyzq, const float* d_vel, const float* d_ew, int n_electrodes,
                                 int64_t n, double* d_out, void* cuda_stream)
{
    if (!c || n_electrodes < 0 || n < 0) return OBEM_EINVAL;
    if (n_electrodes == 0) return OBEM_OK;
    if (!d_out || (((uintptr_t)d_out) & 7u)) return OBEM_EINVAL;
    if (n > 0 && (!d_xyzq || !d_vel || !d_ew || !aligned16(d_xyzq) || !aligned16(d_vel) || !aligned16(d_ew))) return OBEM_EINVAL;
    DeviceGuard g(c->device);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (n == 0) {
        OBEM_CUDA(c, cudaMemsetAsync(d_out, 0, (size_t)n_electrodes * 2 * sizeof(double), st));
        return OBEM_OK;
    }
    long long blocks = ceil_div(n, 4LL * R_THREADS);
    if (blocks > 1024) blocks = 1024;
    const long long chunk = ceil_div(ceil_div(n, blocks), R_THREADS) * R_THREADS;
    blocks = ceil_div(n, chunk);
    const size_t need = (size_t)n_electrodes * (size_t)blocks * 2;
    if (need > c->ramo_cap) {
        double* p = nullptr;
        OBEM_CUDA(c, cudaMalloc(&p, need * sizeof(double)));
        if (c->d_ramo) cudaFree(c->d_ramo);
        c->d_ramo = p;
        c->ramo_cap = need;
    }
    ramo_partial_kernel<<<dim3((unsigned)blocks, (unsigned)n_electrodes), R_THREADS, 0, st>>>(
        (const float4*)d_xyzq, (const float4*)d_vel, (const float4*)d_ew, n, chunk, c->d_ramo);
    OBEM_CUDA(c, cudaGetLastError());
    ramo_final_kernel<<<(unsigned)n_electrodes, R_THREADS, 0, st>>>(c->d_ramo, (int)blocks, n_electrodes, d_out);
    OBEM_CUDA(c, cudaGetLastError());
    c->launches += 2;
    return OBEM_OK;
}
