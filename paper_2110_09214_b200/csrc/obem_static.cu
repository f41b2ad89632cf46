/*
 * obem_static.cu -- ONE entry point that allocates nothing: obem_nbody_at_points_static.
 *
 * Why: every other evaluate call of libobem.so works on a context whose buffers (blocked sources, split-tile
 * workspace) come from cudaMalloc at obem_create / obem_set_*.  Some callers cannot call cudaMalloc at all: code under
 * CUDA graph capture, tight serving loops, harnesses that forbid it.  For them this file evaluates the N-body sum of
 * Eq (3.8) (softened, reading A2; no index exclusion, zero distance contributes 0, reading A4 --
 * what obem_eval_at_points(OBEM_NBODY) computes) straight from the caller's arrays, without a context.
 *
 * How: a variant of the evaluation kernel's split-source scheme.  The hot path splits the sources of a target tile
 * between CTAs and keeps the partial sums in a cudaMalloc'ed workspace (obem.cu, d_ws); here the partial sums live in
 * a file-scope `static __device__` array of FIXED size (g_static_scratch below: OBEM_STATIC_MAX_POINTS targets x
 * OBEM_STATIC_MAX_SPLITS source splits x 4 doubles = 8 MiB), which every GPU that loads the library holds until the
 * process exits.  Kernel 1 (nbody_static_kernel): CTA (tile, split) sums its share of the sources for 1024 targets
 * (256 threads x 2 packed f32x2 pairs; fp32 inside a block of 256 sources, fp64 across blocks, like the hot path) and
 * writes fp64 partials to the scratch.  Kernel 2 (nbody_static_reduce_kernel): sums the splits of every target in a
 * fixed order, multiplies by k_e, writes the result.  Deterministic; no atomics.
 *
 * The scratch is shared by ALL calls on a device and keeps the last call's contents.  Every slot kernel 2 reads was
 * written by kernel 1 of the SAME call (all splits of all targets, also for empty splits), so nothing has to start at
 * zero and nothing is cleared.  Two calls that overlap on the GPU (different streams, or graphs replayed concurrently)
 * race on the scratch: serialise them.
 *
 * In host code `g_static_scratch` is a host-side stand-in, not a device address; the device address is taken once per
 * device with cudaGetSymbolAddress (with that device current) and passed to the kernels.
 *
 * Part of libobem.so; shares nothing with oracle/.
 */
#include <mutex>

#include "obem_internal.cuh"

namespace {

constexpr int S_THREADS = 256;
constexpr int S_NP = 2;                          /* packed target pairs per thread              */
constexpr int S_TT = S_THREADS * 2 * S_NP;       /* targets per tile: 1024                      */
constexpr int S_SB = 256;                        /* sources per shared-memory block             */
constexpr int S_MAX_DEVICES = 64;
constexpr double S_KE = 1.0 / (4.0 * 3.14159265358979323846 * 8.8541878128e-12); /* reading A7 */

/* [split][target][Ex, Ey, Ez, phi] fp64 partial sums; target stride = the call's padded target count */
static __device__ __align__(256) double g_static_scratch[(size_t)OBEM_STATIC_MAX_POINTS * OBEM_STATIC_MAX_SPLITS * 4];

struct StaticSetup {
    bool ready = false;
    double* scratch = nullptr; /* device address of g_static_scratch on this device */
    int sm_count = 0;
};
StaticSetup g_setup[S_MAX_DEVICES];
std::mutex g_setup_mutex;

/* CTA (tile, split): targets [tile * S_TT, +S_TT), source blocks [split * bps, (split + 1) * bps) */
__global__ void __launch_bounds__(S_THREADS) nbody_static_kernel(const float4* __restrict__ chg, long long n,
                                                                 const float4* __restrict__ pts, long long m,
                                                                 long long m_pad, float eps2, int bps,
                                                                 double* __restrict__ scratch)
{
    __shared__ float4 sh[S_SB];
    const int tid = threadIdx.x;
    const long long tile = blockIdx.x, split = blockIdx.y;
    const long long nblk = (n + S_SB - 1) / S_SB;
    const long long b0 = split * bps, b1 = (b0 + bps < nblk) ? b0 + bps : nblk;
    const long long tbase = tile * (long long)S_TT + tid;

    u64 X[S_NP], Y[S_NP], Z[S_NP];
#pragma unroll
    for (int p = 0; p < S_NP; ++p) {
        const long long i0 = tbase + (2 * p) * S_THREADS, i1 = i0 + S_THREADS;
        const float4 a = (i0 < m) ? pts[i0] : make_float4(0.f, 0.f, 0.f, 0.f);
        const float4 b = (i1 < m) ? pts[i1] : make_float4(0.f, 0.f, 0.f, 0.f);
        X[p] = pk(a.x, b.x);
        Y[p] = pk(a.y, b.y);
        Z[p] = pk(a.z, b.z);
    }
    double R[S_NP][2][4];
#pragma unroll
    for (int p = 0; p < S_NP; ++p)
#pragma unroll
        for (int h = 0; h < 2; ++h) R[p][h][0] = R[p][h][1] = R[p][h][2] = R[p][h][3] = 0.0;
    const u64 e2 = pk(eps2, eps2);

    for (long long b = b0; b < b1; ++b) {
        __syncthreads(); /* everyone is done with the previous block */
        const long long j = b * S_SB + tid;
        /* padding: weight 0, parked far away (never at zero distance from a target) */
        sh[tid] = (j < n) ? chg[j] : make_float4(1.0e15f, 1.0e15f, 1.0e15f, 0.f);
        __syncthreads();
        u64 aX[S_NP], aY[S_NP], aZ[S_NP], aP[S_NP];
#pragma unroll
        for (int p = 0; p < S_NP; ++p) aX[p] = aY[p] = aZ[p] = aP[p] = 0ull;
#pragma unroll 4
        for (int k = 0; k < S_SB; ++k) {
            const float4 q = sh[k]; /* warp-uniform address: broadcast */
            const u64 w = pk(q.w, q.w);
#pragma unroll
            for (int p = 0; p < S_NP; ++p) {
                const u64 dx = sub2(X[p], pk(q.x, q.x));
                const u64 dy = sub2(Y[p], pk(q.y, q.y));
                const u64 dz = sub2(Z[p], pk(q.z, q.z));
                u64 r2 = fma2(dx, dx, e2);
                r2 = fma2(dy, dy, r2);
                r2 = fma2(dz, dz, r2);
                float r2l, r2h;
                upk(r2, r2l, r2h);
                /* reading A4: a source at zero (softened) distance contributes 0 */
                const float ul = (r2l > 0.f) ? rsqrt_approx(r2l) : 0.f;
                const float uh = (r2h > 0.f) ? rsqrt_approx(r2h) : 0.f;
                const u64 u = pk(ul, uh);
                const u64 t = mul2(u, w);
                aP[p] = add2(aP[p], t);
                const u64 sE = mul2(t, mul2(u, u));
                aX[p] = fma2(sE, dx, aX[p]);
                aY[p] = fma2(sE, dy, aY[p]);
                aZ[p] = fma2(sE, dz, aZ[p]);
            }
        }
        /* second accumulation level: fp64 across the blocks */
#pragma unroll
        for (int p = 0; p < S_NP; ++p) {
            float l, h;
            upk(aX[p], l, h);
            R[p][0][0] += (double)l, R[p][1][0] += (double)h;
            upk(aY[p], l, h);
            R[p][0][1] += (double)l, R[p][1][1] += (double)h;
            upk(aZ[p], l, h);
            R[p][0][2] += (double)l, R[p][1][2] += (double)h;
            upk(aP[p], l, h);
            R[p][0][3] += (double)l, R[p][1][3] += (double)h;
        }
    }
    /* every (split, target < m_pad) slot is written, also by a split with no block: the reducer reads them all */
#pragma unroll
    for (int p = 0; p < S_NP; ++p)
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const long long i = tbase + (long long)(2 * p + h) * S_THREADS;
            double2* dst = reinterpret_cast<double2*>(scratch + ((size_t)split * (size_t)m_pad + (size_t)i) * 4);
            dst[0] = make_double2(R[p][h][0], R[p][h][1]);
            dst[1] = make_double2(R[p][h][2], R[p][h][3]);
        }
}

/* one thread per target: the splits in ascending order (fixed), times k_e */
__global__ void __launch_bounds__(256) nbody_static_reduce_kernel(const double* __restrict__ scratch, long long m,
                                                                  long long m_pad, int splits, float4* __restrict__ out)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= m) return;
    double ex = 0.0, ey = 0.0, ez = 0.0, ph = 0.0;
    for (int s = 0; s < splits; ++s) {
        const double2* src = reinterpret_cast<const double2*>(scratch + ((size_t)s * (size_t)m_pad + (size_t)i) * 4);
        const double2 a = src[0], b = src[1];
        ex += a.x, ey += a.y, ez += b.x, ph += b.y;
    }
    out[i] = make_float4((float)(S_KE * ex), (float)(S_KE * ey), (float)(S_KE * ez), (float)(S_KE * ph));
}

/* once per device, with that device current: the device address of the scratch and the SM count */
int static_setup(int dev, StaticSetup& out)
{
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    StaticSetup& s = g_setup[dev];
    if (!s.ready) {
        void* ptr = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&ptr, g_static_scratch);
        int sms = 0;
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess || !ptr || sms < 1) {
            cudaGetLastError();
            return OBEM_ECUDA;
        }
        s.scratch = (double*)ptr;
        s.sm_count = sms;
        s.ready = true;
    }
    out = s;
    return OBEM_OK;
}

} /* namespace */

extern "C" int obem_nbody_at_points_static(const float* d_xyzq, int64_t n, const float* d_pts, int64_t m, float eps_pp_m,
                                           float* d_out, void* cuda_stream)
{
    if (n < 0 || m < 0 || !(eps_pp_m >= 0.f) || isinf(eps_pp_m)) return OBEM_EINVAL;
    if (m > OBEM_STATIC_MAX_POINTS) return OBEM_ELIMIT;
    if (m == 0) return OBEM_OK;
    if (!d_pts || !d_out || !aligned16(d_pts) || !aligned16(d_out)) return OBEM_EINVAL;
    if (n > 0 && (!d_xyzq || !aligned16(d_xyzq))) return OBEM_EINVAL;
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= S_MAX_DEVICES) {
        cudaGetLastError();
        return OBEM_ECUDA;
    }
    StaticSetup su;
    const int rc = static_setup(dev, su);
    if (rc != OBEM_OK) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;

    const long long tiles = (m + S_TT - 1) / S_TT, m_pad = tiles * S_TT;
    const long long nblk = (n + S_SB - 1) / S_SB;
    /* enough CTAs for two per SM, no empty split, at most OBEM_STATIC_MAX_SPLITS */
    long long splits = (2LL * su.sm_count + tiles - 1) / tiles;
    if (splits > OBEM_STATIC_MAX_SPLITS) splits = OBEM_STATIC_MAX_SPLITS;
    if (splits > nblk) splits = nblk;
    if (splits < 1) splits = 1;
    const long long bps = (nblk + splits - 1) / splits > 0 ? (nblk + splits - 1) / splits : 1;
    splits = nblk > 0 ? (nblk + bps - 1) / bps : 1;
    if (bps > 0x7fffffffLL) return OBEM_EINVAL;

    nbody_static_kernel<<<dim3((unsigned)tiles, (unsigned)splits), S_THREADS, 0, st>>>(
        (const float4*)d_xyzq, n, (const float4*)d_pts, m, m_pad, eps_pp_m * eps_pp_m, (int)bps, su.scratch);
    if (cudaGetLastError() != cudaSuccess) return OBEM_ECUDA;
    nbody_static_reduce_kernel<<<(unsigned)((m + 255) / 256), 256, 0, st>>>(su.scratch, m, m_pad, (int)splits,
                                                                          (float4*)d_out);
    if (cudaGetLastError() != cudaSuccess) return OBEM_ECUDA;
    return OBEM_OK;
}
