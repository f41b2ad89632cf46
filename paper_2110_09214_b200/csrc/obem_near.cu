/*
 * obem_near.cu -- near-field-accurate panels (the cell
 * integrals of Eq (2.13)/(2.14) "are calculated analytically").
 *
 * The hot path sums 7 quadrature sources per panel; that is the exact integral to ~(h/r)^6.  For the few panels
 * within near_factor * h_p of a target this file replaces the 7-point value by the closed-form integral over the
 * flat triangle, as a correction added after the evaluation kernel:
 *
 *     out[t] += k_e sum_{p near t} sigma_p ( I_exact(p, t) - A_p sum_k w_k K(t - x_pk) )
 *
 * Closed form (uniformly charged planar polygon, edge by edge): with n the unit normal, d = n.(r - v0) the signed
 * height, rho the foot of r on the plane and, per edge a -> b: l the unit tangent, u = l x n the outward in-plane
 * normal, P0 = (a - rho).u, l- = (a - rho).l, l+ = (b - rho).l, R0^2 = P0^2 + d^2, R-+ = |r - a|, |r - b|,
 *     f = ln((R+ + l+)/(R- + l-)),   beta = atan(P0 l+/(R0^2 + |d| R+)) - atan(P0 l-/(R0^2 + |d| R-)),
 *     Int dS/R = sum (P0 f - |d| beta),      Int (r - r')/R^3 dS = sum u f + n sgn(d) sum beta.
 * All of it in fp64 from the fp32 vertices: the terms cancel strongly between edges once r is a few h away.
 *
 * Finding the near pairs: a uniform grid of cubic cells over the panels' near spheres (centre = centroid, radius
 * R_p = near_factor * longest edge); every cell lists, in ascending order, the panels whose sphere overlaps it.
 * Built once per geometry (count -> exclusive scan -> fill -> per-cell sort); a target looks at its own cell only.
 *
 * Part of libobem.so; shares nothing with oracle/.
 */
#include <cub/device/device_scan.cuh>

#include "obem_internal.cuh"

namespace {

constexpr double KE_NEAR = 1.0 / (4.0 * 3.14159265358979323846 * 8.8541878128e-12);
constexpr long long MAX_CELLS = 1LL << 24;

struct NearGrid {
    double lo[3];
    double s, inv_s;
    int n[3];
};

/* centroid and near radius of every panel */
__global__ void near_prep_kernel(const float* __restrict__ verts, float4* __restrict__ pcr, long long np, float factor)
{
    const long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= np) return;
    double v[3][3];
#pragma unroll
    for (int j = 0; j < 3; ++j)
#pragma unroll
        for (int k = 0; k < 3; ++k) v[j][k] = (double)verts[(p * 3 + j) * 3 + k];
    double h2 = 0.0;
#pragma unroll
    for (int j = 0; j < 3; ++j) {
        const int j1 = (j + 1) % 3;
        const double ex = v[j1][0] - v[j][0], ey = v[j1][1] - v[j][1], ez = v[j1][2] - v[j][2];
        h2 = fmax(h2, ex * ex + ey * ey + ez * ez);
    }
    const double ax = v[1][0] - v[0][0], ay = v[1][1] - v[0][1], az = v[1][2] - v[0][2];
    const double bx = v[2][0] - v[0][0], by = v[2][1] - v[0][1], bz = v[2][2] - v[0][2];
    const double cx = ay * bz - az * by, cy = az * bx - ax * bz, cz = ax * by - ay * bx;
    const bool flat = (cx * cx + cy * cy + cz * cz) > 0.0; /* a degenerate panel contributes 0 either way */
    float4 o;
    o.x = (float)((v[0][0] + v[1][0] + v[2][0]) / 3.0);
    o.y = (float)((v[0][1] + v[1][1] + v[2][1]) / 3.0);
    o.z = (float)((v[0][2] + v[1][2] + v[2][2]) / 3.0);
    const double R = (double)factor * sqrt(h2);
    o.w = (flat && isfinite(R)) ? (float)R : 0.f;
    pcr[p] = o;
}

/* one block: bounding box of the near spheres, sum and count of the positive radii -> red[0..7] */
__global__ void __launch_bounds__(1024) near_reduce_kernel(const float4* __restrict__ pcr, long long np,
                                                           double* __restrict__ red)
{
    __shared__ double sh[8][32];
    double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300}, sum = 0.0, cnt = 0.0;
    for (long long p = threadIdx.x; p < np; p += blockDim.x) {
        const float4 c = pcr[p];
        if (!(c.w > 0.f)) continue;
        const double R = c.w, q[3] = {c.x, c.y, c.z};
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            lo[a] = fmin(lo[a], q[a] - R);
            hi[a] = fmax(hi[a], q[a] + R);
        }
        sum += R;
        cnt += 1.0;
    }
    double v[8] = {lo[0], lo[1], lo[2], hi[0], hi[1], hi[2], sum, cnt};
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        for (int o = 16; o > 0; o >>= 1) {
            const double x = __shfl_xor_sync(0xffffffffu, v[k], o);
            v[k] = (k < 3) ? fmin(v[k], x) : ((k < 6) ? fmax(v[k], x) : v[k] + x);
        }
        if (lane == 0) sh[k][w] = v[k];
    }
    __syncthreads();
    if (w == 0) {
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            double x = sh[k][lane];
            for (int o = 16; o > 0; o >>= 1) {
                const double y = __shfl_xor_sync(0xffffffffu, x, o);
                x = (k < 3) ? fmin(x, y) : ((k < 6) ? fmax(x, y) : x + y);
            }
            if (lane == 0) red[k] = x;
        }
    }
}

/* cells [c0, c1] per axis that the (slightly inflated) sphere's bounding cube touches */
__device__ __forceinline__ void sphere_cells(const NearGrid& g, const float4 c, double& R, int (&c0)[3], int (&c1)[3])
{
    R = (double)c.w * (1.0 + 1e-6) + g.s * 1e-6; /* margin: the target's cell index is a rounded quotient */
    const double q[3] = {c.x, c.y, c.z};
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        int i0 = (int)floor((q[a] - R - g.lo[a]) * g.inv_s), i1 = (int)floor((q[a] + R - g.lo[a]) * g.inv_s);
        c0[a] = i0 < 0 ? 0 : i0;
        c1[a] = i1 > g.n[a] - 1 ? g.n[a] - 1 : i1;
    }
}
/* squared distance from the point q to the cell (ix, iy, iz) (an axis-aligned cube) */
__device__ __forceinline__ double cell_dist2(const NearGrid& g, const double (&q)[3], int ix, int iy, int iz)
{
    const int id[3] = {ix, iy, iz};
    double d2 = 0.0;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const double lo = g.lo[a] + id[a] * g.s, hi = lo + g.s;
        const double d = q[a] < lo ? lo - q[a] : (q[a] > hi ? q[a] - hi : 0.0);
        d2 += d * d;
    }
    return d2;
}

/* FILL = false: count the panels per cell;  FILL = true: write them (order fixed afterwards by near_sort_kernel) */
template <bool FILL>
__global__ void near_bin_kernel(NearGrid g, const float4* __restrict__ pcr, long long np, int* __restrict__ counts,
                                const int* __restrict__ start, int* __restrict__ list)
{
    const long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= np) return;
    const float4 c = pcr[p];
    if (!(c.w > 0.f)) return;
    double R;
    int c0[3], c1[3];
    sphere_cells(g, c, R, c0, c1);
    const double q[3] = {c.x, c.y, c.z};
    for (int ix = c0[0]; ix <= c1[0]; ++ix)
        for (int iy = c0[1]; iy <= c1[1]; ++iy)
            for (int iz = c0[2]; iz <= c1[2]; ++iz) {
                if (cell_dist2(g, q, ix, iy, iz) > R * R) continue;
                const long long cell = ((long long)ix * g.n[1] + iy) * g.n[2] + iz;
                const int k = atomicAdd(&counts[cell], 1);
                if (FILL) list[start[cell] + k] = (int)p;
            }
}

/* ascending panel index inside every cell: the correction is then summed in an order that does not depend on
 * how the atomics of the fill pass were scheduled */
__global__ void near_sort_kernel(const int* __restrict__ start, int* __restrict__ list, long long ncells)
{
    const long long cell = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (cell >= ncells) return;
    const int a = start[cell], b = start[cell + 1];
    for (int i = a + 1; i < b; ++i) {
        const int v = list[i];
        int j = i - 1;
        while (j >= a && list[j] > v) {
            list[j + 1] = list[j];
            --j;
        }
        list[j + 1] = v;
    }
}

} /* namespace */

namespace {

/* Int dS/R and Int (r - r')/R^3 dS over the flat triangle v[0..2] at r (header comment).  Zero-area: 0. */
__device__ void tri_exact(const double (&v)[3][3], const double (&r)[3], double& I_phi, double (&I_E)[3])
{
    I_phi = 0.0;
    I_E[0] = I_E[1] = I_E[2] = 0.0;
    const double e1x = v[1][0] - v[0][0], e1y = v[1][1] - v[0][1], e1z = v[1][2] - v[0][2];
    const double e2x = v[2][0] - v[0][0], e2y = v[2][1] - v[0][1], e2z = v[2][2] - v[0][2];
    double nx = e1y * e2z - e1z * e2y, ny = e1z * e2x - e1x * e2z, nz = e1x * e2y - e1y * e2x;
    const double nn = sqrt(nx * nx + ny * ny + nz * nz);
    if (!(nn > 0.0)) return;
    nx /= nn, ny /= nn, nz /= nn;
    const double d = nx * (r[0] - v[0][0]) + ny * (r[1] - v[0][1]) + nz * (r[2] - v[0][2]);
    const double ad = fabs(d);
    double sb = 0.0;
    /* NOT unrolled, and one log call site: the fp64 log / atan routines are inlined wherever they are called, and
     * with three copies of the edge body the correction kernel spent most of its issue slots waiting for instructions
     * (ncu: stall "no instruction" 15.9 per issue) */
#pragma unroll 1
    for (int i = 0; i < 3; ++i) {
        const int i1 = (i == 2) ? 0 : i + 1;
        /* vectors from r to the two ends of the edge; their in-plane parts are (a - rho), (b - rho) */
        const double ax = v[i][0] - r[0], ay = v[i][1] - r[1], az = v[i][2] - r[2];
        const double bx = v[i1][0] - r[0], by = v[i1][1] - r[1], bz = v[i1][2] - r[2];
        double lx = bx - ax, ly = by - ay, lz = bz - az;
        const double len = sqrt(lx * lx + ly * ly + lz * lz);
        if (!(len > 0.0)) continue;
        lx /= len, ly /= len, lz /= len;
        const double ux = ly * nz - lz * ny, uy = lz * nx - lx * nz, uz = lx * ny - ly * nx;
        /* u and l are orthogonal to n, so the normal part of (a - r) drops out of these dot products */
        const double P0 = ax * ux + ay * uy + az * uz;
        const double lm = ax * lx + ay * ly + az * lz, lp = bx * lx + by * ly + bz * lz;
        const double Rm = sqrt(ax * ax + ay * ay + az * az), Rp = sqrt(bx * bx + by * by + bz * bz);
        const double R02 = P0 * P0 + d * d;
        double num, den; /* the same three forms as before, the operands selected first */
        if (lm >= 0.0) {
            num = Rp + lp, den = Rm + lm;
        } else if (lp <= 0.0) {
            num = Rm - lm, den = Rp - lp;
        } else {
            num = (Rp + lp) * (Rm - lm), den = R02;
        }
        if (!(den > 0.0)) continue;
        const double f = log(num / den);
        double beta = 0.0;
        if (P0 != 0.0) beta = atan(P0 * lp / (R02 + ad * Rp)) - atan(P0 * lm / (R02 + ad * Rm));
        I_phi += P0 * f - ad * beta;
        sb += beta;
        I_E[0] += ux * f;
        I_E[1] += uy * f;
        I_E[2] += uz * f;
    }
    const double sg = d > 0.0 ? 1.0 : (d < 0.0 ? -1.0 : 0.0);
    I_E[0] += nx * sg * sb;
    I_E[1] += ny * sg * sb;
    I_E[2] += nz * sg * sb;
}

struct NearParams {
    NearGrid g;
    const int* start;
    const int* list;
    const float4* pcr;
    const float4* porg;
    const float4* qrel;
    const float* verts;
    const float* sigma;
    const float4* tgt;
    float4* out;
    long long nt;
    double eps2;  /* softening of the 7-point panel sum (what the evaluation kernel used) */
    double crit2; /* (VERY_NEAR / near_factor)^2: a source closer than VERY_NEAR * h_p sends the target to the redo list */
    int* redo_list;
    unsigned* redo_count;
};

/* sigma_p (exact - 7-point) of panel p at target t, added to acc = (Ex, Ey, Ez, phi) in units of 1/k_e */
__device__ __forceinline__ bool near_pair(const NearParams& P, int p, const float4 t, double (&acc)[4])
{
    double v[3][3];
#pragma unroll
    for (int j = 0; j < 3; ++j)
#pragma unroll
        for (int k = 0; k < 3; ++k) v[j][k] = (double)__ldg(P.verts + ((long long)p * 3 + j) * 3 + k);
    const double r[3] = {(double)t.x, (double)t.y, (double)t.z};
    double Iphi, IE[3];
    tri_exact(v, r, Iphi, IE);
    /* the 7-point value as the evaluation kernel formed it: target shifted into the panel's frame in fp32 */
    const float4 o = __ldg(P.porg + p);
    const double TX = (double)__fsub_rn(t.x, o.x), TY = (double)__fsub_rn(t.y, o.y), TZ = (double)__fsub_rn(t.z, o.z);
    double r2min = 1e300;
#pragma unroll 1
    for (int k = 0; k < 7; ++k) {
        const float4 q = __ldg(P.qrel + (long long)p * 7 + k);
        const double dx = TX - (double)q.x, dy = TY - (double)q.y, dz = TZ - (double)q.z;
        const double g2 = dx * dx + dy * dy + dz * dz;
        r2min = fmin(r2min, g2);
        const double r2 = g2 + P.eps2;
        if (!(r2 > 0.0)) continue;
        const double u = 1.0 / sqrt(r2), wu = (double)q.w * u, s3 = wu * u * u;
        Iphi -= wu;
        IE[0] -= s3 * dx;
        IE[1] -= s3 * dy;
        IE[2] -= s3 * dz;
    }
    const double s = (double)__ldg(P.sigma + p);
    acc[0] += s * IE[0];
    acc[1] += s * IE[1];
    acc[2] += s * IE[2];
    acc[3] += s * Iphi;
    const double R = (double)__ldg(&P.pcr[p].w);
    return r2min < P.crit2 * R * R;
}

#ifndef OBEM_NEAR_WARPS
#define OBEM_NEAR_WARPS 2
#endif
#ifndef OBEM_NEAR_MINB
#define OBEM_NEAR_MINB 24
#endif
constexpr int NEAR_WARPS = OBEM_NEAR_WARPS; /* small CTAs: most warps leave at once (no near panel): 14.5 -> 12.3 ms on config 3 against 8 warps */
/* A target closer than VERY_NEAR * h_p to a quadrature source of panel p: that one 7-point term exceeds the whole
 * local field by more than 0.013 / VERY_NEAR^2 (= 13 at 1/32), and what it cost the fp32 accumulation of the
 * evaluation kernel (an ulp of ITS size) cannot be corrected afterwards.  Such targets are recomputed from scratch
 * in fp64 by near_redo_kernel. */
constexpr double VERY_NEAR = 1.0 / 32.0;

/* cell of a target, -1 if it lies outside the grid (no near panel can exist; also NaN) */
__device__ __forceinline__ long long near_cell_of(const NearGrid& g, const float4 t)
{
    const double tq[3] = {(double)t.x, (double)t.y, (double)t.z};
    int ci[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const double u = floor((tq[a] - g.lo[a]) * g.inv_s);
        if (!(u >= 0.0 && u < (double)g.n[a])) return -1;
        ci[a] = (int)u;
    }
    return ((long long)ci[0] * g.n[1] + ci[1]) * g.n[2] + ci[2];
}
/* cell of every target (-1: none, or an empty cell) and the number of targets per cell */
__global__ void __launch_bounds__(256) near_tcount_kernel(const NearParams P, int* __restrict__ tcell, int* __restrict__ tcount)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P.nt) return;
    long long cell = near_cell_of(P.g, P.tgt[i]);
    if (cell >= 0 && P.start[cell] == P.start[cell + 1]) cell = -1;
    tcell[i] = (int)cell;
    if (cell >= 0) atomicAdd(tcount + cell, 1);
}
/* the targets grouped by cell (any order inside a cell: it enters no result) */
__global__ void __launch_bounds__(256) near_tfill_kernel(const int* __restrict__ tcell, const int* __restrict__ tstart,
                                                        int* __restrict__ cursor, int* __restrict__ tlist, long long nt)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nt) return;
    const int cell = tcell[i];
    if (cell >= 0) tlist[tstart[cell] + atomicAdd(cursor + cell, 1)] = (int)i;
}

/* one warp per target: the lanes test 32 candidates of the target's cell at a time; the near ones are compacted
 * into a per-warp queue so that the expensive closed form always runs on full warps */
/* Round 1: latency-bound (dependent fp64 log / atan chains, per-pair loads): more resident warps beat fewer spills --
 * A/B on config 3 with the register cap of 2..32 CTAs/SM: 12.4 (108 registers), 11.0 (96), 10.1 (72), 8.8 (48), 8.1 (40),
 * 8.6 (32) ms.  Round 2 (config 3): 8.05 ms -> 5.4 with the targets in cell order (panel records hit L1) -> 3.45 with the
 * edge loop of tri_exact rolled and one log call site -> 3.03 with the 7-point loop rolled too (the kernel was waiting
 * for INSTRUCTIONS: 14,000 SASS lines of inlined fp64 log / atan / sqrt copies; now 5,000); warps per CTA and the
 * register cap no longer matter (3.0 .. 3.3 ms over 1..8 warps, 4..32 CTAs/SM). */
/* Round 2: the warps take the targets in CELL order (order[], from near_tcount / near_tfill below), not in the
 * caller's order: the warps that are resident together then walk the same cell's panel list and read the same panel
 * records, so those loads hit L1 instead of going to L2 one by one; and the targets that have no cell (3 of 4 in
 * config 3) never get a warp.  Which warp handles a target enters no result: each target still sums its own panels
 * in ascending order, alone. */
__global__ void __launch_bounds__(NEAR_WARPS * 32, OBEM_NEAR_MINB) near_correct_kernel(const NearParams P, const int* __restrict__ order,
                                                                          const int* __restrict__ n_order)
{
    __shared__ int queue[NEAR_WARPS][64];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const long long slot = (long long)blockIdx.x * NEAR_WARPS + w;
    if (slot >= (long long)*n_order) return;
    const long long t_idx = order[slot];
    const float4 t = P.tgt[t_idx];
    int ci[3];
    const double tq[3] = {(double)t.x, (double)t.y, (double)t.z};
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const double u = floor((tq[a] - P.g.lo[a]) * P.g.inv_s);
        if (!(u >= 0.0 && u < (double)P.g.n[a])) return; /* outside every near sphere (also NaN) */
        ci[a] = (int)u;
    }
    const long long cell = ((long long)ci[0] * P.g.n[1] + ci[1]) * P.g.n[2] + ci[2];
    const int beg = P.start[cell], end = P.start[cell + 1];
    if (beg == end) return;
    double acc[4] = {0.0, 0.0, 0.0, 0.0};
    int qn = 0;
    int* q = queue[w];
    bool redo = false;
    for (int base = beg; base < end; base += 32) {
        const int k = base + lane;
        int p = -1;
        bool near = false;
        if (k < end) {
            p = P.list[k];
            const float4 c = __ldg(P.pcr + p);
            const double dx = tq[0] - (double)c.x, dy = tq[1] - (double)c.y, dz = tq[2] - (double)c.z;
            near = dx * dx + dy * dy + dz * dz < (double)c.w * (double)c.w;
        }
        const unsigned m = __ballot_sync(0xffffffffu, near);
        if (near) q[qn + __popc(m & ((1u << lane) - 1u))] = p;
        qn += __popc(m);
        __syncwarp();
        if (qn >= 32) {
            redo |= near_pair(P, q[lane], t, acc);
            __syncwarp();
            const int rest = qn - 32;
            const int moved = (lane < rest) ? q[32 + lane] : 0;
            __syncwarp();
            if (lane < rest) q[lane] = moved;
            qn = rest;
            __syncwarp();
        }
    }
    if (lane < qn) redo |= near_pair(P, q[lane], t, acc);
    if (__any_sync(0xffffffffu, redo)) { /* near_redo_kernel overwrites out[t_idx] */
        if (lane == 0) P.redo_list[atomicAdd(P.redo_count, 1u)] = (int)t_idx;
        return;
    }
#pragma unroll
    for (int k = 0; k < 4; ++k)
        for (int o = 16; o > 0; o >>= 1) acc[k] += __shfl_xor_sync(0xffffffffu, acc[k], o);
    if (lane == 0) {
        float4 h = P.out[t_idx];
        h.x = (float)((double)h.x + KE_NEAR * acc[0]);
        h.y = (float)((double)h.y + KE_NEAR * acc[1]);
        h.z = (float)((double)h.z + KE_NEAR * acc[2]);
        h.w = (float)((double)h.w + KE_NEAR * acc[3]);
        P.out[t_idx] = h;
    }
}

/* Targets of the redo list: the whole panel sum again, in fp64, one CTA per target -- the closed form for the
 * near panels, the 7-point rule (fp64 differences, so no frame is needed) for all others.  Overwrites out[t]. */
__global__ void __launch_bounds__(256) near_redo_kernel(const NearParams P, long long np)
{
    __shared__ double red[4][256];
    const unsigned n = *P.redo_count;
    const int tid = threadIdx.x;
    for (unsigned r = blockIdx.x; r < n; r += gridDim.x) {
        const int ti = P.redo_list[r];
        const float4 t = P.tgt[ti];
        const double tq[3] = {(double)t.x, (double)t.y, (double)t.z};
        double acc[4] = {0.0, 0.0, 0.0, 0.0};
        for (long long p = tid; p < np; p += 256) {
            const float4 c = __ldg(P.pcr + p);
            if (!(c.w > 0.f)) continue; /* zero-area panel: all its weights are 0 */
            const double cx = tq[0] - (double)c.x, cy = tq[1] - (double)c.y, cz = tq[2] - (double)c.z;
            const double s = (double)__ldg(P.sigma + p);
            if (cx * cx + cy * cy + cz * cz < (double)c.w * (double)c.w) {
                double v[3][3], Iphi, IE[3];
#pragma unroll
                for (int j = 0; j < 3; ++j)
#pragma unroll
                    for (int k = 0; k < 3; ++k) v[j][k] = (double)__ldg(P.verts + (p * 3 + j) * 3 + k);
                tri_exact(v, tq, Iphi, IE);
                acc[0] += s * IE[0], acc[1] += s * IE[1], acc[2] += s * IE[2], acc[3] += s * Iphi;
            } else {
                const float4 o = __ldg(P.porg + p);
                const double TX = tq[0] - (double)o.x, TY = tq[1] - (double)o.y, TZ = tq[2] - (double)o.z;
#pragma unroll
                for (int k = 0; k < 7; ++k) {
                    const float4 q = __ldg(P.qrel + p * 7 + k);
                    const double dx = TX - (double)q.x, dy = TY - (double)q.y, dz = TZ - (double)q.z;
                    const double r2 = dx * dx + dy * dy + dz * dz + P.eps2;
                    if (!(r2 > 0.0)) continue;
                    const double u = 1.0 / sqrt(r2), wu = s * (double)q.w * u, s3 = wu * u * u;
                    acc[0] += s3 * dx, acc[1] += s3 * dy, acc[2] += s3 * dz, acc[3] += wu;
                }
            }
        }
#pragma unroll
        for (int k = 0; k < 4; ++k) red[k][tid] = acc[k];
        __syncthreads();
        for (int h = 128; h > 0; h >>= 1) {
            if (tid < h)
#pragma unroll
                for (int k = 0; k < 4; ++k) red[k][tid] += red[k][tid + h];
            __syncthreads();
        }
        if (tid == 0)
            P.out[ti] = make_float4((float)(KE_NEAR * red[0][0]), (float)(KE_NEAR * red[1][0]),
                                    (float)(KE_NEAR * red[2][0]), (float)(KE_NEAR * red[3][0]));
        __syncthreads();
    }
}

__global__ void near_combine_kernel(float4* __restrict__ out, const float4* __restrict__ pan, long long nt)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nt) return;
    const float4 a = out[i], b = pan[i];
    out[i] = make_float4(a.x + b.x, a.y + b.y, a.z + b.z, a.w + b.w);
}

} /* namespace */

namespace {

int near_grow_panels(obem_ctx* c, long long np)
{
    const long long need = np > 0 ? np : 1;
    if (need <= c->near_cap) return OBEM_OK;
    float *v = nullptr, *s = nullptr;
    float4 *o = nullptr, *r = nullptr;
    cudaError_t e = cudaMalloc(&v, (size_t)need * 9 * sizeof(float));
    if (e == cudaSuccess) e = cudaMalloc(&s, (size_t)need * sizeof(float));
    if (e == cudaSuccess) e = cudaMalloc(&o, (size_t)need * sizeof(float4));
    if (e == cudaSuccess) e = cudaMalloc(&r, (size_t)need * sizeof(float4));
    if (e != cudaSuccess) {
        if (v) cudaFree(v);
        if (s) cudaFree(s);
        if (o) cudaFree(o);
        if (r) cudaFree(r);
        return cuda_fail(c, e);
    }
    if (c->d_pverts) cudaFree(c->d_pverts);
    if (c->d_psigma) cudaFree(c->d_psigma);
    if (c->d_porg) cudaFree(c->d_porg);
    if (c->d_pcr) cudaFree(c->d_pcr);
    c->d_pverts = v, c->d_psigma = s, c->d_porg = o, c->d_pcr = r;
    c->near_cap = need;
    return OBEM_OK;
}

/* (Re)build the cell lists for the current panels and near_factor.  Allocates and synchronises `st`. */
int near_build(obem_ctx* c, cudaStream_t st)
{
    const long long np = c->n_pan;
    c->near_n[0] = c->near_n[1] = c->near_n[2] = 0;
    int rc = obem_panel_origins(c, c->d_porg, st);
    if (rc != OBEM_OK) return rc;
    near_prep_kernel<<<(unsigned)ceil_div(np, 256), 256, 0, st>>>(c->d_pverts, c->d_pcr, np, c->near_factor);
    OBEM_CUDA(c, cudaGetLastError());
    if (!c->d_near_red) OBEM_CUDA(c, cudaMalloc(&c->d_near_red, 8 * sizeof(double)));
    near_reduce_kernel<<<1, 1024, 0, st>>>(c->d_pcr, np, c->d_near_red);
    OBEM_CUDA(c, cudaGetLastError());
    c->launches += 2;
    double red[8];
    OBEM_CUDA(c, cudaMemcpyAsync(red, c->d_near_red, sizeof(red), cudaMemcpyDeviceToHost, st));
    OBEM_CUDA(c, cudaStreamSynchronize(st));
    if (!(red[7] >= 1.0)) { /* no panel with a positive near radius: nothing is ever near */
        c->near_valid = 1;
        return OBEM_OK;
    }
    NearGrid g;
    double s = red[6] / red[7]; /* mean near radius */
    long long n[3];
    for (;;) {
        long long cells = 1;
        for (int a = 0; a < 3; ++a) {
            n[a] = (long long)floor((red[3 + a] - red[a]) / s) + 1;
            cells *= n[a];
        }
        if (cells <= MAX_CELLS) break;
        s *= 1.25992104989487; /* 2^(1/3): halves the cell count */
    }
    for (int a = 0; a < 3; ++a) g.lo[a] = red[a], g.n[a] = (int)n[a];
    g.s = s, g.inv_s = 1.0 / s;
    const long long ncells = n[0] * n[1] * n[2];
    if (ncells + 1 > c->cell_cap) {
        if (c->d_cell_start) cudaFree(c->d_cell_start);
        if (c->d_cell_fill) cudaFree(c->d_cell_fill);
        c->d_cell_start = c->d_cell_fill = nullptr, c->cell_cap = 0;
        OBEM_CUDA(c, cudaMalloc(&c->d_cell_start, (size_t)(ncells + 1) * sizeof(int)));
        OBEM_CUDA(c, cudaMalloc(&c->d_cell_fill, (size_t)(ncells + 1) * sizeof(int)));
        c->cell_cap = ncells + 1;
    }
    /* count (the extra last element stays 0 so that the exclusive scan's last output is the total) */
    OBEM_CUDA(c, cudaMemsetAsync(c->d_cell_fill, 0, (size_t)(ncells + 1) * sizeof(int), st));
    near_bin_kernel<false><<<(unsigned)ceil_div(np, 128), 128, 0, st>>>(g, c->d_pcr, np, c->d_cell_fill, nullptr, nullptr);
    OBEM_CUDA(c, cudaGetLastError());
    size_t tmp = 0;
    OBEM_CUDA(c, cub::DeviceScan::ExclusiveSum(nullptr, tmp, c->d_cell_fill, c->d_cell_start, (int)(ncells + 1), st));
    if (tmp > c->scan_tmp_cap) {
        if (c->d_scan_tmp) cudaFree(c->d_scan_tmp);
        c->d_scan_tmp = nullptr, c->scan_tmp_cap = 0;
        OBEM_CUDA(c, cudaMalloc(&c->d_scan_tmp, tmp));
        c->scan_tmp_cap = tmp;
    }
    OBEM_CUDA(c, cub::DeviceScan::ExclusiveSum(c->d_scan_tmp, tmp, c->d_cell_fill, c->d_cell_start, (int)(ncells + 1), st));
    int total = 0;
    OBEM_CUDA(c, cudaMemcpyAsync(&total, c->d_cell_start + ncells, sizeof(int), cudaMemcpyDeviceToHost, st));
    OBEM_CUDA(c, cudaStreamSynchronize(st));
    if (total < 0) return OBEM_ENOMEM; /* more than 2^31 entries: the lists do not fit their int offsets */
    if ((long long)total > c->list_cap) {
        if (c->d_cell_list) cudaFree(c->d_cell_list);
        c->d_cell_list = nullptr, c->list_cap = 0;
        OBEM_CUDA(c, cudaMalloc(&c->d_cell_list, (size_t)(total > 0 ? total : 1) * sizeof(int)));
        c->list_cap = total > 0 ? total : 1;
    }
    OBEM_CUDA(c, cudaMemsetAsync(c->d_cell_fill, 0, (size_t)(ncells + 1) * sizeof(int), st));
    near_bin_kernel<true><<<(unsigned)ceil_div(np, 128), 128, 0, st>>>(g, c->d_pcr, np, c->d_cell_fill, c->d_cell_start,
                                                                       c->d_cell_list);
    OBEM_CUDA(c, cudaGetLastError());
    near_sort_kernel<<<(unsigned)ceil_div(ncells, 128), 128, 0, st>>>(c->d_cell_start, c->d_cell_list, ncells);
    OBEM_CUDA(c, cudaGetLastError());
    c->launches += 5;
    for (int a = 0; a < 3; ++a) c->near_lo[a] = g.lo[a], c->near_n[a] = g.n[a];
    c->near_s = s;
    c->near_entries = total;
    c->near_valid = 1;
    return OBEM_OK;
}

} /* namespace */

int obem_near_store_panels(obem_ctx* c, const float* d_verts, const float* d_sigma, long long np, cudaStream_t st)
{
    c->near_valid = 0;
    c->near_entries = -1;
    if (np <= 0) return OBEM_OK;
    int rc = near_grow_panels(c, np);
    if (rc != OBEM_OK) return rc;
    OBEM_CUDA(c, cudaMemcpyAsync(c->d_pverts, d_verts, (size_t)np * 9 * sizeof(float), cudaMemcpyDeviceToDevice, st));
    OBEM_CUDA(c, cudaMemcpyAsync(c->d_psigma, d_sigma, (size_t)np * sizeof(float), cudaMemcpyDeviceToDevice, st));
    return OBEM_OK;
}

int obem_near_store_sigma(obem_ctx* c, const float* d_sigma, long long np, cudaStream_t st)
{
    if (np <= 0 || !c->d_psigma) return OBEM_OK;
    OBEM_CUDA(c, cudaMemcpyAsync(c->d_psigma, d_sigma, (size_t)np * sizeof(float), cudaMemcpyDeviceToDevice, st));
    return OBEM_OK;
}

int obem_near_correct(obem_ctx* c, const float4* tgt, long long nt, float4* out, cudaStream_t st)
{
    if (nt <= 0 || c->n_pan <= 0) return OBEM_OK;
    if (nt > 0x7fffffffLL) return OBEM_EINVAL;
    if (!c->near_valid) {
        int rc = near_build(c, st);
        if (rc != OBEM_OK) return rc;
    }
    if (c->near_n[0] == 0) return OBEM_OK;
    if (nt > c->redo_cap) {
        if (c->d_redo_list) cudaFree(c->d_redo_list);
        c->d_redo_list = nullptr, c->redo_cap = 0;
        OBEM_CUDA(c, cudaMalloc(&c->d_redo_list, (size_t)nt * sizeof(int)));
        c->redo_cap = nt;
    }
    if (!c->d_redo_count) OBEM_CUDA(c, cudaMalloc(&c->d_redo_count, 256));
    OBEM_CUDA(c, cudaMemsetAsync(c->d_redo_count, 0, sizeof(unsigned), st));
    NearParams P;
    for (int a = 0; a < 3; ++a) P.g.lo[a] = c->near_lo[a], P.g.n[a] = c->near_n[a];
    P.g.s = c->near_s, P.g.inv_s = 1.0 / c->near_s;
    P.start = c->d_cell_start, P.list = c->d_cell_list;
    P.pcr = c->d_pcr, P.porg = c->d_porg, P.qrel = c->d_qrel;
    P.verts = c->d_pverts, P.sigma = c->d_psigma;
    P.tgt = tgt, P.out = out, P.nt = nt;
    P.eps2 = (double)c->eps_panel * (double)c->eps_panel;
    P.crit2 = (VERY_NEAR / (double)c->near_factor) * (VERY_NEAR / (double)c->near_factor);
    P.redo_list = c->d_redo_list, P.redo_count = c->d_redo_count;
    /* the targets in cell order: count, scan, fill (three O(nt) passes) */
    const long long ncells = (long long)c->near_n[0] * c->near_n[1] * c->near_n[2];
    if (nt > c->near_t_cap) {
        if (c->d_near_tcell) cudaFree(c->d_near_tcell);
        if (c->d_near_tlist) cudaFree(c->d_near_tlist);
        c->d_near_tcell = c->d_near_tlist = nullptr, c->near_t_cap = 0;
        OBEM_CUDA(c, cudaMalloc(&c->d_near_tcell, (size_t)nt * sizeof(int)));
        OBEM_CUDA(c, cudaMalloc(&c->d_near_tlist, (size_t)nt * sizeof(int)));
        c->near_t_cap = nt;
    }
    if (ncells + 1 > c->near_c_cap) {
        if (c->d_near_tcount) cudaFree(c->d_near_tcount);
        if (c->d_near_tstart) cudaFree(c->d_near_tstart);
        c->d_near_tcount = c->d_near_tstart = nullptr, c->near_c_cap = 0;
        OBEM_CUDA(c, cudaMalloc(&c->d_near_tcount, (size_t)(ncells + 1) * sizeof(int)));
        OBEM_CUDA(c, cudaMalloc(&c->d_near_tstart, (size_t)(ncells + 1) * sizeof(int)));
        c->near_c_cap = ncells + 1;
    }
    size_t tmp = 0;
    OBEM_CUDA(c, cub::DeviceScan::ExclusiveSum(nullptr, tmp, c->d_near_tcount, c->d_near_tstart, (int)(ncells + 1), st));
    if (tmp > c->scan_tmp_cap) {
        if (c->d_scan_tmp) cudaFree(c->d_scan_tmp);
        c->d_scan_tmp = nullptr, c->scan_tmp_cap = 0;
        OBEM_CUDA(c, cudaMalloc(&c->d_scan_tmp, tmp));
        c->scan_tmp_cap = tmp;
    }
    OBEM_CUDA(c, cudaMemsetAsync(c->d_near_tcount, 0, (size_t)(ncells + 1) * sizeof(int), st));
    near_tcount_kernel<<<(unsigned)ceil_div(nt, 256), 256, 0, st>>>(P, c->d_near_tcell, c->d_near_tcount);
    OBEM_CUDA(c, cudaGetLastError());
    tmp = c->scan_tmp_cap;
    OBEM_CUDA(c, cub::DeviceScan::ExclusiveSum(c->d_scan_tmp, tmp, c->d_near_tcount, c->d_near_tstart, (int)(ncells + 1), st));
    OBEM_CUDA(c, cudaMemsetAsync(c->d_near_tcount, 0, (size_t)(ncells + 1) * sizeof(int), st)); /* now the fill cursor */
    near_tfill_kernel<<<(unsigned)ceil_div(nt, 256), 256, 0, st>>>(c->d_near_tcell, c->d_near_tstart, c->d_near_tcount,
                                                                 c->d_near_tlist, nt);
    OBEM_CUDA(c, cudaGetLastError());
    c->launches += 3;
    /* grid for the worst case (every target has a cell); warps beyond tstart[ncells] leave at once */
    near_correct_kernel<<<(unsigned)ceil_div(nt, NEAR_WARPS), NEAR_WARPS * 32, 0, st>>>(P, c->d_near_tlist,
                                                                                       c->d_near_tstart + ncells);
    OBEM_CUDA(c, cudaGetLastError());
    near_redo_kernel<<<4 * c->sm_count, 256, 0, st>>>(P, c->n_pan);
    OBEM_CUDA(c, cudaGetLastError());
    c->launches += 2;
    return OBEM_OK;
}

int obem_eval_exact(obem_ctx* c, const float4* tgt, long long nt, float4* out, unsigned flags, long long self_first,
                    float eps_nbody, cudaStream_t st, float2* trk_out)
{
    float4* pan = out;
    int rc;
    if (flags & OBEM_NBODY) {
        rc = obem_eval_internal(c, tgt, nt, out, OBEM_NBODY, self_first, eps_nbody, st, trk_out);
        if (rc != OBEM_OK) return rc;
        if (nt > c->exact_tmp_cap) {
            if (c->d_exact_tmp) cudaFree(c->d_exact_tmp);
            c->d_exact_tmp = nullptr, c->exact_tmp_cap = 0;
            OBEM_CUDA(c, cudaMalloc(&c->d_exact_tmp, (size_t)nt * sizeof(float4)));
            c->exact_tmp_cap = nt;
        }
        pan = c->d_exact_tmp;
    }
    rc = obem_eval_internal(c, tgt, nt, pan, OBEM_PANELS, -1, eps_nbody, st, nullptr);
    if (rc == OBEM_OK) rc = obem_near_correct(c, tgt, nt, pan, st);
    if (rc != OBEM_OK || pan == out) return rc;
    near_combine_kernel<<<(unsigned)ceil_div(nt, 256), 256, 0, st>>>(out, pan, nt);
    OBEM_CUDA(c, cudaGetLastError());
    c->launches += 1;
    return OBEM_OK;
}

void obem_near_free(obem_ctx* c)
{
    void* ptrs[] = {c->d_pverts, c->d_psigma, c->d_porg, c->d_pcr, c->d_cell_start, c->d_cell_fill, c->d_cell_list,
                    c->d_near_red, c->d_scan_tmp, c->d_redo_list, c->d_redo_count, c->d_exact_tmp, c->d_near_tcell,
                    c->d_near_tlist, c->d_near_tcount, c->d_near_tstart};
    for (void* p : ptrs)
        if (p) cudaFree(p);
}

extern "C" {

int obem_set_near_field(obem_ctx* c, float near_factor)
{
    if (!c || !(near_factor > 0.f) || !isfinite(near_factor)) return OBEM_EINVAL;
    if (near_factor != c->near_factor) c->near_valid = 0, c->near_entries = -1;
    c->near_factor = near_factor;
    return OBEM_OK;
}

int64_t obem_near_list_size(const obem_ctx* c) { return c ? c->near_entries : -1; }

int64_t obem_near_cells(const obem_ctx* c)
{
    if (!c || c->near_entries < 0) return -1;
    return (int64_t)c->near_n[0] * c->near_n[1] * c->near_n[2];
}

} /* extern "C" */
