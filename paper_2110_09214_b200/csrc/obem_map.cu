/*
 * obem_map.cu -- the static field option (section 3.2.1):
 * "the field components are computed only once at some predefined spatial coordinates located on a uniform 3D
 * grid map ... During the transport, the field components at each particle location are then interpolated in this
 * 3D map."
 *
 *   obem_field_map   fills the map: node coordinates generated on the device, evaluated by the hot path's
 *                    evaluation kernel (obem.cu) -- config 5 of BASELINE.json is exactly this call.
 *   obem_interp_map  trilinear interpolation (reading A18) of (Ex, Ey, Ez, phi) at M positions: a gather of
 *                    8 float4 nodes per position; bound by HBM / L2 (32 B streamed per position + the touched
 *                    part of the map).
 *
 * Part of libobem.so; shares nothing with oracle/.
 */
#include "obem_internal.cuh"

namespace {

struct MapGeom {
    double o[3];   /* origin: coordinates of node (0,0,0) [m] */
    double d[3];   /* spacing [m] */
    double inv[3]; /* 1/spacing, 0 along an axis with a single node */
    int n[3];      /* nodes per axis (nx, ny, nz); z is the fastest index */
};

/* node (ix, iy, iz) -> float4 (x, y, z, 0), rounded once to fp32 from the fp64 value o + i*d (a multiply and an
 * add, each rounded: no contraction, so a host that computes the same expression in fp64 gets the same bits) */
__global__ void __launch_bounds__(256) map_nodes_kernel(MapGeom g, float4* __restrict__ pts, long long total)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= total) return;
    const int iz = (int)(i % g.n[2]);
    const long long r = i / g.n[2];
    const int iy = (int)(r % g.n[1]);
    const int ix = (int)(r / g.n[1]);
    float4 p;
    p.x = (float)__dadd_rn(g.o[0], __dmul_rn((double)ix, g.d[0]));
    p.y = (float)__dadd_rn(g.o[1], __dmul_rn((double)iy, g.d[1]));
    p.z = (float)__dadd_rn(g.o[2], __dmul_rn((double)iz, g.d[2]));
    p.w = 0.f;
    pts[i] = p;
}

/* cell index and fraction along one axis; the position is clamped to the node lattice (reading A18).  fp64: the
 * fraction f and its complement g = 1 - f are then exact to one fp32 rounding each, whatever the size of the map
 * (4 fp64 operations per axis against 8 16-byte gathers per position) */
__device__ __forceinline__ void axis_cell(double p, double o, double inv, int n, int& i0, int& i1, float& f,
                                          float& g)
{
    double u = (p - o) * inv;
    const double top = (double)(n - 1);
    u = u < 0.0 ? 0.0 : (u > top ? top : u); /* NaN positions fall to node 0 */
    if (!(u == u)) u = 0.0;
    int i = (int)u; /* u >= 0: truncation is floor */
    if (i > n - 2) i = n - 2 > 0 ? n - 2 : 0;
    i0 = i;
    i1 = i + 1 < n ? i + 1 : n - 1;
    const double fd = u - (double)i;
    f = (float)fd;
    g = (float)(1.0 - fd); /* both weights of the axis carry a RELATIVE error of one fp32 rounding */
}

template <bool ACCUM>
__global__ void __launch_bounds__(256) map_interp_kernel(MapGeom g, const float4* __restrict__ map,
                                                         const float4* __restrict__ pts, float4* __restrict__ out,
                                                         long long m)
{
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= m) return;
    const float4 p = __ldcs(pts + t); /* streamed once: keep the map, not the positions, in L2 */
    int x0, x1, y0, y1, z0, z1;
    float fx, fy, fz, gx, gy, gz;
    axis_cell((double)p.x, g.o[0], g.inv[0], g.n[0], x0, x1, fx, gx);
    axis_cell((double)p.y, g.o[1], g.inv[1], g.n[1], y0, y1, fy, gy);
    axis_cell((double)p.z, g.o[2], g.inv[2], g.n[2], z0, z1, fz, gz);
    const long long sy = g.n[2], sx = (long long)g.n[1] * g.n[2];
    const float4* b00 = map + x0 * sx + y0 * sy;
    const float4* b01 = map + x0 * sx + y1 * sy;
    const float4* b10 = map + x1 * sx + y0 * sy;
    const float4* b11 = map + x1 * sx + y1 * sy;
    /* 8 independent 16-byte gathers; the two z neighbours of a row share a 32-byte sector */
    const float4 c000 = __ldg(b00 + z0), c001 = __ldg(b00 + z1);
    const float4 c010 = __ldg(b01 + z0), c011 = __ldg(b01 + z1);
    const float4 c100 = __ldg(b10 + z0), c101 = __ldg(b10 + z1);
    const float4 c110 = __ldg(b11 + z0), c111 = __ldg(b11 + z1);
    const float w000 = gx * gy * gz, w001 = gx * gy * fz, w010 = gx * fy * gz, w011 = gx * fy * fz;
    const float w100 = fx * gy * gz, w101 = fx * gy * fz, w110 = fx * fy * gz, w111 = fx * fy * fz;
    float4 r;
#define OBEM_TRI(comp)                                                                                             \
    r.comp = w000 * c000.comp + w001 * c001.comp + w010 * c010.comp + w011 * c011.comp + w100 * c100.comp +        \
             w101 * c101.comp + w110 * c110.comp + w111 * c111.comp;
    OBEM_TRI(x) OBEM_TRI(y) OBEM_TRI(z) OBEM_TRI(w)
#undef OBEM_TRI
    if (ACCUM) {
        const float4 a = out[t];
        r.x += a.x, r.y += a.y, r.z += a.z, r.w += a.w;
    }
    __stcs(out + t, r);
}

int map_geom(MapGeom& g, int nx, int ny, int nz, const double* h_origin, const double* h_spacing)
{
    if (nx < 1 || ny < 1 || nz < 1 || !h_origin || !h_spacing) return OBEM_EINVAL;
    const int n[3] = {nx, ny, nz};
    for (int a = 0; a < 3; ++a) {
        if (!isfinite(h_origin[a]) || !isfinite(h_spacing[a])) return OBEM_EINVAL;
        if (n[a] > 1 && !(h_spacing[a] > 0.0)) return OBEM_EINVAL;
        g.o[a] = h_origin[a];
        g.d[a] = h_spacing[a];
        g.inv[a] = (n[a] > 1) ? 1.0 / h_spacing[a] : 0.0;
        g.n[a] = n[a];
    }
    return OBEM_OK;
}

} /* namespace */

extern "C" {

int obem_field_map(obem_ctx* c, int nx, int ny, int nz, const double* h_origin, const double* h_spacing,
                   float* d_map, unsigned flags, void* cuda_stream)
{
    if (!c) return OBEM_EINVAL;
    MapGeom g;
    int rc = map_geom(g, nx, ny, nz, h_origin, h_spacing);
    if (rc != OBEM_OK) return rc;
    if (!d_map || !aligned16(d_map)) return OBEM_EINVAL;
    const long long total = (long long)nx * ny * nz;
    DeviceGuard dg(c->device);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if ((size_t)total * sizeof(float4) > c->map_pts_cap) {
        if (c->d_map_pts) OBEM_CUDA(c, cudaFree(c->d_map_pts));
        c->d_map_pts = nullptr, c->map_pts_cap = 0;
        OBEM_CUDA(c, cudaMalloc(&c->d_map_pts, (size_t)total * sizeof(float4)));
        c->map_pts_cap = (size_t)total * sizeof(float4);
    }
    map_nodes_kernel<<<(unsigned)ceil_div(total, 256), 256, 0, st>>>(g, c->d_map_pts, total);
    OBEM_CUDA(c, cudaGetLastError());
    c->launches += 1;
    return obem_eval_at_points(c, (const float*)c->d_map_pts, total, d_map, flags, cuda_stream);
}

int obem_interp_map(obem_ctx* c, const float* d_map, int nx, int ny, int nz, const double* h_origin,
                    const double* h_spacing, const float* d_pts, int64_t m, float* d_out, int accumulate,
                    void* cuda_stream)
{
    if (!c || m < 0) return OBEM_EINVAL;
    MapGeom g;
    int rc = map_geom(g, nx, ny, nz, h_origin, h_spacing);
    if (rc != OBEM_OK) return rc;
    if (m == 0) return OBEM_OK;
    if (!d_map || !d_pts || !d_out || !aligned16(d_map) || !aligned16(d_pts) || !aligned16(d_out)) return OBEM_EINVAL;
    DeviceGuard dg(c->device);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const unsigned grid = (unsigned)ceil_div(m, 256);
    if (accumulate)
        map_interp_kernel<true><<<grid, 256, 0, st>>>(g, (const float4*)d_map, (const float4*)d_pts, (float4*)d_out, m);
    else
        map_interp_kernel<false><<<grid, 256, 0, st>>>(g, (const float4*)d_map, (const float4*)d_pts, (float4*)d_out, m);
    OBEM_CUDA(c, cudaGetLastError());
    c->launches += 1;
    return OBEM_OK;
}

} /* extern "C" */
