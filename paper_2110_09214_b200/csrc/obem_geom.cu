/*
 * obem_geom.cu -- geometry conveniences of SURVEY.md section 8(f), NEXT-3:
 *
 *   quadrilateral cells   PAPER.md:119, :167: "flat polygonal cells (triangles, quadrangles, etc.)", each with one
 *                         constant sigma.  A flat quadrilateral (v0, v1, v2, v3) is the two triangles (v0, v1, v2) and
 *                         (v0, v2, v3) carrying the same sigma: its integrals of Eq (2.13)/(2.14) are their sum.
 *   symmetry planes       PAPER.md:165: "up to three symmetry planes can also be included".  A plane x_a = c with
 *                         parity s = +1 (mirror images carry the same charge) or -1 (opposite charge: a grounded
 *                         plane) adds the field of the mirrored sources.  By symmetry of the kernel,
 *                             E_image(r) = s M E_orig(M r),   phi_image(r) = s phi_orig(M r),
 *                         M the reflection, so the images are evaluated as REFLECTED TARGETS on the original sources:
 *                         nothing is duplicated in memory, and an image of charge i acts on charge i itself.
 *
 * Part of libobem.so; shares nothing with oracle/.
 */
#include "obem_internal.cuh"

namespace {

/* cell (v0, v1, v2, v3) -> triangles 2i = (v0, v1, v2), 2i + 1 = (v0, v2, v3); nvert[i] == 3: the second one is
 * the degenerate (v0, v2, v2), which contributes 0 (reading A8) */
__global__ void split_cells_kernel(const float* __restrict__ verts4, const int* __restrict__ nvert,
                                   const float* __restrict__ sigma, float* __restrict__ tri, float* __restrict__ tsig,
                                   long long nc)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nc) return;
    const float* v = verts4 + i * 12;
    const bool quad = nvert == nullptr || nvert[i] == 4;
    float* t = tri + i * 18;
    for (int d = 0; d < 3; ++d) {
        t[0 + d] = v[0 + d], t[3 + d] = v[3 + d], t[6 + d] = v[6 + d];
        t[9 + d] = v[0 + d], t[12 + d] = v[6 + d], t[15 + d] = quad ? v[9 + d] : v[6 + d];
    }
    if (sigma) tsig[2 * i] = tsig[2 * i + 1] = sigma[i];
}

__global__ void dup_sigma_kernel(const float* __restrict__ sigma, float* __restrict__ tsig, long long nc)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < nc) tsig[2 * i] = tsig[2 * i + 1] = sigma[i];
}

struct Mirror {
    double two_c[3]; /* 2 c along the reflected axes */
    int flip[3];     /* 1: this axis is reflected */
    float sign;      /* product of the parities */
};

__global__ void reflect_targets_kernel(const float4* __restrict__ in, float4* __restrict__ out, long long n, Mirror m)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float4 p = in[i];
    if (m.flip[0]) p.x = (float)(m.two_c[0] - (double)p.x);
    if (m.flip[1]) p.y = (float)(m.two_c[1] - (double)p.y);
    if (m.flip[2]) p.z = (float)(m.two_c[2] - (double)p.z);
    out[i] = p;
}

__global__ void add_image_kernel(float4* __restrict__ out, const float4* __restrict__ img, long long n, Mirror m)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float4 o = out[i];
    const float4 e = img[i];
    o.x += (m.flip[0] ? -m.sign : m.sign) * e.x;
    o.y += (m.flip[1] ? -m.sign : m.sign) * e.y;
    o.z += (m.flip[2] ? -m.sign : m.sign) * e.z;
    o.w += m.sign * e.w;
    out[i] = o;
}

template <typename T>
int geom_grow(obem_ctx* c, T*& p, size_t& cap, size_t count)
{
    const size_t bytes = count * sizeof(T);
    if (bytes <= cap) return OBEM_OK;
    if (p) cudaFree(p);
    p = nullptr, cap = 0;
    OBEM_CUDA(c, cudaMalloc(&p, bytes));
    cap = bytes;
    return OBEM_OK;
}

} /* namespace */

/* the evaluation with symmetry planes: the direct term, then one reflected-target evaluation per image */
int obem_eval_symmetric(obem_ctx* c, const float4* tgt, long long nt, float4* out, unsigned flags, long long self_first,
                        float eps_nbody, cudaStream_t st, float2* trk_out)
{
    c->sym_busy = 1;
    int rc = obem_eval_internal(c, tgt, nt, out, flags, self_first, eps_nbody, st, trk_out);
    if (rc == OBEM_OK && nt > 0) {
        rc = geom_grow(c, c->d_sym_pts, c->sym_pts_cap, (size_t)nt);
        if (rc == OBEM_OK) rc = geom_grow(c, c->d_sym_out, c->sym_out_cap, (size_t)nt);
    }
    const unsigned grid = (unsigned)ceil_div(nt > 0 ? nt : 1, 256);
    for (int mask = 1; rc == OBEM_OK && nt > 0 && mask < (1 << c->sym_n); ++mask) {
        Mirror m;
        m.sign = 1.f;
        for (int a = 0; a < 3; ++a) m.flip[a] = 0, m.two_c[a] = 0.0;
        for (int k = 0; k < c->sym_n; ++k)
            if (mask & (1 << k)) {
                m.flip[c->sym_axis[k]] = 1;
                m.two_c[c->sym_axis[k]] = 2.0 * c->sym_coord[k];
                m.sign *= (float)c->sym_sign[k];
            }
        reflect_targets_kernel<<<grid, 256, 0, st>>>(tgt, c->d_sym_pts, nt, m);
        if (cudaGetLastError() != cudaSuccess) rc = OBEM_ECUDA;
        /* an image never coincides with its original by index: no exclusion, no partner tracking */
        if (rc == OBEM_OK) rc = obem_eval_internal(c, c->d_sym_pts, nt, c->d_sym_out, flags, -1, eps_nbody, st, nullptr);
        if (rc == OBEM_OK) {
            add_image_kernel<<<grid, 256, 0, st>>>(out, c->d_sym_out, nt, m);
            if (cudaGetLastError() != cudaSuccess) rc = OBEM_ECUDA;
            c->launches += 2;
        }
    }
    c->sym_busy = 0;
    return rc;
}

void obem_geom_free(obem_ctx* c)
{
    void* ptrs[] = {c->d_sym_pts, c->d_sym_out, c->d_cell_tri, c->d_cell_sig};
    for (void* p : ptrs)
        if (p) cudaFree(p);
}

extern "C" {

int obem_set_symmetry(obem_ctx* c, int n_planes, const int* h_axis, const double* h_coord, const int* h_parity)
{
    if (!c || n_planes < 0 || n_planes > 3) return OBEM_EINVAL;
    if (n_planes > 0 && (!h_axis || !h_coord || !h_parity)) return OBEM_EINVAL;
    int seen[3] = {0, 0, 0};
    for (int k = 0; k < n_planes; ++k) {
        if (h_axis[k] < 0 || h_axis[k] > 2 || seen[h_axis[k]]) return OBEM_EINVAL; /* one plane per axis */
        if (!isfinite(h_coord[k]) || (h_parity[k] != 1 && h_parity[k] != -1)) return OBEM_EINVAL;
        seen[h_axis[k]] = 1;
    }
    c->sym_n = n_planes;
    for (int k = 0; k < n_planes; ++k) {
        c->sym_axis[k] = h_axis[k];
        c->sym_coord[k] = h_coord[k];
        c->sym_sign[k] = h_parity[k];
    }
    return OBEM_OK;
}

int obem_set_panels_cells(obem_ctx* c, const float* d_verts4, const int32_t* d_nvert, const float* d_sigma,
                          int64_t n_cells, void* cuda_stream)
{
    if (!c || n_cells < 0) return OBEM_EINVAL;
    if (n_cells > 0 && (!d_verts4 || !d_sigma || !aligned4(d_verts4) || !aligned4(d_sigma) ||
                        (d_nvert && !aligned4(d_nvert))))
        return OBEM_EINVAL;
    DeviceGuard g(c->device);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (n_cells == 0) return obem_set_panels(c, nullptr, nullptr, 0, cuda_stream);
    int rc = geom_grow(c, c->d_cell_tri, c->cell_tri_cap, (size_t)n_cells * 18);
    if (rc == OBEM_OK) rc = geom_grow(c, c->d_cell_sig, c->cell_sig_cap, (size_t)n_cells * 2);
    if (rc != OBEM_OK) return rc;
    split_cells_kernel<<<(unsigned)ceil_div(n_cells, 256), 256, 0, st>>>(d_verts4, d_nvert, d_sigma, c->d_cell_tri,
                                                                         c->d_cell_sig, n_cells);
    OBEM_CUDA(c, cudaGetLastError());
    c->launches += 1;
    return obem_set_panels(c, c->d_cell_tri, c->d_cell_sig, 2 * n_cells, cuda_stream);
}

int obem_set_sigma_cells(obem_ctx* c, const float* d_sigma, int64_t n_cells, void* cuda_stream)
{
    if (!c || n_cells < 0) return OBEM_EINVAL;
    if (c->n_pan < 0) return OBEM_ESTATE;
    if (2 * n_cells != c->n_pan) return OBEM_EINVAL;
    if (n_cells == 0) return OBEM_OK;
    if (!d_sigma || !aligned4(d_sigma)) return OBEM_EINVAL;
    DeviceGuard g(c->device);
    int rc = geom_grow(c, c->d_cell_sig, c->cell_sig_cap, (size_t)n_cells * 2);
    if (rc != OBEM_OK) return rc;
    dup_sigma_kernel<<<(unsigned)ceil_div(n_cells, 256), 256, 0, (cudaStream_t)cuda_stream>>>(d_sigma, c->d_cell_sig,
                                                                                              n_cells);
    OBEM_CUDA(c, cudaGetLastError());
    c->launches += 1;
    return obem_set_sigma(c, c->d_cell_sig, 2 * n_cells, cuda_stream);
}

} /* extern "C" */
