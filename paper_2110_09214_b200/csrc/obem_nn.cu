/*
 * obem_nn.cu -- the nearest-neighbour (NN) approximation of the N-body sum (
 * PAPER.md:279-296, section 3.2.4): "evaluating the exact Coulombian field following (3.8) for each of the closest
 * particles to the particle of interest while the field from the particles further away is approximated by their
 * centre of charges with a barycentric method."  The paper says no more; the algorithm is DESIGN.md reading A19:
 *
 *   1. k-d partition with equal-count leaves: level by level, every segment of more than 256 charges is sorted
 *      (stably) along the longest axis of its bounding box and cut at a multiple of 256 -- one radix sort per level
 *      over the whole array with key = (segment rank, coordinate).  A leaf = 256 charges = one source block of the
 *      evaluation kernel; a target group = 8 consecutive leaves = one 2048-target tile.
 *   2. Per leaf, and per super-leaf (64 consecutive leaves): bounding box and two pseudo-particles (the centres of
 *      charge of its positive and of its negative members).
 *   3. A box B is FAR from tile t iff theta^2 dist2(box_t, B) > diag2(B), decided in fp64 with individually rounded
 *      operations (the oracle takes the same decisions bit for bit).  A super-leaf that is far at theta / 2 stands for
 *      all its leaves; the leaves of the other super-leaves are classified one by one at theta.
 *   4. Tile t's source list = its near leaves (the charges themselves, exact Eq 3.8, self excluded by index) + its
 *      own far blocks: the pseudo-particles of its far super-leaves and far leaves, compacted -- run by the LIST
 *      instantiation of the hot path's evaluation kernel (obem.cu), stream-K over all (tile, block) units.
 *   5. Results are scattered back to the input order.
 *
 * Every step is enqueued on the caller's stream; nothing is read back to the host (all sizes follow from n).
 * Part of libobem.so; shares nothing with oracle/.
 */
#include <cub/block/block_radix_sort.cuh>
#include <cub/device/device_radix_sort.cuh>

#include "obem_internal.cuh"

namespace {

typedef unsigned long long u64k;
constexpr int LEAF = OBEM_SB;        /* 256 */
constexpr int GROUP = OBEM_TT;       /* 2048 */
constexpr int LPG = GROUP / LEAF;    /* leaves per group */
constexpr int SUPER = 64;            /* leaves per super-leaf */
constexpr int MAX_SUPER = 32768;     /* super-leaves the list kernel keeps flags for (5.4e8 charges) */
constexpr float NN_PAD_FAR = 1.0e15f;

__host__ __device__ __forceinline__ long long nn_split(long long a, long long b)
{
    const long long leaves = (b - a + LEAF - 1) / LEAF;
    return a + (long long)LEAF * ((leaves + 1) / 2);
}
/* segment [a, b) that holds position i after `level` rounds of cuts; rank = its `level`-bit path (0 = left, 1 = right
 * at every cut, 0 once a segment is final): ascending in position, so it can stand for the segment in a sort key */
__device__ __forceinline__ void nn_segment(long long n, long long i, int level, long long& a, long long& b,
                                           unsigned& rank)
{
    a = 0, b = n;
    rank = 0u;
    for (int t = 0; t < level; ++t) {
        rank <<= 1;
        if (b - a <= LEAF) continue;
        const long long m = nn_split(a, b);
        if (i < m) b = m;
        else a = m, rank |= 1u;
    }
}
__device__ __forceinline__ void nn_segment(long long n, long long i, int level, long long& a, long long& b)
{
    unsigned rank;
    nn_segment(n, i, level, a, b, rank);
}
/* fp32 bits -> unsigned whose order is the IEEE total order of the floats */
__device__ __forceinline__ unsigned nn_ordered(float f)
{
    const unsigned u = __float_as_uint(f);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float nn_unordered(unsigned k)
{
    return __uint_as_float((k & 0x80000000u) ? (k & 0x7fffffffu) : ~k);
}

__global__ void nn_iota_kernel(int* __restrict__ perm, long long n)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) perm[i] = (int)i;
}

/* segmin[s][0..2], segmax[s][0..2] = min, max of the ordered coordinates of segment s = (segment start)/256
 * (initialised to 0xffffffff and 0 by the caller).  min / max
 * are order independent, so the atomics do not make the result depend on scheduling. */
__global__ void __launch_bounds__(256) nn_segbox_kernel(const float4* __restrict__ x, const int* __restrict__ perm,
                                                        long long n, int level, unsigned* __restrict__ segmin,
                                                        unsigned* __restrict__ segmax)
{
    __shared__ unsigned sh[6][8];
    __shared__ long long sh_a[8];
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    long long a = -1, b = -1;
    unsigned k[6] = {0xffffffffu, 0xffffffffu, 0xffffffffu, 0u, 0u, 0u};
    if (i < n) {
        nn_segment(n, i, level, a, b);
        if (b - a <= LEAF) a = -1; /* final: not sorted again */
        else {
            const float4 p = x[perm[i]];
            k[0] = k[3] = nn_ordered(p.x), k[1] = k[4] = nn_ordered(p.y), k[2] = k[5] = nn_ordered(p.z);
        }
    }
    /* a warp that lies inside one segment (almost all do) reduces first; so does a block of such warps */
    const long long a0 = __shfl_sync(0xffffffffu, a, 0);
    const bool warp_same = __all_sync(0xffffffffu, a == a0);
    if (!warp_same) {
        if (a >= 0) {
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                atomicMin(segmin + (a / LEAF) * 3 + d, k[d]);
                atomicMax(segmax + (a / LEAF) * 3 + d, k[3 + d]);
            }
        }
    } else {
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            k[d] = __reduce_min_sync(0xffffffffu, k[d]);
            k[3 + d] = __reduce_max_sync(0xffffffffu, k[3 + d]);
        }
    }
    if (lane == 0) {
        sh_a[w] = warp_same ? a0 : -2; /* -2: this warp has already written */
#pragma unroll
        for (int d = 0; d < 6; ++d) sh[d][w] = k[d];
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        /* merge runs of consecutive warps of the same segment, one atomic per run and component */
        int w0 = 0;
        while (w0 < 8) {
            const long long sa = sh_a[w0];
            int w1 = w0 + 1;
            unsigned m[6];
            for (int d = 0; d < 6; ++d) m[d] = sh[d][w0];
            while (w1 < 8 && sh_a[w1] == sa) {
                for (int d = 0; d < 3; ++d) {
                    m[d] = min(m[d], sh[d][w1]);
                    m[3 + d] = max(m[3 + d], sh[3 + d][w1]);
                }
                ++w1;
            }
            if (sa >= 0) {
                for (int d = 0; d < 3; ++d) {
                    atomicMin(segmin + (sa / LEAF) * 3 + d, m[d]);
                    atomicMax(segmax + (sa / LEAF) * 3 + d, m[3 + d]);
                }
            }
            w0 = w1;
        }
    }
}

__global__ void nn_key_kernel(const float4* __restrict__ x, const int* __restrict__ perm, long long n, int level,
                              const unsigned* __restrict__ segmin, const unsigned* __restrict__ segmax,
                              u64k* __restrict__ keys)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    long long a, b;
    unsigned rank;
    nn_segment(n, i, level, a, b, rank);
    unsigned low;
    if (b - a <= LEAF) {
        low = (unsigned)(i - a); /* keep the order of a final segment */
    } else {
        double ext[3];
#pragma unroll
        for (int d = 0; d < 3; ++d)
            ext[d] = (double)nn_unordered(segmax[(a / LEAF) * 3 + d]) - (double)nn_unordered(segmin[(a / LEAF) * 3 + d]);
        int ax = 0; /* the first axis of the largest extent */
        if (ext[1] > ext[ax]) ax = 1;
        if (ext[2] > ext[ax]) ax = 2;
        const float4 p = x[perm[i]];
        low = nn_ordered(ax == 0 ? p.x : (ax == 1 ? p.y : p.z));
    }
    keys[i] = ((u64k)rank << 32) | (u64k)low; /* `level` bits of segment rank + 32 of coordinate: 4-6 radix passes */
}

/*
 * The last levels of the k-d order, one CTA per segment.  Once every segment holds at most KD_LOCAL_LEAVES leaves
 * (8192 charges) the remaining cuts touch nothing outside it: the CTA keeps the segment's 8192 (key, index) pairs in
 * registers and runs the same rounds as the global loop -- boxes of the current sub-segments, axis = first of the
 * largest extents (fp64), STABLE sort by (sub-segment rank, ordered coordinate), cut at nn_split -- with a block-wide
 * radix sort instead of a device-wide one: the same order, bit for bit (a stable sort by the same keys), in one launch
 * instead of three launches + 5-6 radix passes per level.  CTA k takes the segment whose l0-bit path is k.
 */
constexpr int KD_LOCAL_LEAVES = 32, KD_THREADS = 512, KD_ITEMS = KD_LOCAL_LEAVES * LEAF / KD_THREADS;
constexpr int KD_MAX_SUB = KD_LOCAL_LEAVES / 2; /* sub-segments that can still be cut in the last round */
typedef cub::BlockRadixSort<u64k, KD_THREADS, KD_ITEMS, int, 6> KdSort; /* 6-bit digits: 6 passes over 33-36 key bits */

__global__ void __launch_bounds__(KD_THREADS, 1) nn_kd_local_kernel(const float4* __restrict__ x, int* __restrict__ perm,
                                                                 long long n, int l0, int levels)
{
    extern __shared__ __align__(16) unsigned char kd_dyn[]; /* sizeof(KdSort::TempStorage): above the static limit */
    typename KdSort::TempStorage& sort_tmp = *reinterpret_cast<typename KdSort::TempStorage*>(kd_dyn);
    __shared__ unsigned smin[2 * KD_MAX_SUB][3], smax[2 * KD_MAX_SUB][3];
    long long a = 0, b = n;
    for (int t = 0; t < l0; ++t) {
        const unsigned bit = ((unsigned)blockIdx.x >> (l0 - 1 - t)) & 1u;
        if (b - a <= LEAF) {
            if (bit) return; /* a final segment has path bits 0 from there on */
            continue;
        }
        const long long m = nn_split(a, b);
        if (bit) a = m;
        else b = m;
    }
    if (b - a <= LEAF) return; /* final already: its order stays */
    const int m = (int)(b - a), tid = threadIdx.x;
    u64k key[KD_ITEMS];
    int val[KD_ITEMS];
#pragma unroll
    for (int j = 0; j < KD_ITEMS; ++j) {
        const int p = tid * KD_ITEMS + j;
        val[j] = p < m ? perm[a + p] : -1;
    }
    /* sub-segment of position p (relative to a) after t more cuts: [ua, ub), its t-bit path r */
    auto sub_of = [&](const int p, const int t, int& ua, int& ub, unsigned& r) {
        ua = 0, ub = m, r = 0u;
        for (int q = 0; q < t; ++q) {
            r <<= 1;
            if (ub - ua <= LEAF) continue;
            const int mid = ua + LEAF * (((ub - ua + LEAF - 1) / LEAF + 1) / 2); /* nn_split: a is a multiple of LEAF */
            if (p < mid) ub = mid;
            else ua = mid, r |= 1u;
        }
    };
    for (int t = 0; t < levels - l0; ++t) {
        if (tid < 2 * KD_MAX_SUB * 3) {
            (&smin[0][0])[tid] = 0xffffffffu;
            (&smax[0][0])[tid] = 0u;
        }
        __syncthreads();
        /* boxes: a thread's 16 consecutive positions lie in at most two sub-segments */
        unsigned run_rank = 0xffffffffu, bmin[3], bmax[3];
#pragma unroll
        for (int j = 0; j < KD_ITEMS; ++j) {
            const int p = tid * KD_ITEMS + j;
            if (p >= m) continue;
            int ua, ub;
            unsigned r;
            sub_of(p, t, ua, ub, r);
            if (ub - ua <= LEAF) continue; /* final */
            const float4 v = x[val[j]];
            const unsigned k0 = nn_ordered(v.x), k1 = nn_ordered(v.y), k2 = nn_ordered(v.z);
            if (r != run_rank) {
                if (run_rank != 0xffffffffu) {
#pragma unroll
                    for (int d = 0; d < 3; ++d) atomicMin(&smin[run_rank][d], bmin[d]), atomicMax(&smax[run_rank][d], bmax[d]);
                }
                run_rank = r;
                bmin[0] = bmax[0] = k0, bmin[1] = bmax[1] = k1, bmin[2] = bmax[2] = k2;
            } else {
                bmin[0] = min(bmin[0], k0), bmax[0] = max(bmax[0], k0);
                bmin[1] = min(bmin[1], k1), bmax[1] = max(bmax[1], k1);
                bmin[2] = min(bmin[2], k2), bmax[2] = max(bmax[2], k2);
            }
        }
        if (run_rank != 0xffffffffu) {
#pragma unroll
            for (int d = 0; d < 3; ++d) atomicMin(&smin[run_rank][d], bmin[d]), atomicMax(&smax[run_rank][d], bmax[d]);
        }
        __syncthreads();
#pragma unroll
        for (int j = 0; j < KD_ITEMS; ++j) {
            const int p = tid * KD_ITEMS + j;
            unsigned low = 0u, r = 1u << t; /* pads: behind every sub-segment */
            if (p < m) {
                int ua, ub;
                sub_of(p, t, ua, ub, r);
                if (ub - ua <= LEAF) {
                    low = (unsigned)(p - ua); /* keep the order of a final sub-segment */
                } else {
                    double ext[3];
#pragma unroll
                    for (int d = 0; d < 3; ++d)
                        ext[d] = (double)nn_unordered(smax[r][d]) - (double)nn_unordered(smin[r][d]);
                    int ax = 0; /* the first axis of the largest extent */
                    if (ext[1] > ext[ax]) ax = 1;
                    if (ext[2] > ext[ax]) ax = 2;
                    const float* v = reinterpret_cast<const float*>(x + val[j]); /* second read: an L1 / L2 hit */
                    low = nn_ordered(__ldg(v + ax));
                }
            }
            key[j] = ((u64k)r << 32) | (u64k)low;
        }
        KdSort(sort_tmp).Sort(key, val, 0, 32 + t + 1);
        __syncthreads();
    }
#pragma unroll
    for (int j = 0; j < KD_ITEMS; ++j) {
        const int p = tid * KD_ITEMS + j;
        if (p < m) perm[a + p] = val[j];
    }
}

/* one CTA per leaf: sorted copy (plain, padded) + blocked copy with header + bounding box + the two pseudo-particles.
 * Inside the leaf the members are put in the order negative weights first (a stable partition: which charges a leaf
 * holds is the k-d order's business, their order inside it enters no result), and perm_out records the final order.
 * Header: .x = the weight all 256 members share, or NaN; .z = |w| if the leaf is full and its members carry exactly
 * -|w| and +|w| (electrons and singly charged ions: the usual leaf), else 0; .w = the number of negative members.
 * The list kernel then sums the negative and the positive run unweighted (12 packed instructions per interaction
 * instead of 13) and only the 4-source group that straddles the sign boundary with weights. */
__global__ void __launch_bounds__(LEAF) nn_leaf_kernel(const float4* __restrict__ x, const int* __restrict__ perm,
                                                        long long n, float4* __restrict__ sorted,
                                                        float4* __restrict__ pool, float* __restrict__ leafbox,
                                                        float4* __restrict__ pseudo, double* __restrict__ leafmom,
                                                        int* __restrict__ perm_out)
{
    __shared__ double red[8][LEAF / 32];
    __shared__ float fred[6][LEAF / 32];
    __shared__ int wneg[LEAF / 32];
    const long long l = blockIdx.x, i = l * LEAF + threadIdx.x;
    const bool valid = i < n;
    const int src = valid ? perm[i] : -1;
    const float4 v = valid ? x[src] : make_float4(NN_PAD_FAR, NN_PAD_FAR, NN_PAD_FAR, 0.f);
    /* stable partition: negatives first */
    const bool neg = valid && v.w < 0.f;
    {
        const unsigned bal = __ballot_sync(0xffffffffu, neg);
        if ((threadIdx.x & 31) == 0) wneg[threadIdx.x >> 5] = __popc(bal);
        __syncthreads();
        int before = 0, total = 0;
        for (int ww = 0; ww < LEAF / 32; ++ww) {
            if (ww < (int)(threadIdx.x >> 5)) before += wneg[ww];
            total += wneg[ww];
        }
        const int in_warp = __popc(bal & ((1u << (threadIdx.x & 31)) - 1u));
        const int rank_neg = before + in_warp;
        const int slot = neg ? rank_neg : total + ((int)threadIdx.x - rank_neg);
        const long long j = l * LEAF + slot;
        sorted[j] = v;
        pool[l * OBEM_SBH + 1 + slot] = v;
        if (j < n) perm_out[j] = src; /* invalid members are the last threads of the last leaf: they stay last */
        const float w0 = x[perm[l * LEAF]].w, m0 = fabsf(w0);
        const int uniform = __syncthreads_and(v.w == w0);
        const int twoval = __syncthreads_and(valid && m0 > 0.f && fabsf(v.w) == m0);
        if (threadIdx.x == 0)
            pool[l * OBEM_SBH] = make_float4(uniform ? w0 : __int_as_float(0x7fc00000), 0.f,
                                             (twoval && !uniform) ? m0 : 0.f, (float)total);
    }
    /* box over the valid members, charge and first moment of the positive and of the negative members */
    const float big = __int_as_float(0x7f800000);
    float lo[3] = {valid ? v.x : big, valid ? v.y : big, valid ? v.z : big};
    float hi[3] = {valid ? v.x : -big, valid ? v.y : -big, valid ? v.z : -big};
    const double q = (double)v.w;
    double m[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    if (valid && v.w > 0.f) m[0] = q, m[1] = q * v.x, m[2] = q * v.y, m[3] = q * v.z;
    if (valid && v.w < 0.f) m[4] = q, m[5] = q * v.x, m[6] = q * v.y, m[7] = q * v.z;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            lo[d] = fminf(lo[d], __shfl_xor_sync(0xffffffffu, lo[d], o));
            hi[d] = fmaxf(hi[d], __shfl_xor_sync(0xffffffffu, hi[d], o));
        }
#pragma unroll
        for (int k = 0; k < 8; ++k) m[k] += __shfl_xor_sync(0xffffffffu, m[k], o);
    }
    if (lane == 0) {
#pragma unroll
        for (int d = 0; d < 3; ++d) fred[d][w] = lo[d], fred[3 + d][w] = hi[d];
#pragma unroll
        for (int k = 0; k < 8; ++k) red[k][w] = m[k];
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int ww = 1; ww < LEAF / 32; ++ww) {
            for (int d = 0; d < 3; ++d) {
                fred[d][0] = fminf(fred[d][0], fred[d][ww]);
                fred[3 + d][0] = fmaxf(fred[3 + d][0], fred[3 + d][ww]);
            }
            for (int k = 0; k < 8; ++k) red[k][0] += red[k][ww];
        }
        for (int d = 0; d < 6; ++d) leafbox[l * 6 + d] = fred[d][0];
        for (int k = 0; k < 8; ++k) leafmom[l * 8 + k] = red[k][0]; /* Q+, Q+ R+ (3), Q-, Q- R- (3): for the super-leaves */
        for (int h = 0; h < 2; ++h) {
            const double Q = red[4 * h][0];
            pseudo[l * 2 + h] = (Q != 0.0) ? make_float4((float)(red[4 * h + 1][0] / Q), (float)(red[4 * h + 2][0] / Q),
                                                         (float)(red[4 * h + 3][0] / Q), (float)Q)
                                           : make_float4(NN_PAD_FAR, NN_PAD_FAR, NN_PAD_FAR, 0.f);
        }
    }
}

/* FAR iff theta^2 * dist2(box_g, box_l) > diag2(box_l); every operation rounded on its own (no contraction), x, y, z
 * in this order -- the oracle forms the same expression in numpy */
__device__ __forceinline__ bool nn_is_far(const float (&g)[6], const float* __restrict__ lb, double theta2)
{
    double dist2 = 0.0, diag2 = 0.0;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const double a = (double)lb[d] - (double)g[3 + d], b = (double)g[d] - (double)lb[3 + d];
        const double gap = fmax(0.0, fmax(a, b));
        const double side = (double)lb[3 + d] - (double)lb[d];
        const double g2 = __dmul_rn(gap, gap), s2 = __dmul_rn(side, side);
        dist2 = (d == 0) ? g2 : __dadd_rn(dist2, g2);
        diag2 = (d == 0) ? s2 : __dadd_rn(diag2, s2);
    }
    return __dmul_rn(theta2, dist2) > diag2;
}

__device__ __forceinline__ void nn_group_box(const float* __restrict__ leafbox, long long g, long long n_leaf, float (&gb)[6])
{
    const float big = __int_as_float(0x7f800000);
    for (int d = 0; d < 3; ++d) gb[d] = big, gb[3 + d] = -big;
    for (long long l = g * LPG; l < (g + 1) * LPG && l < n_leaf; ++l)
        for (int d = 0; d < 3; ++d) {
            gb[d] = fminf(gb[d], leafbox[l * 6 + d]);
            gb[3 + d] = fmaxf(gb[3 + d], leafbox[l * 6 + 3 + d]);
        }
}

/* one CTA of SUPER threads per super-leaf: union of its leaves' boxes (min / max: exact in any order), centres of
 * charge from their fp64 moments, summed in leaf order by one thread per moment (from shared memory) */
__global__ void __launch_bounds__(SUPER) nn_super_kernel(const float* __restrict__ leafbox,
                                                         const double* __restrict__ leafmom, long long n_leaf,
                                                         long long n_super, float* __restrict__ superbox,
                                                         float4* __restrict__ superpseudo)
{
    __shared__ double mom[SUPER][9]; /* stride 9: the 8 summing threads read down the columns */
    __shared__ float box[SUPER / 32][6];
    __shared__ double tot[8];
    const long long sidx = blockIdx.x;
    const int t = threadIdx.x;
    const long long l = sidx * SUPER + t;
    const float big = __int_as_float(0x7f800000);
    float b[6] = {big, big, big, -big, -big, -big};
    if (l < n_leaf) {
#pragma unroll
        for (int d = 0; d < 6; ++d) b[d] = leafbox[l * 6 + d];
#pragma unroll
        for (int k = 0; k < 8; ++k) mom[t][k] = leafmom[l * 8 + k];
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            b[d] = fminf(b[d], __shfl_xor_sync(0xffffffffu, b[d], o));
            b[3 + d] = fmaxf(b[3 + d], __shfl_xor_sync(0xffffffffu, b[3 + d], o));
        }
    }
    if ((t & 31) == 0) {
#pragma unroll
        for (int d = 0; d < 6; ++d) box[t >> 5][d] = b[d];
    }
    __syncthreads();
    const int cnt = (int)min((long long)SUPER, n_leaf - sidx * SUPER);
    if (t < 8) {
        double m = 0.0;
        for (int j = 0; j < cnt; ++j) m += mom[j][t];
        tot[t] = m;
    }
    if (t >= 32 && t < 38) {
        const int d = t - 32;
        float v = box[0][d];
        for (int w = 1; w < SUPER / 32; ++w) v = d < 3 ? fminf(v, box[w][d]) : fmaxf(v, box[w][d]);
        superbox[sidx * 6 + d] = v;
    }
    __syncthreads();
    if (t < 2) {
        const double Q = tot[4 * t];
        superpseudo[sidx * 2 + t] = (Q != 0.0) ? make_float4((float)(tot[4 * t + 1] / Q), (float)(tot[4 * t + 2] / Q),
                                                             (float)(tot[4 * t + 3] / Q), (float)Q)
                                               : make_float4(NN_PAD_FAR, NN_PAD_FAR, NN_PAD_FAR, 0.f);
    }
}

/* entry e of a tile's far area (blocks of 256 entries, each behind a header) */
__device__ __forceinline__ float4* nn_far_slot(float4* far, long long e) { return far + (e >> 8) * OBEM_SBH + 1 + (e & 255); }

/* block-wide rank of the threads whose flag is set (ascending thread order) and their total; wsum: 8 ints of scratch */
__device__ __forceinline__ int nn_block_rank(bool flag, int* wsum, int& total)
{
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const unsigned bal = __ballot_sync(0xffffffffu, flag);
    __syncthreads(); /* wsum is free again */
    if (lane == 0) wsum[w] = __popc(bal);
    __syncthreads();
    int before = 0;
    total = 0;
    for (int ww = 0; ww < 8; ++ww) {
        if (ww < w) before += wsum[ww];
        total += wsum[ww];
    }
    return before + __popc(bal & ((1u << lane) - 1u));
}

/* one CTA per tile.  FILL = false: cnt[g] = (near leaves) + (far blocks).  FILL = true: write the tile's list (near
 * leaf blocks in ascending order, then its far blocks) and its far blocks: the pseudo-particles of its far
 * super-leaves (ascending), then of its far leaves (ascending), padded with blanks to a whole block. */
template <bool FILL>
__global__ void __launch_bounds__(256) nn_lists_kernel(const float* __restrict__ leafbox, const float4* __restrict__ pseudo,
                                                       const float* __restrict__ superbox,
                                                       const float4* __restrict__ superpseudo, long long n_leaf,
                                                       long long n_super, long long far_cap, double theta2,
                                                       double theta2_super,
                                                       long long* __restrict__ cnt, const long long* __restrict__ tile_ptr,
                                                       int* __restrict__ list, float4* __restrict__ pool)
{
    __shared__ int wsum[8];
    __shared__ unsigned sflag[MAX_SUPER / 32]; /* bit s: super-leaf s is far from this tile */
    const long long g = blockIdx.x;
    float gb[6];
    nn_group_box(leafbox, g, n_leaf, gb);
    const int lane = threadIdx.x & 31;
    float4* far = FILL ? pool + (n_leaf + g * far_cap) * OBEM_SBH : nullptr;
    int* out = FILL ? list + tile_ptr[g] : nullptr;
    long long n_far = 0; /* pairs of pseudo-particles in the far area so far (same value in every thread) */
    int n_near = 0;
    /* super-leaves */
    for (long long s0 = 0; s0 < n_super; s0 += 256) {
        const long long sidx = s0 + threadIdx.x;
        const bool isfar = sidx < n_super && nn_is_far(gb, superbox + sidx * 6, theta2_super);
        const unsigned bal = __ballot_sync(0xffffffffu, isfar);
        if (lane == 0 && (s0 + (threadIdx.x & ~31)) < n_super) sflag[(s0 + threadIdx.x) >> 5] = bal;
        int total;
        const int rank = nn_block_rank(isfar, wsum, total);
        if (FILL && isfar) {
            *nn_far_slot(far, 2 * (n_far + rank)) = superpseudo[sidx * 2];
            *nn_far_slot(far, 2 * (n_far + rank) + 1) = superpseudo[sidx * 2 + 1];
        }
        n_far += total;
    }
    __syncthreads();
    /* leaves of the super-leaves that are not far */
    for (long long l0 = 0; l0 < n_leaf; l0 += 256) {
        const long long l = l0 + threadIdx.x;
        bool near = false, farleaf = false;
        if (l < n_leaf && !((sflag[(l / SUPER) >> 5] >> ((l / SUPER) & 31)) & 1u)) {
            farleaf = nn_is_far(gb, leafbox + l * 6, theta2);
            near = !farleaf;
        }
        int tn, tf;
        const int rn = nn_block_rank(near, wsum, tn);
        const int rf = nn_block_rank(farleaf, wsum, tf);
        if (FILL) {
            if (near) out[n_near + rn] = (int)l;
            if (farleaf) {
                *nn_far_slot(far, 2 * (n_far + rf)) = pseudo[l * 2];
                *nn_far_slot(far, 2 * (n_far + rf) + 1) = pseudo[l * 2 + 1];
            }
        }
        n_near += tn;
        n_far += tf;
    }
    const long long entries = 2 * n_far, blocks = (entries + 255) >> 8;
    if (FILL) {
        const float4 blank = make_float4(NN_PAD_FAR, NN_PAD_FAR, NN_PAD_FAR, 0.f);
        for (long long e = entries + threadIdx.x; e < blocks * 256; e += 256) *nn_far_slot(far, e) = blank;
        for (long long k = threadIdx.x; k < blocks; k += 256) {
            far[k * OBEM_SBH] = make_float4(__int_as_float(0x7fc00000), 0.f, 0.f, 0.f); /* header: weights differ */
            out[n_near + k] = (int)(n_leaf + g * far_cap + k);
        }
    } else if (threadIdx.x == 0) {
        cnt[g] = n_near + blocks;
    }
}

/* tile_ptr = exclusive prefix sum of cnt, U = the total.  One CTA: every thread sums a run of consecutive tiles,
 * the runs' totals are scanned across the block, then every thread writes its run (integers: exact in any order). */
constexpr int SCAN_THREADS = 1024;
__global__ void __launch_bounds__(SCAN_THREADS) nn_scan_kernel(const long long* __restrict__ cnt, long long n_group,
                                                               long long* __restrict__ tile_ptr, long long* __restrict__ U)
{
    __shared__ long long wtot[SCAN_THREADS / 32];
    const int t = threadIdx.x, lane = t & 31, w = t >> 5;
    const long long per = (n_group + SCAN_THREADS - 1) / SCAN_THREADS;
    const long long g0 = min(n_group, (long long)t * per), g1 = min(n_group, g0 + per);
    long long s = 0;
    for (long long g = g0; g < g1; ++g) s += cnt[g];
    long long inc = s; /* inclusive scan of the runs' totals: inside the warp, then across the warps */
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const long long v = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += v;
    }
    if (lane == 31) wtot[w] = inc;
    __syncthreads();
    long long before = 0;
    for (int ww = 0; ww < w; ++ww) before += wtot[ww];
    long long run = before + inc - s;
    for (long long g = g0; g < g1; ++g) {
        tile_ptr[g] = run;
        run += cnt[g];
    }
    if (t == SCAN_THREADS - 1) {
        tile_ptr[n_group] = before + inc;
        *U = before + inc;
    }
}

__global__ void nn_scatter_kernel(const float4* __restrict__ sorted_out, const int* __restrict__ perm, long long n,
                                  float4* __restrict__ out)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[perm[i]] = sorted_out[i];
}

__global__ void nn_add_kernel(float4* __restrict__ out, const float4* __restrict__ b, long long n)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float4 p = out[i], q = b[i];
    out[i] = make_float4(p.x + q.x, p.y + q.y, p.z + q.z, p.w + q.w);
}

} /* namespace */

namespace {

template <typename T>
int nn_grow(obem_ctx* c, T*& p, size_t& cap, size_t count)
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

void obem_nn_free(obem_ctx* c)
{
    void* ptrs[] = {c->nn.perm[0], c->nn.perm[1], c->nn.key[0], c->nn.key[1], c->nn.seg, c->nn.sorted, c->nn.pool,
                    c->nn.leafbox, c->nn.pseudo, c->nn.leafmom, c->nn.superbox, c->nn.superpseudo, c->nn.cnt, c->nn.tile_ptr, c->nn.list, c->nn.out_sorted, c->nn.tmp,
                    c->nn.pan};
    for (void* p : ptrs)
        if (p) cudaFree(p);
}

extern "C" {

int obem_set_nn_theta(obem_ctx* c, float theta)
{
    if (!c || !(theta >= 0.f) || !isfinite(theta)) return OBEM_EINVAL;
    c->nn.theta = theta;
    return OBEM_OK;
}

int obem_eval_at_charges_nn(obem_ctx* c, float* d_out, unsigned flags, void* cuda_stream)
{
    if (!c) return OBEM_EINVAL;
    if (flags & ~(OBEM_NBODY | OBEM_PANELS | OBEM_PANELS_EXACT)) return OBEM_EINVAL;
    if (!(flags & OBEM_NBODY)) return OBEM_EINVAL;
    if ((flags & OBEM_PANELS_EXACT) && !(flags & OBEM_PANELS)) return OBEM_EINVAL;
    if (c->n_chg < 0) return OBEM_ESTATE;
    if ((flags & OBEM_PANELS) && c->n_pan < 0) return OBEM_ESTATE;
    if (c->sym_n > 0) return OBEM_EINVAL; /* the lists hold no image leaves */
    const long long n = c->n_chg;
    if (n == 0) return OBEM_OK;
    if (!d_out || !aligned16(d_out)) return OBEM_EINVAL;
    if (n > 0x7fffffffLL - GROUP) return OBEM_EINVAL;
    DeviceGuard dg(c->device);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    obem_nn_state& S = c->nn;
    const long long n_leaf = ceil_div(n, LEAF), n_group = ceil_div(n, GROUP);
    const long long n_super = ceil_div(n_leaf, SUPER);
    if (n_super > MAX_SUPER) return OBEM_EINVAL;
    const long long far_cap = ceil_div(2 * (n_leaf + n_super), LEAF); /* far blocks a tile can need at most */
    int levels = 0;
    while ((1LL << levels) < n_leaf) ++levels;
    int nbits = 1; /* bits of a segment's leaf index */
    while ((1LL << nbits) <= n_leaf) ++nbits;

    int rc = OBEM_OK;
    for (int k = 0; k < 2 && rc == OBEM_OK; ++k) {
        rc = nn_grow(c, S.perm[k], S.perm_cap[k], (size_t)n);
        if (rc == OBEM_OK) rc = nn_grow(c, S.key[k], S.key_cap[k], (size_t)n);
    }
    if (rc == OBEM_OK) rc = nn_grow(c, S.seg, S.seg_cap, (size_t)n_leaf * 6);
    if (rc == OBEM_OK) rc = nn_grow(c, S.sorted, S.sorted_cap, (size_t)n_leaf * LEAF);
    if (rc == OBEM_OK) rc = nn_grow(c, S.pool, S.pool_cap, (size_t)(n_leaf + n_group * far_cap) * OBEM_SBH);
    if (rc == OBEM_OK) rc = nn_grow(c, S.leafbox, S.leafbox_cap, (size_t)n_leaf * 6);
    if (rc == OBEM_OK) rc = nn_grow(c, S.pseudo, S.pseudo_cap, (size_t)n_leaf * 2);
    if (rc == OBEM_OK) rc = nn_grow(c, S.leafmom, S.leafmom_cap, (size_t)n_leaf * 8);
    if (rc == OBEM_OK) rc = nn_grow(c, S.superbox, S.superbox_cap, (size_t)n_super * 6);
    if (rc == OBEM_OK) rc = nn_grow(c, S.superpseudo, S.superpseudo_cap, (size_t)n_super * 2);
    if (rc == OBEM_OK) rc = nn_grow(c, S.cnt, S.cnt_cap, (size_t)n_group);
    if (rc == OBEM_OK) rc = nn_grow(c, S.tile_ptr, S.tile_ptr_cap, (size_t)n_group + 2); /* [n_group + 1] + U */
    if (rc == OBEM_OK) rc = nn_grow(c, S.list, S.list_cap, (size_t)n_group * (size_t)(n_leaf + far_cap));
    if (rc == OBEM_OK) rc = nn_grow(c, S.out_sorted, S.out_sorted_cap, (size_t)n);
    if (rc != OBEM_OK) return rc;
    size_t tmp_bytes = 0;
    OBEM_CUDA(c, cub::DeviceRadixSort::SortPairs(nullptr, tmp_bytes, S.key[0], S.key[1], S.perm[0], S.perm[1], (int)n, 0,
                                                 32 + nbits, st));
    {
        unsigned char* t = (unsigned char*)S.tmp;
        rc = nn_grow(c, t, S.tmp_cap, tmp_bytes);
        S.tmp = t;
        if (rc != OBEM_OK) return rc;
    }

    const unsigned gn = (unsigned)ceil_div(n, 256);
    /* 1. k-d order */
    nn_iota_kernel<<<gn, 256, 0, st>>>(S.perm[0], n);
    OBEM_CUDA(c, cudaGetLastError());
    int cur = 0;
    unsigned* segmin = S.seg;
    unsigned* segmax = S.seg + n_leaf * 3;
    /* device-wide rounds while a segment can exceed KD_LOCAL_LEAVES leaves, then one launch for the rest */
    int l0 = 0;
    for (long long lv = n_leaf; lv > KD_LOCAL_LEAVES; lv = (lv + 1) / 2) ++l0;
    if (l0 > levels) l0 = levels;
    for (int level = 0; level < l0; ++level) {
        OBEM_CUDA(c, cudaMemsetAsync(segmin, 0xff, (size_t)n_leaf * 3 * sizeof(unsigned), st));
        OBEM_CUDA(c, cudaMemsetAsync(segmax, 0x00, (size_t)n_leaf * 3 * sizeof(unsigned), st));
        nn_segbox_kernel<<<gn, 256, 0, st>>>(c->d_chg, S.perm[cur], n, level, segmin, segmax);
        OBEM_CUDA(c, cudaGetLastError());
        nn_key_kernel<<<gn, 256, 0, st>>>(c->d_chg, S.perm[cur], n, level, segmin, segmax, S.key[cur]);
        OBEM_CUDA(c, cudaGetLastError());
        OBEM_CUDA(c, cub::DeviceRadixSort::SortPairs(S.tmp, tmp_bytes, S.key[cur], S.key[cur ^ 1], S.perm[cur],
                                                     S.perm[cur ^ 1], (int)n, 0, 32 + level, st));
        cur ^= 1;
        c->launches += 3;
    }
    if (l0 < levels) {
        OBEM_CUDA(c, cudaFuncSetAttribute(nn_kd_local_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          (int)sizeof(KdSort::TempStorage)));
        nn_kd_local_kernel<<<1u << l0, KD_THREADS, sizeof(KdSort::TempStorage), st>>>(c->d_chg, S.perm[cur], n, l0, levels);
        OBEM_CUDA(c, cudaGetLastError());
        c->launches += 1;
    }
    const int* perm = S.perm[cur];
    /* 2. leaves */
    nn_leaf_kernel<<<(unsigned)n_leaf, LEAF, 0, st>>>(c->d_chg, perm, n, S.sorted, S.pool, S.leafbox, S.pseudo,
                                                      S.leafmom, S.perm[cur ^ 1]);
    perm = S.perm[cur ^ 1]; /* the k-d order with the sign partition inside the leaves */
    OBEM_CUDA(c, cudaGetLastError());
    nn_super_kernel<<<(unsigned)n_super, SUPER, 0, st>>>(S.leafbox, S.leafmom, n_leaf, n_super, S.superbox,
                                                                    S.superpseudo);
    OBEM_CUDA(c, cudaGetLastError());
    /* 3. + 4. per-tile lists and far blocks */
    const double theta2 = (double)S.theta * (double)S.theta;
    const double theta_s = 0.5 * (double)S.theta, theta2s = theta_s * theta_s; /* super-leaves: accepted at theta / 2 */
    long long* U_dev = S.tile_ptr + n_group + 1;
    nn_lists_kernel<false><<<(unsigned)n_group, 256, 0, st>>>(S.leafbox, S.pseudo, S.superbox, S.superpseudo, n_leaf,
                                                              n_super, far_cap, theta2, theta2s, S.cnt, nullptr, nullptr, nullptr);
    OBEM_CUDA(c, cudaGetLastError());
    nn_scan_kernel<<<1, SCAN_THREADS, 0, st>>>(S.cnt, n_group, S.tile_ptr, U_dev);
    OBEM_CUDA(c, cudaGetLastError());
    nn_lists_kernel<true><<<(unsigned)n_group, 256, 0, st>>>(S.leafbox, S.pseudo, S.superbox, S.superpseudo, n_leaf,
                                                             n_super, far_cap, theta2, theta2s, S.cnt, S.tile_ptr, S.list, S.pool);
    OBEM_CUDA(c, cudaGetLastError());
    c->launches += 6;
    /* 5. the sums, in sorted order, then back to the input order */
    rc = obem_eval_list(c, S.sorted, n, S.out_sorted, S.pool, S.tile_ptr, S.list, U_dev, n_leaf, c->eps_pp, st);
    if (rc != OBEM_OK) return rc;
    nn_scatter_kernel<<<gn, 256, 0, st>>>(S.out_sorted, perm, n, (float4*)d_out);
    OBEM_CUDA(c, cudaGetLastError());
    c->launches += 1;
    S.last_n = n;
    if (flags & OBEM_PANELS) {
        rc = nn_grow(c, S.pan, S.pan_cap, (size_t)n);
        if (rc != OBEM_OK) return rc;
        rc = obem_eval_internal(c, c->d_chg, n, S.pan, flags & ~OBEM_NBODY, -1, c->eps_pp, st);
        if (rc != OBEM_OK) return rc;
        nn_add_kernel<<<gn, 256, 0, st>>>((float4*)d_out, S.pan, n);
        OBEM_CUDA(c, cudaGetLastError());
        c->launches += 1;
    }
    return OBEM_OK;
}

int64_t obem_nn_last_units(obem_ctx* c, void* cuda_stream)
{
    if (!c || c->nn.last_n <= 0 || !c->nn.tile_ptr) return -1;
    DeviceGuard dg(c->device);
    long long U = -1;
    const long long n_group = ceil_div(c->nn.last_n, GROUP);
    if (cudaMemcpyAsync(&U, c->nn.tile_ptr + n_group + 1, sizeof(U), cudaMemcpyDeviceToHost, (cudaStream_t)cuda_stream) !=
            cudaSuccess ||
        cudaStreamSynchronize((cudaStream_t)cuda_stream) != cudaSuccess) {
        cudaGetLastError();
        return -1;
    }
    return U;
}

} /* extern "C" */
