// bvh.cu -- GPU LBVH build over the triangle soup (SURVEY.md 8(a) A0 + A1).
//
// The paper's implementation takes its BVH from a library; here
// it is built on the device: vertex AABB -> 63-bit Morton keys of the face
// centroids -> stable radix sort -> binary radix tree (Karras 2012, restated;
// equal keys are split by their sorted position) -> bottom-up refit with one
// arrival counter per internal node -> 64-byte two-child-box nodes.
// Nothing here assumes a manifold, consistently oriented, non-degenerate or
// connected mesh: every face is a leaf (all triangles absorb).
//
// Sliver splitting (Fig. 8: CAD models "made of sliver triangles").
// The box of a long thin triangle that is not axis-aligned is almost all empty space: on BASELINE config 3 the
// 42 000 strips of the rotated cylinders (length 1.4-2, width 3e-4) have boxes of side ~1, a query point inside
// such a box must test the strip, and a point inside a cylinder's box tests thousands of them (measured: 145
// triangle tests and 95 wide nodes per query against 6 and 13 on the icosphere).  A face that is long (longest
// edge > `split_length` mean edge lengths) and thin (aspect L^2 / 2A > 8) therefore enters the tree as several
// LEAF REFERENCES: it is cut into slabs across its longest edge, each reference carries the box of one slab and
// the whole triangle (the point-triangle test is the exact one, so the query result cannot change; a triangle
// reached through two of its references is simply tested twice).  The number of extra references is bounded by
// `split_budget` per face on average: the piece length is raised until the budget holds.
#include "common.cuh"

#include <limits.h>
#include <new>
#include <string.h>

namespace {

constexpr int BT = 256;

__device__ __forceinline__ int float_to_ordered(float f)
{
    int i = __float_as_int(f);
    return i >= 0 ? i : i ^ 0x7FFFFFFF;
}
__device__ __forceinline__ float ordered_to_float(int i)
{
    return __int_as_float(i >= 0 ? i : i ^ 0x7FFFFFFF);
}

struct BuildScratch {
    int      flags;          // bit 0: face index out of range; bit 1: non-finite vertex
    int      n_degenerate;
    int      max_depth;
    int      pad;
    int      lo[3], hi[3];   // ordered-int AABB
    double   area;
};

// Pass 1: validate faces, AABB of the referenced vertices, per-block area partials.
__global__ void __launch_bounds__(BT)
face_bounds_kernel(const float* __restrict__ verts, int64_t V, const int32_t* __restrict__ faces, int64_t F,
                   BuildScratch* __restrict__ sc, double* __restrict__ area_partials)
{
    __shared__ double s_area[BT];
    __shared__ int s_lo[3], s_hi[3];
    if (threadIdx.x < 3) { s_lo[threadIdx.x] = 0x7FFFFFFF; s_hi[threadIdx.x] = (int)0x80000000; }
    __syncthreads();
    const int64_t f = (int64_t)blockIdx.x * BT + threadIdx.x;
    double area = 0.0;
    if (f < F) {
        const int i0 = faces[3 * f], i1 = faces[3 * f + 1], i2 = faces[3 * f + 2];
        if (i0 < 0 || i1 < 0 || i2 < 0 || i0 >= V || i1 >= V || i2 >= V) {
            atomicOr(&sc->flags, 1);
        } else {
            float p[3][3];
            const int idx[3] = { i0, i1, i2 };
            bool finite = true;
            for (int k = 0; k < 3; ++k)
                for (int d = 0; d < 3; ++d) { p[k][d] = verts[3 * (int64_t)idx[k] + d]; finite = finite && isfinite(p[k][d]); }
            if (!finite) {
                atomicOr(&sc->flags, 2);
            } else {
                for (int d = 0; d < 3; ++d) {
                    float lo = fminf(p[0][d], fminf(p[1][d], p[2][d]));
                    float hi = fmaxf(p[0][d], fmaxf(p[1][d], p[2][d]));
                    atomicMin(&s_lo[d], float_to_ordered(lo));
                    atomicMax(&s_hi[d], float_to_ordered(hi));
                }
                const double ax = (double)p[1][0] - p[0][0], ay = (double)p[1][1] - p[0][1], az = (double)p[1][2] - p[0][2];
                const double bx = (double)p[2][0] - p[0][0], by = (double)p[2][1] - p[0][1], bz = (double)p[2][2] - p[0][2];
                const double cx = ay * bz - az * by, cy = az * bx - ax * bz, cz = ax * by - ay * bx;
                area = 0.5 * sqrt(cx * cx + cy * cy + cz * cz);
                if (!(area > 0.0)) atomicAdd(&sc->n_degenerate, 1);
            }
        }
    }
    s_area[threadIdx.x] = area;
    __syncthreads();
    for (int s = BT / 2; s > 0; s >>= 1) {          // fixed-shape tree: deterministic
        if (threadIdx.x < s) s_area[threadIdx.x] += s_area[threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x == 0) area_partials[blockIdx.x] = s_area[0];
    if (threadIdx.x < 3) {
        atomicMin(&sc->lo[threadIdx.x], s_lo[threadIdx.x]);
        atomicMax(&sc->hi[threadIdx.x], s_hi[threadIdx.x]);
    }
}

__global__ void area_total_kernel(const double* __restrict__ partials, int n, BuildScratch* sc)
{
    double t = 0.0;
    for (int i = 0; i < n; ++i) t += partials[i];   // one thread, fixed order
    sc->area = t;
}

__device__ __forceinline__ uint64_t spread21(uint64_t x)
{
    x &= 0x1FFFFFull;
    x = (x | x << 32) & 0x1F00000000FFFFull;
    x = (x | x << 16) & 0x1F0000FF0000FFull;
    x = (x | x << 8)  & 0x100F00F00F00F00Full;
    x = (x | x << 4)  & 0x10C30C30C30C30C3ull;
    x = (x | x << 2)  & 0x1249249249249249ull;
    return x;
}

// ---------------------------------------------------------------------------
// Sliver splitting: pieces per face, leaf references with the boxes of the slabs.
// ---------------------------------------------------------------------------
constexpr float SPLIT_MIN_ASPECT = 8.0f;     // L^2 / (2 A): only thin faces are cut (an isotropic one gains nothing from slabs)
constexpr int   SPLIT_BINS = 64;             // histogram of L / unit in quarter octaves

struct FaceGeom { float3 A, B, C; float L2, tC, area2; };   // longest edge A->B, apex C, tC = parameter of C's foot on AB

__device__ __forceinline__ FaceGeom face_geom(const float* __restrict__ verts, const int32_t* __restrict__ faces, int64_t f)
{
    float3 p[3];
    for (int k = 0; k < 3; ++k) {
        const int64_t v = faces[3 * f + k];
        p[k] = make_float3(verts[3 * v], verts[3 * v + 1], verts[3 * v + 2]);
    }
    float l2[3];
    for (int k = 0; k < 3; ++k) {
        const float3 a = p[k], b = p[(k + 1) % 3];
        l2[k] = (b.x - a.x) * (b.x - a.x) + (b.y - a.y) * (b.y - a.y) + (b.z - a.z) * (b.z - a.z);
    }
    const int e = (l2[0] >= l2[1] && l2[0] >= l2[2]) ? 0 : (l2[1] >= l2[2] ? 1 : 2);
    FaceGeom g;
    g.A = p[e]; g.B = p[(e + 1) % 3]; g.C = p[(e + 2) % 3]; g.L2 = l2[e];
    const float3 ab = make_float3(g.B.x - g.A.x, g.B.y - g.A.y, g.B.z - g.A.z), ac = make_float3(g.C.x - g.A.x, g.C.y - g.A.y, g.C.z - g.A.z);
    const float t = g.L2 > 0.0f ? (ab.x * ac.x + ab.y * ac.y + ab.z * ac.z) / g.L2 : 0.0f;
    g.tC = fminf(fmaxf(t, 0.0f), 1.0f);
    const float cx = ab.y * ac.z - ab.z * ac.y, cy = ab.z * ac.x - ab.x * ac.z, cz = ab.x * ac.y - ab.y * ac.x;
    g.area2 = sqrtf(cx * cx + cy * cy + cz * cz);                 // 2 A
    return g;
}

// pieces of a face for a piece length `unit`: 1 unless the face is long AND thin
__device__ __forceinline__ int face_pieces(const FaceGeom& g, float unit, int max_pieces)
{
    if (!(g.L2 > unit * unit) || !(g.L2 > SPLIT_MIN_ASPECT * g.area2)) return 1;
    const float n = ceilf(sqrtf(g.L2) / unit);
    return n < 2.0f ? 1 : (n > (float)max_pieces ? max_pieces : (int)n);
}

__global__ void __launch_bounds__(BT)
split_hist_kernel(const float* __restrict__ verts, const int32_t* __restrict__ faces, int64_t F, float mean_edge,
                  unsigned int* __restrict__ hist)
{
    __shared__ unsigned int s_h[SPLIT_BINS];
    if (threadIdx.x < SPLIT_BINS) s_h[threadIdx.x] = 0;
    __syncthreads();
    const int64_t f = (int64_t)blockIdx.x * BT + threadIdx.x;
    if (f < F) {
        const FaceGeom g = face_geom(verts, faces, f);
        const float q = sqrtf(g.L2) / mean_edge;
        if (q > 1.0f && g.L2 > SPLIT_MIN_ASPECT * g.area2) {
            const int bin = min(SPLIT_BINS - 1, (int)(4.0f * log2f(q)));
            atomicAdd(&s_h[bin], 1u);
        }
    }
    __syncthreads();
    if (threadIdx.x < SPLIT_BINS && s_h[threadIdx.x]) atomicAdd(&hist[threadIdx.x], s_h[threadIdx.x]);
}

__global__ void __launch_bounds__(BT)
split_count_kernel(const float* __restrict__ verts, const int32_t* __restrict__ faces, int64_t F, float unit, int max_pieces,
                   uint32_t* __restrict__ counts)
{
    const int64_t f = (int64_t)blockIdx.x * BT + threadIdx.x;
    if (f >= F) return;
    counts[f] = unit > 0.0f ? (uint32_t)face_pieces(face_geom(verts, faces, f), unit, max_pieces) : 1u;
}

__device__ __forceinline__ void grow(float* box, float3 p)
{
    box[0] = fminf(box[0], p.x); box[1] = fminf(box[1], p.y); box[2] = fminf(box[2], p.z);
    box[3] = fmaxf(box[3], p.x); box[4] = fmaxf(box[4], p.y); box[5] = fmaxf(box[5], p.z);
}

// One leaf reference per piece: the face, the box of the slab t in [i/n, (i+1)/n] across the longest edge, and the
// Morton key of the box centre.  The slab is the convex hull of its two end cross-sections (a point X(t) on AB and
// a point Y(t) on AC or CB) and of C when its foot lies in the slab; the box is padded by a few ulps of the
// coordinates so that rounding cannot open a gap between neighbouring slabs or leave a point of the face outside.
__global__ void __launch_bounds__(BT)
ref_emit_kernel(const float* __restrict__ verts, const int32_t* __restrict__ faces, int64_t F, float unit, int max_pieces,
                const uint32_t* __restrict__ offs, const BuildScratch* __restrict__ sc,
                int32_t* __restrict__ ref_face, float* __restrict__ ref_box, uint64_t* __restrict__ keys, uint32_t* __restrict__ vals)
{
    const int64_t f = (int64_t)blockIdx.x * BT + threadIdx.x;
    if (f >= F) return;
    const FaceGeom g = face_geom(verts, faces, f);
    const int n = unit > 0.0f ? face_pieces(g, unit, max_pieces) : 1;
    float lo3[3], ext3[3];
    for (int d = 0; d < 3; ++d) { lo3[d] = ordered_to_float(sc->lo[d]); ext3[d] = ordered_to_float(sc->hi[d]) - lo3[d]; }
    for (int i = 0; i < n; ++i) {
        float box[6] = { CUDART_INF_F, CUDART_INF_F, CUDART_INF_F, -CUDART_INF_F, -CUDART_INF_F, -CUDART_INF_F };
        if (n == 1) {
            grow(box, g.A); grow(box, g.B); grow(box, g.C);                  // exactly the min/max of the vertices
        } else {
            const float t0 = (float)i / (float)n, t1 = (float)(i + 1) / (float)n;
            for (int e = 0; e < 2; ++e) {
                const float t = e ? t1 : t0;
                grow(box, make_float3(fmaf(t, g.B.x - g.A.x, g.A.x), fmaf(t, g.B.y - g.A.y, g.A.y), fmaf(t, g.B.z - g.A.z, g.A.z)));
                float3 y;
                if (t < g.tC) { const float u = t / g.tC; y = make_float3(fmaf(u, g.C.x - g.A.x, g.A.x), fmaf(u, g.C.y - g.A.y, g.A.y), fmaf(u, g.C.z - g.A.z, g.A.z)); }
                else if (g.tC < 1.0f) { const float u = (1.0f - t) / (1.0f - g.tC); y = make_float3(fmaf(u, g.C.x - g.B.x, g.B.x), fmaf(u, g.C.y - g.B.y, g.B.y), fmaf(u, g.C.z - g.B.z, g.B.z)); }
                else y = g.C;
                grow(box, y);
            }
            if (t0 <= g.tC && g.tC <= t1) grow(box, g.C);
            if (i == 0) grow(box, g.A);
            if (i == n - 1) grow(box, g.B);
            for (int d = 0; d < 3; ++d) {
                const float pad = 4e-6f * fmaxf(fabsf(box[d]), fabsf(box[3 + d])) + 1e-30f;
                box[d] -= pad; box[3 + d] += pad;
            }
        }
        const int64_t r = (int64_t)offs[f] + i;
        ref_face[r] = (int32_t)f;
        for (int q = 0; q < 6; ++q) ref_box[6 * r + q] = box[q];
        uint64_t key = 0;
        const float cen[3] = { (g.A.x + g.B.x + g.C.x) * (1.0f / 3.0f), (g.A.y + g.B.y + g.C.y) * (1.0f / 3.0f), (g.A.z + g.B.z + g.C.z) * (1.0f / 3.0f) };
        for (int d = 0; d < 3; ++d) {
            const float c = n == 1 ? cen[d] : 0.5f * (box[d] + box[3 + d]);  // whole face: its centroid; slab: the box centre
            float t = ext3[d] > 0.0f ? (c - lo3[d]) / ext3[d] : 0.0f;
            t = fminf(fmaxf(t, 0.0f), 1.0f);
            const uint64_t qd = (uint64_t)fminf(t * 2097152.0f, 2097151.0f);
            key |= spread21(qd) << (2 - d);                                  // x is the most significant axis
        }
        keys[r] = key;
        vals[r] = (uint32_t)r;
    }
}

// Length of the common prefix of the (key, position) pairs at sorted positions i, j.
__device__ __forceinline__ int delta(const uint64_t* __restrict__ keys, int64_t F, int64_t i, int64_t j)
{
    if (j < 0 || j >= F) return -1;
    const uint64_t ki = keys[i], kj = keys[j];
    if (ki == kj) return 64 + __clz((unsigned)(i ^ j));
    return __clzll((long long)(ki ^ kj));
}

// Binary radix tree: internal node i covers a range of sorted leaves that has i at one end.
// node words: [0..5] box of child 0, [6..11] box of child 1, [12] child0, [13] child1, [14] parent.
__global__ void __launch_bounds__(BT)
radix_tree_kernel(const uint64_t* __restrict__ keys, int64_t F, int32_t* __restrict__ node_words,
                  int32_t* __restrict__ leaf_parent)
{
    const int64_t i = (int64_t)blockIdx.x * BT + threadIdx.x;
    if (i >= F - 1) return;
    const int d = (delta(keys, F, i, i + 1) - delta(keys, F, i, i - 1)) >= 0 ? 1 : -1;
    const int dmin = delta(keys, F, i, i - d);
    int64_t lmax = 2;
    while (delta(keys, F, i, i + lmax * d) > dmin) lmax *= 2;
    int64_t l = 0;
    for (int64_t t = lmax / 2; t >= 1; t /= 2)
        if (delta(keys, F, i, i + (l + t) * d) > dmin) l += t;
    const int64_t j = i + l * d;
    const int dnode = delta(keys, F, i, j);
    int64_t s = 0, t = l;
    do {
        t = (t + 1) / 2;
        if (delta(keys, F, i, i + (s + t) * d) > dnode) s += t;
    } while (t > 1);
    const int64_t gamma = i + s * d + (d < 0 ? -1 : 0);
    const int64_t lo = i < j ? i : j, hi = i < j ? j : i;
    int32_t* w = node_words + 16 * i;
    if (lo == gamma) { w[12] = ~(int32_t)gamma; leaf_parent[gamma] = (int32_t)i; }
    else             { w[12] = (int32_t)gamma;  node_words[16 * gamma + 14] = (int32_t)i; }
    if (hi == gamma + 1) { w[13] = ~(int32_t)(gamma + 1); leaf_parent[gamma + 1] = (int32_t)i; }
    else                 { w[13] = (int32_t)(gamma + 1);  node_words[16 * (gamma + 1) + 14] = (int32_t)i; }
    if (i == 0) w[14] = -1;
    w[15] = 0;
}

// Pack the sorted leaf references and refit boxes bottom-up.  The second thread to reach
// a node owns it (arrival counter), reads both child boxes and carries their
// union to the parent.  Leaf k holds the WHOLE triangle of its face (PackedTri) and the box of its slab.
__global__ void __launch_bounds__(BT)
pack_refit_kernel(const float* __restrict__ verts, const int32_t* __restrict__ faces, int64_t R,
                  const uint32_t* __restrict__ sorted_ref, const int32_t* __restrict__ ref_face, const float* __restrict__ ref_box,
                  const uint32_t* __restrict__ offs, const int32_t* __restrict__ leaf_parent,
                  int32_t* node_words, int* __restrict__ arrivals, PackedTri* __restrict__ tris,
                  int32_t* __restrict__ leaf_tri, int32_t* __restrict__ face_slot, BuildScratch* sc)
{
    const int64_t k = (int64_t)blockIdx.x * BT + threadIdx.x;
    if (k >= R) return;
    const uint32_t ref = sorted_ref[k];
    const int32_t f = ref_face[ref];
    leaf_tri[k] = f;
    atomicMin(&face_slot[f], (int32_t)k);           // the first (in Morton order) leaf of the face: deterministic
    float p[3][3];
    for (int v = 0; v < 3; ++v)
        for (int d = 0; d < 3; ++d) p[v][d] = verts[3 * (int64_t)faces[3 * (int64_t)f + v] + d];
    PackedTri t;
    {
        const double abx = (double)p[1][0] - p[0][0], aby = (double)p[1][1] - p[0][1], abz = (double)p[1][2] - p[0][2];
        const double acx = (double)p[2][0] - p[0][0], acy = (double)p[2][1] - p[0][1], acz = (double)p[2][2] - p[0][2];
        const float nx = (float)(aby * acz - abz * acy), ny = (float)(abz * acx - abx * acz), nz = (float)(abx * acy - aby * acx);
        const float nn = nx * nx + ny * ny + nz * nz;
        const float e2 = fmaxf((float)(abx * abx + aby * aby + abz * abz), (float)(acx * acx + acy * acy + acz * acz));
        const bool degenerate = !(nn > 1e-12f * e2 * e2) || !(nn > 0.0f) || !isfinite(1.0f / nn);
        const int flags = (degenerate ? 1 : 0) | (ref != offs[f] ? 2 : 0);   // bit 1: not the face's first reference
        t.t0 = make_float4(p[0][0], p[0][1], p[0][2], __int_as_float(f));
        t.t1 = make_float4(p[1][0], p[1][1], p[1][2], degenerate ? 0.0f : nn);
        t.t2 = make_float4(p[2][0], p[2][1], p[2][2], degenerate ? 0.0f : 1.0f / nn);
        t.t3 = make_float4(nx, ny, nz, __int_as_float(flags));
    }
    tris[k] = t;
    float box[6];
    for (int q = 0; q < 6; ++q) box[q] = ref_box[6 * (int64_t)ref + q];
    if (R == 1) {                                   // single leaf: node 0 holds it twice
        float* w = reinterpret_cast<float*>(node_words);
        for (int c = 0; c < 2; ++c) for (int q = 0; q < 6; ++q) w[6 * c + q] = box[q];
        node_words[12] = ~0; node_words[13] = ~0; node_words[14] = -1; node_words[15] = 0;
        sc->max_depth = 1;
        return;
    }
    int32_t child = ~(int32_t)k;
    int32_t node = leaf_parent[k];
    int depth = 1;
    for (;;) {
        volatile float* w = reinterpret_cast<volatile float*>(node_words + 16 * (int64_t)node);
        volatile int32_t* wi = reinterpret_cast<volatile int32_t*>(node_words + 16 * (int64_t)node);
        const int side = (wi[12] == child) ? 0 : 1;
        for (int q = 0; q < 6; ++q) w[6 * side + q] = box[q];
        __threadfence();
        const int old = atomicAdd(&arrivals[node], 1);
        if (old == 0) return;                       // first arrival: the sibling will carry on
        __threadfence();
        const int other = 1 - side;
        for (int d = 0; d < 3; ++d) {
            box[d] = fminf(box[d], w[6 * other + d]);
            box[3 + d] = fmaxf(box[3 + d], w[6 * other + 3 + d]);
        }
        const int32_t parent = wi[14];
        if (parent < 0) return;                     // root done
        child = node;
        node = parent;
        ++depth;
    }
}

// Surface-area cost of the packed tree (a quality readout, mcs_bvh_info_t.sah_cost): sum over all child slots of
// area(box) x (1 for an inner child, C_LEAF for a leaf), to be divided by the area of the root box: the expected
// number of box tests plus C_LEAF x triangle tests of a random line -- the usual proxy for query cost.
constexpr double SAH_C_LEAF = 80.0 / 18.0;          // flop model of DESIGN.md section 6: triangle test / box test
__global__ void __launch_bounds__(BT)
sah_partial_kernel(const int32_t* __restrict__ node_words, int64_t n_nodes, double* __restrict__ partials)
{
    __shared__ double s_c[BT];
    const int64_t i = (int64_t)blockIdx.x * BT + threadIdx.x;
    double c = 0.0;
    if (i < n_nodes) {
        const float* w = reinterpret_cast<const float*>(node_words + 16 * i);
        for (int side = 0; side < 2; ++side) {
            const double ex = (double)w[6 * side + 3] - w[6 * side], ey = (double)w[6 * side + 4] - w[6 * side + 1], ez = (double)w[6 * side + 5] - w[6 * side + 2];
            const double sa = 2.0 * (ex * ey + ey * ez + ez * ex);
            c += node_words[16 * i + 12 + side] < 0 ? SAH_C_LEAF * sa : sa;
        }
    }
    s_c[threadIdx.x] = c;
    __syncthreads();
    for (int s = BT / 2; s > 0; s >>= 1) {          // fixed-shape tree: deterministic
        if (threadIdx.x < s) s_c[threadIdx.x] += s_c[threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x == 0) partials[blockIdx.x] = s_c[0];
}

__global__ void __launch_bounds__(BT)
depth_kernel(const int32_t* __restrict__ node_words, const int32_t* __restrict__ leaf_parent, int64_t F, BuildScratch* sc)
{
    const int64_t k = (int64_t)blockIdx.x * BT + threadIdx.x;
    int depth = 0;
    if (k < F && F > 1) {
        depth = 1;
        int32_t node = leaf_parent[k];
        while (node_words[16 * (int64_t)node + 14] >= 0) { node = node_words[16 * (int64_t)node + 14]; ++depth; }
    }
    for (int o = 16; o > 0; o >>= 1) depth = max(depth, __shfl_xor_sync(0xFFFFFFFFu, depth, o));
    if ((threadIdx.x & 31) == 0 && depth > 0) atomicMax(&sc->max_depth, depth);
}

// ---------------------------------------------------------------------------
// 4-wide collapse for the walk kernel: binary nodes at even depth become wide nodes.
// ---------------------------------------------------------------------------
__global__ void __launch_bounds__(BT)
even_depth_kernel(const int32_t* __restrict__ node_words, int64_t n_nodes, uint32_t* __restrict__ even)
{
    const int64_t i = (int64_t)blockIdx.x * BT + threadIdx.x;
    if (i >= n_nodes) return;
    int depth = 0;
    for (int32_t p = node_words[16 * i + 14]; p >= 0; p = node_words[16 * (int64_t)p + 14]) ++depth;
    even[i] = (depth & 1) ? 0u : 1u;
}

__global__ void __launch_bounds__(BT)
wide_pack_kernel(const int32_t* __restrict__ node_words, int64_t n_nodes, const uint32_t* __restrict__ even,
                 const uint32_t* __restrict__ widx, WideNode* __restrict__ wide)
{
    const int64_t i = (int64_t)blockIdx.x * BT + threadIdx.x;
    if (i >= n_nodes || !even[i]) return;
    const float* fw = reinterpret_cast<const float*>(node_words);
    WideNode w;
    int n = 0;
    for (int side = 0; side < 2; ++side) {
        const int32_t c = node_words[16 * i + 12 + side];
        if (c < 0) {                                           // leaf child: its box is stored in i
            for (int q = 0; q < 6; ++q) w.f[6 * n + q] = fw[16 * i + 6 * side + q];
            w.c[n++] = c;
        } else {                                               // inner child at odd depth: take its two children
            for (int s2 = 0; s2 < 2; ++s2) {
                const int32_t g = node_words[16 * (int64_t)c + 12 + s2];
                for (int q = 0; q < 6; ++q) w.f[6 * n + q] = fw[16 * (int64_t)c + 6 * s2 + q];
                w.c[n++] = g < 0 ? g : (int32_t)widx[g];
            }
        }
    }
    for (; n < 4; ++n) {
        for (int q = 0; q < 3; ++q) { w.f[6 * n + q] = CUDART_INF_F; w.f[6 * n + 3 + q] = -CUDART_INF_F; }
        w.c[n] = INT_MIN;
    }
    for (int k = 0; k < 4; ++k) {                                  // squared diagonal of every child box (far-field test of the walk kernel)
        const float ex = w.f[6 * k + 3] - w.f[6 * k], ey = w.f[6 * k + 4] - w.f[6 * k + 1], ez = w.f[6 * k + 5] - w.f[6 * k + 2];
        const float g = w.c[k] == INT_MIN ? CUDART_INF_F : (ex * ex + ey * ey + ez * ez) * (1.0f + 4e-7f);   // rounded up
        w.pad[k] = __float_as_int(g);
    }
    wide[widx[i]] = w;
}

}  // namespace

// Device memory of a tree comes from the device's stream-ordered pool (cudaMallocAsync) with the release threshold
// raised, so that building and freeing a tree per mesh (BASELINE config 4: 1024 meshes) recycles the same memory
// instead of going to the driver: cudaFree blocks the host, measured at up to 0.5 s per call on this pool's boxes.
static void keep_pool_memory()
{
    int dev = 0; cudaMemPool_t pool;
    if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetDefaultMemPool(&pool, dev) == cudaSuccess) {
        unsigned long long keep = ~0ull;
        cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
        // Memory freed on one stream may be handed to an allocation on another only when that free has COMPLETED
        // (opportunistic reuse), never by making the allocating stream wait for it: with several meshes in flight on
        // their own streams (mcs_estimate_dtn_batch) such inserted dependencies serialised the workers.
        int off = 0;
        cudaMemPoolSetAttribute(pool, cudaMemPoolReuseAllowInternalDependencies, &off);
    }
}

void mcs_bvh_touch(const mcs_bvh* b, cudaStream_t st)
{
    if (!b || !b->last_use) return;
    // Under stream capture the record would become a node of the caller's graph and the event could no longer order
    // mcs_free_bvh: skip it (the caller keeps the handle alive for as long as the graph may run, include/mcdtn.h).
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(st, &cs) != cudaSuccess) { (void)cudaGetLastError(); return; }
    if (cs == cudaStreamCaptureStatusNone) cudaEventRecord(b->last_use, st);
}

// Frees the handle's memory in the order of `st`, which must be a stream the handle's last use is ordered before
// (the batch workers and the host entry points free on the stream they worked on: no detour through stream 0).
void mcs_free_bvh_on(mcs_bvh* b, cudaStream_t st)
{
    if (!b) return;
    int cur = 0;
    cudaGetDevice(&cur);
    if (cur != b->device) cudaSetDevice(b->device);
    if (b->last_use) cudaStreamWaitEvent(st, b->last_use, 0);
    void* ptrs[11] = { b->verts, b->faces, b->nodes, b->wide, b->tris, b->leaf_tri, b->face_slot, b->morton,
                       b->wn_nodes, b->wn_order, b->wn_face_pos };
    for (void* p : ptrs) if (p) cudaFreeAsync(p, st);
    if (b->last_use) cudaEventDestroy(b->last_use);
    if (cur != b->device) cudaSetDevice(cur);
    delete b;
}

extern "C" void mcs_free_bvh(mcs_bvh* b)
{
    if (!b) return;
    int cur = 0;
    cudaGetDevice(&cur);
    if (cur != b->device) cudaSetDevice(b->device);
    // The memory goes back to the pool in the order of the legacy default stream, which is first made to wait for the
    // last call that used the handle: stream 0 orders itself after BLOCKING streams only, and PyTorch's side streams
    // (like this library's own) are non-blocking, so without the event a kernel still queued on such a stream could
    // read the tree after the pool had handed its memory to someone else.
    if (b->last_use) cudaStreamWaitEvent((cudaStream_t)0, b->last_use, 0);
    void* ptrs[11] = { b->verts, b->faces, b->nodes, b->wide, b->tris, b->leaf_tri, b->face_slot, b->morton,
                       b->wn_nodes, b->wn_order, b->wn_face_pos };
    for (void* p : ptrs) if (p) cudaFreeAsync(p, (cudaStream_t)0);
    if (b->last_use) cudaEventDestroy(b->last_use);
    if (cur != b->device) cudaSetDevice(cur);
    delete b;
}

extern "C" int mcs_build_bvh(const float* verts, int64_t V, const int32_t* faces, int64_t F,
                             const mcs_build_opts* opts, void* stream, mcs_bvh** out)
{
    if (!out) return MCS_EINVAL;
    *out = nullptr;
    if (!verts || !faces || V < 1 || F < 1 || V >= (int64_t)1 << 31 || F >= (int64_t)1 << 30) return MCS_EINVAL;
    const bool split = !(opts && opts->no_split);
    const int max_pieces = (opts && opts->max_pieces > 0) ? opts->max_pieces : 64;
    const float split_length = (opts && opts->split_length > 0.0f) ? opts->split_length : 4.0f;
    const float split_budget = (opts && opts->split_budget > 0.0f) ? opts->split_budget : 1.0f;
    if (opts && (opts->max_pieces < 0 || opts->max_pieces > 1024 || opts->split_length < 0.0f || opts->split_budget < 0.0f)) return MCS_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    mcs_bvh* b = new (std::nothrow) mcs_bvh();
    if (!b) return MCS_ENOMEM;
    b->V = V; b->F = F; b->root = 0;
    cudaGetDevice(&b->device);

    const size_t nb_verts = (size_t)V * 3 * sizeof(float), nb_faces = (size_t)F * 3 * sizeof(int32_t);
    BuildScratch* sc = nullptr; double* partials = nullptr; uint32_t* vals = nullptr; uint32_t* counts = nullptr;
    int32_t* leaf_parent = nullptr; int* arrivals = nullptr; void* sort_ws = nullptr; void* scan_ws = nullptr;
    int32_t* ref_face = nullptr; float* ref_box = nullptr; double* sah_partials = nullptr;
    const int nblk = (int)ceil_div64(F, BT);
    int rc = MCS_OK;
    int64_t R = F;                                        // leaf references
    float unit = 0.0f;                                    // piece length of the sliver splitting (0: none)
    size_t nb_nodes = 0, nb_tris = 0, sort_bytes = 0;
    int nblk_r = 0, nblk_n = 0;
    cudaError_t e = cudaSuccess;
    keep_pool_memory();
    if (cudaEventCreateWithFlags(&b->last_use, cudaEventDisableTiming) != cudaSuccess) b->last_use = nullptr;
#define ALLOC(ptr, bytes) if (e == cudaSuccess) e = cudaMallocAsync((void**)&(ptr), (bytes), st)
    ALLOC(b->verts, nb_verts); ALLOC(b->faces, nb_faces); ALLOC(b->face_slot, (size_t)F * 4);
    ALLOC(sc, sizeof(BuildScratch) + 512); ALLOC(partials, (size_t)nblk * 8);
    ALLOC(counts, (size_t)(F + 1) * 4); ALLOC(scan_ws, scan_workspace_bytes(F) + 256);
    BuildScratch h;
    if (e != cudaSuccess) { rc = (e == cudaErrorMemoryAllocation) ? MCS_ENOMEM : MCS_ECUDA; mcs_set_last_cuda_error((int)e); goto done; }

    cudaMemcpyAsync(b->verts, verts, nb_verts, cudaMemcpyDeviceToDevice, st);
    cudaMemcpyAsync(b->faces, faces, nb_faces, cudaMemcpyDeviceToDevice, st);
    memset(&h, 0, sizeof h);
    for (int d = 0; d < 3; ++d) { h.lo[d] = 0x7FFFFFFF; h.hi[d] = (int)0x80000000; }
    cudaMemcpyAsync(sc, &h, sizeof h, cudaMemcpyHostToDevice, st);
    cudaMemsetAsync((char*)sc + sizeof(BuildScratch), 0, 512, st);                 // histogram + scratch words

    mcs_note_launch(), face_bounds_kernel<<<nblk, BT, 0, st>>>(b->verts, V, b->faces, F, sc, partials);
    mcs_note_launch(), area_total_kernel<<<1, 1, 0, st>>>(partials, nblk, sc);
    unsigned int hist[SPLIT_BINS];
    {
        unsigned int* hist_dev = (unsigned int*)((char*)sc + sizeof(BuildScratch));
        e = cudaMemcpyAsync(&h, sc, sizeof h, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) { rc = MCS_ECUDA; mcs_set_last_cuda_error((int)e); goto done; }
        if (h.flags & 1) { rc = MCS_EINVAL; goto done; }
        if ((h.flags & 2) || !(h.area > 0.0)) { rc = MCS_EDEGENERATE; goto done; }
        // ---- sliver splitting: piece length = split_length mean edge lengths, raised until the budget holds
        const float mean_edge = (float)sqrt(2.0 * h.area / (double)F);            // edge of a triangle of the mean area
        if (split && F > 1 && mean_edge > 0.0f) {
            mcs_note_launch(), split_hist_kernel<<<nblk, BT, 0, st>>>(b->verts, b->faces, F, mean_edge, hist_dev);
            e = cudaMemcpyAsync(hist, hist_dev, sizeof hist, cudaMemcpyDeviceToHost, st);
            if (e == cudaSuccess) e = cudaStreamSynchronize(st);
            if (e != cudaSuccess) { rc = MCS_ECUDA; mcs_set_last_cuda_error((int)e); goto done; }
            double m = split_length;
            for (int it = 0; it < 96; ++it, m *= 1.189207115) {                   // quarter octaves
                double extra = 0.0;
                for (int bin = 0; bin < SPLIT_BINS; ++bin) {
                    if (!hist[bin]) continue;
                    const double q_hi = pow(2.0, (bin + 1) / 4.0);                  // upper edge of the bin: an over-estimate
                    double n = ceil(q_hi / m);
                    if (bin == SPLIT_BINS - 1 || n > max_pieces) n = max_pieces;
                    if (q_hi > m && n > 1.0) extra += (n - 1.0) * hist[bin];
                }
                if (extra <= (double)split_budget * (double)F) break;
            }
            unit = (float)(m * mean_edge);
        }
    }
    mcs_note_launch(), split_count_kernel<<<nblk, BT, 0, st>>>(b->verts, b->faces, F, unit, max_pieces, counts);
    {
        uint32_t total = 0;
        rc = exclusive_scan_u32(counts, counts, F, counts + F, scan_ws, scan_workspace_bytes(F) + 256, st);
        if (rc != MCS_OK) goto done;
        e = cudaMemcpyAsync(&total, counts + F, 4, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) { rc = MCS_ECUDA; mcs_set_last_cuda_error((int)e); goto done; }
        R = (int64_t)total;
        if (R < F || R >= (int64_t)1 << 30) { rc = MCS_ECUDA; goto done; }
    }
    b->n_leaves = R;
    b->n_nodes = R > 1 ? R - 1 : 1;
    nb_nodes = (size_t)b->n_nodes * sizeof(BvhNode); nb_tris = (size_t)R * sizeof(PackedTri);
    sort_bytes = sort_workspace_bytes(R, 8);
    nblk_r = (int)ceil_div64(R, BT); nblk_n = (int)ceil_div64(b->n_nodes, BT);
    ALLOC(b->nodes, nb_nodes); ALLOC(b->tris, nb_tris); ALLOC(b->leaf_tri, (size_t)R * 4); ALLOC(b->morton, (size_t)R * 8);
    ALLOC(vals, (size_t)R * 4); ALLOC(leaf_parent, (size_t)R * 4); ALLOC(arrivals, (size_t)b->n_nodes * 4);
    ALLOC(ref_face, (size_t)R * 4); ALLOC(ref_box, (size_t)R * 24); ALLOC(sort_ws, sort_bytes); ALLOC(sah_partials, (size_t)nblk_n * 8);
#undef ALLOC
    if (e != cudaSuccess) { rc = (e == cudaErrorMemoryAllocation) ? MCS_ENOMEM : MCS_ECUDA; mcs_set_last_cuda_error((int)e); goto done; }
    b->device_bytes = nb_verts + nb_faces + nb_nodes + nb_tris + (size_t)R * 12 + (size_t)F * 4;
    cudaMemsetAsync(arrivals, 0, (size_t)b->n_nodes * 4, st);
    cudaMemsetAsync(b->nodes, 0, nb_nodes, st);
    cudaMemsetAsync(b->face_slot, 0x7F, (size_t)F * 4, st);                        // atomicMin target

    mcs_note_launch(), ref_emit_kernel<<<nblk, BT, 0, st>>>(b->verts, b->faces, F, unit, max_pieces, counts, sc, ref_face, ref_box, b->morton, vals);
    rc = sort_pairs_u64(b->morton, vals, R, 63, sort_ws, sort_bytes, st);
    if (rc != MCS_OK) goto done;
    if (R > 1)
        mcs_note_launch(), radix_tree_kernel<<<(int)ceil_div64(R - 1, BT), BT, 0, st>>>(b->morton, R, (int32_t*)b->nodes, leaf_parent);
    mcs_note_launch(), pack_refit_kernel<<<nblk_r, BT, 0, st>>>(b->verts, b->faces, R, vals, ref_face, ref_box, counts, leaf_parent,
                                             (int32_t*)b->nodes, arrivals, b->tris, b->leaf_tri, b->face_slot, sc);
    mcs_note_launch(), depth_kernel<<<nblk_r, BT, 0, st>>>((const int32_t*)b->nodes, leaf_parent, R, sc);
    {   // surface-area cost readout (one double per block, summed in order by one thread into sc->area)
        mcs_note_launch(), sah_partial_kernel<<<nblk_n, BT, 0, st>>>((const int32_t*)b->nodes, b->n_nodes, sah_partials);
        const double area_keep = h.area;
        mcs_note_launch(), area_total_kernel<<<1, 1, 0, st>>>(sah_partials, nblk_n, sc);
        e = cudaMemcpyAsync(&h, sc, sizeof h, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e == cudaSuccess) e = cudaGetLastError();
        if (e != cudaSuccess) { rc = MCS_ECUDA; mcs_set_last_cuda_error((int)e); goto done; }
        double ext[3];
        for (int d = 0; d < 3; ++d) {
            int lo = h.lo[d], hi = h.hi[d];
            lo = lo >= 0 ? lo : lo ^ 0x7FFFFFFF; hi = hi >= 0 ? hi : hi ^ 0x7FFFFFFF;
            float flo, fhi; memcpy(&flo, &lo, 4); memcpy(&fhi, &hi, 4);
            ext[d] = (double)fhi - (double)flo;
        }
        const double root_sa = 2.0 * (ext[0] * ext[1] + ext[1] * ext[2] + ext[2] * ext[0]);
        b->sah_cost = root_sa > 0.0 ? h.area / root_sa : 0.0;                      // h.area holds the cost sum here
        h.area = area_keep;
    }
    {   // 4-wide collapse (binary nodes at even depth), compacted with a prefix sum
        uint32_t* even = (uint32_t*)arrivals;                  // arrivals are done: reuse as flags
        uint32_t* widx = vals;                                 // sorted reference ids are packed: reuse (n_nodes <= R)
        uint32_t n_wide = 0;
        mcs_note_launch(), even_depth_kernel<<<nblk_n, BT, 0, st>>>((const int32_t*)b->nodes, b->n_nodes, even);
        uint32_t* total_dev = (uint32_t*)((char*)sc + sizeof(BuildScratch) + 256);   // scratch word behind the histogram
        rc = exclusive_scan_u32(even, widx, b->n_nodes, total_dev, sort_ws, sort_bytes, st);
        if (rc != MCS_OK) goto done;
        e = cudaMemcpyAsync(&n_wide, total_dev, 4, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e == cudaSuccess) e = cudaMallocAsync((void**)&b->wide, (size_t)(n_wide ? n_wide : 1) * sizeof(WideNode), st);
        if (e != cudaSuccess) { rc = (e == cudaErrorMemoryAllocation) ? MCS_ENOMEM : MCS_ECUDA; mcs_set_last_cuda_error((int)e); goto done; }
        b->n_wide = n_wide;
        b->device_bytes += (size_t)n_wide * sizeof(WideNode);
        mcs_note_launch(), wide_pack_kernel<<<nblk_n, BT, 0, st>>>((const int32_t*)b->nodes, b->n_nodes, even, widx, b->wide);
        e = cudaStreamSynchronize(st);
        if (e == cudaSuccess) e = cudaGetLastError();
        if (e != cudaSuccess) { rc = MCS_ECUDA; mcs_set_last_cuda_error((int)e); goto done; }
    }
    b->max_depth = h.max_depth;
    b->n_degenerate = h.n_degenerate;
    b->area = h.area;
    for (int d = 0; d < 3; ++d) {
        int lo = h.lo[d], hi = h.hi[d];
        lo = lo >= 0 ? lo : lo ^ 0x7FFFFFFF; hi = hi >= 0 ? hi : hi ^ 0x7FFFFFFF;
        memcpy(&b->aabb_lo[d], &lo, 4); memcpy(&b->aabb_hi[d], &hi, 4);
    }
done:
    { void* tmp[11] = { sc, partials, vals, counts, leaf_parent, arrivals, sort_ws, scan_ws, ref_face, ref_box, sah_partials }; for (void* p : tmp) if (p) cudaFreeAsync(p, st); }
    if (rc != MCS_OK) { mcs_free_bvh(b); return rc; }
    mcs_bvh_touch(b, st);
    *out = b;
    return MCS_OK;
}

extern "C" int mcs_bvh_info(const mcs_bvh* b, mcs_bvh_info_t* o)
{
    if (!b || !o) return MCS_EINVAL;
    o->V = b->V; o->F = b->F; o->n_nodes = b->n_nodes; o->max_depth = b->max_depth;
    o->n_leaves = b->n_leaves; o->sah_cost = b->sah_cost;
    o->n_degenerate = b->n_degenerate;
    for (int d = 0; d < 3; ++d) { o->aabb_lo[d] = b->aabb_lo[d]; o->aabb_hi[d] = b->aabb_hi[d]; }
    o->area = b->area; o->device_bytes = b->device_bytes;
    return MCS_OK;
}

extern "C" int mcs_bvh_dump(const mcs_bvh* b, uint32_t* nodes, int32_t* leaf_tri, uint64_t* morton, void* stream)
{
    if (!b) return MCS_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    if (nodes) MCS_CUDA_TRY(cudaMemcpyAsync(nodes, b->nodes, (size_t)b->n_nodes * sizeof(BvhNode), cudaMemcpyDeviceToDevice, st));
    if (leaf_tri) MCS_CUDA_TRY(cudaMemcpyAsync(leaf_tri, b->leaf_tri, (size_t)b->n_leaves * 4, cudaMemcpyDeviceToDevice, st));
    if (morton) MCS_CUDA_TRY(cudaMemcpyAsync(morton, b->morton, (size_t)b->n_leaves * 8, cudaMemcpyDeviceToDevice, st));
    MCS_CUDA_TRY(cudaStreamSynchronize(st));
    return MCS_OK;
}
