// winding.cu -- generalised winding number of the mesh at query points, and the sidedness of boundary samples
// ("we repair normals using generalized winding numbers"; DESIGN.md G-R1).
//     w(p) = (1 / 4 pi) sum_f Omega_f(p),
//     tan(Omega_f / 2) = a.(b x c) / (|a||b||c| + (a.b)|c| + (b.c)|a| + (c.a)|b|),   a, b, c = vertices - p
// (Van Oosterom & Strackee 1983).  The sum is exhaustive: every (point, face) pair is evaluated -- an all-pairs
// kernel, compute-bound (about 60 flops and one atan2 per pair against 48 bytes per face per 128 points).  A block
// holds 128 query points in registers (one per thread) and streams its chunk of the faces through shared memory in
// tiles of 128; faces are split in chunks over blockIdx.y so that a handful of points still fills the device; the
// per-chunk partial sums (compensated fp32) are added in chunk order in fp64: deterministic.
#include "common.cuh"
#include "traverse.cuh"

#include <mutex>

namespace {

constexpr int WQ = 128;           // query points per block = faces per tile

__global__ void __launch_bounds__(WQ)
winding_partial_kernel(const float* __restrict__ verts, const int32_t* __restrict__ faces, long long F, const float* __restrict__ pts,
                       const int32_t* __restrict__ exclude, long long n, long long faces_per_chunk,
                       float* __restrict__ partial)
{
    __shared__ float4 sA[WQ], sB[WQ], sC[WQ];
    const long long q = (long long)blockIdx.x * WQ + threadIdx.x;
    const bool live = q < n;
    const float px = live ? pts[3 * q] : 0.0f, py = live ? pts[3 * q + 1] : 0.0f, pz = live ? pts[3 * q + 2] : 0.0f;
    const int ex = (live && exclude) ? exclude[q] : -1;
    const long long f0 = (long long)blockIdx.y * faces_per_chunk;
    const long long f1 = f0 + faces_per_chunk < F ? f0 + faces_per_chunk : F;
    float sum = 0.0f, comp = 0.0f;                                    // Kahan: a chunk holds up to ~10^5 terms
    for (long long t0 = f0; t0 < f1; t0 += WQ) {
        const long long k = t0 + threadIdx.x;
        if (k < f1) {                                                 // every face once, from the mesh itself (the tree's
            const long long i0 = faces[3 * k], i1 = faces[3 * k + 1], i2 = faces[3 * k + 2];   // leaves hold split faces several times)
            sA[threadIdx.x] = make_float4(verts[3 * i0], verts[3 * i0 + 1], verts[3 * i0 + 2], __int_as_float((int)k));
            sB[threadIdx.x] = make_float4(verts[3 * i1], verts[3 * i1 + 1], verts[3 * i1 + 2], 0.0f);
            sC[threadIdx.x] = make_float4(verts[3 * i2], verts[3 * i2 + 1], verts[3 * i2 + 2], 0.0f);
        }
        __syncthreads();
        const int cnt = (int)((f1 - t0) < WQ ? (f1 - t0) : WQ);
#pragma unroll 4
        for (int j = 0; j < cnt; ++j) {
            const float4 A = sA[j], B = sB[j], C = sC[j];             // broadcast reads
            const float ax = A.x - px, ay = A.y - py, az = A.z - pz;
            const float bx = B.x - px, by = B.y - py, bz = B.z - pz;
            const float cx = C.x - px, cy = C.y - py, cz = C.z - pz;
            const float la = sqrtf(fmaf(ax, ax, fmaf(ay, ay, az * az)));
            const float lb = sqrtf(fmaf(bx, bx, fmaf(by, by, bz * bz)));
            const float lc = sqrtf(fmaf(cx, cx, fmaf(cy, cy, cz * cz)));
            const float det = ax * (by * cz - bz * cy) - ay * (bx * cz - bz * cx) + az * (bx * cy - by * cx);
            const float ab = fmaf(ax, bx, fmaf(ay, by, az * bz));
            const float bc = fmaf(bx, cx, fmaf(by, cy, bz * cz));
            const float ca = fmaf(cx, ax, fmaf(cy, ay, cz * az));
            const float den = fmaf(la * lb, lc, fmaf(ab, lc, fmaf(bc, la, ca * lb)));
            float om = atan2f(det, den);
            if (__float_as_int(A.w) == ex) om = 0.0f;                 // the excluded face (original index in A.w)
            const float y = om - comp, s2 = sum + y;
            comp = (s2 - sum) - y; sum = s2;
        }
        __syncthreads();
    }
    if (live) partial[(long long)blockIdx.y * n + q] = sum;
}

__global__ void winding_reduce_kernel(const float* __restrict__ partial, long long n, int n_chunks, float* __restrict__ w)
{
    const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= n) return;
    double s = 0.0;
    for (int c = 0; c < n_chunks; ++c) s += (double)partial[(long long)c * n + q];
    w[q] = (float)(s * (2.0 / (4.0 * 3.14159265358979323846)));     // Omega = 2 atan2(...), w = sum Omega / 4 pi
}

// back and front probe points of every sample: s -/+ h n_f, h = h_scale sqrt(area_f); both exclude the sample's face
__global__ void orient_points_kernel(const float* __restrict__ verts, const int32_t* __restrict__ faces, long long F,
                                     const int32_t* __restrict__ tri, const float* __restrict__ bary, long long n,
                                     float h_scale, float* __restrict__ pts, int32_t* __restrict__ excl,
                                     float* __restrict__ normal_out, int* __restrict__ err)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int f = tri[i];
    if (f < 0 || f >= F) { *err = 1; return; }
    const int i0 = faces[3 * f], i1 = faces[3 * f + 1], i2 = faces[3 * f + 2];
    const float3 a = f3(verts[3 * i0], verts[3 * i0 + 1], verts[3 * i0 + 2]);
    const float3 b = f3(verts[3 * i1], verts[3 * i1 + 1], verts[3 * i1 + 2]);
    const float3 c = f3(verts[3 * i2], verts[3 * i2 + 1], verts[3 * i2 + 2]);
    const float b0 = bary[3 * i], b1 = bary[3 * i + 1], b2 = bary[3 * i + 2];
    const float3 s = f3(b0 * a.x + b1 * b.x + b2 * c.x, b0 * a.y + b1 * b.y + b2 * c.y, b0 * a.z + b1 * b.z + b2 * c.z);
    float3 nr = cross3(b - a, c - a);
    const float nn = sqrtf(dot3(nr, nr));
    const float inv = nn > 0.0f ? 1.0f / nn : 0.0f;
    nr = inv * nr;
    const float h = h_scale * sqrtf(0.5f * nn);
    pts[6 * i] = s.x - h * nr.x; pts[6 * i + 1] = s.y - h * nr.y; pts[6 * i + 2] = s.z - h * nr.z;
    pts[6 * i + 3] = s.x + h * nr.x; pts[6 * i + 4] = s.y + h * nr.y; pts[6 * i + 5] = s.z + h * nr.z;
    excl[2 * i] = f; excl[2 * i + 1] = f;
    normal_out[3 * i] = nr.x; normal_out[3 * i + 1] = nr.y; normal_out[3 * i + 2] = nr.z;
}

__global__ void orient_finish_kernel(const float* __restrict__ w, long long n, float* __restrict__ normal_out, float* __restrict__ d_out)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float d = w[2 * i] - w[2 * i + 1];                          // back minus front
    if (d_out) d_out[i] = d;
    if (d < 0.0f) { normal_out[3 * i] = -normal_out[3 * i]; normal_out[3 * i + 1] = -normal_out[3 * i + 1]; normal_out[3 * i + 2] = -normal_out[3 * i + 2]; }
}

int winding_chunks(long long F, long long n)
{
    const long long q_blocks = ceil_div64(n, WQ);
    long long want = ceil_div64(4 * 148, q_blocks);                   // about four blocks per SM
    const long long most = ceil_div64(F, 4 * WQ);                     // at least four tiles per chunk
    if (want > most) want = most;
    if (want > 1024) want = 1024;
    return (int)(want < 1 ? 1 : want);
}

size_t partial_bytes(long long F, long long n) { return (size_t)winding_chunks(F, n) * (size_t)n * 4; }

int winding_run(const mcs_bvh* b, const float* pts, const int32_t* excl, long long n, float* w, float* partial, cudaStream_t st)
{
    const int n_chunks = winding_chunks(b->F, n);
    const long long fpc = ceil_div64(ceil_div64(b->F, n_chunks), WQ) * WQ;
    const dim3 grid((unsigned)ceil_div64(n, WQ), (unsigned)n_chunks);
    mcs_note_launch(), winding_partial_kernel<<<grid, WQ, 0, st>>>(b->verts, b->faces, b->F, pts, excl, n, fpc, partial);
    mcs_note_launch(), winding_reduce_kernel<<<(unsigned)ceil_div64(n, 256), 256, 0, st>>>(partial, n, n_chunks, w);
    mcs_bvh_touch(b, st);
    MCS_CUDA_TRY(cudaGetLastError());
    return MCS_OK;
}

// ---------------------------------------------------------------------------
// Hierarchical evaluation for the sidedness decision (mcs_orient_samples_fast).
//
// d_i = w_-f(s - h n) - w_-f(s + h n) is a difference of the winding number at two points 2h apart, so only the
// surface NEAR the sample decides it; far parts contribute almost the same solid angle to both probes.  The faces
// are sorted along a Z-order curve and cut into groups of 32; a complete binary tree over the groups stores for
// every node the sum of its area vectors N = sum (b-a)x(c-a)/2, its area-weighted centroid c and the radius R of a
// ball about c that holds its faces.  Seen from a point p farther than beta R from c, a node is replaced by its
// dipole, Omega ~ N.(c - p) / |c - p|^3 (first term of the multipole expansion of the solid angle; Barill et al.
// 2018 use the same hierarchy for generalised winding numbers); nearer nodes are opened, and the faces of an opened
// group are summed exactly (Van Oosterom-Strackee, as above).  BOTH probes of a sample use the same cut, decided from
// the sample point itself, so the truncation error is a smooth function evaluated at two points 2h apart and largely
// cancels in d.  The node that holds the sample's own face is always opened (the face must be left out).
// One warp per sample: a warp-shared node stack, up to 32 nodes tested per pass (one per lane), opened groups go to a
// list and are summed with one face per lane.  Per-lane compensated sums, reduced in lane order: deterministic.
// ---------------------------------------------------------------------------
constexpr int WG = 32;                 // faces per leaf group
constexpr int WT_WARPS = 4;
constexpr int WT_NCAP = 1024;          // node stack per warp
constexpr int WT_GCAP = 160;           // opened-group list per warp (drained one group per pass)

__device__ __forceinline__ unsigned wn_spread10(unsigned x)
{
    x &= 0x3FFu;
    x = (x | (x << 16)) & 0x030000FFu;
    x = (x | (x << 8))  & 0x0300F00Fu;
    x = (x | (x << 4))  & 0x030C30C3u;
    x = (x | (x << 2))  & 0x09249249u;
    return x;
}

__global__ void wn_keys_kernel(const float* __restrict__ verts, const int32_t* __restrict__ faces, long long F,
                               float3 lo, float3 ext, uint32_t* __restrict__ keys, uint32_t* __restrict__ vals)
{
    const long long f = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (f >= F) return;
    float c[3];
    for (int d = 0; d < 3; ++d)
        c[d] = (verts[3 * (long long)faces[3 * f] + d] + verts[3 * (long long)faces[3 * f + 1] + d] + verts[3 * (long long)faces[3 * f + 2] + d]) * (1.0f / 3.0f);
    const float tx = ext.x > 0.f ? fminf(fmaxf((c[0] - lo.x) / ext.x, 0.f), 1.f) : 0.f;
    const float ty = ext.y > 0.f ? fminf(fmaxf((c[1] - lo.y) / ext.y, 0.f), 1.f) : 0.f;
    const float tz = ext.z > 0.f ? fminf(fmaxf((c[2] - lo.z) / ext.z, 0.f), 1.f) : 0.f;
    keys[f] = (wn_spread10((unsigned)fminf(tx * 1024.f, 1023.f)) << 2) | (wn_spread10((unsigned)fminf(ty * 1024.f, 1023.f)) << 1) |
              wn_spread10((unsigned)fminf(tz * 1024.f, 1023.f));
    vals[f] = (uint32_t)f;
}

__global__ void wn_pos_kernel(const uint32_t* __restrict__ order, long long F, int32_t* __restrict__ face_pos)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < F) face_pos[order[i]] = (int32_t)i;
}

// leaf groups: node G + g from the faces at sorted positions [32 g, 32 g + 32)
__global__ void __launch_bounds__(128)
wn_leaf_kernel(const float* __restrict__ verts, const int32_t* __restrict__ faces, const uint32_t* __restrict__ order, long long F,
               long long n_groups, long long G, float4* __restrict__ nodes)
{
    const unsigned FULL = 0xFFFFFFFFu;
    const int lane = threadIdx.x & 31;
    const long long g = (long long)blockIdx.x * 4 + (threadIdx.x >> 5);
    if (g >= G) return;
    const long long k = g * WG + lane;
    float3 a = f3(0, 0, 0), b = a, c = a;
    const bool live = g < n_groups && k < F;
    if (live) {
        const long long f = order[k];
        const long long i0 = faces[3 * f], i1 = faces[3 * f + 1], i2 = faces[3 * f + 2];
        a = f3(verts[3 * i0], verts[3 * i0 + 1], verts[3 * i0 + 2]);
        b = f3(verts[3 * i1], verts[3 * i1 + 1], verts[3 * i1 + 2]);
        c = f3(verts[3 * i2], verts[3 * i2 + 1], verts[3 * i2 + 2]);
    }
    float3 nv = 0.5f * cross3(b - a, c - a);
    float area = sqrtf(dot3(nv, nv));
    float3 ac = f3(area * (a.x + b.x + c.x) * (1.0f / 3.0f), area * (a.y + b.y + c.y) * (1.0f / 3.0f), area * (a.z + b.z + c.z) * (1.0f / 3.0f));
    float3 sum_pt = live ? f3((a.x + b.x + c.x) * (1.0f / 3.0f), (a.y + b.y + c.y) * (1.0f / 3.0f), (a.z + b.z + c.z) * (1.0f / 3.0f)) : f3(0, 0, 0);
    float cnt = live ? 1.0f : 0.0f;
    for (int off = 16; off > 0; off >>= 1) {
        nv.x += __shfl_xor_sync(FULL, nv.x, off); nv.y += __shfl_xor_sync(FULL, nv.y, off); nv.z += __shfl_xor_sync(FULL, nv.z, off);
        ac.x += __shfl_xor_sync(FULL, ac.x, off); ac.y += __shfl_xor_sync(FULL, ac.y, off); ac.z += __shfl_xor_sync(FULL, ac.z, off);
        sum_pt.x += __shfl_xor_sync(FULL, sum_pt.x, off); sum_pt.y += __shfl_xor_sync(FULL, sum_pt.y, off); sum_pt.z += __shfl_xor_sync(FULL, sum_pt.z, off);
        area += __shfl_xor_sync(FULL, area, off);
        cnt += __shfl_xor_sync(FULL, cnt, off);
    }
    // centre: area-weighted centroid; zero-area groups fall back to the mean of the face centroids
    float3 cen = area > 0.0f ? (1.0f / area) * ac : (cnt > 0.0f ? (1.0f / cnt) * sum_pt : f3(0, 0, 0));
    float r = 0.0f;
    if (live) {
        const float3 da = a - cen, db = b - cen, dc = c - cen;
        r = sqrtf(fmaxf(dot3(da, da), fmaxf(dot3(db, db), dot3(dc, dc))));
    }
    for (int off = 16; off > 0; off >>= 1) r = fmaxf(r, __shfl_xor_sync(FULL, r, off));
    if (lane == 0) {
        nodes[2 * (G + g)] = make_float4(cen.x, cen.y, cen.z, cnt > 0.0f ? r * (1.0f + 1e-6f) : -1.0f);   // R < 0: empty
        nodes[2 * (G + g) + 1] = make_float4(nv.x, nv.y, nv.z, area);
    }
}

// one level of inner nodes [first, first + n): from the two children 2 i, 2 i + 1
__global__ void wn_inner_kernel(long long first, long long n, float4* __restrict__ nodes)
{
    const long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    const long long i = first + j;
    const float4 c0 = nodes[4 * i], n0 = nodes[4 * i + 1], c1 = nodes[4 * i + 2], n1 = nodes[4 * i + 3];
    float4 oc, on;
    if (c0.w < 0.0f && c1.w < 0.0f) { oc = make_float4(0, 0, 0, -1.0f); on = make_float4(0, 0, 0, 0); }
    else if (c1.w < 0.0f) { oc = c0; on = n0; }
    else if (c0.w < 0.0f) { oc = c1; on = n1; }
    else {
        const float A = n0.w + n1.w;
        float3 cen = A > 0.0f ? f3((n0.w * c0.x + n1.w * c1.x) / A, (n0.w * c0.y + n1.w * c1.y) / A, (n0.w * c0.z + n1.w * c1.z) / A)
                              : f3(0.5f * (c0.x + c1.x), 0.5f * (c0.y + c1.y), 0.5f * (c0.z + c1.z));
        const float3 d0 = f3(c0.x, c0.y, c0.z) - cen, d1 = f3(c1.x, c1.y, c1.z) - cen;
        const float r = fmaxf(sqrtf(dot3(d0, d0)) + c0.w, sqrtf(dot3(d1, d1)) + c1.w) * (1.0f + 1e-6f);
        oc = make_float4(cen.x, cen.y, cen.z, r);
        on = make_float4(n0.x + n1.x, n0.y + n1.y, n0.z + n1.z, A);
    }
    nodes[2 * i] = oc; nodes[2 * i + 1] = on;
}

struct Kahan { float s, c; };
__device__ __forceinline__ void kadd(Kahan& k, float x) { const float y = x - k.c, t = k.s + y; k.c = (t - k.s) - y; k.s = t; }

__device__ __forceinline__ float half_solid_angle(float3 a, float3 b, float3 c)        // Omega / 2 of the triangle seen from the origin
{
    const float la = sqrtf(dot3(a, a)), lb = sqrtf(dot3(b, b)), lc = sqrtf(dot3(c, c));
    const float det = a.x * (b.y * c.z - b.z * c.y) - a.y * (b.x * c.z - b.z * c.x) + a.z * (b.x * c.y - b.y * c.x);
    const float den = fmaf(la * lb, lc, fmaf(dot3(a, b), lc, fmaf(dot3(b, c), la, dot3(c, a) * lb)));
    return atan2f(det, den);
}

__global__ void __launch_bounds__(WT_WARPS * 32)
orient_tree_kernel(const float* __restrict__ verts, const int32_t* __restrict__ faces, long long F,
                   const float4* __restrict__ nodes, const uint32_t* __restrict__ order, const int32_t* __restrict__ face_pos,
                   long long G, int levels, const int32_t* __restrict__ tri, const float* __restrict__ bary, long long n,
                   float h_scale, float beta, float* __restrict__ normal_out, float* __restrict__ d_out, int* __restrict__ err)
{
    __shared__ int s_nodes[WT_WARPS][WT_NCAP];
    __shared__ int s_groups[WT_WARPS][WT_GCAP];
    const unsigned FULL = 0xFFFFFFFFu;
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const unsigned lt = (1u << lane) - 1u;
    int* nstack = s_nodes[wib];
    int* glist = s_groups[wib];
    const long long n_warps = (long long)gridDim.x * WT_WARPS;
    for (long long i = (long long)blockIdx.x * WT_WARPS + wib; i < n; i += n_warps) {
        const int f = tri[i];
        if (f < 0 || f >= F) { if (lane == 0) *err = 1; continue; }
        const long long i0 = faces[3 * (long long)f], i1 = faces[3 * (long long)f + 1], i2 = faces[3 * (long long)f + 2];
        const float3 a = f3(verts[3 * i0], verts[3 * i0 + 1], verts[3 * i0 + 2]);
        const float3 b = f3(verts[3 * i1], verts[3 * i1 + 1], verts[3 * i1 + 2]);
        const float3 c = f3(verts[3 * i2], verts[3 * i2 + 1], verts[3 * i2 + 2]);
        const float b0 = bary[3 * i], b1 = bary[3 * i + 1], b2 = bary[3 * i + 2];
        const float3 s = f3(b0 * a.x + b1 * b.x + b2 * c.x, b0 * a.y + b1 * b.y + b2 * c.y, b0 * a.z + b1 * b.z + b2 * c.z);
        float3 nr = cross3(b - a, c - a);
        const float nn = sqrtf(dot3(nr, nr));
        nr = (nn > 0.0f ? 1.0f / nn : 0.0f) * nr;
        const float h = h_scale * sqrtf(0.5f * nn);
        const float3 pb = f3(s.x - h * nr.x, s.y - h * nr.y, s.z - h * nr.z), pf = f3(s.x + h * nr.x, s.y + h * nr.y, s.z + h * nr.z);
        const int own_group = face_pos[f] / WG;
        Kahan wb = { 0.0f, 0.0f }, wf = { 0.0f, 0.0f };              // sums of Omega / 2 at the back and front probe
        int ncount = 1, gcount = 0;
        if (lane == 0) nstack[0] = 1;                                 // root
        __syncwarp();
        while (ncount > 0 || gcount > 0) {
            if (gcount > 0 && (gcount >= WT_GCAP - 64 || ncount == 0)) {
                // ---- one opened group: one face per lane, exact solid angles ------------------------
                const long long k = (long long)glist[gcount - 1] * WG + lane;
                --gcount;
                if (k < F) {
                    const long long ff = order[k];
                    if (ff != f) {
                        const long long j0 = faces[3 * ff], j1 = faces[3 * ff + 1], j2 = faces[3 * ff + 2];
                        const float3 va = f3(verts[3 * j0], verts[3 * j0 + 1], verts[3 * j0 + 2]);
                        const float3 vb = f3(verts[3 * j1], verts[3 * j1 + 1], verts[3 * j1 + 2]);
                        const float3 vc = f3(verts[3 * j2], verts[3 * j2 + 1], verts[3 * j2 + 2]);
                        kadd(wb, half_solid_angle(va - pb, vb - pb, vc - pb));
                        kadd(wf, half_solid_angle(va - pf, vb - pf, vc - pf));
                    }
                }
                __syncwarp();
            } else {
                // ---- node pass: far nodes contribute their dipole, near ones are opened ---------------
                int np = ncount < 32 ? ncount : 32;
                if (ncount > WT_NCAP - 96) np = 1;                    // nearly full: depth-first (+1 per level)
                bool open_inner = false, open_leaf = false;
                int node = 0;
                if (lane < np) {
                    node = nstack[ncount - np + lane];
                    const float4 cn = nodes[2 * (long long)node], nv = nodes[2 * (long long)node + 1];
                    if (cn.w >= 0.0f) {                               // not empty
                        const int level = 31 - __clz(node);           // root: 0
                        const int span = (int)(G >> level);           // groups under the node
                        const int first = (node - (1 << level)) * span;
                        const float3 r = f3(cn.x - s.x, cn.y - s.y, cn.z - s.z);
                        const bool holds_own = own_group >= first && own_group < first + span;
                        if (!holds_own && dot3(r, r) > beta * beta * cn.w * cn.w) {
                            const float3 rb = f3(cn.x - pb.x, cn.y - pb.y, cn.z - pb.z), rf = f3(cn.x - pf.x, cn.y - pf.y, cn.z - pf.z);
                            const float db2 = dot3(rb, rb), df2 = dot3(rf, rf);
                            kadd(wb, 0.5f * (nv.x * rb.x + nv.y * rb.y + nv.z * rb.z) * rsqrtf(db2) / db2);
                            kadd(wf, 0.5f * (nv.x * rf.x + nv.y * rf.y + nv.z * rf.z) * rsqrtf(df2) / df2);
                        } else if (level == levels) open_leaf = true;
                        else open_inner = true;
                    }
                }
                ncount -= np;
                __syncwarp();                                         // all pops read before any push writes
                const unsigned mi = __ballot_sync(FULL, open_inner), ml = __ballot_sync(FULL, open_leaf);
                if (open_inner) { const int o = ncount + 2 * __popc(mi & lt); nstack[o] = 2 * node; nstack[o + 1] = 2 * node + 1; }
                if (open_leaf) glist[gcount + __popc(ml & lt)] = node - (int)G;
                ncount += 2 * __popc(mi); gcount += __popc(ml);
                __syncwarp();
            }
        }
        float sb = wb.s, sf = wf.s;
        for (int off = 16; off > 0; off >>= 1) { sb += __shfl_xor_sync(FULL, sb, off); sf += __shfl_xor_sync(FULL, sf, off); }
        if (lane == 0) {
            const float d = (sb - sf) * (2.0f / (4.0f * CUDART_PI_F));            // Omega = 2 x, w = Omega / 4 pi
            if (d_out) d_out[i] = d;
            const float sg = d < 0.0f ? -1.0f : 1.0f;
            normal_out[3 * i] = sg * nr.x; normal_out[3 * i + 1] = sg * nr.y; normal_out[3 * i + 2] = sg * nr.z;
        }
        __syncwarp();
    }
}

}  // namespace

extern "C" size_t mcs_winding_workspace_bytes(const mcs_bvh* b, int64_t n)
{
    if (!b || n < 1) return 0;
    // partial sums (n points, or the 2n probe points of mcs_orient_samples) + probe coordinates, exclusions, values
    const long long m = 2 * n;
    const size_t pb = partial_bytes(b->F, n) > partial_bytes(b->F, m) ? partial_bytes(b->F, n) : partial_bytes(b->F, m);
    return align_up(pb) + align_up((size_t)m * 12) + align_up((size_t)m * 4) * 2 + 256;
}

extern "C" int mcs_winding_number(const mcs_bvh* b, const float* points, const int32_t* exclude, int64_t n,
                                  float* w_out, void* ws, size_t ws_bytes, void* stream)
{
    if (!b || !points || !w_out || n < 1) return MCS_EINVAL;
    if (!ws || ws_bytes < mcs_winding_workspace_bytes(b, n)) return MCS_ENOMEM;
    return winding_run(b, points, exclude, n, w_out, (float*)ws, (cudaStream_t)stream);
}

extern "C" int mcs_orient_samples(const mcs_bvh* b, const mcs_samples* s, float h_scale, float* normal_out, float* d_out,
                                  void* ws, size_t ws_bytes, void* stream)
{
    if (!b || !s || !s->tri || !s->bary || !normal_out || s->n_s < 1 || !(h_scale > 0.0f)) return MCS_EINVAL;
    const long long n = s->n_s, m = 2 * n;
    if (!ws || ws_bytes < mcs_winding_workspace_bytes(b, n)) return MCS_ENOMEM;
    cudaStream_t st = (cudaStream_t)stream;
    char* p = (char*)ws;
    float* partial = (float*)p;   p += align_up(partial_bytes(b->F, n) > partial_bytes(b->F, m) ? partial_bytes(b->F, n) : partial_bytes(b->F, m));
    float* pts = (float*)p;       p += align_up((size_t)m * 12);
    int32_t* excl = (int32_t*)p;  p += align_up((size_t)m * 4);
    float* w = (float*)p;         p += align_up((size_t)m * 4);
    int* err = (int*)p;
    MCS_CUDA_TRY(cudaMemsetAsync(err, 0, 4, st));
    mcs_note_launch(), orient_points_kernel<<<(unsigned)ceil_div64(n, 256), 256, 0, st>>>(b->verts, b->faces, b->F, s->tri, s->bary, n,
                                                                                     h_scale, pts, excl, normal_out, err);
    int rc = winding_run(b, pts, excl, m, w, partial, st);
    if (rc != MCS_OK) return rc;
    mcs_note_launch(), orient_finish_kernel<<<(unsigned)ceil_div64(n, 256), 256, 0, st>>>(w, n, normal_out, d_out);
    int h_err = 0;
    MCS_CUDA_TRY(cudaMemcpyAsync(&h_err, err, 4, cudaMemcpyDeviceToHost, st));
    MCS_CUDA_TRY(cudaStreamSynchronize(st));
    return h_err ? MCS_EINVAL : MCS_OK;
}

// Builds the face hierarchy of mcs_orient_samples_fast once per handle (stream-ordered; the arrays belong to the handle).
static int wn_tree_build(const mcs_bvh* b, cudaStream_t st)
{
    std::lock_guard<std::mutex> lock(b->wn_mutex);
    if (b->wn_nodes) return MCS_OK;
    const long long F = b->F;
    const long long n_groups = ceil_div64(F, WG);
    long long G = 1; int levels = 0;
    while (G < n_groups) { G <<= 1; ++levels; }
    float4* nodes = nullptr; uint32_t* keys = nullptr; uint32_t* order = nullptr; int32_t* face_pos = nullptr; void* sort_ws = nullptr;
    const size_t sort_bytes = sort_workspace_bytes(F, 4);
    cudaError_t e = cudaMallocAsync((void**)&nodes, (size_t)(2 * G) * 2 * sizeof(float4), st);
    if (e == cudaSuccess) e = cudaMallocAsync((void**)&keys, (size_t)F * 4, st);
    if (e == cudaSuccess) e = cudaMallocAsync((void**)&order, (size_t)F * 4, st);
    if (e == cudaSuccess) e = cudaMallocAsync((void**)&face_pos, (size_t)F * 4, st);
    if (e == cudaSuccess) e = cudaMallocAsync(&sort_ws, sort_bytes, st);
    int rc = MCS_OK;
    if (e != cudaSuccess) { mcs_set_last_cuda_error((int)e); rc = MCS_ENOMEM; }
    if (rc == MCS_OK) {
        const float3 lo = f3(b->aabb_lo[0], b->aabb_lo[1], b->aabb_lo[2]);
        const float3 ext = f3(b->aabb_hi[0] - lo.x, b->aabb_hi[1] - lo.y, b->aabb_hi[2] - lo.z);
        mcs_note_launch(), wn_keys_kernel<<<(unsigned)ceil_div64(F, 256), 256, 0, st>>>(b->verts, b->faces, F, lo, ext, keys, order);
        rc = sort_pairs_u32(keys, order, F, 30, sort_ws, sort_bytes, st);
    }
    if (rc == MCS_OK) {
        mcs_note_launch(), wn_pos_kernel<<<(unsigned)ceil_div64(F, 256), 256, 0, st>>>(order, F, face_pos);
        mcs_note_launch(), wn_leaf_kernel<<<(unsigned)ceil_div64(G, 4), 128, 0, st>>>(b->verts, b->faces, order, F, n_groups, G, nodes);
        for (long long first = G >> 1; first >= 1; first >>= 1)
            mcs_note_launch(), wn_inner_kernel<<<(unsigned)ceil_div64(first, 256), 256, 0, st>>>(first, first, nodes);
        e = cudaGetLastError();
        if (e != cudaSuccess) { mcs_set_last_cuda_error((int)e); rc = MCS_ECUDA; }
    }
    if (keys) cudaFreeAsync(keys, st);
    if (sort_ws) cudaFreeAsync(sort_ws, st);
    if (rc != MCS_OK) {
        if (nodes) cudaFreeAsync(nodes, st);
        if (order) cudaFreeAsync(order, st);
        if (face_pos) cudaFreeAsync(face_pos, st);
        return rc;
    }
    // later calls may come on other streams: the tree must be complete before the handle advertises it
    e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) { mcs_set_last_cuda_error((int)e); return MCS_ECUDA; }
    b->wn_order = order; b->wn_face_pos = face_pos; b->wn_G = G; b->wn_levels = levels;
    b->wn_nodes = nodes;
    return MCS_OK;
}

extern "C" int mcs_orient_samples_fast(const mcs_bvh* b, const mcs_samples* s, float h_scale, float beta, float* normal_out,
                                       float* d_out, void* stream)
{
    if (!b || !s || !s->tri || !s->bary || !normal_out || s->n_s < 1 || !(h_scale > 0.0f) || !(beta >= 1.5f)) return MCS_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    int rc = wn_tree_build(b, st);
    if (rc != MCS_OK) return rc;
    int* err = nullptr;
    cudaError_t e = cudaMallocAsync((void**)&err, 4, st);
    if (e != cudaSuccess) { mcs_set_last_cuda_error((int)e); return MCS_ENOMEM; }
    cudaMemsetAsync(err, 0, 4, st);
    const long long n = s->n_s;
    long long blocks = ceil_div64(n, WT_WARPS);
    if (blocks > 148 * 8) blocks = 148 * 8;
    mcs_note_launch(), orient_tree_kernel<<<(unsigned)blocks, WT_WARPS * 32, 0, st>>>(
        b->verts, b->faces, b->F, (const float4*)b->wn_nodes, b->wn_order, b->wn_face_pos, b->wn_G, b->wn_levels,
        s->tri, s->bary, n, h_scale, beta, normal_out, d_out, err);
    mcs_bvh_touch(b, st);
    int h_err = 0;
    e = cudaMemcpyAsync(&h_err, err, 4, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    cudaFreeAsync(err, st);
    if (e != cudaSuccess) { mcs_set_last_cuda_error((int)e); return MCS_ECUDA; }
    return h_err ? MCS_EINVAL : MCS_OK;
}
