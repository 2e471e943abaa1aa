// query.cu -- closest-point entry points (SURVEY.md 8(b) mcs_closest_point):
// the BVH query kernel and the exhaustive device-side cross-check.
#include "traverse.cuh"

#include <limits.h>

namespace {

constexpr int QT = 128;

__global__ void __launch_bounds__(QT)
closest_point_kernel(const BvhNode* __restrict__ nodes, const PackedTri* __restrict__ tris,
                     const float* __restrict__ q, int64_t Q, float mesh_scale,
                     float* __restrict__ dist, int32_t* __restrict__ tri, float* __restrict__ bary)
{
    const int64_t i = (int64_t)blockIdx.x * QT + threadIdx.x;
    if (i >= Q) return;
    const float3 p = f3(q[3 * i], q[3 * i + 1], q[3 * i + 2]);
    ClosestHit h; h.d2 = CUDART_INF_F; h.tri = INT_MAX; h.k = -1; h.v = 0.0f; h.w = 0.0f;
    TraversalCounters cnt;
    bvh_closest_point<false, false>(nodes, tris, p, h, cnt, mesh_scale);
    if (dist) dist[i] = sqrtf(h.d2);
    if (tri) tri[i] = h.k >= 0 ? h.tri : -1;
    if (bary) { bary[3 * i] = fmaxf(1.0f - h.v - h.w, 0.0f); bary[3 * i + 1] = h.v; bary[3 * i + 2] = h.w; }
}

// Exhaustive scan: every thread tests every face; faces staged through shared memory.
constexpr int BF_TILE = 128;
__global__ void __launch_bounds__(QT)
closest_point_bruteforce_kernel(const PackedTri* __restrict__ tris, int64_t F,
                                const float* __restrict__ q, int64_t Q,
                                float* __restrict__ dist, int32_t* __restrict__ tri, float* __restrict__ bary)
{
    __shared__ float4 s_tri[BF_TILE * 4];
    const int64_t i = (int64_t)blockIdx.x * QT + threadIdx.x;
    const bool active = i < Q;
    const float3 p = active ? f3(q[3 * i], q[3 * i + 1], q[3 * i + 2]) : f3(0.f, 0.f, 0.f);
    ClosestHit h; h.d2 = CUDART_INF_F; h.tri = INT_MAX; h.k = -1; h.v = 0.0f; h.w = 0.0f;
    for (int64_t base = 0; base < F; base += BF_TILE) {
        const int n = (int)min((int64_t)BF_TILE, F - base);
        __syncthreads();
        for (int j = threadIdx.x; j < n * 4; j += QT)
            s_tri[j] = reinterpret_cast<const float4*>(tris + base)[j];
        __syncthreads();
        if (active) {
            for (int j = 0; j < n; ++j) {
                const TriData T = unpack_tri(s_tri[4 * j], s_tri[4 * j + 1], s_tri[4 * j + 2], s_tri[4 * j + 3]);
                float v = 0.0f, w = 0.0f;
                const float d2 = closest_point_triangle(p, T, CUDART_INF_F, v, w);
                const int orig = T.orig;
                if (d2 < h.d2 || (d2 == h.d2 && orig < h.tri)) { h.d2 = d2; h.tri = orig; h.k = (int)(base + j); h.v = v; h.w = w; }
            }
        }
    }
    if (!active) return;
    if (dist) dist[i] = sqrtf(h.d2);
    if (tri) tri[i] = h.tri;
    if (bary) { bary[3 * i] = fmaxf(1.0f - h.v - h.w, 0.0f); bary[3 * i + 1] = h.v; bary[3 * i + 2] = h.w; }
}

__global__ void philox_kernel(const uint32_t* __restrict__ ctr, int64_t n, uint2 key, uint32_t* __restrict__ out)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const uint4 c = make_uint4(ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3]);
    const uint4 o = philox4x32_10(c, key);
    out[4 * i] = o.x; out[4 * i + 1] = o.y; out[4 * i + 2] = o.z; out[4 * i + 3] = o.w;
}

}  // namespace

extern "C" int mcs_closest_point(const mcs_bvh* b, const float* q, int64_t Q,
                                 float* dist, int32_t* tri, float* bary, void* stream)
{
    if (!b || Q < 0 || (Q > 0 && !q)) return MCS_EINVAL;
    if (Q == 0) return MCS_OK;
    float scale = 0.0f;                                // |coordinates|_1 bound of the mesh (prune_limit)
    for (int d = 0; d < 3; ++d) scale += fmaxf(fabsf(b->aabb_lo[d]), fabsf(b->aabb_hi[d]));
    mcs_note_launch(), closest_point_kernel<<<(unsigned)ceil_div64(Q, QT), QT, 0, (cudaStream_t)stream>>>(b->nodes, b->tris, q, Q, scale, dist, tri, bary);
    mcs_bvh_touch(b, (cudaStream_t)stream);
    MCS_CUDA_TRY(cudaGetLastError());
    return MCS_OK;
}

extern "C" int mcs_closest_point_bruteforce(const mcs_bvh* b, const float* q, int64_t Q,
                                            float* dist, int32_t* tri, float* bary, void* stream)
{
    if (!b || Q < 0 || (Q > 0 && !q)) return MCS_EINVAL;
    if (Q == 0) return MCS_OK;
    mcs_note_launch(), closest_point_bruteforce_kernel<<<(unsigned)ceil_div64(Q, QT), QT, 0, (cudaStream_t)stream>>>(b->tris, b->n_leaves, q, Q, dist, tri, bary);
    mcs_bvh_touch(b, (cudaStream_t)stream);
    MCS_CUDA_TRY(cudaGetLastError());
    return MCS_OK;
}

extern "C" int mcs_philox4x32_10(const uint32_t* counters, int64_t n, const uint32_t* key, uint32_t* out, void* stream)
{
    if (n < 0 || !key || (n > 0 && (!counters || !out))) return MCS_EINVAL;
    if (n == 0) return MCS_OK;
    mcs_note_launch(), philox_kernel<<<(unsigned)ceil_div64(n, 256), 256, 0, (cudaStream_t)stream>>>(counters, n, make_uint2(key[0], key[1]), out);
    MCS_CUDA_TRY(cudaGetLastError());
    return MCS_OK;
}
