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
