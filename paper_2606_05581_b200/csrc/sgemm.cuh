// sgemm.cuh -- plain fp32 SIMT matrix product with split-K, shared by project.cu (reduced Galerkin matrix) and eigs.cu
// (subspace iteration for the smallest eigenpairs at large K).  Included inside an anonymous namespace.
#pragma once

constexpr int GT = 64;     // C tile is GT x GT
constexpr int GK = 16;     // depth of one slab

// C[M][N] = op(A) B, row-major.  TA = false: A is [M][Kd]; TA = true: A is stored [Kd][M] (op(A) = A^T).
template <bool TA>
__global__ void __launch_bounds__(256)
sgemm_kernel(const float* __restrict__ A, const float* __restrict__ B, float* __restrict__ C, int M, int N, int Kd,
             int k_per_z)   // split-K: block z takes k in [z k_per_z, (z+1) k_per_z) and writes C + z M N
{
    __shared__ float As[GK][GT + 4], Bs[GK][GT + 4];
    const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
    const int m0 = blockIdx.y * GT, n0 = blockIdx.x * GT;
    float acc[4][4] = {};
    const int k_lo = blockIdx.z * k_per_z;
    const int k_hi = k_lo + k_per_z < Kd ? k_lo + k_per_z : Kd;
    C += (size_t)blockIdx.z * M * N;
    for (int k0 = k_lo; k0 < k_hi; k0 += GK) {
        for (int i = threadIdx.x; i < GK * GT; i += 256) {
            if (TA) {                                   // A^T tile: consecutive threads along m (contiguous in memory)
                const int kk = i / GT, mm = i - kk * GT;
                const int gm = m0 + mm, gk = k0 + kk;
                As[kk][mm] = (gm < M && gk < k_hi) ? A[(size_t)gk * M + gm] : 0.0f;
            } else {                                    // A tile: consecutive threads along k
                const int mm = i / GK, kk = i - mm * GK;
                const int gm = m0 + mm, gk = k0 + kk;
                As[kk][mm] = (gm < M && gk < k_hi) ? A[(size_t)gm * Kd + gk] : 0.0f;
            }
            const int kb = i / GT, nn = i - kb * GT;
            const int gn = n0 + nn, gkb = k0 + kb;
            Bs[kb][nn] = (gn < N && gkb < k_hi) ? B[(size_t)gkb * N + gn] : 0.0f;
        }
        __syncthreads();
#pragma unroll
        for (int kk = 0; kk < GK; ++kk) {
            float a[4], b[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) { a[i] = As[kk][ty * 4 + i]; b[i] = Bs[kk][tx * 4 + i]; }
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(a[i], b[j], acc[i][j]);
        }
        __syncthreads();
    }
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int gm = m0 + ty * 4 + i, gn = n0 + tx * 4 + j;
            if (gm < M && gn < N) C[(size_t)gm * N + gn] = acc[i][j];
        }
}


// The tall product of the subspace iteration: C [M][N] = A [M][Kd] B [Kd][N] (row-major, N a multiple of 4), split-K as
// above.  128 x 128 tile, 256 threads, 8 x 8 outputs per thread as four 4 x 4 quadrants (two LDS.128 of A and two of B
// feed 64 FMAs, against 16 for the 64 x 64 kernel above, which is bound by shared-memory bandwidth), depth 8 per slab,
// the next slab's global loads in flight while the current one is multiplied (registers), two shared-memory buffers, one
// barrier per slab.  A's rows are only 4-byte aligned in general (Kd = 2562): scalar loads; B's are 16-byte aligned.
constexpr int TT = 128;    // tile edge
constexpr int TK = 8;      // depth of one slab

__global__ void __launch_bounds__(256, 2)
sgemm_tall_kernel(const float* __restrict__ A, const float* __restrict__ B, float* __restrict__ C, int M, int N, int Kd, int k_per_z)
{
    __shared__ __align__(16) float As[2][TK][TT], Bs[2][TK][TT];
    const int t = threadIdx.x;
    const int tx = t & 15, ty = t >> 4;
    const int m0 = blockIdx.y * TT, n0 = blockIdx.x * TT;
    const int k_lo = blockIdx.z * k_per_z;
    const int k_hi = k_lo + k_per_z < Kd ? k_lo + k_per_z : Kd;
    C += (size_t)blockIdx.z * M * N;
    // global -> register staging: A: row t / 2, four k's starting at (t & 1) * 4; B: k = t / 32, four columns at (t & 31) * 4
    const int a_row = m0 + (t >> 1), a_k = (t & 1) * 4;
    const int b_k = t >> 5, b_col = n0 + (t & 31) * 4;
    const float* a_ptr = A + (size_t)(a_row < M ? a_row : 0) * Kd;
    float ra[4];
    float4 rb;
    auto load = [&](int k0) {
#pragma unroll
        for (int i = 0; i < 4; ++i) { const int k = k0 + a_k + i; ra[i] = (a_row < M && k < k_hi) ? a_ptr[k] : 0.0f; }
        const int kb = k0 + b_k;
        rb = (kb < k_hi && b_col < N) ? *reinterpret_cast<const float4*>(B + (size_t)kb * N + b_col) : make_float4(0.f, 0.f, 0.f, 0.f);
    };
    auto stage = [&](int buf) {
#pragma unroll
        for (int i = 0; i < 4; ++i) As[buf][a_k + i][t >> 1] = ra[i];
        *reinterpret_cast<float4*>(&Bs[buf][b_k][(t & 31) * 4]) = rb;
    };
    float acc[8][8] = {};
    int buf = 0;
    if (k_lo < k_hi) { load(k_lo); stage(0); }
    __syncthreads();
    for (int k0 = k_lo; k0 < k_hi; k0 += TK) {
        const bool more = k0 + TK < k_hi;
        if (more) load(k0 + TK);
#pragma unroll
        for (int kk = 0; kk < TK; ++kk) {
            const float4 a0 = *reinterpret_cast<const float4*>(&As[buf][kk][ty * 4]);
            const float4 a1 = *reinterpret_cast<const float4*>(&As[buf][kk][64 + ty * 4]);
            const float4 b0 = *reinterpret_cast<const float4*>(&Bs[buf][kk][tx * 4]);
            const float4 b1 = *reinterpret_cast<const float4*>(&Bs[buf][kk][64 + tx * 4]);
            const float a[8] = { a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w };
            const float b[8] = { b0.x, b0.y, b0.z, b0.w, b1.x, b1.y, b1.z, b1.w };
#pragma unroll
            for (int i = 0; i < 8; ++i)
#pragma unroll
                for (int j = 0; j < 8; ++j) acc[i][j] = fmaf(a[i], b[j], acc[i][j]);
        }
        if (more) stage(buf ^ 1);
        __syncthreads();
        buf ^= 1;
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const int gm = m0 + (i < 4 ? ty * 4 + i : 64 + ty * 4 + (i - 4));
        if (gm >= M) continue;
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int gn = n0 + h * 64 + tx * 4;
            if (gn < N) *reinterpret_cast<float4*>(C + (size_t)gm * N + gn) = make_float4(acc[i][h * 4], acc[i][h * 4 + 1], acc[i][h * 4 + 2], acc[i][h * 4 + 3]);
        }
    }
}
