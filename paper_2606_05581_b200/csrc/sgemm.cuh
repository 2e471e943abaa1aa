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

