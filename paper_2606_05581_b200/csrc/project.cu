// project.cu -- reduced Ritz-Galerkin DtN matrix.
// With basis functions phi_k = sum_v Phi[v][k] hat_v the paper evaluates the dense vector b(p) = Phi^T iota(p) at both ends
// of every walk and defers the outer products d d^T to a batched contraction D^T diag(w) D over the walks
// (N K^2 multiply-adds: 2.7e11 for configs[1] at K = 160).  The same matrix is Phi^T S Phi for the nodal matrix S
// that the hat-basis accumulation of this library has already reduced to V x V (exactly, by linearity; pinned in
// the oracle), i.e. two small products of 2 V^2 K + 2 V K^2 flops (2.2e9): the outer products are deferred past the
// nodal reduction instead of being batched over walks.  Plain fp32 SIMT tiles: at this size the products take a
// fraction of a millisecond, and the eigenvalues wanted from the result need fp32 accumulation.
#include "common.cuh"

namespace {

constexpr int GT = 64;     // C tile is GT x GT
constexpr int GK = 16;     // depth of one slab

// C[M][N] = op(A) B, row-major.  TA = false: A is [M][Kd]; TA = true: A is stored [Kd][M] (op(A) = A^T).
template <bool TA>
__global__ void __launch_bounds__(256)
sgemm_kernel(const float* __restrict__ A, const float* __restrict__ B, float* __restrict__ C, int M, int N, int Kd)
{
    __shared__ float As[GK][GT + 4], Bs[GK][GT + 4];
    const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
    const int m0 = blockIdx.y * GT, n0 = blockIdx.x * GT;
    float acc[4][4] = {};
    for (int k0 = 0; k0 < Kd; k0 += GK) {
        for (int i = threadIdx.x; i < GK * GT; i += 256) {
            if (TA) {                                   // A^T tile: consecutive threads along m (contiguous in memory)
                const int kk = i / GT, mm = i - kk * GT;
                const int gm = m0 + mm, gk = k0 + kk;
                As[kk][mm] = (gm < M && gk < Kd) ? A[(size_t)gk * M + gm] : 0.0f;
            } else {                                    // A tile: consecutive threads along k
                const int mm = i / GK, kk = i - mm * GK;
                const int gm = m0 + mm, gk = k0 + kk;
                As[kk][mm] = (gm < M && gk < Kd) ? A[(size_t)gm * Kd + gk] : 0.0f;
            }
            const int kb = i / GT, nn = i - kb * GT;
            const int gn = n0 + nn, gkb = k0 + kb;
            Bs[kb][nn] = (gn < N && gkb < Kd) ? B[(size_t)gkb * N + gn] : 0.0f;
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

__global__ void symmetrise_kernel(float* __restrict__ R, int K)
{
    const int i = blockIdx.y * 16 + threadIdx.y, j = blockIdx.x * 16 + threadIdx.x;
    if (i < K && j < K && i < j) {
        const float m = 0.5f * (R[(size_t)i * K + j] + R[(size_t)j * K + i]);
        R[(size_t)i * K + j] = m; R[(size_t)j * K + i] = m;
    }
}

}  // namespace

extern "C" size_t mcs_project_workspace_bytes(int64_t V, int64_t K)
{
    if (V < 1 || K < 1) return 0;
    return align_up((size_t)V * K * 4) + 256;
}

extern "C" int mcs_project_galerkin(const float* S, const float* Phi, int64_t V, int64_t K, float* out,
                                    void* ws, size_t ws_bytes, void* stream)
{
    if (!S || !Phi || !out || V < 1 || K < 1 || V > 65535 || K > 65535) return MCS_EINVAL;
    if (!ws || ws_bytes < mcs_project_workspace_bytes(V, K)) return MCS_ENOMEM;
    cudaStream_t st = (cudaStream_t)stream;
    float* Y = (float*)ws;                                                   // Y = S Phi  [V][K]
    const dim3 g1((unsigned)ceil_div64(K, GT), (unsigned)ceil_div64(V, GT));
    mcs_note_launch(), sgemm_kernel<false><<<g1, 256, 0, st>>>(S, Phi, Y, (int)V, (int)K, (int)V);
    const dim3 g2((unsigned)ceil_div64(K, GT), (unsigned)ceil_div64(K, GT));
    mcs_note_launch(), sgemm_kernel<true><<<g2, 256, 0, st>>>(Phi, Y, out, (int)K, (int)K, (int)V);      // Phi^T Y
    const dim3 g3((unsigned)ceil_div64(K, 16), (unsigned)ceil_div64(K, 16));
    mcs_note_launch(), symmetrise_kernel<<<g3, dim3(16, 16), 0, st>>>(out, (int)K);
    MCS_CUDA_TRY(cudaGetLastError());
    return MCS_OK;
}
