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

#include "sgemm.cuh"

// R = sum over z of P[z] (in order), then R = R + R^T: for U' = Phi^T Y' with the diagonal entries of S halved in Y'
__global__ void splitk_sum_symmetric_kernel(const float* __restrict__ P, int n_z, int K, float* __restrict__ R)
{
    const int i = blockIdx.y * 16 + threadIdx.y, j = blockIdx.x * 16 + threadIdx.x;
    if (i >= K || j >= K || i > j) return;
    float a = 0.0f, b = 0.0f;
    for (int z = 0; z < n_z; ++z) { a += P[((size_t)z * K + i) * K + j]; b += P[((size_t)z * K + j) * K + i]; }
    const float r = a + b;
    R[(size_t)i * K + j] = r; R[(size_t)j * K + i] = r;
}

// first entry of every row of a (row, col)-sorted COO list: row_ptr[r] = number of entries with row < r
__global__ void coo_row_ptr_kernel(const int32_t* __restrict__ row, long long nnz, long long V, int32_t* __restrict__ row_ptr, int* __restrict__ err)
{
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e > nnz) return;
    const long long prev = e == 0 ? -1 : row[e - 1];
    const long long cur = e == nnz ? V : row[e];
    if (cur < prev || cur > V || (e < nnz && cur >= V)) { *err = 1; return; }
    for (long long r = prev + 1; r <= cur; ++r) row_ptr[r] = (int32_t)e;
}

// Y'[r][:] = sum over the entries (r, c, v) of row r, in list order, of v Phi[c][:]  (diagonal entries halved).
// One warp per row, lanes over the K columns: no atomics, fixed order.
__global__ void __launch_bounds__(256)
coo_spmm_rows_kernel(const int32_t* __restrict__ row_ptr, const int32_t* __restrict__ col, const float* __restrict__ val,
                     const float* __restrict__ Phi, long long V, int K, float* __restrict__ Y, int* __restrict__ err)
{
    const long long r = (long long)blockIdx.x * 8 + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (r >= V) return;
    const int e0 = row_ptr[r], e1 = row_ptr[r + 1];
    for (int k0 = 0; k0 < K; k0 += 128) {                    // 4 columns per lane per sweep
        float acc[4] = { 0.f, 0.f, 0.f, 0.f };
        for (int e = e0; e < e1; ++e) {
            const int c = col[e];
            if (c < r || c >= V) { *err = 1; continue; }    // upper triangle expected
            const float v = (c == r ? 0.5f : 1.0f) * val[e];
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const int k = k0 + q * 32 + lane;
                if (k < K) acc[q] = fmaf(v, Phi[(size_t)c * K + k], acc[q]);
            }
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int k = k0 + q * 32 + lane;
            if (k < K) Y[(size_t)r * K + k] = acc[q];
        }
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
    mcs_note_launch(), sgemm_kernel<false><<<g1, 256, 0, st>>>(S, Phi, Y, (int)V, (int)K, (int)V, (int)V);
    const dim3 g2((unsigned)ceil_div64(K, GT), (unsigned)ceil_div64(K, GT));
    mcs_note_launch(), sgemm_kernel<true><<<g2, 256, 0, st>>>(Phi, Y, out, (int)K, (int)K, (int)V, (int)V);      // Phi^T Y
    const dim3 g3((unsigned)ceil_div64(K, 16), (unsigned)ceil_div64(K, 16));
    mcs_note_launch(), symmetrise_kernel<<<g3, dim3(16, 16), 0, st>>>(out, (int)K);
    MCS_CUDA_TRY(cudaGetLastError());
    return MCS_OK;
}

// The same matrix from the sparse output (mcs_matrix kind 1: upper triangle, sorted by (row, col), one entry per
// position): R = U' + U'^T with U' = Phi^T Y', Y' = S_upper Phi with the diagonal halved.  Y' by one warp per row
// (segments of the sorted list), U' by a split-K product whose partial matrices are added in order: deterministic.
static int coo_split(long long V, long long K)
{
    const long long tiles = ceil_div64(K, GT) * ceil_div64(K, GT);
    long long z = ceil_div64(4 * 148, tiles);
    const long long most = ceil_div64(V, 8 * GK);
    if (z > most) z = most;
    if (z > 512) z = 512;
    return (int)(z < 1 ? 1 : z);
}

extern "C" size_t mcs_project_coo_workspace_bytes(int64_t V, int64_t K)
{
    if (V < 1 || K < 1) return 0;
    return align_up((size_t)(V + 2) * 4) + align_up((size_t)V * K * 4) + align_up((size_t)coo_split(V, K) * K * K * 4) + 256;
}

extern "C" int mcs_project_galerkin_coo(const int32_t* row, const int32_t* col, const float* val, int64_t nnz,
                                        const float* Phi, int64_t V, int64_t K, float* out,
                                        void* ws, size_t ws_bytes, void* stream)
{
    if (!Phi || !out || V < 1 || K < 1 || K > 65535 || nnz < 0 || nnz >= ((int64_t)1 << 31) || V >= ((int64_t)1 << 31)) return MCS_EINVAL;
    if (nnz > 0 && (!row || !col || !val)) return MCS_EINVAL;
    if (!ws || ws_bytes < mcs_project_coo_workspace_bytes(V, K)) return MCS_ENOMEM;
    cudaStream_t st = (cudaStream_t)stream;
    char* p = (char*)ws;
    int32_t* row_ptr = (int32_t*)p;  p += align_up((size_t)(V + 2) * 4);
    float* Y = (float*)p;            p += align_up((size_t)V * K * 4);
    float* partial = (float*)p;      p += align_up((size_t)coo_split(V, K) * K * K * 4);
    int* err = (int*)p;
    MCS_CUDA_TRY(cudaMemsetAsync(err, 0, 4, st));
    mcs_note_launch(), coo_row_ptr_kernel<<<(unsigned)ceil_div64(nnz + 1, 256), 256, 0, st>>>(row, nnz, V, row_ptr, err);
    mcs_note_launch(), coo_spmm_rows_kernel<<<(unsigned)ceil_div64(V, 8), 256, 0, st>>>(row_ptr, col, val, Phi, V, (int)K, Y, err);
    const int n_z = coo_split(V, K);
    const int k_per_z = (int)(ceil_div64(ceil_div64(V, n_z), GK) * GK);
    const dim3 g((unsigned)ceil_div64(K, GT), (unsigned)ceil_div64(K, GT), (unsigned)n_z);
    mcs_note_launch(), sgemm_kernel<true><<<g, 256, 0, st>>>(Phi, Y, partial, (int)K, (int)K, (int)V, k_per_z);
    const dim3 g3((unsigned)ceil_div64(K, 16), (unsigned)ceil_div64(K, 16));
    mcs_note_launch(), splitk_sum_symmetric_kernel<<<g3, dim3(16, 16), 0, st>>>(partial, n_z, (int)K, out);
    int h_err = 0;
    MCS_CUDA_TRY(cudaMemcpyAsync(&h_err, err, 4, cudaMemcpyDeviceToHost, st));
    MCS_CUDA_TRY(cudaStreamSynchronize(st));
    return h_err ? MCS_EINVAL : MCS_OK;
}
