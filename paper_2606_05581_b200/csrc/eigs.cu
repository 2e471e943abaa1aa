// eigs.cu -- smallest Steklov eigenpairs of an estimated DtN matrix:
//     S psi = lambda M psi,   M = diag(mass)  (lumped boundary mass).
// With A = M^-1/2 S M^-1/2 (symmetric, PSD up to Monte Carlo noise) the problem is the ordinary symmetric one.
// A is diagonalised by one-sided Jacobi (Hestenes) on the ROWS of G = A: plane rotations that make pairs of
// rows orthogonal are applied to G and accumulated in Q (initially I).  At convergence the rows of G are
// mutually orthogonal, so Q A A^T Q^T is diagonal: the rows of Q are eigenvectors of A and |lambda_i| = |g_i|.
// The sign comes from the Rayleigh quotient g_i . q_i.  Every round of a sweep rotates K/2 disjoint row pairs
// (round-robin tournament), one thread block per pair, all pairs of all matrices of a batch in one launch; a
// rotation reads and writes two contiguous rows of G and of Q (coalesced), nothing else.
// fp32 throughout; Jacobi's rotations are orthogonal to rounding, so eigenvalues are good to ~1e-6 |A|.
#include "common.cuh"

#include <string.h>

namespace {

constexpr int ET = 256;

struct EigArgs {
    float* G;           // [B][K][K]
    float* Q;           // [B][K][K]
    long long K;
    int Kp;             // K rounded up to even (a dummy player sits out)
    int round;
    unsigned* not_converged;   // [1]: max over pairs of |gamma| / sqrt(alpha beta) > tol
    const unsigned* scale_bits; // [B]: bits of max_i |A_ii| (rows below 1e-6 of it are null rows)
    float tol;
};

__device__ __forceinline__ float block_sum(float v, float* s_red)
{
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, o);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    __syncthreads();
    if (lane == 0) s_red[warp] = v;
    __syncthreads();
    float t = 0.0f;
    for (int w = 0; w < ET / 32; ++w) t += s_red[w];      // fixed order: deterministic
    return t;
}

// A = M^-1/2 S M^-1/2 symmetrised, Q = I
__global__ void __launch_bounds__(ET)
eig_init_kernel(const float* __restrict__ S, const float* __restrict__ mass, long long K, float* __restrict__ G, float* __restrict__ Q)
{
    const long long b = blockIdx.y;
    const long long i = (long long)blockIdx.x * ET + threadIdx.x;
    if (i >= K * K) return;
    const long long r = i / K, c = i - r * K;
    const float* Sb = S + b * K * K;
    const float* mb = mass + b * K;
    const float a = 0.5f * (Sb[r * K + c] + Sb[c * K + r]) * rsqrtf(mb[r]) * rsqrtf(mb[c]);
    G[b * K * K + i] = a;
    Q[b * K * K + i] = r == c ? 1.0f : 0.0f;
}

__global__ void __launch_bounds__(ET)
eig_scale_kernel(const float* __restrict__ G, long long K, unsigned* __restrict__ scale_bits)
{
    const long long b = blockIdx.y;
    const long long i = (long long)blockIdx.x * ET + threadIdx.x;
    if (i >= K) return;
    atomicMax(&scale_bits[b], __float_as_uint(fabsf(G[(b * K + i) * K + i])));      // non-negative floats order as unsigned
}

// round-robin tournament: pair `i` of round `r` among Kp (even) players
__device__ __forceinline__ void tournament_pair(int Kp, int r, int i, int& p, int& q)
{
    const int m = Kp - 1;
    if (i == 0) { p = m; q = r % m; }
    else { p = (r + i) % m; q = (r + m - i) % m; }
    if (p > q) { const int t = p; p = q; q = t; }
}

__global__ void __launch_bounds__(ET)
eig_rotate_kernel(EigArgs a)
{
    __shared__ float s_red[ET / 32];
    const long long b = blockIdx.y;
    int p, q;
    tournament_pair(a.Kp, a.round, blockIdx.x, p, q);
    if (q >= a.K) return;                                   // the dummy player of an odd K
    float* gp = a.G + (b * a.K + p) * a.K;
    float* gq = a.G + (b * a.K + q) * a.K;
    float al = 0.0f, be = 0.0f, ga = 0.0f;
    for (long long j = threadIdx.x; j < a.K; j += ET) {
        const float x = gp[j], y = gq[j];
        al = fmaf(x, x, al); be = fmaf(y, y, be); ga = fmaf(x, y, ga);
    }
    al = block_sum(al, s_red); be = block_sum(be, s_red); ga = block_sum(ga, s_red);
    const float den = sqrtf(al * be);
    const float nul = 1e-6f * __uint_as_float(a.scale_bits[b]);
    if (al < nul * nul || be < nul * nul) return;            // a null row (eigenvalue 0 to fp32): orthogonal to everything
    if (!(fabsf(ga) > a.tol * den)) return;                  // already orthogonal
    if (threadIdx.x == 0) *a.not_converged = 1u;
    // rotation that zeroes g_p . g_q
    const float zeta = (be - al) / (2.0f * ga);
    const float t = copysignf(1.0f, zeta) / (fabsf(zeta) + sqrtf(fmaf(zeta, zeta, 1.0f)));
    const float c = 1.0f / sqrtf(fmaf(t, t, 1.0f)), s = c * t;       // correctly rounded: c^2 + s^2 stays at 1 over many rotations
    float* qp = a.Q + (b * a.K + p) * a.K;
    float* qq = a.Q + (b * a.K + q) * a.K;
    for (long long j = threadIdx.x; j < a.K; j += ET) {
        const float x = gp[j], y = gq[j];
        gp[j] = fmaf(c, x, -s * y); gq[j] = fmaf(s, x, c * y);
        const float u = qp[j], v = qq[j];
        qp[j] = fmaf(c, u, -s * v); qq[j] = fmaf(s, u, c * v);
    }
}

// Blocked form of the same sweep.  Rows are grouped in blocks of BR; a thread block takes a PAIR of row blocks
// (outer round-robin over the blocks), stages their 2 BR rows of G and of Q in shared memory, and runs a complete
// inner tournament over those rows -- 2 BR - 1 rounds, one warp per row pair, lanes strided over the row so that
// shared-memory accesses are conflict-free -- before writing the rows back.  Global traffic per sweep drops from
// 16 K^3 bytes to 16 K^3 / BR; the rotations themselves are unchanged (same formulas, same thresholds).
template <int BR>
__global__ void __launch_bounds__(32 * BR)
eig_block_rotate_kernel(EigArgs a, int nblk_p)
{
    extern __shared__ float s_rows[];                        // [2 BR][K] of G, then [2 BR][K] of Q
    const long long K = a.K, b = blockIdx.y;
    float* sG = s_rows;
    float* sQ = s_rows + 2 * BR * K;
    int I, J;
    tournament_pair(nblk_p, a.round, blockIdx.x, I, J);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    auto global_row = [&](int r) -> long long {               // slot r of the staged rows -> row of the matrix, or -1
        const long long g = (long long)(r < BR ? I : J) * BR + (r < BR ? r : r - BR);
        return g < K ? g : -1;
    };
    for (int r = warp; r < 2 * BR; r += BR) {
        const long long g = global_row(r);
        if (g < 0) continue;
        const float* src_g = a.G + (b * K + g) * K;
        const float* src_q = a.Q + (b * K + g) * K;
        for (long long j = lane; j < K; j += 32) { sG[r * K + j] = src_g[j]; sQ[r * K + j] = src_q[j]; }
    }
    __syncthreads();
    const float nul = 1e-6f * __uint_as_float(a.scale_bits[b]);
    bool rotated = false;
    for (int round = 0; round < 2 * BR - 1; ++round) {
        int p, q;
        tournament_pair(2 * BR, round, warp, p, q);
        if (global_row(p) >= 0 && global_row(q) >= 0) {
            float* gp = sG + p * K;
            float* gq = sG + q * K;
            float al = 0.0f, be = 0.0f, ga = 0.0f;
            for (long long j = lane; j < K; j += 32) {
                const float x = gp[j], y = gq[j];
                al = fmaf(x, x, al); be = fmaf(y, y, be); ga = fmaf(x, y, ga);
            }
            for (int o = 16; o > 0; o >>= 1) {
                al += __shfl_xor_sync(0xFFFFFFFFu, al, o);
                be += __shfl_xor_sync(0xFFFFFFFFu, be, o);
                ga += __shfl_xor_sync(0xFFFFFFFFu, ga, o);
            }
            if (!(al < nul * nul || be < nul * nul) && fabsf(ga) > a.tol * sqrtf(al * be)) {
                rotated = true;
                const float zeta = (be - al) / (2.0f * ga);
                const float t = copysignf(1.0f, zeta) / (fabsf(zeta) + sqrtf(fmaf(zeta, zeta, 1.0f)));
                const float c = 1.0f / sqrtf(fmaf(t, t, 1.0f)), sn = c * t;
                float* qp = sQ + p * K;
                float* qq = sQ + q * K;
                for (long long j = lane; j < K; j += 32) {
                    const float x = gp[j], y = gq[j];
                    gp[j] = fmaf(c, x, -sn * y); gq[j] = fmaf(sn, x, c * y);
                    const float u = qp[j], v = qq[j];
                    qp[j] = fmaf(c, u, -sn * v); qq[j] = fmaf(sn, u, c * v);
                }
            }
        }
        __syncthreads();
    }
    if (rotated && lane == 0) *a.not_converged = 1u;
    for (int r = warp; r < 2 * BR; r += BR) {
        const long long g = global_row(r);
        if (g < 0) continue;
        float* dst_g = a.G + (b * K + g) * K;
        float* dst_q = a.Q + (b * K + g) * K;
        for (long long j = lane; j < K; j += 32) { dst_g[j] = sG[r * K + j]; dst_q[j] = sQ[r * K + j]; }
    }
}

// The same blocked sweep for K <= 128 NV with the row stride fixed at compile time (128 NV floats, zero padded):
// a lane holds its 4 NV elements of both rows in registers between the dot products and the rotation, and every
// shared-memory access is a conflict-free 128-bit one.
template <int BR, int NV>
__global__ void __launch_bounds__(32 * BR)
eig_block_rotate_vec_kernel(EigArgs a, int nblk_p)
{
    extern __shared__ float4 s_rows4[];                      // [2 BR][32 NV] float4 of G, then of Q
    constexpr int RS = 32 * NV;                              // row stride in float4
    const long long K = a.K, b = blockIdx.y;
    float4* sG = s_rows4;
    float4* sQ = s_rows4 + 2 * BR * RS;
    int I, J;
    tournament_pair(nblk_p, a.round, blockIdx.x, I, J);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    auto global_row = [&](int r) -> long long {
        const long long g = (long long)(r < BR ? I : J) * BR + (r < BR ? r : r - BR);
        return g < K ? g : -1;
    };
    for (int r = warp; r < 2 * BR; r += BR) {
        const long long g = global_row(r);
        if (g < 0) continue;
        const float* src_g = a.G + (b * K + g) * K;
        const float* src_q = a.Q + (b * K + g) * K;
        float* dg = (float*)(sG + r * RS);
        float* dq = (float*)(sQ + r * RS);
        for (int j = lane; j < 4 * RS; j += 32) { dg[j] = j < K ? src_g[j] : 0.0f; dq[j] = j < K ? src_q[j] : 0.0f; }
    }
    __syncthreads();
    const float nul = 1e-6f * __uint_as_float(a.scale_bits[b]);
    bool rotated = false;
    for (int round = 0; round < 2 * BR - 1; ++round) {
        int p, q;
        tournament_pair(2 * BR, round, warp, p, q);
        if (global_row(p) >= 0 && global_row(q) >= 0) {
            float4* gp = sG + p * RS + lane;
            float4* gq = sG + q * RS + lane;
            float4 x[NV], y[NV];
            float al = 0.0f, be = 0.0f, ga = 0.0f;
#pragma unroll
            for (int i = 0; i < NV; ++i) { x[i] = gp[32 * i]; y[i] = gq[32 * i]; }
#pragma unroll
            for (int i = 0; i < NV; ++i) {
                al = fmaf(x[i].x, x[i].x, al); be = fmaf(y[i].x, y[i].x, be); ga = fmaf(x[i].x, y[i].x, ga);
                al = fmaf(x[i].y, x[i].y, al); be = fmaf(y[i].y, y[i].y, be); ga = fmaf(x[i].y, y[i].y, ga);
                al = fmaf(x[i].z, x[i].z, al); be = fmaf(y[i].z, y[i].z, be); ga = fmaf(x[i].z, y[i].z, ga);
                al = fmaf(x[i].w, x[i].w, al); be = fmaf(y[i].w, y[i].w, be); ga = fmaf(x[i].w, y[i].w, ga);
            }
            for (int o = 16; o > 0; o >>= 1) {
                al += __shfl_xor_sync(0xFFFFFFFFu, al, o);
                be += __shfl_xor_sync(0xFFFFFFFFu, be, o);
                ga += __shfl_xor_sync(0xFFFFFFFFu, ga, o);
            }
            if (!(al < nul * nul || be < nul * nul) && fabsf(ga) > a.tol * sqrtf(al * be)) {
                rotated = true;
                const float zeta = (be - al) / (2.0f * ga);
                const float t = copysignf(1.0f, zeta) / (fabsf(zeta) + sqrtf(fmaf(zeta, zeta, 1.0f)));
                const float c = 1.0f / sqrtf(fmaf(t, t, 1.0f)), sn = c * t;
                auto rot = [&](float4 u, float4 v, float4& ru, float4& rv) {
                    ru.x = fmaf(c, u.x, -sn * v.x); rv.x = fmaf(sn, u.x, c * v.x);
                    ru.y = fmaf(c, u.y, -sn * v.y); rv.y = fmaf(sn, u.y, c * v.y);
                    ru.z = fmaf(c, u.z, -sn * v.z); rv.z = fmaf(sn, u.z, c * v.z);
                    ru.w = fmaf(c, u.w, -sn * v.w); rv.w = fmaf(sn, u.w, c * v.w);
                };
                float4* qp = sQ + p * RS + lane;
                float4* qq = sQ + q * RS + lane;
#pragma unroll
                for (int i = 0; i < NV; ++i) {
                    float4 ru, rv;
                    rot(x[i], y[i], ru, rv);
                    gp[32 * i] = ru; gq[32 * i] = rv;
                    rot(qp[32 * i], qq[32 * i], ru, rv);
                    qp[32 * i] = ru; qq[32 * i] = rv;
                }
            }
        }
        __syncthreads();
    }
    if (rotated && lane == 0) *a.not_converged = 1u;
    for (int r = warp; r < 2 * BR; r += BR) {
        const long long g = global_row(r);
        if (g < 0) continue;
        float* dst_g = a.G + (b * K + g) * K;
        float* dst_q = a.Q + (b * K + g) * K;
        const float* sg = (const float*)(sG + r * RS);
        const float* sq = (const float*)(sQ + r * RS);
        for (int j = lane; j < K; j += 32) { dst_g[j] = sg[j]; dst_q[j] = sq[j]; }
    }
}

template <int BR, int NV>
int eig_block_sweep_vec(EigArgs a, int64_t batch, cudaStream_t st)
{
    const size_t smem = (size_t)4 * BR * 128 * NV * sizeof(float);
    static bool attr_set = false;
    if (!attr_set) {
        MCS_CUDA_TRY(cudaFuncSetAttribute(eig_block_rotate_vec_kernel<BR, NV>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        attr_set = true;
    }
    const int nblk = (int)ceil_div64(a.K, BR);
    const int nblk_p = nblk < 2 ? 2 : nblk + (nblk & 1);
    for (int r = 0; r < nblk_p - 1; ++r) {
        a.round = r;
        mcs_note_launch(), eig_block_rotate_vec_kernel<BR, NV><<<dim3((unsigned)(nblk_p / 2), (unsigned)batch), 32 * BR, smem, st>>>(a, nblk_p);
    }
    return MCS_OK;
}

// Gram form of the blocked sweep (K <= 768).  For the 32 staged rows X of G the inner tournament is run on their
// 32 x 32 Gram matrix W = X X^T instead of on the rows: a one-sided rotation of rows p, q is the two-sided rotation
// W <- R W R^T (same alpha = W_pp, beta = W_qq, gamma = W_pq, same c and s), so the same rotations come out, at
// 32 numbers per row instead of K.  They are accumulated in J (32 x 32); the rows of G and of Q are then updated
// once, X <- J X, Q <- J Q, as register-tiled products written straight to global memory.  Shared-memory traffic
// per block pair: about 25 passes over the staged rows instead of 250.  Convergence is judged on the freshly
// computed Gram matrix of every visit, so rounding inside W cannot accumulate from visit to visit.
template <int NV>
__global__ void __launch_bounds__(512)
eig_block_gram_kernel(EigArgs a, int nblk_p)
{
    constexpr int BR = 16, R2 = 32, RS = 32 * NV;             // rows per block, staged rows, row stride in float4
    extern __shared__ float4 s_rows4[];
    float4* sX = s_rows4;
    float4* sQ = s_rows4 + R2 * RS;
    float (*sW)[R2 + 1] = reinterpret_cast<float (*)[R2 + 1]>(s_rows4 + 2 * R2 * RS);
    float (*sJ)[R2 + 1] = sW + R2;
    const long long K = a.K, b = blockIdx.y;
    int I, Jb;
    tournament_pair(nblk_p, a.round, blockIdx.x, I, Jb);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    auto global_row = [&](int r) -> long long {
        const long long g = (long long)(r < BR ? I : Jb) * BR + (r < BR ? r : r - BR);
        return g < K ? g : -1;
    };
    for (int r = warp; r < R2; r += BR) {
        const long long g = global_row(r);
        float* dg = (float*)(sX + r * RS);
        float* dq = (float*)(sQ + r * RS);
        if (g < 0) { for (int j = lane; j < 4 * RS; j += 32) { dg[j] = 0.0f; dq[j] = 0.0f; } continue; }
        const float* src_g = a.G + (b * K + g) * K;
        const float* src_q = a.Q + (b * K + g) * K;
        if ((K & 3) == 0) {                                   // rows are 16-byte aligned: 128-bit loads
            const float4 z4 = make_float4(0.f, 0.f, 0.f, 0.f);
            for (int j = lane; j < RS; j += 32) {
                const bool in = 4 * j < K;
                sX[r * RS + j] = in ? reinterpret_cast<const float4*>(src_g)[j] : z4;
                sQ[r * RS + j] = in ? reinterpret_cast<const float4*>(src_q)[j] : z4;
            }
        } else {
            for (int j = lane; j < 4 * RS; j += 32) { dg[j] = j < K ? src_g[j] : 0.0f; dq[j] = j < K ? src_q[j] : 0.0f; }
        }
    }
    for (int i = threadIdx.x; i < R2 * (R2 + 1); i += 512) { (&sJ[0][0])[i] = 0.0f; }
    __syncthreads();
    if (threadIdx.x < R2) sJ[threadIdx.x][threadIdx.x] = 1.0f;
    // W = X X^T: warp w owns rows w and w + 16 (kept in registers), against every row j >= its own
    for (int i = warp; i < R2; i += BR) {
        float4 x[NV];
#pragma unroll
        for (int v = 0; v < NV; ++v) x[v] = sX[i * RS + lane + 32 * v];
        for (int j0 = i; j0 < R2; j0 += 4) {                  // four dot products in flight
            float d[4] = { 0.f, 0.f, 0.f, 0.f };
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int j = j0 + u < R2 ? j0 + u : R2 - 1;
#pragma unroll
                for (int v = 0; v < NV; ++v) {
                    const float4 y = sX[j * RS + lane + 32 * v];
                    d[u] = fmaf(x[v].x, y.x, d[u]); d[u] = fmaf(x[v].y, y.y, d[u]); d[u] = fmaf(x[v].z, y.z, d[u]); d[u] = fmaf(x[v].w, y.w, d[u]);
                }
            }
            for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
                for (int u = 0; u < 4; ++u) d[u] += __shfl_xor_sync(0xFFFFFFFFu, d[u], o);
            }
            if (lane < 4 && j0 + lane < R2) { const float dv = lane == 0 ? d[0] : lane == 1 ? d[1] : lane == 2 ? d[2] : d[3]; sW[i][j0 + lane] = dv; sW[j0 + lane][i] = dv; }
        }
    }
    __syncthreads();
    const float nul = 1e-6f * __uint_as_float(a.scale_bits[b]);
    bool rotated = false;
    for (int round = 0; round < R2 - 1; ++round) {
        int p = 0, q = 1;
        float c = 1.0f, sn = 0.0f;
        if (warp < BR) {
            tournament_pair(R2, round, warp, p, q);
            const float al = sW[p][p], be = sW[q][q], ga = sW[p][q];
            if (global_row(p) >= 0 && global_row(q) >= 0 && !(al < nul * nul || be < nul * nul) && fabsf(ga) > a.tol * sqrtf(al * be)) {
                rotated = true;
                const float zeta = (be - al) / (2.0f * ga);
                const float t = copysignf(1.0f, zeta) / (fabsf(zeta) + sqrtf(fmaf(zeta, zeta, 1.0f)));
                c = 1.0f / sqrtf(fmaf(t, t, 1.0f)); sn = c * t;
            }
        }
        __syncthreads();                                      // every pair has read its alpha, beta, gamma
        if (sn != 0.0f) {                                     // rows p, q of W and of J (lane = column)
            const float wp = sW[p][lane], wq = sW[q][lane];
            sW[p][lane] = fmaf(c, wp, -sn * wq); sW[q][lane] = fmaf(sn, wp, c * wq);
            const float jp = sJ[p][lane], jq = sJ[q][lane];
            sJ[p][lane] = fmaf(c, jp, -sn * jq); sJ[q][lane] = fmaf(sn, jp, c * jq);
        }
        __syncthreads();
        if (sn != 0.0f) {                                     // columns p, q of W (lane = row)
            const float wp = sW[lane][p], wq = sW[lane][q];
            sW[lane][p] = fmaf(c, wp, -sn * wq); sW[lane][q] = fmaf(sn, wp, c * wq);
        }
        __syncthreads();
    }
    if (rotated && lane == 0) *a.not_converged = 1u;
    const unsigned any = __syncthreads_or(rotated ? 1 : 0);
    if (!any) return;                                         // nothing rotated in this block pair: rows unchanged
    // X <- J X, Q <- J Q: warp w computes output rows w and w + 16 over all columns, reading every staged row once
    for (int m = 0; m < 2; ++m) {
        const float4* src = m == 0 ? sX : sQ;
        float* dst_base = m == 0 ? a.G : a.Q;
        float4 acc0[NV], acc1[NV];
#pragma unroll
        for (int v = 0; v < NV; ++v) { acc0[v] = make_float4(0.f, 0.f, 0.f, 0.f); acc1[v] = acc0[v]; }
        for (int j = 0; j < R2; ++j) {
            const float j0 = sJ[warp][j], j1 = sJ[warp + BR][j];
#pragma unroll
            for (int v = 0; v < NV; ++v) {
                const float4 y = src[j * RS + lane + 32 * v];
                acc0[v].x = fmaf(j0, y.x, acc0[v].x); acc0[v].y = fmaf(j0, y.y, acc0[v].y); acc0[v].z = fmaf(j0, y.z, acc0[v].z); acc0[v].w = fmaf(j0, y.w, acc0[v].w);
                acc1[v].x = fmaf(j1, y.x, acc1[v].x); acc1[v].y = fmaf(j1, y.y, acc1[v].y); acc1[v].z = fmaf(j1, y.z, acc1[v].z); acc1[v].w = fmaf(j1, y.w, acc1[v].w);
            }
        }
#pragma unroll
        for (int half = 0; half < 2; ++half) {
            const long long g = global_row(warp + half * BR);
            if (g < 0) continue;
            float* dst = dst_base + (b * K + g) * K;
#pragma unroll
            for (int v = 0; v < NV; ++v) {
                const float4 o = half == 0 ? acc0[v] : acc1[v];
                const int col = 4 * (lane + 32 * v);
                if ((K & 3) == 0) { if (col < K) reinterpret_cast<float4*>(dst)[lane + 32 * v] = o; continue; }
                if (col < K) dst[col] = o.x;
                if (col + 1 < K) dst[col + 1] = o.y;
                if (col + 2 < K) dst[col + 2] = o.z;
                if (col + 3 < K) dst[col + 3] = o.w;
            }
        }
    }
}

template <int NV>
int eig_block_sweep_gram(EigArgs a, int64_t batch, cudaStream_t st)
{
    const size_t smem = (size_t)4 * 16 * 128 * NV * sizeof(float) + (size_t)2 * 32 * 33 * sizeof(float);
    static bool attr_set = false;
    if (!attr_set) {
        MCS_CUDA_TRY(cudaFuncSetAttribute(eig_block_gram_kernel<NV>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        attr_set = true;
    }
    const int nblk = (int)ceil_div64(a.K, 16);
    const int nblk_p = nblk < 2 ? 2 : nblk + (nblk & 1);
    for (int r = 0; r < nblk_p - 1; ++r) {
        a.round = r;
        mcs_note_launch(), eig_block_gram_kernel<NV><<<dim3((unsigned)(nblk_p / 2), (unsigned)batch), 512, smem, st>>>(a, nblk_p);
    }
    return MCS_OK;
}

template <int BR>
int eig_block_sweep(EigArgs a, int64_t batch, cudaStream_t st)
{
    const size_t smem = (size_t)4 * BR * a.K * sizeof(float);
    static bool attr_set = false;
    if (!attr_set) {
        MCS_CUDA_TRY(cudaFuncSetAttribute(eig_block_rotate_kernel<BR>, cudaFuncAttributeMaxDynamicSharedMemorySize, 220 * 1024));
        attr_set = true;
    }
    const int nblk = (int)ceil_div64(a.K, BR);
    const int nblk_p = nblk < 2 ? 2 : nblk + (nblk & 1);
    for (int r = 0; r < nblk_p - 1; ++r) {
        a.round = r;
        mcs_note_launch(), eig_block_rotate_kernel<BR><<<dim3((unsigned)(nblk_p / 2), (unsigned)batch), 32 * BR, smem, st>>>(a, nblk_p);
    }
    return MCS_OK;
}

// lambda_i = g_i . q_i / q_i . q_i (Rayleigh quotient); sort key = order-preserving bits of lambda
__global__ void __launch_bounds__(ET)
eig_values_kernel(const float* __restrict__ G, const float* __restrict__ Q, long long K, float* __restrict__ lam,
                  uint32_t* __restrict__ keys, uint32_t* __restrict__ vals)
{
    __shared__ float s_red[ET / 32];
    const long long b = blockIdx.y, i = blockIdx.x;
    const float* g = G + (b * K + i) * K;
    const float* q = Q + (b * K + i) * K;
    float v = 0.0f, n2 = 0.0f;
    for (long long j = threadIdx.x; j < K; j += ET) { v = fmaf(g[j], q[j], v); n2 = fmaf(q[j], q[j], n2); }
    v = block_sum(v, s_red); n2 = block_sum(n2, s_red);
    v /= n2;                                                 // |q| drifts from 1 by rounding over ~K sweeps rotations
    if (threadIdx.x == 0) {
        lam[b * K + i] = v;
        const uint32_t u = __float_as_uint(v);
        keys[b * K + i] = (u & 0x80000000u) ? ~u : (u | 0x80000000u);      // total order of floats as unsigned
        vals[b * K + i] = (uint32_t)i;
    }
}

// psi_e = M^-1/2 q_(order[e]) : M-orthonormal eigenvectors (q renormalised)
__global__ void __launch_bounds__(ET)
eig_vectors_kernel(const float* __restrict__ Q, const float* __restrict__ mass, const float* __restrict__ lam,
                   const uint32_t* __restrict__ order, long long K, int n_eig, float* __restrict__ evals, float* __restrict__ evecs)
{
    __shared__ float s_red[ET / 32];
    __shared__ float s_sign;
    const long long b = blockIdx.y;
    const int e = blockIdx.x;
    const long long i = order[b * K + e];
    const float* q = Q + (b * K + i) * K;
    // sign convention: make sum_j q_j^3 positive (a smooth, deterministic rule); falls back to + when it vanishes
    float v = 0.0f, n2 = 0.0f;
    for (long long j = threadIdx.x; j < K; j += ET) { v += q[j] * q[j] * q[j]; n2 = fmaf(q[j], q[j], n2); }
    v = block_sum(v, s_red); n2 = block_sum(n2, s_red);
    if (threadIdx.x == 0) { s_sign = (v < 0.0f ? -1.0f : 1.0f) / sqrtf(n2); evals[b * n_eig + e] = lam[b * K + i]; }
    __syncthreads();
    const float sg = s_sign;
    for (long long j = threadIdx.x; j < K; j += ET)
        evecs[(b * n_eig + e) * K + j] = sg * q[j] * rsqrtf(mass[b * K + j]);
}

}  // namespace

// Sorts the K (key, index) pairs of one matrix per block: bitonic network on 64-bit (key << 32 | index) words in shared
// memory, so equal keys keep index order (what the stable radix sort gave).
__global__ void __launch_bounds__(256)
eig_sort_kernel(uint32_t* __restrict__ keys, uint32_t* __restrict__ vals, int K, int P)
{
    extern __shared__ unsigned long long s_kv[];
    uint32_t* k = keys + (size_t)blockIdx.x * K;
    uint32_t* v = vals + (size_t)blockIdx.x * K;
    for (int i = threadIdx.x; i < P; i += blockDim.x)
        s_kv[i] = i < K ? ((unsigned long long)k[i] << 32) | (unsigned long long)v[i] : ~0ull;
    __syncthreads();
    for (int size = 2; size <= P; size <<= 1)
        for (int stride = size >> 1; stride > 0; stride >>= 1) {
            for (int i = threadIdx.x; i < P; i += blockDim.x) {
                const int j = i ^ stride;
                if (j > i) {
                    const unsigned long long a = s_kv[i], b = s_kv[j];
                    const bool up = (i & size) == 0;
                    if ((a > b) == up) { s_kv[i] = b; s_kv[j] = a; }
                }
            }
            __syncthreads();
        }
    for (int i = threadIdx.x; i < K; i += blockDim.x) { k[i] = (uint32_t)(s_kv[i] >> 32); v[i] = (uint32_t)s_kv[i]; }
}

extern "C" size_t mcs_steklov_eigs_workspace_bytes(int64_t K, int64_t batch)
{
    if (K < 1 || batch < 1) return 0;
    const size_t n = (size_t)batch * K;
    return 2 * align_up((size_t)batch * K * K * 4) + align_up(n * 4) * 3 + align_up(sort_workspace_bytes(K, 4)) +
           align_up((size_t)batch * 4) + 1024;
}

extern "C" int mcs_steklov_eigs(const float* S, const float* mass, int64_t K, int64_t batch, int32_t n_eig,
                                float* evals, float* evecs, void* ws, size_t ws_bytes, int32_t* sweeps_out, void* stream)
{
    if (!S || !mass || !evals || K < 1 || batch < 1 || n_eig < 1 || n_eig > K || K > 16384) return MCS_EINVAL;
    if (!ws || ws_bytes < mcs_steklov_eigs_workspace_bytes(K, batch)) return MCS_ENOMEM;
    cudaStream_t st = (cudaStream_t)stream;
    char* p = (char*)ws;
    float* G = (float*)p;           p += align_up((size_t)batch * K * K * 4);
    float* Q = (float*)p;           p += align_up((size_t)batch * K * K * 4);
    float* lam = (float*)p;         p += align_up((size_t)batch * K * 4);
    uint32_t* keys = (uint32_t*)p;  p += align_up((size_t)batch * K * 4);
    uint32_t* vals = (uint32_t*)p;  p += align_up((size_t)batch * K * 4);
    void* sort_ws = p;              p += align_up(sort_workspace_bytes(K, 4));
    unsigned* scale_bits = (unsigned*)p; p += align_up((size_t)batch * 4);
    unsigned* flag = (unsigned*)p;

    const dim3 g_init((unsigned)ceil_div64(K * K, ET), (unsigned)batch);
    mcs_note_launch(), eig_init_kernel<<<g_init, ET, 0, st>>>(S, mass, K, G, Q);
    EigArgs a;
    MCS_CUDA_TRY(cudaMemsetAsync(scale_bits, 0, (size_t)batch * 4, st));
    mcs_note_launch(), eig_scale_kernel<<<dim3((unsigned)ceil_div64(K, ET), (unsigned)batch), ET, 0, st>>>(G, K, scale_bits);
    a.G = G; a.Q = Q; a.K = K; a.Kp = (int)(K + (K & 1)); a.not_converged = flag; a.scale_bits = scale_bits;
    a.tol = fmaxf(1e-6f, 2e-7f * sqrtf((float)K));           // fp32 dot products of length K cannot resolve less
    int sweep = 0;
    unsigned last_flag = 0;
    const int max_sweeps = 30;
    if (K > 1)
        for (; sweep < max_sweeps; ++sweep) {
            MCS_CUDA_TRY(cudaMemsetAsync(flag, 0, 4, st));
            // rows staged in shared memory while 2 x 2 BR rows fit (BR = 16 to K = 896, BR = 8 to K = 1760); else row pairs from L2/HBM
            int rc = MCS_OK;
            if (K <= 128) rc = eig_block_sweep_gram<1>(a, batch, st);
            else if (K <= 256) rc = eig_block_sweep_gram<2>(a, batch, st);
            else if (K <= 384) rc = eig_block_sweep_gram<3>(a, batch, st);
            else if (K <= 512) rc = eig_block_sweep_gram<4>(a, batch, st);
            else if (K <= 640) rc = eig_block_sweep_gram<5>(a, batch, st);
            else if (K <= 768) rc = eig_block_sweep_gram<6>(a, batch, st);
            else if (K <= 896) rc = eig_block_sweep_vec<16, 7>(a, batch, st);
            else if (K <= 1760) rc = eig_block_sweep<8>(a, batch, st);
            else
                for (int r = 0; r < a.Kp - 1; ++r) {
                    a.round = r;
                    mcs_note_launch(), eig_rotate_kernel<<<dim3((unsigned)(a.Kp / 2), (unsigned)batch), ET, 0, st>>>(a);
                }
            if (rc != MCS_OK) return rc;
            unsigned h = 0;
            MCS_CUDA_TRY(cudaMemcpyAsync(&h, flag, 4, cudaMemcpyDeviceToHost, st));
            MCS_CUDA_TRY(cudaStreamSynchronize(st));
            last_flag = h;
            if (!h) { ++sweep; break; }
        }
    if (sweeps_out) *sweeps_out = sweep;
    const bool converged = K <= 1 || sweep < max_sweeps || last_flag == 0;
    mcs_note_launch(), eig_values_kernel<<<dim3((unsigned)K, (unsigned)batch), ET, 0, st>>>(G, Q, K, lam, keys, vals);
    if (K <= 4096) {
        // one block per matrix: (eigenvalue, index) pairs sorted in shared memory -- the same order as the stable sort
        int P = 1; while (P < K) P <<= 1;
        mcs_note_launch(), eig_sort_kernel<<<(unsigned)batch, 256, (size_t)P * 8, st>>>(keys, vals, (int)K, P);
    } else
    for (int64_t b = 0; b < batch; ++b) {
        int rc = sort_pairs_u32(keys + b * K, vals + b * K, K, 32, sort_ws, sort_workspace_bytes(K, 4), st);
        if (rc != MCS_OK) return rc;
    }
    if (evecs)
        mcs_note_launch(), eig_vectors_kernel<<<dim3((unsigned)n_eig, (unsigned)batch), ET, 0, st>>>(Q, mass, lam, vals, K, n_eig, evals, evecs);
    else {
        // eigenvalues only: reuse the vector kernel's first part through a tiny launch writing into G's first row
        mcs_note_launch(), eig_vectors_kernel<<<dim3((unsigned)n_eig, (unsigned)batch), ET, 0, st>>>(Q, mass, lam, vals, K, n_eig, evals, G);
    }
    MCS_CUDA_TRY(cudaGetLastError());
    return converged ? MCS_OK : MCS_WNOTCONVERGED;
}
