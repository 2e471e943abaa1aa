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

#include <math.h>
#include <string.h>
#include <vector>

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

namespace {

// ---------------------------------------------------------------------------
// Large K, few eigenpairs: Chebyshev-filtered subspace iteration.
// One-sided Jacobi computes ALL K eigenpairs (O(K^3) per sweep: 0.52 s at K = 2562, out of reach at the 2^14 points of
// the paper's point-based discretisation); the applications want the lowest 64-128 modes (PAPER.md:357,
// 401).  For n_eig << K a block X [K][m] (m = n_eig + guard columns) is iterated instead:
//   filter      Y = p(A) X, p = the degree-d Chebyshev polynomial that is small on [a, b] (the unwanted part of the
//               spectrum: a = the largest Ritz value of the block, b >= lambda_max by Gershgorin) and grows fast below
//               a; three-term recurrence, one product A Y per degree, scaled so that nothing overflows;
//   orthonormalise  shifted Cholesky QR, three passes: G = Y^T Y (+ shift) = R^T R in one block, Y <- Y R^-1;
//   Rayleigh-Ritz   H = Y^T A Y = W Theta W^T (m x m, same solver), X <- Y W: Ritz pairs (Theta, X);
//   stop when the residuals |A x_i - theta_i x_i| of the n_eig lowest pairs are below tol * b.
// fp32 throughout.  The Gram matrix squares the condition number of Y, and the filter spreads the columns' scales by
// p(0) / p(a), so the degree is kept low enough (p(0) / p(a) <= ~1e3) for fp32 and the loop runs a few more times.
// (A first version orthonormalised through the eigen-decomposition of the Gram matrix, twice per iteration: three
// 1 ms Jacobi solves of an m x m matrix per iteration were 55 % of the run; Cholesky QR leaves one.)
// All products are the plain SIMT tiles of sgemm.cuh with split-K (the block is tall and thin: K/64 row tiles alone
// do not fill 148 SMs); a dense contraction on tensor cores would need TF32 inputs, which the filter tolerates but
// the Rayleigh-Ritz step does not -- left as fp32 CUDA cores (2 K^2 m flops per product: 1.7 GFLOP at K = 2562).
// ---------------------------------------------------------------------------
#include "sgemm.cuh"

// row sums of |A|: Gershgorin bound of the largest eigenvalue (max over rows; non-negative floats order like their bits)
__global__ void __launch_bounds__(ET)
sub_gershgorin_kernel(const float* __restrict__ A, long long K, unsigned* __restrict__ bound_bits)
{
    __shared__ float s_red[ET / 32];
    const float* row = A + (long long)blockIdx.x * K;
    float v = 0.0f;
    for (long long j = threadIdx.x; j < K; j += ET) v += fabsf(row[j]);
    v = block_sum(v, s_red);
    if (threadIdx.x == 0) atomicMax(bound_bits, __float_as_uint(v));
}

// deterministic start block: a hash of (row, column) mapped to (-1, 1)
__global__ void sub_init_kernel(float* __restrict__ X, long long n, unsigned seed)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    unsigned h = (unsigned)i * 0x9E3779B1u + seed;
    h ^= h >> 16; h *= 0x85EBCA6Bu; h ^= h >> 13; h *= 0xC2B2AE35u; h ^= h >> 16;
    X[i] = (float)(h >> 8) * (2.0f / 16777216.0f) - 1.0f;
}

// out = alpha * (P[0] + P[1] + ... in order) + beta * D1 + gamma * D2   (D1, D2 may be NULL; out may alias D2)
__global__ void sub_combine_kernel(const float* __restrict__ P, int n_z, long long n, float alpha,
                                   const float* __restrict__ D1, float beta, const float* D2, float gamma, float* out)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float s = 0.0f;
    for (int z = 0; z < n_z; ++z) s += P[(long long)z * n + i];
    float r = alpha * s;
    if (D1) r = fmaf(beta, D1[i], r);
    if (D2) r = fmaf(gamma, D2[i], r);
    out[i] = r;
}

// B[j][i] = VT[i][j] * s_i: the eigenvectors of a small problem come as rows (VT[i] = i-th vector); the products above
// want them as columns, scaled by d_i^-1/2 after the Gram step (scale = NULL: no scaling).  d_i below rel * d_max: the
// column is dropped (rank-deficient block), its scale is 0.
__global__ void sub_transpose_scale_kernel(const float* __restrict__ VT, const float* __restrict__ d, int m, int use_scale,
                                           float* __restrict__ B)
{
    const int i = blockIdx.y * 16 + threadIdx.y, j = blockIdx.x * 16 + threadIdx.x;
    if (i >= m || j >= m) return;
    float s = 1.0f;
    if (use_scale) {
        const float dmax = d[m - 1];                   // ascending
        s = d[i] > 1e-10f * dmax ? rsqrtf(d[i]) : 0.0f;
    }
    B[(long long)j * m + i] = VT[(long long)i * m + j] * s;
}

// residual norms: r2[i] = | AX[:, i] - theta_i X[:, i] |^2, one block per column, fixed order
__global__ void __launch_bounds__(ET)
sub_residual_kernel(const float* __restrict__ AX, const float* __restrict__ X, const float* __restrict__ theta, long long K, int m,
                    float* __restrict__ r2)
{
    __shared__ float s_red[ET / 32];
    const int i = blockIdx.x;
    const float th = theta[i];
    float v = 0.0f;
    for (long long k = threadIdx.x; k < K; k += ET) { const float r = fmaf(-th, X[k * m + i], AX[k * m + i]); v = fmaf(r, r, v); }
    v = block_sum(v, s_red);
    if (threadIdx.x == 0) r2[i] = v;
}

// output: eigenvalue e and psi_e = M^-1/2 x_e with the sign rule of eig_vectors_kernel, rows [n_eig][K]
__global__ void __launch_bounds__(ET)
sub_output_kernel(const float* __restrict__ X, const float* __restrict__ theta, const float* __restrict__ mass, long long K, int m,
                  float* __restrict__ evals, float* __restrict__ evecs)
{
    __shared__ float s_red[ET / 32];
    __shared__ float s_sign;
    const int e = blockIdx.x;
    float v = 0.0f, n2 = 0.0f;
    for (long long j = threadIdx.x; j < K; j += ET) { const float q = X[j * m + e]; v += q * q * q; n2 = fmaf(q, q, n2); }
    v = block_sum(v, s_red); n2 = block_sum(n2, s_red);
    if (threadIdx.x == 0) { s_sign = (v < 0.0f ? -1.0f : 1.0f) / sqrtf(n2); evals[e] = theta[e]; }
    __syncthreads();
    if (!evecs) return;
    const float sg = s_sign;
    for (long long j = threadIdx.x; j < K; j += ET) evecs[(long long)e * K + j] = sg * X[j * m + e] * rsqrtf(mass[j]);
}

// Cholesky G = L L^T of an m x m Gram matrix and Linv = L^-1 (written to global memory, full rows, zeros above the
// diagonal), one block.  SMEM: L and Linv live in shared memory as packed lower triangles (m <= 192: 2 x 74 KB);
// otherwise everything stays in global memory (slow, m up to 320 only).  shift_rel > 0 adds shift_rel * trace(G) to the
// diagonal first (shifted Cholesky QR: the first pass on a block whose Gram matrix is numerically singular in fp32);
// pivots are clamped at 1e-12 of the largest diagonal entry.
template <bool SMEM>
__global__ void __launch_bounds__(1024)
sub_chol_inv_kernel(float* __restrict__ G, int m, float shift_rel, float* __restrict__ Linv)
{
    extern __shared__ float s_tri[];
    __shared__ float s_red[32];
    __shared__ float s_piv, s_floor;
    const int tid = threadIdx.x, T = blockDim.x;
    const int tri = m * (m + 1) / 2;
    float* L = SMEM ? s_tri : G;                     // element (i, k), k <= i
    float* X = SMEM ? s_tri + tri : Linv;            // Linv while it is built
#define LIDX(i, k) (SMEM ? ((i) * ((i) + 1) / 2 + (k)) : ((i) * m + (k)))
    if (SMEM) {
        for (int e = tid; e < m * m; e += T) { const int i = e / m, k = e - i * m; if (k <= i) L[LIDX(i, k)] = G[e]; }
        __syncthreads();
    }
    {
        float tr = 0.0f, mx = 0.0f;
        for (int i = tid; i < m; i += T) { const float d = L[LIDX(i, i)]; tr += d; mx = fmaxf(mx, d); }
        for (int o = 16; o > 0; o >>= 1) { tr += __shfl_xor_sync(0xFFFFFFFFu, tr, o); mx = fmaxf(mx, __shfl_xor_sync(0xFFFFFFFFu, mx, o)); }
        if ((tid & 31) == 0) s_red[tid >> 5] = tr;
        __syncthreads();
        float trace = 0.0f;
        for (int w = 0; w < (T + 31) / 32; ++w) trace += s_red[w];
        __syncthreads();
        if ((tid & 31) == 0) s_red[tid >> 5] = mx;
        __syncthreads();
        float dmax = 0.0f;
        for (int w = 0; w < (T + 31) / 32; ++w) dmax = fmaxf(dmax, s_red[w]);
        if (tid == 0) s_floor = 1e-12f * dmax;
        const float sh = shift_rel * trace;
        if (sh > 0.0f) for (int i = tid; i < m; i += T) L[LIDX(i, i)] += sh;
    }
    for (int j = 0; j < m; ++j) {
        __syncthreads();
        if (tid == 0) { const float piv = sqrtf(fmaxf(L[LIDX(j, j)], s_floor)); L[LIDX(j, j)] = piv; s_piv = piv; }
        __syncthreads();
        const float inv = 1.0f / s_piv;
        for (int i = j + 1 + tid; i < m; i += T) L[LIDX(i, j)] *= inv;
        __syncthreads();
        // trailing update of the lower triangle: a warp takes rows, its lanes the columns of a row
        const int warp = tid >> 5, lane = tid & 31, n_warps = T >> 5;
        for (int i = j + 1 + warp; i < m; i += n_warps) {
            const float lij = L[LIDX(i, j)];
            for (int k = j + 1 + lane; k <= i; k += 32) L[LIDX(i, k)] = fmaf(-lij, L[LIDX(k, j)], L[LIDX(i, k)]);
        }
    }
    __syncthreads();
    // Linv: thread c solves L x = e_c for column c
    for (int c = tid; c < m; c += T) {
        X[LIDX(c, c)] = 1.0f / L[LIDX(c, c)];
        for (int i = c + 1; i < m; ++i) {
            float acc = 0.0f;
            for (int k = c; k < i; ++k) acc = fmaf(L[LIDX(i, k)], X[LIDX(k, c)], acc);
            X[LIDX(i, c)] = -acc / L[LIDX(i, i)];
        }
    }
    __syncthreads();
    if (SMEM) {
        for (int e = tid; e < m * m; e += T) { const int i = e / m, k = e - i * m; Linv[e] = k <= i ? X[LIDX(i, k)] : 0.0f; }
    } else {
        for (int e = tid; e < m * m; e += T) { const int i = e / m, k = e - i * m; if (k > i) Linv[e] = 0.0f; }
    }
#undef LIDX
}

__global__ void __launch_bounds__(ET)
sub_matrix_kernel(const float* __restrict__ S, const float* __restrict__ mass, long long K, float* __restrict__ A)
{
    const long long i = (long long)blockIdx.x * ET + threadIdx.x;
    if (i >= K * K) return;
    const long long r = i / K, c = i - r * K;
    A[i] = 0.5f * (S[r * K + c] + S[c * K + r]) * rsqrtf(mass[r]) * rsqrtf(mass[c]);     // as eig_init_kernel
}

__global__ void sub_fill_kernel(float* __restrict__ x, int n, float v)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) x[i] = v;
}

constexpr int SUB_MIN_K = 1024;        // below: one-sided Jacobi (all eigenpairs) is as fast
constexpr int SUB_M_MAX = 320;         // widest block: n_eig <= 256
constexpr int SUB_MAX_ITERS = 40;

int sub_block_width(int n_eig)
{
    const int guard = n_eig / 4 > 16 ? n_eig / 4 : 16;
    return ((n_eig + guard + 63) / 64) * 64;
}

int sub_split(long long tiles, long long Kd, int cap)
{
    long long nz = (296 + tiles - 1) / tiles;                 // about two blocks per SM
    const long long by_depth = Kd / 128 > 1 ? Kd / 128 : 1;    // at least 128 of depth per slice
    if (nz > by_depth) nz = by_depth;
    if (nz > cap) nz = cap;
    return nz < 1 ? 1 : (int)nz;
}

// capacity of the split-K partials: n_z <= 296 / tiles + 1 slices of tiles * 4096 entries each (tall products), or 64 slices
// of an m x m product
size_t sub_partial_floats(long long K)
{
    const size_t tall = (size_t)297 * TT * TT + (size_t)(K + TT) * (SUB_M_MAX + TT);
    const size_t small = (size_t)64 * SUB_M_MAX * SUB_M_MAX;
    return tall > small ? tall : small;
}

size_t sub_extra_bytes(long long K)
{
    if (K < SUB_MIN_K) return 0;
    const size_t m = SUB_M_MAX;
    return align_up(sub_partial_floats(K) * 4) + 5 * align_up((size_t)K * m * 4) + 3 * align_up(m * m * 4) + 6 * align_up(m * 4) + 256
         + align_up(mcs_steklov_eigs_workspace_bytes(SUB_M_MAX, 1));
}

struct SubBuffers {
    float *A, *P, *X, *Y, *Z, *T, *U, *Gm, *VT, *Bm, *d, *theta, *r2, *ones;
    unsigned* bound;
    void* small_ws; size_t small_bytes;
};

// C [M][N] = op(A) B through split-K partials in `P`, then C = the ordered sum of the partials
template <bool TA>
int sub_gemm(const float* A, const float* B, float* C, int M, int N, int Kd, int n_z, float* P, cudaStream_t st)
{
    const int k_per_z = (int)(ceil_div64(ceil_div64(Kd, n_z), GK) * GK);
    const dim3 g((unsigned)ceil_div64(N, GT), (unsigned)ceil_div64(M, GT), (unsigned)n_z);
    mcs_note_launch(), sgemm_kernel<TA><<<g, 256, 0, st>>>(A, B, n_z == 1 ? C : P, M, N, Kd, k_per_z);
    if (n_z > 1) {
        const long long n = (long long)M * N;
        mcs_note_launch(), sub_combine_kernel<<<(unsigned)ceil_div64(n, 256), 256, 0, st>>>(P, n_z, n, 1.0f, nullptr, 0.0f, nullptr, 0.0f, C);
    }
    MCS_CUDA_TRY(cudaGetLastError());
    return MCS_OK;
}

// One pass of Cholesky QR: out = Y R^-1 with Y^T Y (+ shift) = R^T R.  Three passes, the first one shifted, orthonormalise a
// block whose Gram matrix has a condition number up to ~1/eps^2... in exact terms: pass 1 brings cond(Y) down to ~1e3,
// pass 2 leaves an orthogonality error of ~cond^2 eps, pass 3 of ~eps (shifted Cholesky QR3).  `Y` is left as it was.
int sub_cholqr_pass(const float* Y, float* out, long long K, int m, float shift_rel, const SubBuffers& w, cudaStream_t st)
{
    const int nz_small = sub_split((long long)(m / 64) * (m / 64), K, 64);
    int rc = sub_gemm<true>(Y, Y, w.Gm, m, m, (int)K, nz_small, w.P, st);
    if (rc != MCS_OK) return rc;
    if (m <= 192) {
        static bool attr_set = false;
        if (!attr_set) {
            MCS_CUDA_TRY(cudaFuncSetAttribute(sub_chol_inv_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 192 * 193 * 4));
            attr_set = true;
        }
        mcs_note_launch(), sub_chol_inv_kernel<true><<<1, 1024, (size_t)m * (m + 1) * 4, st>>>(w.Gm, m, shift_rel, w.VT);
    } else {
        mcs_note_launch(), sub_chol_inv_kernel<false><<<1, 1024, 0, st>>>(w.Gm, m, shift_rel, w.VT);
    }
    const dim3 gt((unsigned)ceil_div64(m, 16), (unsigned)ceil_div64(m, 16));
    mcs_note_launch(), sub_transpose_scale_kernel<<<gt, dim3(16, 16), 0, st>>>(w.VT, w.d, m, 0, w.Bm);      // R^-1 = (L^-1)^T
    return sub_gemm<false>(Y, w.Bm, out, (int)K, m, m, 1, w.P, st);
}

// Smallest n_eig eigenpairs of ONE matrix.  evals [n_eig], evecs [n_eig][K] or NULL.  Returns MCS_OK, MCS_WNOTCONVERGED or an error.
int sub_eigs_one(const float* S, const float* mass, long long K, int n_eig, float* evals, float* evecs,
                 const SubBuffers& w, int* iters_out, cudaStream_t st)
{
    const int m = sub_block_width(n_eig);
    const long long n = K * (long long)m;
    mcs_note_launch(), sub_matrix_kernel<<<(unsigned)ceil_div64(K * K, ET), ET, 0, st>>>(S, mass, K, w.A);
    MCS_CUDA_TRY(cudaMemsetAsync(w.bound, 0, 4, st));
    mcs_note_launch(), sub_gershgorin_kernel<<<(unsigned)K, ET, 0, st>>>(w.A, K, w.bound);
    mcs_note_launch(), sub_fill_kernel<<<(unsigned)ceil_div64(m, 256), 256, 0, st>>>(w.ones, m, 1.0f);
    mcs_note_launch(), sub_init_kernel<<<(unsigned)ceil_div64(n, 256), 256, 0, st>>>(w.Y, n, 0x1234567u);
    float b = 0.0f;
    MCS_CUDA_TRY(cudaMemcpyAsync(&b, w.bound, 4, cudaMemcpyDeviceToHost, st));
    MCS_CUDA_TRY(cudaStreamSynchronize(st));
    if (!(b > 0.0f) || !(b < 3.0e38f)) {               // the zero matrix (every vector is an eigenvector) or a non-finite entry
        if (!(b == 0.0f)) return MCS_EINVAL;
        b = 1.0f;
    }
    b *= 1.01f;
    const int nz_tall = sub_split(ceil_div64(m, TT) * ceil_div64(K, TT), K, 8);
    const int nz_small = sub_split((long long)(m / 64) * (m / 64), K, 64);
    if ((size_t)nz_tall * K * m > sub_partial_floats(K) || (size_t)nz_small * m * m > sub_partial_floats(K)) return MCS_ENOMEM;
    const dim3 gt((unsigned)ceil_div64(m, 16), (unsigned)ceil_div64(m, 16));
    std::vector<float> theta((size_t)m), r2((size_t)m);
    const float tol = 2.0e-5f;
    float a = 0.0f, a_low = 0.0f;
    bool converged = false;
    int it = 0;
    for (; it <= SUB_MAX_ITERS; ++it) {
        if (it > 0) {
            // ---- filter: Y = p(A) X, scaled three-term recurrence (X, Y, T rotate) ----
            const float e = 0.5f * (b - a), c = 0.5f * (b + a);
            const float x0 = (c - a_low) / e;                                        // > 1: where the wanted end of the spectrum sits
            int deg = (int)(7.6 / acosh((double)x0));                                // p(a_low) / p(a) <= ~1e3 (fp32 Gram step)
            deg = deg < 4 ? 4 : (deg > 40 ? 40 : deg);
            float sigma = e / (a_low - c);
            const float sigma1 = sigma;
            float *px = w.X, *py = w.Y, *pt = w.T;
            // py = (sigma1 / e) (A px - c px)
            {
                const int k_per_z = (int)(ceil_div64(ceil_div64(K, nz_tall), TK) * TK);
                const dim3 g((unsigned)ceil_div64(m, TT), (unsigned)ceil_div64(K, TT), (unsigned)nz_tall);
                mcs_note_launch(), sgemm_tall_kernel<<<g, 256, 0, st>>>(w.A, px, w.P, (int)K, m, (int)K, k_per_z);
                mcs_note_launch(), sub_combine_kernel<<<(unsigned)ceil_div64(n, 256), 256, 0, st>>>(w.P, nz_tall, n, sigma1 / e, px, -c * sigma1 / e, nullptr, 0.0f, py);
                for (int i = 2; i <= deg; ++i) {
                    const float sigma2 = 1.0f / (2.0f / sigma1 - sigma);
                    // pt = 2 (sigma2 / e) (A py - c py) - sigma sigma2 px
                    mcs_note_launch(), sgemm_tall_kernel<<<g, 256, 0, st>>>(w.A, py, w.P, (int)K, m, (int)K, k_per_z);
                    mcs_note_launch(), sub_combine_kernel<<<(unsigned)ceil_div64(n, 256), 256, 0, st>>>(
                        w.P, nz_tall, n, 2.0f * sigma2 / e, py, -2.0f * c * sigma2 / e, px, -sigma * sigma2, pt);
                    float* t = px; px = py; py = pt; pt = t;
                    sigma = sigma2;
                }
            }
            MCS_CUDA_TRY(cudaGetLastError());
            if (py != w.Y) MCS_CUDA_TRY(cudaMemcpyAsync(w.Y, py, (size_t)n * 4, cudaMemcpyDeviceToDevice, st));
        }
        // ---- orthonormalise Y: shifted Cholesky QR, three passes (Y -> U -> Z -> Y) ----
        int rc = sub_cholqr_pass(w.Y, w.U, K, m, 3.0e-6f, w, st);
        if (rc == MCS_OK) rc = sub_cholqr_pass(w.U, w.Z, K, m, 0.0f, w, st);
        if (rc == MCS_OK) rc = sub_cholqr_pass(w.Z, w.Y, K, m, 0.0f, w, st);
        if (rc != MCS_OK) return rc;
        // ---- Rayleigh-Ritz: Z = A Y, H = Y^T Z = W Theta W^T, X = Y W, AX = Z W ----
        {
            const int k_per_z = (int)(ceil_div64(ceil_div64(K, nz_tall), TK) * TK);
            const dim3 g((unsigned)ceil_div64(m, TT), (unsigned)ceil_div64(K, TT), (unsigned)nz_tall);
            mcs_note_launch(), sgemm_tall_kernel<<<g, 256, 0, st>>>(w.A, w.Y, w.P, (int)K, m, (int)K, k_per_z);
            mcs_note_launch(), sub_combine_kernel<<<(unsigned)ceil_div64(n, 256), 256, 0, st>>>(w.P, nz_tall, n, 1.0f, nullptr, 0.0f, nullptr, 0.0f, w.Z);
            rc = cudaGetLastError() == cudaSuccess ? MCS_OK : MCS_ECUDA;
        }
        if (rc == MCS_OK) rc = sub_gemm<true>(w.Y, w.Z, w.Gm, m, m, (int)K, nz_small, w.P, st);
        if (rc != MCS_OK) return rc;
        rc = mcs_steklov_eigs_method(w.Gm, w.ones, m, 1, m, 1, w.theta, w.VT, w.small_ws, w.small_bytes, nullptr, st);
        if (rc < 0) return rc;
        mcs_note_launch(), sub_transpose_scale_kernel<<<gt, dim3(16, 16), 0, st>>>(w.VT, w.theta, m, 0, w.Bm);
        rc = sub_gemm<false>(w.Y, w.Bm, w.X, (int)K, m, m, 1, w.P, st);
        if (rc == MCS_OK) rc = sub_gemm<false>(w.Z, w.Bm, w.U, (int)K, m, m, 1, w.P, st);
        if (rc != MCS_OK) return rc;
        mcs_note_launch(), sub_residual_kernel<<<(unsigned)m, ET, 0, st>>>(w.U, w.X, w.theta, K, m, w.r2);
        MCS_CUDA_TRY(cudaMemcpyAsync(theta.data(), w.theta, (size_t)m * 4, cudaMemcpyDeviceToHost, st));
        MCS_CUDA_TRY(cudaMemcpyAsync(r2.data(), w.r2, (size_t)m * 4, cudaMemcpyDeviceToHost, st));
        MCS_CUDA_TRY(cudaStreamSynchronize(st));
        float worst = 0.0f;
        for (int i = 0; i < n_eig; ++i) worst = fmaxf(worst, sqrtf(fmaxf(r2[(size_t)i], 0.0f)));
        if (!(worst == worst)) return MCS_EINVAL;                                        // NaN: non-finite input
        if (it > 0 && worst <= tol * b) { converged = true; ++it; break; }
        a = theta[(size_t)m - 1];
        a_low = theta[0] < 0.0f ? theta[0] : 0.0f;
        if (!(a > a_low + 1e-6f * b)) a = a_low + 1e-6f * b;                             // a flat block: keep the interval proper
        if (a > 0.999f * b) a = 0.999f * b;
    }
    if (iters_out) *iters_out = it;
    mcs_note_launch(), sub_output_kernel<<<(unsigned)n_eig, ET, 0, st>>>(w.X, w.theta, mass, K, m, evals, evecs);
    MCS_CUDA_TRY(cudaGetLastError());
    return converged ? MCS_OK : MCS_WNOTCONVERGED;
}

}  // namespace

extern "C" size_t mcs_steklov_eigs_workspace_bytes(int64_t K, int64_t batch)
{
    if (K < 1 || batch < 1) return 0;
    const size_t n = (size_t)batch * K;
    return 2 * align_up((size_t)batch * K * K * 4) + align_up(n * 4) * 3 + align_up(sort_workspace_bytes(K, 4)) +
           align_up((size_t)batch * 4) + 1024 + sub_extra_bytes(K);
}

extern "C" int mcs_steklov_eigs(const float* S, const float* mass, int64_t K, int64_t batch, int32_t n_eig,
                                float* evals, float* evecs, void* ws, size_t ws_bytes, int32_t* sweeps_out, void* stream)
{
    return mcs_steklov_eigs_method(S, mass, K, batch, n_eig, 0, evals, evecs, ws, ws_bytes, sweeps_out, stream);
}

extern "C" int mcs_steklov_eigs_method(const float* S, const float* mass, int64_t K, int64_t batch, int32_t n_eig, int32_t method,
                                       float* evals, float* evecs, void* ws, size_t ws_bytes, int32_t* sweeps_out, void* stream)
{
    if (!S || !mass || !evals || K < 1 || batch < 1 || n_eig < 1 || n_eig > K || K > 16384) return MCS_EINVAL;
    if (method < 0 || method > 2) return MCS_EINVAL;
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
    unsigned* flag = (unsigned*)p;  p += 1024;

    // Few eigenpairs of a large matrix: subspace iteration, one matrix after the other (see above)
    const bool sub_ok = K >= SUB_MIN_K && n_eig <= 256 && 2 * (int64_t)sub_block_width(n_eig) <= K;
    if (method == 2 && !sub_ok) return MCS_EINVAL;
    if (sub_ok && method != 1) {
        const size_t mm = SUB_M_MAX;
        SubBuffers w;
        w.A = G;
        w.P = (float*)p;  p += align_up(sub_partial_floats(K) * 4);
        float** tall[5] = { &w.X, &w.Y, &w.Z, &w.T, &w.U };
        for (float** t : tall) { *t = (float*)p; p += align_up((size_t)K * mm * 4); }
        w.Gm = (float*)p; p += align_up(mm * mm * 4);
        w.VT = (float*)p; p += align_up(mm * mm * 4);
        w.Bm = (float*)p; p += align_up(mm * mm * 4);
        float** vec[4] = { &w.d, &w.theta, &w.r2, &w.ones };
        for (float** t : vec) { *t = (float*)p; p += align_up(mm * 4); }
        w.bound = (unsigned*)p; p += align_up(mm * 4) * 2 + 256;
        w.small_ws = p; w.small_bytes = mcs_steklov_eigs_workspace_bytes(SUB_M_MAX, 1);
        int worst_rc = MCS_OK, iters = 0;
        for (int64_t bi = 0; bi < batch; ++bi) {
            int it_b = 0;
            const int rc = sub_eigs_one(S + bi * K * K, mass + bi * K, K, n_eig, evals + bi * n_eig, evecs ? evecs + bi * n_eig * K : nullptr,
                                        w, &it_b, st);
            if (rc < 0) return rc;
            if (rc > worst_rc) worst_rc = rc;
            if (it_b > iters) iters = it_b;
        }
        if (sweeps_out) *sweeps_out = iters;
        // automatic choice: a spectrum the filter cannot separate within its iteration cap (eigenvalues crowded at the low
        // end) falls through to the Jacobi solver below, which does not care
        if (worst_rc == MCS_OK || method == 2) return worst_rc;
    }

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
