// walk.cu -- sample preparation (A2), walk initialisation (A3), the
// walk-on-spheres loop (A4), termination records (A5) and killing walks (A6) of
// SURVEY.md 8(a).  Follows Alg. 2 for the interior operator
// and Eq. 32 for the exterior one, in fp32.
//
// Scheduling: a persistent grid (a multiple of the SM count).  A warp takes a
// chunk of consecutive walk indices from one global counter; every lane runs
// one walk and, when it terminates, takes the next index of the warp's chunk
// (wavefront compaction at lane granularity), so a warp never idles behind its
// longest walk.  Results do not depend on the schedule: the RNG is
// Philox4x32-10 keyed by (seed; sample, walk, step, purpose) and each walk
// writes its record to the fixed slot sample*W + walk.
#include "traverse.cuh"
#include "walk.cuh"

#include <limits.h>
#include <stdlib.h>
#include <vector>

namespace {

constexpr int WT = 128;                 // threads per block of the walk kernel
constexpr int PT = 128;                 // threads per block of the per-sample kernels

__device__ __forceinline__ int float_to_ordered(float f)
{
    int i = __float_as_int(f);
    return i >= 0 ? i : i ^ 0x7FFFFFFF;
}

// ---------------------------------------------------------------------------
// Exterior prerequisites: AABB of the Kelvin-inverted vertices (r_max rule,
// PAPER.md:642) and R_max = max |v - o| (reading E3).
// out: int[7] = ordered lo[3], hi[3], ordered max norm.
// ---------------------------------------------------------------------------
__global__ void __launch_bounds__(PT)
kelvin_bounds_kernel(const float* __restrict__ verts, int64_t V, float3 o, int* __restrict__ out)
{
    const int64_t i = (int64_t)blockIdx.x * PT + threadIdx.x;
    float lo[3] = { CUDART_INF_F, CUDART_INF_F, CUDART_INF_F }, hi[3] = { -CUDART_INF_F, -CUDART_INF_F, -CUDART_INF_F };
    float nrm = 0.0f;
    if (i < V) {
        const float3 w = f3(verts[3 * i] - o.x, verts[3 * i + 1] - o.y, verts[3 * i + 2] - o.z);
        const float s = dot3(w, w);
        nrm = sqrtf(s);
        if (s > 0.0f) {
            lo[0] = hi[0] = w.x / s; lo[1] = hi[1] = w.y / s; lo[2] = hi[2] = w.z / s;
        } else {
            out[7] = 1;                 // a vertex at the Kelvin origin
        }
    }
    for (int off = 16; off > 0; off >>= 1) {
        for (int d = 0; d < 3; ++d) {
            lo[d] = fminf(lo[d], __shfl_xor_sync(0xFFFFFFFFu, lo[d], off));
            hi[d] = fmaxf(hi[d], __shfl_xor_sync(0xFFFFFFFFu, hi[d], off));
        }
        nrm = fmaxf(nrm, __shfl_xor_sync(0xFFFFFFFFu, nrm, off));
    }
    if ((threadIdx.x & 31) == 0) {
        for (int d = 0; d < 3; ++d) {
            if (lo[d] <= hi[d]) { atomicMin(&out[d], float_to_ordered(lo[d])); atomicMax(&out[3 + d], float_to_ordered(hi[d])); }
        }
        atomicMax(&out[6], float_to_ordered(nrm));
    }
}

__global__ void kelvin_bounds_init_kernel(int* __restrict__ out)
{
    const int d = threadIdx.x;
    if (d < 8) out[d] = d < 3 ? 0x7FFFFFFF : (d < 7 ? (int)0x80000000 : 0);
}

__device__ __forceinline__ float ordered_to_float(int h)
{
    return __int_as_float(h >= 0 ? h : h ^ 0x7FFFFFFF);
}

// r_max (rmax_scale x half the shortest side of the domain's bounding box; exterior: of the box of the
// Kelvin-inverted vertices) and R_max, written where the later kernels of the call read them.  bounds = the int[8] of
// kelvin_bounds_kernel (exterior) or unused (interior: `side` comes from the handle's AABB).
__global__ void walk_dyn_kernel(const int* __restrict__ bounds, int exterior, float side, float rmax_scale, float rmax_override,
                                WalkDyn* __restrict__ dyn)
{
    float Rmax = 0.0f;
    int err = 0;
    if (exterior) {
        float f[7];
        for (int d = 0; d < 7; ++d) f[d] = ordered_to_float(bounds[d]);
        side = fminf(f[3] - f[0], fminf(f[4] - f[1], f[5] - f[2]));
        Rmax = f[6];
        if (bounds[7] || !(Rmax > 0.0f)) err = WALK_ERR_DEGENERATE;
    }
    dyn->rmax = rmax_override > 0.0f ? rmax_override : rmax_scale * (0.5f * side);
    dyn->Rmax = Rmax;
    dyn->err = err;
}

// ---------------------------------------------------------------------------
// Z-order keys of the sample points ("sort sample points s via
// Z-order curves, which greatly reduces warp divergence").
// ---------------------------------------------------------------------------
__device__ __forceinline__ unsigned spread10(unsigned x)
{
    x &= 0x3FFu;
    x = (x | (x << 16)) & 0x030000FFu;
    x = (x | (x << 8))  & 0x0300F00Fu;
    x = (x | (x << 4))  & 0x030C30C3u;
    x = (x | (x << 2))  & 0x09249249u;
    return x;
}

__device__ __forceinline__ void sample_point(const float* __restrict__ verts, const int32_t* __restrict__ faces,
                                             const int32_t* __restrict__ tri, const float* __restrict__ bary, int64_t i,
                                             float3& s, float3& n)
{
    const int64_t f = tri[i];
    const int i0 = faces[3 * f], i1 = faces[3 * f + 1], i2 = faces[3 * f + 2];
    const float3 a = f3(verts[3 * (int64_t)i0], verts[3 * (int64_t)i0 + 1], verts[3 * (int64_t)i0 + 2]);
    const float3 b = f3(verts[3 * (int64_t)i1], verts[3 * (int64_t)i1 + 1], verts[3 * (int64_t)i1 + 2]);
    const float3 c = f3(verts[3 * (int64_t)i2], verts[3 * (int64_t)i2 + 1], verts[3 * (int64_t)i2 + 2]);
    const float b0 = bary[3 * i], b1 = bary[3 * i + 1], b2 = bary[3 * i + 2];
    s = f3(fmaf(b0, a.x, fmaf(b1, b.x, b2 * c.x)), fmaf(b0, a.y, fmaf(b1, b.y, b2 * c.y)), fmaf(b0, a.z, fmaf(b1, b.z, b2 * c.z)));
    n = cross3(b - a, c - a);
    const float l = sqrtf(dot3(n, n));
    if (l > 0.0f) n = (1.0f / l) * n;
}

__global__ void __launch_bounds__(PT)
sample_keys_kernel(const float* __restrict__ verts, const int32_t* __restrict__ faces, int64_t F,
                   const int32_t* __restrict__ tri, const float* __restrict__ bary, int64_t n_s,
                   float3 lo, float3 hi, uint32_t* __restrict__ keys, uint32_t* __restrict__ vals, int* __restrict__ err)
{
    const int64_t i = (int64_t)blockIdx.x * PT + threadIdx.x;
    if (i >= n_s) return;
    vals[i] = (uint32_t)i;
    if (tri[i] < 0 || tri[i] >= F) { atomicOr(err, WALK_ERR_SAMPLE_FACE); keys[i] = 0; return; }
    float3 s, n;
    sample_point(verts, faces, tri, bary, i, s, n);
    const float ex = hi.x - lo.x, ey = hi.y - lo.y, ez = hi.z - lo.z;
    const float tx = ex > 0.f ? fminf(fmaxf((s.x - lo.x) / ex, 0.f), 1.f) : 0.f;
    const float ty = ey > 0.f ? fminf(fmaxf((s.y - lo.y) / ey, 0.f), 1.f) : 0.f;
    const float tz = ez > 0.f ? fminf(fmaxf((s.z - lo.z) / ez, 0.f), 1.f) : 0.f;
    keys[i] = (spread10((unsigned)fminf(tx * 1024.f, 1023.f)) << 2) | (spread10((unsigned)fminf(ty * 1024.f, 1023.f)) << 1) |
              spread10((unsigned)fminf(tz * 1024.f, 1023.f));
}

// ---------------------------------------------------------------------------
// LargestTangentBall: the bisection of PAPER.md:383 with `iters`
// iterations, radius clamped to r_max (R4).
//
// The bisection probes radii on the grid r_j = j * hi / 2^iters and, because the
// probed balls B(s - r n, r - eps/2) are nested (tangent at s), returns the largest
// grid radius whose ball no face enters:  r = r_J,  J = min over faces T of
// j_T = max{ j : T outside ball_j }.  Instead of `iters` separate emptiness proofs
// (each one visits every node its ball touches), ONE traversal with a shrinking ball
// computes that minimum: keep the current candidate J, visit only nodes whose box
// enters ball_J, and when a face enters ball_J find its own j_T by bisection over j
// on that single face (<= iters point-triangle tests) and shrink J.
//
// One warp per sample: the warp shares a node stack and a leaf list in shared
// memory, pops up to 32 nodes (or 32 leaves) per pass, one per lane, and pushes the
// surviving children with warp-aggregated offsets.  J is a minimum, so the result
// does not depend on the order of the traversal.
// Exterior: the ball lives in the inverted domain and is probed through its primal
// image (E2), which preserves the nesting.
// ---------------------------------------------------------------------------
constexpr int TB_WARPS = 4;
constexpr int TB_NCAP = 2048;          // node stack entries per warp
constexpr int TB_LCAP = 128;           // leaf list entries per warp (drained at 32)

struct BallFamily {
    float3 base, pole, o;
    float step, ss2, sdn, eps;
};

// Probe ball of grid index j: centre c and squared threshold thr2 (< 0: nothing can be closer).
template <bool EXT>
__device__ __forceinline__ void probe_ball(const BallFamily& f, int j, float3& c, float& thr2)
{
    const float r = (float)j * f.step;
    c = f3(fmaf(-r, f.pole.x, f.base.x), fmaf(-r, f.pole.y, f.base.y), fmaf(-r, f.pole.z, f.base.z));
    float thr;
    if (EXT) {
        // the Kelvin ball B(c*, r - eps/2) through its own primal image (R4 / E2): centre c* / den, radius rk / den
        const float rk = r - 0.5f * f.eps;
        const float den = (f.ss2 - 2.0f * r * f.sdn) + (r - rk) * (r + rk);   // |c*|^2 - rk^2,  |c*|^2 = ss2 - 2 r sdn + r^2
        c = f3(f.o.x + c.x / den, f.o.y + c.y / den, f.o.z + c.z / den);
        thr = rk / den;
    } else {
        thr = r - 0.5f * f.eps;
    }
    thr2 = (j > 0 && thr > 0.0f) ? thr * thr : -1.0f;
}

template <bool EXT>
__global__ void __launch_bounds__(TB_WARPS * 32)
tangent_ball_kernel(WalkGeom g, const int32_t* __restrict__ tri, const float* __restrict__ bary,
                    const float* __restrict__ normal, const uint32_t* __restrict__ order, int64_t n_s,
                    const WalkDyn* __restrict__ dyn, float eps, int iters, float3 o, float mesh_scale,
                    float4* __restrict__ balls, unsigned long long* __restrict__ stats)
{
    __shared__ int s_nodes[TB_WARPS][TB_NCAP];
    __shared__ int s_leaves[TB_WARPS][TB_LCAP];
    const unsigned FULL = 0xFFFFFFFFu;
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    if (dyn->err) {                                   // poisoned call: every sample is discarded (radius 0), no geometry is read
        for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < 2 * n_s; i += (int64_t)gridDim.x * blockDim.x)
            balls[i] = make_float4(0.f, 0.f, 0.f, 0.f);
        return;
    }
    const float rmax = dyn->rmax;
    const unsigned lt = (1u << lane) - 1u;
    int* nstack = s_nodes[wib];
    int* lstack = s_leaves[wib];
    const int64_t n_warps = (int64_t)gridDim.x * TB_WARPS;
    unsigned cnt_nodes = 0, cnt_tris = 0, cnt_queries = 0, cnt_discarded = 0;

    for (int64_t jj = (int64_t)blockIdx.x * TB_WARPS + wib; jj < n_s; jj += n_warps) {
        const int64_t i = order[jj];
        float3 s, n;
        sample_point(g.verts, g.faces, tri, bary, i, s, n);
        int own_face = tri[i];
        if (normal) {
            const float3 nf = n;
            n = f3(normal[3 * i], normal[3 * i + 1], normal[3 * i + 2]);
            if (!(fabsf(dot3(n, nf)) > 0.999999f)) own_face = -1;      // an override off the face's normal line: the ball is not tangent to the face
        }
        BallFamily fam;
        fam.base = s; fam.pole = n; fam.o = o; fam.ss2 = 1.0f; fam.sdn = 0.0f; fam.eps = eps;
        float hi = rmax, sstar_norm = 1.0f;
        bool ok = true;
        if (EXT) {
            const float3 st = s - o;
            const float sig = dot3(st, st);
            ok = sig > 0.0f;
            if (ok) {
                fam.base = (1.0f / sig) * st;                              // s* = kappa(s - o)
                const float sn = dot3(st, n) / sig;
                fam.pole = f3(-(n.x - 2.0f * st.x * sn), -(n.y - 2.0f * st.y * sn), -(n.z - 2.0f * st.z * sn));   // Eq. 54
                fam.ss2 = dot3(fam.base, fam.base);
                fam.sdn = dot3(fam.base, fam.pole);
                if (fam.sdn > 0.0f) hi = fminf(hi, 0.45f * fam.ss2 / fam.sdn);   // keep 0 = kappa(inf) outside the ball
                sstar_norm = sqrtf(fam.ss2);
            }
        }
        const int NJ = 1 << iters;
        fam.step = hi / (float)NJ;
        int J = ok ? NJ - 1 : 0;
        float3 cJ; float thr2J;
        probe_ball<EXT>(fam, J, cJ, thr2J);
        int ncount = 0, lcount = 0;
        if (J > 0 && thr2J > 0.0f) { if (lane == 0) nstack[0] = 0; ncount = 1; }
        if (lane == 0) ++cnt_queries;
        __syncwarp();
        while (J > 0 && (ncount > 0 || lcount > 0)) {
            if (lcount >= 32 || ncount == 0) {
                // ---- leaf pass: does the face enter ball_J? ---------------------------
                const int nl = lcount < 32 ? lcount : 32;
                int myJ = J;
                if (lane < nl) {
                    const int kk = lstack[lcount - nl + lane];
                    const TriData T = load_tri(g.tris, kk);
                    float v, w;
                    ++cnt_tris;
                    // The sample's own face is tangent to every ball of the family at s (distance exactly r): it can never
                    // enter one.  In fp32 s sits up to ~2e-7 off its plane, which is more than eps/2 at the paper's
                    // eps = 1e-6 and made the face "enter" every ball (38 of 41 000 samples discarded on
                    // the unit icosphere; none in the fp64 oracle).  It is left out.
                    if (T.orig != own_face && closest_point_triangle(cJ, T, thr2J, v, w) < thr2J) {
                        int lo_j = 0, hi_j = J;                           // ball_0 is empty by definition
                        while (hi_j - lo_j > 1) {
                            const int mid = (lo_j + hi_j) >> 1;
                            float3 cm; float t2;
                            probe_ball<EXT>(fam, mid, cm, t2);
                            ++cnt_tris;
                            if (closest_point_triangle(cm, T, t2, v, w) < t2) hi_j = mid; else lo_j = mid;
                        }
                        myJ = lo_j;
                    }
                }
                lcount -= nl;
                for (int off = 16; off > 0; off >>= 1) myJ = min(myJ, __shfl_xor_sync(FULL, myJ, off));
                if (myJ < J) { J = myJ; probe_ball<EXT>(fam, J, cJ, thr2J); }
                __syncwarp();
            } else {
                // ---- node pass: which children enter ball_J? ---------------------------
                int np = ncount < 32 ? ncount : 32;
                if (ncount > TB_NCAP - 256) np = 1;                       // nearly full: plain depth-first (+1 per level of the binary tree)
                bool in0 = false, in1 = false;
                int c0 = 0, c1 = 0;
                if (lane < np) {
                    const int node = nstack[ncount - np + lane];
                    const Vec8 n0 = ldg256(g.nodes + node), n1 = ldg256(reinterpret_cast<const char*>(g.nodes + node) + 32);
                    const float4 w0 = n0.lo, w1 = n0.hi, w2 = n1.lo;
                    const int2 ch = make_int2(__float_as_int(n1.hi.x), __float_as_int(n1.hi.y));
                    ++cnt_nodes;
                    c0 = ch.x; c1 = ch.y;
                    // same limit as the walk kernel's queries: a face whose COMPUTED distance enters the ball is reached
                    // whatever its box distance rounds to, so J is the minimum over all faces and does not depend on the tree
                    const float lim = prune_limit(thr2J, cJ, mesh_scale);
                    in0 = box_dist2(cJ, w0.x, w0.y, w0.z, w0.w, w1.x, w1.y) <= lim;
                    in1 = box_dist2(cJ, w1.z, w1.w, w2.x, w2.y, w2.z, w2.w) <= lim;
                }
                ncount -= np;
                __syncwarp();                                             // all pops read before any push writes
                const unsigned mn0 = __ballot_sync(FULL, in0 && c0 >= 0), mn1 = __ballot_sync(FULL, in1 && c1 >= 0);
                const unsigned ml0 = __ballot_sync(FULL, in0 && c0 < 0), ml1 = __ballot_sync(FULL, in1 && c1 < 0);
                if (in0 && c0 >= 0) nstack[ncount + __popc(mn0 & lt)] = c0;
                if (in1 && c1 >= 0) nstack[ncount + __popc(mn0) + __popc(mn1 & lt)] = c1;
                if (in0 && c0 < 0) lstack[lcount + __popc(ml0 & lt)] = ~c0;
                if (in1 && c1 < 0) lstack[lcount + __popc(ml0) + __popc(ml1 & lt)] = ~c1;
                ncount += __popc(mn0) + __popc(mn1);
                lcount += __popc(ml0) + __popc(ml1);
                __syncwarp();
            }
        }
        const float r = (float)J * fam.step;
        if (lane == 0) {
            if (!(r > 0.0f)) ++cnt_discarded;
            balls[2 * i] = make_float4(fmaf(-r, fam.pole.x, fam.base.x), fmaf(-r, fam.pole.y, fam.base.y),
                                       fmaf(-r, fam.pole.z, fam.base.z), r);
            balls[2 * i + 1] = make_float4(fam.pole.x, fam.pole.y, fam.pole.z, ok ? sstar_norm : 0.0f);
        }
        __syncwarp();
    }
    // statistics (integer atomics: order-independent)
    unsigned vals[4] = { cnt_queries, cnt_discarded, cnt_nodes, cnt_tris };
    for (int q = 0; q < 4; ++q) {
        unsigned v = vals[q];
        for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(FULL, v, off);
        vals[q] = v;
    }
    if (lane == 0) {
        if (vals[0]) { atomicAdd(&stats[ST_QUERIES], (unsigned long long)vals[0]); atomicAdd(&stats[ST_PREP_QUERIES], (unsigned long long)vals[0]); }
        if (vals[1]) atomicAdd(&stats[ST_DISCARDED], (unsigned long long)vals[1]);
        if (vals[2]) { atomicAdd(&stats[ST_NODES], (unsigned long long)vals[2]); atomicAdd(&stats[ST_PREP_NODES], (unsigned long long)vals[2]); }
        if (vals[3]) { atomicAdd(&stats[ST_TRIS], (unsigned long long)vals[3]); atomicAdd(&stats[ST_PREP_TRIS], (unsigned long long)vals[3]); }
    }
}

// Alg. 1: no tangent ball; the walk of sample i starts at the inset point
// x = s - inset * n_s.  Written in the layout of the tangent balls: (x, 1), (n, 1).
__global__ void __launch_bounds__(PT)
naive_start_kernel(WalkGeom g, const int32_t* __restrict__ tri, const float* __restrict__ bary,
                   const float* __restrict__ normal, int64_t n_s, float inset, const WalkDyn* __restrict__ dyn,
                   float4* __restrict__ balls)
{
    const int64_t i = (int64_t)blockIdx.x * PT + threadIdx.x;
    if (i >= n_s) return;
    if (dyn->err) { balls[2 * i] = balls[2 * i + 1] = make_float4(0.f, 0.f, 0.f, 0.f); return; }      // poisoned call
    float3 s, n;
    sample_point(g.verts, g.faces, tri, bary, i, s, n);
    if (normal) n = f3(normal[3 * i], normal[3 * i + 1], normal[3 * i + 2]);
    balls[2 * i] = make_float4(fmaf(-inset, n.x, s.x), fmaf(-inset, n.y, s.y), fmaf(-inset, n.z, s.z), 1.0f);
    balls[2 * i + 1] = make_float4(n.x, n.y, n.z, 1.0f);
}

// Orthonormal frame (e1, e2, n) of a unit vector n: branchless construction of
// Duff et al. (JCGT 2017), restated (R6b: the frame rule is part of
// the definition of a walk's start point).
__device__ __forceinline__ void frame_from_normal(float3 n, float3& e1, float3& e2)
{
    const float sign = copysignf(1.0f, n.z);
    const float a = -1.0f / (sign + n.z);
    const float b = n.x * n.y * a;
    e1 = f3(1.0f + sign * n.x * n.x * a, sign * b, -sign * n.x);
    e2 = f3(b, sign + n.y * n.y * a, -n.y);
}

// ---------------------------------------------------------------------------
// The walk kernel: a per-lane state machine with warp-level phase voting.
//
// Every lane owns one walk and, inside it, one closest-point query.  A query is a
// stack of pending items (inner nodes and leaves of the LBVH, each with the fp32
// squared distance of its box); the lane's next item decides what KIND of work it
// wants to do:   NODE (visit an inner node: two box tests, push the far child),
// TRI (one point-triangle test), TRANS (the query is finished: terminate the walk or
// take the next WoS jump, refill from the work queue, start the next query).
// Each pass of the single loop the warp votes and executes ONE kind, the one most
// lanes wait for; the others keep their state and wait.  No lane ever waits for
// another lane's query to finish, so a query near the medial axis that visits a
// thousand nodes costs its own lane only (wavefront compaction at the granularity of
// single node visits).  What a lane computes does not depend on the vote, so results
// are independent of the schedule.
//
// The traversal stack lives in shared memory ([depth][thread]: a lane always hits its
// own bank); entries beyond WSTACK spill to local memory (deep LBVH chains only).
// ---------------------------------------------------------------------------
constexpr int WALK_MIN_BLOCKS = 8;                  // 64 registers per thread; 10 (48 registers, spills) measured 9 % slower
// Blocks per SM of the variants with the warp-cooperative path (large or messy meshes): they need ~96 registers; at
// 8 blocks (64 registers) ncu counted 19 G spill instructions and more local-memory sectors than global ones on BASELINE
// config 3 (profiles/r02_cfg3_walk_kernel.md).  Measured on that workload (both operators, W = 1024): 8 blocks 358 ms,
// 6: 308, 5: 284, 4: 314.
#ifndef WALK_COOP_BLOCKS
#define WALK_COOP_BLOCKS 5
#endif
// Shared-memory stack entries per lane (the rest of a deep stack lives in local memory).  BASELINE config 3 (tree depth 41),
// walks of both operators at W = 1024: 12 -> 186.7 ms, 16 -> 179.6, 20 -> 175.8, 24 -> 174.4, 28 -> 173.4, 32 -> 175.8;
// configs[1] (depth 14) is flat up to 24 and loses 3-5 % at 28-32 (8 blocks per SM: the stacks take the L1's room).
#ifndef MCS_WSTACK
#define MCS_WSTACK 24
#endif
constexpr int WSTACK = MCS_WSTACK;
constexpr int CUR_NONE = INT_MIN;
#ifndef VOTE_NODE
#define VOTE_NODE 8
#endif
#ifndef VOTE_TRI
#define VOTE_TRI 8
#endif
#ifndef VOTE_TRANS
#define VOTE_TRANS 20
#endif
#ifndef VOTE_AGE
#define VOTE_AGE 32
#endif

struct LaneStack {
    int*   s_ref;      // shared: [WSTACK][block threads], this lane's column
    float* s_d;
    int    l_ref[MCS_STACK - WSTACK];            // local-memory spill
    float  l_d[MCS_STACK - WSTACK];
};

template <int TW>
__device__ __forceinline__ void stack_push(LaneStack& st, int& sp, int ref, float d)
{
    if (sp < WSTACK) { st.s_ref[sp * TW] = ref; st.s_d[sp * TW] = d; }
    else if (sp < MCS_STACK) { st.l_ref[sp - WSTACK] = ref; st.l_d[sp - WSTACK] = d; }
    ++sp;                                        // sp > MCS_STACK cannot happen: depth <= 63 + log2(F)
}

template <int TW>
__device__ __forceinline__ void stack_pop(LaneStack& st, int& sp, int& ref, float& d)
{
    --sp;
    if (sp < WSTACK) { ref = st.s_ref[sp * TW]; d = st.s_d[sp * TW]; }
    else { ref = st.l_ref[sp - WSTACK]; d = st.l_d[sp - WSTACK]; }
}

enum { KIND_IDLE = 0, KIND_NODE = 1, KIND_TRI = 2, KIND_TRANS = 3 };


// ---------------------------------------------------------------------------
// Warp-cooperative completion of ONE heavy query.  A query that has already visited COOP_MIN nodes
// (near a medial axis every box is about equally far: hundreds to thousands of nodes) would keep its
// lane busy for as many passes while the kernel's run time is the longest single-lane chain.  The whole
// warp takes such a query over: its pending items move to a warp-shared node stack and leaf list, every
// pass 32 lanes test 32 wide nodes (or 32 triangles), children are pushed with warp-aggregated offsets,
// and the best hit is a warp arg-min under the tie rule (smaller d2, then smaller face index).  The
// result is the same minimum the lane would have found; the order of the traversal does not matter.
// ---------------------------------------------------------------------------
// Thresholds measured on BASELINE config 3 at W = 1024 (walk kernels only): interior, exact queries (28 nodes per query on
// average): 24 -> 99.7 ms, 32 -> 96.8, 40 -> 98.4; exterior with the far-field cut (24 nodes per query on average): 24 ->
// 158.9 ms, 32 -> 140.5, 40 -> 134.3, 48 -> 133.7, 56 -> 133.2, 64 -> 134.2, 80 -> 135.8, 96 -> 138.5.  At 24 the take-over
// fired for every query above the exterior's MEAN length -- a warp-wide pass for what one lane finishes in a few visits; it
// belongs to the tail.  (Results do not depend on the threshold: the cooperative path finds the same minimum.)
#ifndef COOP_MIN_NODES
#define COOP_MIN_NODES 32
#endif
#ifndef COOP_MIN_EXT_NODES
#define COOP_MIN_EXT_NODES 56
#endif
#ifndef COOP_MIN_MERGED_NODES
#define COOP_MIN_MERGED_NODES 8
#endif
constexpr int COOP_MIN_MERGED = COOP_MIN_MERGED_NODES;     // the same in the merged-pass variant (small jobs: idle lanes are free)
constexpr int COOP_MIN = COOP_MIN_NODES;                      // nodes visited by a lane's query before the warp takes it over
constexpr int COOP_MIN_EXT = COOP_MIN_EXT_NODES;              // the same for the exterior operator
// Capacities.  Nodes: a 32-node pass runs only while ncount <= COOP_SOFT, so it leaves at most COOP_SOFT - 32 + 128
// = 480 entries; above COOP_SOFT the warp goes depth-first (one node per pass: net +3 per level of the wide tree,
// whose depth is at most (63 + log2 F) / 2 < 48), so ncount < 480 + 3 * 48 = 624 < COOP_NCAP.  Leaves: the lane's
// own stack hands over at most MCS_STACK + 1 = 161 entries; afterwards a node pass starts with < 32 and adds <= 128.
constexpr int COOP_NCAP = 1024;                   // warp node stack
constexpr int COOP_SOFT = 384;                    // above this: depth-first
constexpr int COOP_LCAP = 192;                    // warp leaf list (drained at 32)

// The hot per-lane variables of the walk kernel are handed over BY VALUE in this struct (a temporary at the
// call site): passing them by reference to a function that is not inlined would pin them in local memory
// for the whole kernel.
struct CoopState {
    float3 xq;
    ClosestHit h;
    float lim;
    float lb2, dnear2, alpha2;               // far-field lower bound (FAR builds): running minimum, near threshold, alpha^2
    int sp, cur;
    unsigned n_nodes, n_tris, q_nodes;       // increments (COUNT builds)
};

template <bool COUNT, bool FAR, int TW>
__device__ __forceinline__ void coop_finish_query(const BvhNode* nodes_unused, const WideNode* __restrict__ wide,
                                               const PackedTri* __restrict__ tris, int L, float mesh_scale,
                                               int* __restrict__ co_nodes, int* __restrict__ co_leaves,
                                               int* s_ref, float* s_d, int* l_ref, float* l_d, CoopState* stp)
{
    (void)nodes_unused;
    const unsigned FULL = 0xFFFFFFFFu;
    const int lane = threadIdx.x & 31;
    const unsigned lt = (1u << lane) - 1u;
    CoopState& S = *stp;
    const float3 xq_own = S.xq;
    ClosestHit& h = S.h;
    float& lim = S.lim;
    int& sp = S.sp;
    int& cur = S.cur;
    unsigned& n_nodes = S.n_nodes;
    unsigned& n_tris = S.n_tris;
    unsigned& q_nodes = S.q_nodes;
    // the query of lane L, known to all lanes
    const float3 xq = f3(__shfl_sync(FULL, xq_own.x, L), __shfl_sync(FULL, xq_own.y, L), __shfl_sync(FULL, xq_own.z, L));
    float bd2 = __shfl_sync(FULL, h.d2, L), bv = __shfl_sync(FULL, h.v, L), bw = __shfl_sync(FULL, h.w, L);
    int btri = __shfl_sync(FULL, h.tri, L), bk = __shfl_sync(FULL, h.k, L);
    float wlim = __shfl_sync(FULL, lim, L);
    float wlb = FAR ? __shfl_sync(FULL, S.lb2, L) : CUDART_INF_F;
    const float wnear2 = FAR ? __shfl_sync(FULL, S.dnear2, L) : 0.0f;
    const float alpha2 = S.alpha2;                                   // warp-uniform
    // lane L moves its pending items to the warp lists
    int ncount = 0, lcount = 0;
    if (lane == L) {
        if (cur != CUR_NONE) { if (cur >= 0) co_nodes[ncount++] = cur; else co_leaves[lcount++] = ~cur; }
        while (sp > 0) {
            int ref; float d;
            --sp;
            if (sp < WSTACK) { ref = s_ref[sp * TW]; d = s_d[sp * TW]; }
            else { ref = l_ref[sp - WSTACK]; d = l_d[sp - WSTACK]; }
            if (d <= lim) { if (ref >= 0) co_nodes[ncount++] = ref; else co_leaves[lcount++] = ~ref; }
        }
        cur = CUR_NONE;
    }
    ncount = __shfl_sync(FULL, ncount, L); lcount = __shfl_sync(FULL, lcount, L);
    __syncwarp();
    unsigned visited = 0;
    while (ncount > 0 || lcount > 0) {
        if (lcount >= 32 || ncount == 0) {
            // ---- leaf pass: 32 triangles, warp arg-min ------------------------------------
            const int nl = lcount < 32 ? lcount : 32;
            float d2 = CUDART_INF_F, v = 0.f, w = 0.f; int orig = INT_MAX, kk = -1;
            if (lane < nl) {
                kk = co_leaves[lcount - nl + lane];
                const TriData T = load_tri(tris, kk);
                d2 = closest_point_triangle(xq, T, CUDART_INF_F, v, w);
                orig = T.orig;
                if (COUNT) ++n_tris;
            }
            lcount -= nl;
            float md2 = d2; int morig = orig, mlane = lane;
            for (int off = 16; off > 0; off >>= 1) {
                const float od2 = __shfl_xor_sync(FULL, md2, off);
                const int oorig = __shfl_xor_sync(FULL, morig, off), olane = __shfl_xor_sync(FULL, mlane, off);
                if (od2 < md2 || (od2 == md2 && oorig < morig)) { md2 = od2; morig = oorig; mlane = olane; }
            }
            if (md2 < bd2 || (md2 == bd2 && morig < btri)) {
                bd2 = md2; btri = morig;
                bk = __shfl_sync(FULL, kk, mlane); bv = __shfl_sync(FULL, v, mlane); bw = __shfl_sync(FULL, w, mlane);
                wlim = prune_limit(FAR ? fminf(bd2, wlb) : bd2, xq, mesh_scale);
            }
            __syncwarp();
        } else {
            // ---- node pass: 32 wide nodes, four boxes each -----------------------------------
            int np = ncount < 32 ? ncount : 32;
            if (ncount > COOP_SOFT) np = 1;                              // depth-first, one node at a time: bounded growth
            bool in0 = false, in1 = false, in2 = false, in3 = false;
            int c0 = 0, c1 = 0, c2 = 0, c3 = 0;
            float mylb = CUDART_INF_F;
            if (lane < np) {
                const char* wn = reinterpret_cast<const char*>(wide + co_nodes[ncount - np + lane]);
                const Vec8 q0 = ldg256(wn), q1 = ldg256(wn + 32), q2 = ldg256(wn + 64), q3 = ldg256(wn + 96);
                if (COUNT) ++n_nodes;
                in0 = box_dist2(xq, q0.lo.x, q0.lo.y, q0.lo.z, q0.lo.w, q0.hi.x, q0.hi.y) <= wlim;
                in1 = box_dist2(xq, q0.hi.z, q0.hi.w, q1.lo.x, q1.lo.y, q1.lo.z, q1.lo.w) <= wlim;
                in2 = box_dist2(xq, q1.hi.x, q1.hi.y, q1.hi.z, q1.hi.w, q2.lo.x, q2.lo.y) <= wlim;
                in3 = box_dist2(xq, q2.lo.z, q2.lo.w, q2.hi.x, q2.hi.y, q2.hi.z, q2.hi.w) <= wlim;
                c0 = __float_as_int(q3.lo.x); c1 = __float_as_int(q3.lo.y); c2 = __float_as_int(q3.lo.z); c3 = __float_as_int(q3.lo.w);
                if (FAR) {
                    // a child whose box is small against its distance stands for its faces: its box distance is a lower
                    // bound of theirs (see walk_kernel); it is not descended / not tested.  INT_MIN marks an empty slot.
                    const float e0 = box_dist2(xq, q0.lo.x, q0.lo.y, q0.lo.z, q0.lo.w, q0.hi.x, q0.hi.y);
                    const float e1 = box_dist2(xq, q0.hi.z, q0.hi.w, q1.lo.x, q1.lo.y, q1.lo.z, q1.lo.w);
                    const float e2 = box_dist2(xq, q1.hi.x, q1.hi.y, q1.hi.z, q1.hi.w, q2.lo.x, q2.lo.y);
                    const float e3 = box_dist2(xq, q2.lo.z, q2.lo.w, q2.hi.x, q2.hi.y, q2.hi.z, q2.hi.w);
                    if (in0 && e0 >= wnear2 && q3.hi.x <= alpha2 * e0) { mylb = fminf(mylb, e0); in0 = false; }
                    if (in1 && e1 >= wnear2 && q3.hi.y <= alpha2 * e1) { mylb = fminf(mylb, e1); in1 = false; }
                    if (in2 && e2 >= wnear2 && q3.hi.z <= alpha2 * e2) { mylb = fminf(mylb, e2); in2 = false; }
                    if (in3 && e3 >= wnear2 && q3.hi.w <= alpha2 * e3) { mylb = fminf(mylb, e3); in3 = false; }
                }
            }
            if (FAR) {
                for (int off = 16; off > 0; off >>= 1) mylb = fminf(mylb, __shfl_xor_sync(FULL, mylb, off));
                if (mylb < wlb) { wlb = mylb; wlim = fminf(wlim, prune_limit(wlb, xq, mesh_scale)); }
            }
            visited += (unsigned)np;
            ncount -= np;
            __syncwarp();                                                // all pops read before any push writes
#define MCS_COOP_PUSH(inj, cj)                                                                      \
            {                                                                                       \
                const bool lf_ = inj && cj < 0 && cj != INT_MIN;               /* INT_MIN marks an empty slot */ \
                const unsigned mn_ = __ballot_sync(FULL, inj && cj >= 0), ml_ = __ballot_sync(FULL, lf_); \
                if (inj && cj >= 0) co_nodes[ncount + __popc(mn_ & lt)] = cj;                         \
                if (lf_) co_leaves[lcount + __popc(ml_ & lt)] = ~cj;                                  \
                ncount += __popc(mn_); lcount += __popc(ml_);                                       \
            }
            MCS_COOP_PUSH(in0, c0) MCS_COOP_PUSH(in1, c1) MCS_COOP_PUSH(in2, c2) MCS_COOP_PUSH(in3, c3)
#undef MCS_COOP_PUSH
            __syncwarp();
        }
    }
    if (lane == L) {
        h.d2 = bd2; h.tri = btri; h.k = bk; h.v = bv; h.w = bw;
        lim = wlim;
        if (FAR) S.lb2 = wlb;
        if (COUNT) q_nodes += visited;
    }
}

// MERGED (small jobs: a few walks per lane, so nearly the whole run is the tail where a warp holds a handful of
// live walkers in different phases and the cost is the number of passes, each one memory round trip): a pass
// serves the lanes that wait for a node AND the lanes that wait for a triangle -- both loads are issued before
// either is used -- and then the lanes that wait for a transition, instead of one kind per pass: every live lane
// advances every pass.  The arithmetic of a visit is unchanged.
// FAR (mcs_params.far_alpha > 0): far-field queries answered by a LOWER BOUND of the distance.  Walk-on-spheres needs a
// ball about the walker that lies inside the domain, not the largest one, and an exact query from far
// away is expensive for a reason no tree removes: every face whose box enters the ball of radius D about the query
// point has to be tested, and on a finely tessellated surface that is hundreds of faces (BASELINE config 3: 70-150
// triangle tests per query; the paper names the exterior's far queries as its bottleneck).  During
// the traversal a child (sub-tree or single face) whose box is small against its distance -- diagonal <= alpha x box
// distance, and box distance >= the near threshold -- is not descended or tested: its box distance stands for its
// faces (they are at most (1 + alpha) times farther).  The query then returns the minimum over a CUT of the tree (such
// boxes, and real faces where neither they nor an ancestor qualified).  Which nodes qualify depends on the query point only, pruning is against that running
// minimum with the usual margin, so the result does not depend on the traversal order or the schedule.  If the
// minimum is a real face the query is exact as before (exit point, termination test); if it is a box the walker
// jumps with that lower bound as its radius, at least 1 / (1 + alpha) of the largest possible one, and the shell test
// is never taken from it: boxes closer than the near threshold (a multiple of eps, in the exterior the distance whose
// Kelvin radius is that multiple) are always descended.  The estimator is the same in expectation; single walks differ
// from the exact run, so record-level parity tests run with far_alpha = 0 and matrices are compared statistically.
// KEX (exterior, mcs_params.exterior_query = 1): the paper's own exterior query, the exact distance from the walker to
// the Kelvin-inverted faces (reading E4), instead of the flat-triangle query with the conservative radius E3.
// The traversal runs on the SAME primal tree: a box is bounded below by box_ratio2, a face is tested by
// inverted_ratio2_triangle; h.d2 holds the best squared ratio, the radius in Kelvin coordinates is ratio / |x - o|.
// Lane path only (no cooperative take-over, no merged passes, no far-field cut): a cross-check variant.
// The kernel itself lives in walk_body.inc, compiled twice: once as walk_kernel (one mesh, one operator per launch;
// operator and far-field mode are template parameters) and once as walk_batch_kernel (many (mesh, operator) segments in
// ONE launch, per-lane context: mcs_estimate_dtn_batch).
#define WK_NAME walk_kernel
#define WK_BATCH 0
#define A_ a
#define G_ g
#define EXT_ EXT
#define FAR_ FAR
#include "walk_body.inc"
#undef WK_NAME
#undef WK_BATCH
#undef A_
#undef G_
#undef EXT_
#undef FAR_
#define WK_NAME walk_batch_kernel
#define WK_BATCH 1
#define A_ (cx->a)
#define G_ (cx->g)
#define EXT_ lext
#define FAR_ lfar
#include "walk_body.inc"
#undef WK_NAME
#undef WK_BATCH
#undef A_
#undef G_
#undef EXT_
#undef FAR_

__global__ void face_slot_lookup_kernel(const int32_t* __restrict__ face_slot, const int32_t* __restrict__ tri, int64_t F,
                                        int64_t n_s, int32_t* __restrict__ sample_slot)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n_s) sample_slot[i] = (tri[i] >= 0 && tri[i] < F) ? face_slot[tri[i]] : -1;      // out of range: the call is poisoned anyway
}

__global__ void balls_export_kernel(const float4* __restrict__ balls, int64_t n_s, float* __restrict__ out)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_s) return;
    const float4 b0 = balls[2 * i], b1 = balls[2 * i + 1];
    float* o = out + 8 * i;
    o[0] = b0.x; o[1] = b0.y; o[2] = b0.z; o[3] = b0.w; o[4] = b1.x; o[5] = b1.y; o[6] = b1.z; o[7] = b1.w;
}

int check_params(const mcs_bvh* b, const mcs_samples* s, const mcs_params* p, int exterior)
{
    if (!b || !s || !p) return MCS_EINVAL;
    if (s->n_s < 1 || !s->tri || !s->bary || !s->weight) return MCS_EINVAL;
    if (p->walks_per_sample < 1 || p->max_steps < 0 || !(p->eps > 0.0f)) return MCS_EINVAL;
    if (!(p->cap_half_angle_deg > 0.0f) || p->cap_half_angle_deg >= 180.0f) return MCS_EINVAL;
    if (p->bisection_iters < 1 || p->bisection_iters > 24) return MCS_EINVAL;
    if (!(p->rmax_scale > 0.0f) && !(p->rmax_override > 0.0f)) return MCS_EINVAL;
    if (s->n_s >= ((int64_t)1 << 32) - 1) return MCS_EINVAL;
    if (p->estimator != 0 && p->estimator != 1) return MCS_EINVAL;
    if (p->estimator == 1 && (exterior || !(p->inset > 0.0f))) return MCS_EINVAL;      // Alg. 1 is the interior estimator
    if (exterior && p->include_killing && (p->n_kill_walks < 1 || p->n_kill_walks >= ((int64_t)1 << 32))) return MCS_EINVAL;
    if (s->n_s * (int64_t)p->walks_per_sample >= ((int64_t)1 << 40)) return MCS_EINVAL;
    if (!(p->far_alpha >= 0.0f) || p->far_alpha > 4.0f || !(p->far_near_factor >= 0.0f)) return MCS_EINVAL;
    if (p->nonblocking != 0 && p->nonblocking != 1) return MCS_EINVAL;
    if (p->exterior_query != 0 && p->exterior_query != 1) return MCS_EINVAL;
    if (p->exterior_query == 1 && (!exterior || p->far_alpha > 0.0f)) return MCS_EINVAL;      // E4 is an exterior query; the far-field cut belongs to E3
    return MCS_OK;
}

}  // namespace

const WalkDyn* walk_dyn_of(const unsigned long long* stats_dev)
{
    return reinterpret_cast<const WalkDyn*>(reinterpret_cast<const char*>(stats_dev) + ST_COUNT * 8 + 32);   // behind the 8 scratch ints
}

int walk_error_code(int err_bits)
{
    if (err_bits & WALK_ERR_DEGENERATE) return MCS_EDEGENERATE;
    if (err_bits & WALK_ERR_SAMPLE_FACE) return MCS_EINVAL;
    return MCS_OK;
}

int64_t walk_num_records(const mcs_samples* s, const mcs_params* p, int exterior)
{
    int64_t n = s->n_s * (int64_t)p->walks_per_sample;
    if (exterior && p->include_killing) n += p->n_kill_walks;
    return n;
}

constexpr int64_t MAX_WALK_BLOCKS = 2048;         // grid cap of the persistent walk kernel (sizes the cooperative scratch)

size_t walk_workspace_bytes(const mcs_samples* s)
{
    const int64_t n = s->n_s;
    return align_up((size_t)MAX_WALK_BLOCKS * (WT / 32) * (COOP_NCAP + COOP_LCAP) * 4)   // cooperative-path warp lists
         + align_up((size_t)n * 32)                 // balls
         + align_up((size_t)n * 4) * 3              // keys, order, sample_slot
         + align_up(ST_COUNT * 8 + 64)              // counters
         + sort_workspace_bytes(n, 4) + 256;
}

// Runs A2-A6.  Layout of `ws`: see walk_workspace_bytes.
int walk_run(const mcs_bvh* b, const mcs_samples* s, const mcs_params* p, int exterior,
             void* ws, size_t ws_bytes, float4* records, int32_t* steps, bool balls_only, float* balls_out,
             bool count, unsigned long long** stats_dev_out, cudaStream_t st, WalkLaunch* defer, bool check_now)
{
    int rc = check_params(b, s, p, exterior);
    if (rc != MCS_OK) return rc;
    if (!ws || ws_bytes < walk_workspace_bytes(s)) return MCS_ENOMEM;
    const int64_t n_s = s->n_s;
    char* ptr = (char*)ws;
    int* coop_scratch = (int*)ptr;                ptr += align_up((size_t)MAX_WALK_BLOCKS * (WT / 32) * (COOP_NCAP + COOP_LCAP) * 4);
    float4* balls = (float4*)ptr;                 ptr += align_up((size_t)n_s * 32);
    uint32_t* keys = (uint32_t*)ptr;              ptr += align_up((size_t)n_s * 4);
    uint32_t* order = (uint32_t*)ptr;             ptr += align_up((size_t)n_s * 4);
    int32_t* sample_slot = (int32_t*)ptr;         ptr += align_up((size_t)n_s * 4);
    unsigned long long* stats = (unsigned long long*)ptr;  ptr += align_up(ST_COUNT * 8 + 64);
    void* sort_ws = ptr;
    const size_t sort_bytes = ws_bytes - (size_t)(ptr - (char*)ws);
    int* ibuf = (int*)(stats + ST_COUNT);         // 8 ints of scratch after the counters
    if (stats_dev_out) *stats_dev_out = stats;

    WalkGeom g;
    g.nodes = b->nodes; g.wide = b->wide; g.tris = b->tris; g.verts = b->verts; g.faces = b->faces;

    MCS_CUDA_TRY(cudaMemsetAsync(stats, 0, ST_COUNT * 8 + 64, st));
    const float3 lo = f3(b->aabb_lo[0], b->aabb_lo[1], b->aabb_lo[2]);
    const float3 hi = f3(b->aabb_hi[0], b->aabb_hi[1], b->aabb_hi[2]);
    const float3 o = exterior ? f3(p->kelvin_origin[0], p->kelvin_origin[1], p->kelvin_origin[2]) : f3(0.f, 0.f, 0.f);
    const unsigned nblk_s = (unsigned)ceil_div64(n_s, PT);
    const float mesh_scale = fmaxf(fabsf(lo.x), fabsf(hi.x)) + fmaxf(fabsf(lo.y), fabsf(hi.y)) + fmaxf(fabsf(lo.z), fabsf(hi.z));

    // r_max and, for the exterior, R_max: computed on the device and read there (WalkDyn), together with
    // the input errors only the device can see
    WalkDyn* dyn = const_cast<WalkDyn*>(walk_dyn_of(stats));
    const float side = fminf(hi.x - lo.x, fminf(hi.y - lo.y, hi.z - lo.z));
    if (exterior) {
        mcs_note_launch(), kelvin_bounds_init_kernel<<<1, 32, 0, st>>>(ibuf);
        mcs_note_launch(), kelvin_bounds_kernel<<<(unsigned)ceil_div64(b->V, PT), PT, 0, st>>>(b->verts, b->V, o, ibuf);
    }
    mcs_note_launch(), walk_dyn_kernel<<<1, 1, 0, st>>>(ibuf, exterior, side, p->rmax_scale, p->rmax_override, dyn);

    // Z-order of the samples
    mcs_note_launch(), sample_keys_kernel<<<nblk_s, PT, 0, st>>>(b->verts, b->faces, b->F, s->tri, s->bary, n_s, lo, hi, keys, order, &dyn->err);
    rc = sort_pairs_u32(keys, order, n_s, 30, sort_ws, sort_bytes, st);
    if (rc != MCS_OK) return rc;
    mcs_note_launch(), face_slot_lookup_kernel<<<(unsigned)ceil_div64(n_s, 256), 256, 0, st>>>(b->face_slot, s->tri, b->F, n_s, sample_slot);

    if (p->estimator == 1) {
        mcs_note_launch(), naive_start_kernel<<<nblk_s, PT, 0, st>>>(g, s->tri, s->bary, s->normal, n_s, p->inset, dyn, balls);
    } else {
        int dev_tb = 0, n_sm_tb = 0;
        MCS_CUDA_TRY(cudaGetDevice(&dev_tb));
        MCS_CUDA_TRY(cudaDeviceGetAttribute(&n_sm_tb, cudaDevAttrMultiProcessorCount, dev_tb));
        int64_t nblk_tb = ceil_div64(n_s, TB_WARPS);
        const int64_t cap_tb = (int64_t)n_sm_tb * 6;                  // 6 resident blocks of 34 KB shared memory per SM
        if (nblk_tb > cap_tb) nblk_tb = cap_tb;
        if (exterior)
            mcs_note_launch(), tangent_ball_kernel<true><<<(unsigned)nblk_tb, TB_WARPS * 32, 0, st>>>(
                g, s->tri, s->bary, s->normal, order, n_s, dyn, p->eps, p->bisection_iters, o, mesh_scale, balls, stats);
        else
            mcs_note_launch(), tangent_ball_kernel<false><<<(unsigned)nblk_tb, TB_WARPS * 32, 0, st>>>(
                g, s->tri, s->bary, s->normal, order, n_s, dyn, p->eps, p->bisection_iters, o, mesh_scale, balls, stats);
    }
    MCS_CUDA_TRY(cudaGetLastError());
    if (check_now) {                                 // one read-back: input errors before the expensive part runs
        WalkDyn hd;
        MCS_CUDA_TRY(cudaMemcpyAsync(&hd, dyn, sizeof hd, cudaMemcpyDeviceToHost, st));
        MCS_CUDA_TRY(cudaStreamSynchronize(st));
        if (hd.err) return walk_error_code(hd.err);
    }
    if (balls_out) mcs_note_launch(), balls_export_kernel<<<(unsigned)ceil_div64(n_s, 256), 256, 0, st>>>(balls, n_s, balls_out);
    MCS_CUDA_TRY(cudaGetLastError());
    if (balls_only) return MCS_OK;

    WalkArgs a;
    a.balls = balls; a.order = order; a.weight = s->weight; a.sample_slot = sample_slot;
    a.n_s = n_s; a.W = p->walks_per_sample;
    a.n_kill = (exterior && p->include_killing) ? p->n_kill_walks : 0;
    a.eps = p->eps; a.max_steps = p->max_steps;
    a.q0 = (float)sin(0.5 * (double)p->cap_half_angle_deg * 3.14159265358979323846 / 180.0);
    a.inv_q0 = 1.0f / a.q0;
    a.importance = p->importance_sample; a.antithetic = p->antithetic;
    a.naive = p->estimator == 1; a.inv_inset = p->estimator == 1 ? 1.0f / p->inset : 0.0f;
    a.ox = o.x; a.oy = o.y; a.oz = o.z; a.dyn = dyn;
    a.mesh_scale = mesh_scale;
    a.far_alpha2 = p->far_alpha * p->far_alpha;
    a.far_near = (p->far_near_factor > 0.0f ? fmaxf(p->far_near_factor, 2.0f) : 16.0f) * p->eps;   // never below 2 eps
    {
        const float dx = hi.x - lo.x, dy = hi.y - lo.y, dz = hi.z - lo.z;
        a.escape = exterior ? 3.0e38f : sqrtf(dx * dx + dy * dy + dz * dz);
    }
    a.key0 = (uint32_t)(p->seed & 0xFFFFFFFFu); a.key1 = (uint32_t)(p->seed >> 32);
    a.records = records; a.steps = steps; a.coop_scratch = coop_scratch;
    a.work_counter = stats + ST_WORK; a.stats = stats;

    // persistent grid: resident blocks per SM x number of SMs
    int dev = 0, n_sm = 0, per_sm = 0;
    MCS_CUDA_TRY(cudaGetDevice(&dev));
    MCS_CUDA_TRY(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
    // The warp-cooperative completion of heavy queries bounds the longest single-lane chain, which is what the
    // kernel's run time is when walks are few or queries are long-tailed (large or messy meshes).  On a small
    // tree with millions of walks (throughput-bound: BASELINE configs 0-1) its code costs registers and nothing
    // is gained, so it is compiled out there.
    const long long total_walks = s->n_s * (long long)p->walks_per_sample + ((exterior && p->include_killing) ? p->n_kill_walks : 0);
    const bool coop = b->F > 20000 || total_walks < (long long)n_sm * 2048 * 16;
    // Small jobs (a few walks per lane) run the merged-pass variant, always with the cooperative path.
    const bool merged = total_walks < (long long)n_sm * 2048 * 4;
    typedef void (*walk_fn)(WalkGeom, WalkArgs);
#define MCS_WK(E, C, P, M) { walk_kernel<E, C, P, M, false>, walk_kernel<E, C, P, M, true> }
    static const walk_fn table[12][2] = {
        MCS_WK(false, false, false, false), MCS_WK(false, false, true, false), MCS_WK(false, true, false, false), MCS_WK(false, true, true, false),
        MCS_WK(true, false, false, false),  MCS_WK(true, false, true, false),  MCS_WK(true, true, false, false),  MCS_WK(true, true, true, false),
        MCS_WK(false, false, true, true),   MCS_WK(false, true, true, true),   MCS_WK(true, false, true, true),   MCS_WK(true, true, true, true) };
#undef MCS_WK
    const int far = p->far_alpha > 0.0f ? 1 : 0;
    static const walk_fn kex_table[2] = { walk_kernel<true, false, false, false, false, true>, walk_kernel<true, true, false, false, false, true> };
    const bool kex = exterior && p->exterior_query == 1;
    const walk_fn fn = kex ? kex_table[count ? 1 : 0]
                     : merged ? table[8 + (exterior ? 2 : 0) + (count ? 1 : 0)][far]
                              : table[(exterior ? 4 : 0) + (count ? 2 : 0) + (coop ? 1 : 0)][far];
    const int tw = (merged && !kex) ? 32 : WT;        // threads per block of the chosen variant
    MCS_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, (const void*)fn, tw, 0));
    if (per_sm < 1) per_sm = 1;
    const long long total = a.n_s * a.W + a.n_kill;
    long long grid = (long long)n_sm * per_sm;
    const long long warps = grid * (tw / 32);
    long long chunk = total / (warps * 8);
    chunk = chunk < 32 ? 32 : (chunk > 256 ? 256 : chunk);
    chunk = (chunk / 32) * 32;
    a.chunk = (int)chunk;
    const long long need_blocks = ceil_div64(ceil_div64(total, chunk), tw / 32);
    if (grid > need_blocks) grid = need_blocks;
    if (grid * (tw / 32) > MAX_WALK_BLOCKS * (WT / 32)) grid = MAX_WALK_BLOCKS * (WT / 32) / (tw / 32);   // the cooperative scratch is sized per warp
    if (grid < 1) grid = 1;
    if (defer) {                                      // the caller launches it (two operators on two streams)
        defer->fn = fn; defer->grid = (unsigned)grid; defer->block = (unsigned)tw; defer->g = g; defer->a = a; defer->coop = coop || merged;
        return MCS_OK;
    }
    mcs_prof_mark(MCS_MARK_WALK_BEGIN, st);
    mcs_note_launch(), fn<<<(unsigned)grid, tw, 0, st>>>(g, a);
    mcs_prof_mark(MCS_MARK_WALK_END, st);
    MCS_CUDA_TRY(cudaGetLastError());
    return MCS_OK;
}

size_t walk_batch_scratch_bytes(int n_launches)
{
    return align_up((size_t)n_launches * sizeof(WalkCtx)) + 256
         + align_up((size_t)MAX_WALK_BLOCKS * (WT / 32) * (COOP_NCAP + COOP_LCAP) * 4);
}

int walk_launch_batch(const WalkLaunch* launches, const int* exterior, const int* far, int n_launches,
                      void* scratch, size_t scratch_bytes, cudaStream_t st)
{
    if (!launches || n_launches < 1 || !scratch || scratch_bytes < walk_batch_scratch_bytes(n_launches)) return MCS_EINVAL;
    const int chunk = 64;
    std::vector<WalkCtx> h((size_t)n_launches);
    long long begin = 0;
    for (int i = 0; i < n_launches; ++i) {
        h[i].g = launches[i].g; h[i].a = launches[i].a; h[i].begin = begin; h[i].ext = exterior[i]; h[i].far = far[i];
        const long long n = h[i].a.n_s * h[i].a.W + h[i].a.n_kill;
        begin += ceil_div64(n, chunk) * chunk;
    }
    char* p = (char*)scratch;
    WalkCtx* d_ctx = (WalkCtx*)p;                              p += align_up((size_t)n_launches * sizeof(WalkCtx));
    unsigned long long* counter = (unsigned long long*)p;      p += 256;
    int* coop_scratch = (int*)p;
    MCS_CUDA_TRY(cudaMemcpyAsync(d_ctx, h.data(), (size_t)n_launches * sizeof(WalkCtx), cudaMemcpyHostToDevice, st));
    MCS_CUDA_TRY(cudaMemsetAsync(counter, 0, 8, st));
    WalkBatch bt;
    bt.total = begin; bt.n_ctx = n_launches; bt.chunk = chunk; bt.work_counter = counter; bt.coop_scratch = coop_scratch;
    int dev = 0, n_sm = 0, per_sm = 0;
    MCS_CUDA_TRY(cudaGetDevice(&dev));
    MCS_CUDA_TRY(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
    // the warp-cooperative path when any segment would use it on its own (large trees or few walks), else the lean variant
    bool coop = false;
    for (int i = 0; i < n_launches; ++i) coop = coop || launches[i].coop;
    auto fn = coop ? walk_batch_kernel<false, true, false, false> : walk_batch_kernel<false, false, false, false>;
    MCS_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, (const void*)fn, WT, 0));
    if (per_sm < 1) per_sm = 1;
    long long grid = (long long)n_sm * per_sm;
    const long long need_blocks = ceil_div64(ceil_div64(begin, chunk), WT / 32);
    if (grid > need_blocks) grid = need_blocks;
    if (grid > MAX_WALK_BLOCKS) grid = MAX_WALK_BLOCKS;
    if (grid < 1) grid = 1;
    mcs_note_launch(), fn<<<(unsigned)grid, WT, 0, st>>>(d_ctx, bt);
    MCS_CUDA_TRY(cudaGetLastError());
    MCS_CUDA_TRY(cudaStreamSynchronize(st));                   // `h` is pageable and leaves scope
    return MCS_OK;
}

int walk_launch(const WalkLaunch* w, cudaStream_t st)
{
    mcs_note_launch(), w->fn<<<w->grid, w->block, 0, st>>>(w->g, w->a);
    MCS_CUDA_TRY(cudaGetLastError());
    return MCS_OK;
}
