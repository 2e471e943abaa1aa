// traverse.cuh -- closest point on the triangle soup through the packed LBVH.
//
// The geometric query under walk-on-spheres: "the nearest boundary point"
// (PAPER.md:155), served by a BVH in the paper's own implementation
// (PAPER.md:383).  fp32 throughout; all differences are taken from the raw
// fp32 inputs relative to the query point, so the error scales with the local
// feature size and not with the absolute coordinates.
//
// Tie rule (R15): smaller fp32 squared distance, then smaller
// ORIGINAL face index.  Sub-trees are pruned only when their box distance exceeds
// prune_limit(best): the best squared distance so far plus an absolute margin that
// covers the rounding of the computed triangle distances, so every face that can hold
// the computed minimum is tested and the result does not depend on the traversal order.
#pragma once
#include "common.cuh"

#define MCS_STACK 160     // binary tree: >= 63 Morton bits + log2(F) index-tie levels; 4-wide walk: 3 pushes per two levels

// 256-bit read-only global load (sm_100: LDG.E.256).  A divergent warp pays one L1
// wavefront per lane and per load instruction whatever its width, and that wavefront rate
// (one per cycle per SM) is what bounds the walk kernel: 32-byte loads halve the wavefronts
// of a 64-byte node or triangle.  p must be 32-byte aligned.
struct __align__(32) Vec8 { float4 lo, hi; };
__device__ __forceinline__ Vec8 ldg256(const void* p)
{
    Vec8 r;
    asm volatile("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=f"(r.lo.x), "=f"(r.lo.y), "=f"(r.lo.z), "=f"(r.lo.w), "=f"(r.hi.x), "=f"(r.hi.y), "=f"(r.hi.z), "=f"(r.hi.w)
                 : "l"(p));
    return r;
}

struct ClosestHit {
    float d2;      // squared distance
    int   tri;     // ORIGINAL face index (-1: none)
    int   k;       // sorted (Morton-order) triangle slot
    float v, w;    // barycentric weights of vertices 1, 2 of the closest point
};

struct TraversalCounters {
    unsigned nodes, tris;
};

__host__ __device__ __forceinline__ float3 f3(float x, float y, float z) { return make_float3(x, y, z); }
__device__ __forceinline__ float3 operator-(float3 a, float3 b) { return f3(a.x - b.x, a.y - b.y, a.z - b.z); }
__device__ __forceinline__ float3 operator+(float3 a, float3 b) { return f3(a.x + b.x, a.y + b.y, a.z + b.z); }
__device__ __forceinline__ float3 operator*(float s, float3 a) { return f3(s * a.x, s * a.y, s * a.z); }
__device__ __forceinline__ float dot3(float3 a, float3 b) { return fmaf(a.x, b.x, fmaf(a.y, b.y, a.z * b.z)); }
__device__ __forceinline__ float3 cross3(float3 a, float3 b)
{
    return f3(a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x);
}

// Squared distance from the ORIGIN to the segment a + t (b - a), t in [0,1].
__device__ __forceinline__ float origin_to_segment(float3 a, float3 b, float& t)
{
    float3 ab = b - a;
    float den = dot3(ab, ab);
    float tt = den > 0.0f ? __fdividef(-dot3(a, ab), den) : 0.0f;
    tt = fminf(fmaxf(tt, 0.0f), 1.0f);
    t = tt;
    float3 c = f3(fmaf(tt, ab.x, a.x), fmaf(tt, ab.y, a.y), fmaf(tt, ab.z, a.z));
    return dot3(c, c);
}

// One packed triangle as the query kernels see it (common.cuh "PackedTri"): the three fp32
// vertices exactly as given, plus the supporting plane precomputed by the build in fp64 and
// rounded once: n = (b-a) x (c-a), nn = |n|^2, rnn = 1/nn.  A sliver (aspect ratio > 100,
// BASELINE.json config 3) loses its plane when the cross product is formed in fp32
// (relative error eps * aspect); with the fp64 normal the error of the plane is one rounding.
struct TriData {
    float3 a, b, c, n;
    float  nn, rnn;
    int    orig;           // original face index
    bool   degenerate;     // zero-area face: absorbs as its three edges (R16)
};

__device__ __forceinline__ TriData unpack_tri(float4 t0, float4 t1, float4 t2, float4 t3)
{
    TriData T;
    T.a = f3(t0.x, t0.y, t0.z); T.b = f3(t1.x, t1.y, t1.z); T.c = f3(t2.x, t2.y, t2.z);
    T.n = f3(t3.x, t3.y, t3.z);
    T.orig = __float_as_int(t0.w); T.nn = t1.w; T.rnn = t2.w; T.degenerate = (__float_as_int(t3.w) & 1) != 0;
    return T;
}

__device__ __forceinline__ TriData load_tri(const PackedTri* __restrict__ tris, int k)
{
    const Vec8 u0 = ldg256(tris + k), u1 = ldg256(reinterpret_cast<const char*>(tris + k) + 32);
    return unpack_tri(u0.lo, u0.hi, u1.lo, u1.hi);
}

// Closest point of triangle T to p, computed on the triangle translated by -p (A, B, C =
// vertices seen from p, so every rounding error scales with the distance to the triangle,
// not with the absolute coordinates):
//   q = projection of p on the plane = ((A.n)/|n|^2) n,
//   edge functions w_b = ((C-q) x (A-q)).n, w_c = ((A-q) x (B-q)).n, w_a = |n|^2 - w_b - w_c
//   (|n|^2-scaled barycentrics of q).  All >= 0: the answer is q.  Otherwise the closest
//   point lies on an edge whose edge function is negative (at most two): clamp onto those.
// Removing the normal component before forming the edge functions keeps them accurate for
// far-away p.  Returns the squared distance; (v, w) are the weights of b and c.
// `bound`: a triangle whose PLANE is already farther than bound cannot matter to the caller;
// +inf is returned for it without the in-plane work (v, w untouched).
__device__ __forceinline__ float closest_point_triangle(float3 p, const TriData& T, float bound, float& v, float& w)
{
    const float3 A = T.a - p, B = T.b - p, C = T.c - p;
    float t, best, d;
    if (T.degenerate) {
        best = origin_to_segment(A, B, t); v = t; w = 0.0f;
        d = origin_to_segment(B, C, t); if (d < best) { best = d; v = 1.0f - t; w = t; }
        d = origin_to_segment(C, A, t); if (d < best) { best = d; v = 0.0f; w = 1.0f - t; }
        return best;
    }
    const float An = dot3(A, T.n);
    const float hq = An * T.rnn;
    const float plane_d2 = An * hq;
    if (plane_d2 > bound) return CUDART_INF_F;
    const float3 q = f3(hq * T.n.x, hq * T.n.y, hq * T.n.z);
    const float3 Aq = A - q, Bq = B - q, Cq = C - q;
    const float wb = dot3(cross3(Cq, Aq), T.n);
    const float wc = dot3(cross3(Aq, Bq), T.n);
    const float wa = T.nn - wb - wc;
    if (wa >= 0.0f && wb >= 0.0f && wc >= 0.0f) {                 // face
        v = fminf(wb * T.rnn, 1.0f);
        w = fminf(wc * T.rnn, 1.0f - v);
        return plane_d2;
    }
    // first edge with a negative edge function (order ab, bc, ca), selected so that all lanes run ONE clamp
    const int e1 = wc < 0.0f ? 0 : (wa < 0.0f ? 1 : 2);
    {
        const float3 P = e1 == 0 ? A : (e1 == 1 ? B : C), Q = e1 == 0 ? B : (e1 == 1 ? C : A);
        best = origin_to_segment(P, Q, t);
        v = e1 == 0 ? t : (e1 == 1 ? 1.0f - t : 0.0f);
        w = e1 == 0 ? 0.0f : (e1 == 1 ? t : 1.0f - t);
    }
    // a second one (vertex regions): ab & bc -> bc, ab & ca -> ca, bc & ca -> ca
    const int e2 = (e1 == 0 && wa < 0.0f) ? 1 : ((e1 < 2 && wb < 0.0f) ? 2 : -1);
    if (e2 >= 0) {
        const float3 P = e2 == 1 ? B : C, Q = e2 == 1 ? C : A;
        d = origin_to_segment(P, Q, t);
        if (d < best) { best = d; v = e2 == 1 ? 1.0f - t : 0.0f; w = e2 == 1 ? t : 1.0f - t; }
    }
    return best;
}

// ---------------------------------------------------------------------------
// Exact distance to the Kelvin image of a flat face (reading E4; the paper's "spherical-triangular
// elements" with "non-planar distance queries").  With x = kappa(y) and the distance identity of the
// inversion, dist(y, kappa(T)) = (1/|x|) min over p in T of |x - p| / |p| (coordinates about the inversion centre), so
// the query minimises the ratio over the FLAT face: where the Apollonius sphere {|x - p| = k |p|} (centre x / (1 - k^2))
// touches the face's plane, if that point lies in the face; else on an edge (N(t)/D(t), two quadratics with the same
// leading coefficient: the stationary points solve a quadratic) or at a vertex.  Every candidate's value is recomputed
// from the candidate point itself, |x - p|^2 / |p|^2 with the differences taken directly, so the cancellation-prone
// closed forms only choose WHERE, not the value.  X, and the vertices in T, are relative to the inversion centre.
// Returns the squared ratio; (v, w) = weights of b and c.
// ---------------------------------------------------------------------------
__device__ __forceinline__ float ratio2_point(float3 X, float3 P)
{
    const float3 d = X - P;
    const float pp = dot3(P, P);
    return pp > 0.0f ? __fdividef(dot3(d, d), pp) : CUDART_INF_F;
}

__device__ __forceinline__ float inverted_ratio2_triangle(float3 X, float3 A, float3 B, float3 C, float3 n, float nn, bool degenerate,
                                                          float& v, float& w)
{
    float best = ratio2_point(X, A); v = 0.0f; w = 0.0f;
    { const float f = ratio2_point(X, B); if (f < best) { best = f; v = 1.0f; w = 0.0f; } }
    { const float f = ratio2_point(X, C); if (f < best) { best = f; v = 0.0f; w = 1.0f; } }
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const float3 P = k == 0 ? A : (k == 1 ? B : C), Q = k == 0 ? B : (k == 1 ? C : A);
        const float3 e = Q - P, xp = X - P;
        const float n0 = dot3(xp, xp), n1 = -2.0f * dot3(xp, e), n2 = dot3(e, e);
        const float d0 = dot3(P, P), d1 = 2.0f * dot3(P, e);
        const float qa = n2 * (d1 - n1), qb = 2.0f * n2 * (d0 - n0), qc = n1 * d0 - n0 * d1;
        const float disc = qb * qb - 4.0f * qa * qc;
        if (disc >= 0.0f) {
            const float q = -0.5f * (qb + copysignf(sqrtf(disc), qb));
            const float t1 = qa != 0.0f ? q / qa : -1.0f, t2 = q != 0.0f ? qc / q : -1.0f;
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                const float t = j ? t2 : t1;
                if (t > 0.0f && t < 1.0f) {
                    const float3 Pt = f3(fmaf(t, e.x, P.x), fmaf(t, e.y, P.y), fmaf(t, e.z, P.z));
                    const float f = ratio2_point(X, Pt);
                    if (f < best) {
                        best = f;
                        v = k == 0 ? t : (k == 1 ? 1.0f - t : 0.0f);
                        w = k == 0 ? 0.0f : (k == 1 ? t : 1.0f - t);
                    }
                }
            }
        }
    }
    if (!degenerate) {
        const float inv = rsqrtf(nn);
        const float3 nh = inv * n;
        const float h = dot3(nh, A), hx = dot3(nh, X), xx = dot3(X, X);
        const float A2 = h * h, B2 = 2.0f * h * (hx - h) - xx, C2 = (hx - h) * (hx - h);
        float u = -1.0f;
        if (A2 > 1e-12f * xx) {
            const float disc = B2 * B2 - 4.0f * A2 * C2;
            if (disc >= 0.0f) { const float q = -0.5f * (B2 - sqrtf(disc)); u = q > 0.0f ? C2 / q : -1.0f; }
        } else if (xx > 0.0f) {
            u = C2 / xx;
        }
        if (u >= 0.0f && fabsf(1.0f - u) > 1e-6f) {
            const float s = 1.0f / (1.0f - u);
            const float3 cc = s * X;
            const float off = dot3(nh, cc) - h;
            const float3 p0 = f3(cc.x - off * nh.x, cc.y - off * nh.y, cc.z - off * nh.z);
            // |n|^2-scaled barycentrics of p0 by edge functions, as in closest_point_triangle
            const float3 Aq = A - p0, Bq = B - p0, Cq = C - p0;
            const float wb = dot3(cross3(Cq, Aq), n), wc = dot3(cross3(Aq, Bq), n), wa = nn - wb - wc;
            if (wa >= 0.0f && wb >= 0.0f && wc >= 0.0f) {
                const float rnn = 1.0f / nn;
                const float vv = fminf(wb * rnn, 1.0f), ww = fminf(wc * rnn, 1.0f - vv);
                const float uu = 1.0f - vv - ww;
                const float3 pt = f3(fmaf(uu, A.x, fmaf(vv, B.x, ww * C.x)), fmaf(uu, A.y, fmaf(vv, B.y, ww * C.y)), fmaf(uu, A.z, fmaf(vv, B.z, ww * C.z)));
                const float f = ratio2_point(X, pt);
                if (f < best) { best = f; v = vv; w = ww; }
            }
        }
    }
    return best;
}

// Lower bound of |x - p|^2 / |p - o|^2 over a box: squared distance of x to the box over the squared distance of the
// box's farthest corner from o.
__device__ __forceinline__ float box_ratio2(float3 x, float3 o, float lx, float ly, float lz, float hx, float hy, float hz)
{
    const float d2 = fmaf(fmaxf(fmaxf(lx - x.x, x.x - hx), 0.0f), fmaxf(fmaxf(lx - x.x, x.x - hx), 0.0f),
                     fmaf(fmaxf(fmaxf(ly - x.y, x.y - hy), 0.0f), fmaxf(fmaxf(ly - x.y, x.y - hy), 0.0f),
                          fmaxf(fmaxf(lz - x.z, x.z - hz), 0.0f) * fmaxf(fmaxf(lz - x.z, x.z - hz), 0.0f)));
    const float fx = fmaxf(fabsf(lx - o.x), fabsf(hx - o.x)), fy = fmaxf(fabsf(ly - o.y), fabsf(hy - o.y)), fz = fmaxf(fabsf(lz - o.z), fabsf(hz - o.z));
    const float far2 = fmaf(fx, fx, fmaf(fy, fy, fz * fz));
    return far2 < 3.0e38f ? __fdividef(d2, far2) * (1.0f - 4e-7f) : CUDART_INF_F;      // empty slot (lo = +inf): never visited
}

__device__ __forceinline__ float box_dist2(float3 p, float lx, float ly, float lz, float hx, float hy, float hz)
{
    const float dx = fmaxf(fmaxf(lx - p.x, p.x - hx), 0.0f);
    const float dy = fmaxf(fmaxf(ly - p.y, p.y - hy), 0.0f);
    const float dz = fmaxf(fmaxf(lz - p.z, p.z - hz), 0.0f);
    return fmaf(dx, dx, fmaf(dy, dy, dz * dz));
}

// Pruning limit for a running best squared distance d2 of query p.  A sub-tree is skipped when its box is farther than
// the limit, so the limit must exceed d2 by more than the error of the COMPUTED triangle distances: otherwise a
// triangle whose computed distance is the minimum can be skipped after a near-tie has been found first and kept when it
// comes first, and the result depends on the traversal order -- which differs between the lane path and the
// warp-cooperative path, i.e. on the schedule (found on the 2 M-face stress mesh: 1 walk in 82 M changed between
// reruns).  The vertices seen from p carry an absolute rounding error of a few ulp of the coordinates involved, whatever
// the distance, so the margin is absolute in the DISTANCE: (sqrt(d2) + eta)^2 with eta = 8 eps32 (|p|_1 + mesh scale).
__device__ __forceinline__ float prune_limit(float d2, float3 p, float scale)
{
    const float eta = 9.6e-7f * (fabsf(p.x) + fabsf(p.y) + fabsf(p.z) + scale);
    return fminf(fmaf(2.0f * eta, sqrtf(d2), d2 * (1.0f + 4e-6f)) + eta * eta, 3.0e38f);
}

// Tests sorted triangle k against the running best h; `lim` = h.d2 with the pruning slack.
__device__ __forceinline__ void test_triangle(const PackedTri* __restrict__ tris, int k, float3 p, ClosestHit& h, float lim)
{
    const TriData T = load_tri(tris, k);
    float v = 0.0f, w = 0.0f;
    (void)lim;     // no plane early-out here: an exact tie (d2 == h.d2, e.g. 0 on a shared edge) must reach the index rule
    const float d2 = closest_point_triangle(p, T, CUDART_INF_F, v, w);
    if (d2 < h.d2 || (d2 == h.d2 && T.orig < h.tri)) { h.d2 = d2; h.tri = T.orig; h.k = k; h.v = v; h.w = w; }
}

// Full closest-point traversal.  `h` carries the initial bound on entry
// (h.d2 = +inf, h.tri = INT_MAX for an unbounded query, or the result of testing
// a guessed triangle first) and the answer on exit.
// ANY = true: stop as soon as any triangle with d2 < h.d2 is found (bounded
// "is anything closer than R" probe of the tangent-ball bisection);
// the caller sets h.tri = -1 so that equal distances do not count.
template <bool COUNT, bool ANY>
__device__ __forceinline__ void bvh_closest_point(const BvhNode* __restrict__ nodes, const PackedTri* __restrict__ tris,
                                                  float3 p, ClosestHit& h, TraversalCounters& cnt, float mesh_scale)
{
    int   stack_n[MCS_STACK];
    float stack_d[MCS_STACK];
    int sp = 0;
    int node = 0;
    const float bound0 = h.d2;
    // A sub-tree is pruned when its box is farther than prune_limit(best): every face that can hold the computed
    // minimum, or tie with it, is reached, so the result equals the exhaustive minimum under the index tie rule.
    float lim = prune_limit(h.d2, p, mesh_scale);
    for (;;) {
        const Vec8 n0 = ldg256(nodes + node), n1 = ldg256(reinterpret_cast<const char*>(nodes + node) + 32);
        const float4 w0 = n0.lo, w1 = n0.hi, w2 = n1.lo;
        const int4 w3 = make_int4(__float_as_int(n1.hi.x), __float_as_int(n1.hi.y), __float_as_int(n1.hi.z), __float_as_int(n1.hi.w));
        if (COUNT) cnt.nodes++;
        const float d0 = box_dist2(p, w0.x, w0.y, w0.z, w0.w, w1.x, w1.y);
        const float d1 = box_dist2(p, w1.z, w1.w, w2.x, w2.y, w2.z, w2.w);
        const int c0 = w3.x, c1 = w3.y;
        bool go0 = d0 <= lim, go1 = d1 <= lim;
        if (go0 && c0 < 0) { test_triangle(tris, ~c0, p, h, lim); if (COUNT) cnt.tris++; go0 = false; lim = prune_limit(h.d2, p, mesh_scale); }
        if (go1 && c1 < 0) {
            if (d1 <= lim) { test_triangle(tris, ~c1, p, h, lim); if (COUNT) cnt.tris++; lim = prune_limit(h.d2, p, mesh_scale); }
            go1 = false;
        }
        if (ANY && h.d2 < bound0) return;
        go0 = go0 && d0 <= lim;
        go1 = go1 && d1 <= lim;
        if (go0 && go1) {
            const bool swap = d1 < d0;
            const int nearc = swap ? c1 : c0, farc = swap ? c0 : c1;
            stack_n[sp] = farc; stack_d[sp] = swap ? d0 : d1; ++sp;
            node = nearc;
        } else if (go0) {
            node = c0;
        } else if (go1) {
            node = c1;
        } else {
            bool found = false;
            while (sp > 0) {
                --sp;
                if (stack_d[sp] <= lim) { node = stack_n[sp]; found = true; break; }
            }
            if (!found) return;
        }
    }
}

// Barycentric position of hit h in the primal mesh.
__device__ __forceinline__ float3 hit_point(const PackedTri* __restrict__ tris, const ClosestHit& h)
{
    const float4* t = reinterpret_cast<const float4*>(tris + h.k);
    const float4 t0 = __ldg(t), t1 = __ldg(t + 1), t2 = __ldg(t + 2);
    const float u = 1.0f - h.v - h.w;
    return f3(fmaf(u, t0.x, fmaf(h.v, t1.x, h.w * t2.x)),
              fmaf(u, t0.y, fmaf(h.v, t1.y, h.w * t2.y)),
              fmaf(u, t0.z, fmaf(h.v, t1.z, h.w * t2.z)));
}

// ---------------------------------------------------------------------------
// Philox4x32-10 (Salmon et al., SC'11), keyed by the seed, counter =
// (sample, walk, step, purpose)  (R18; BASELINE.json north_star).
// ---------------------------------------------------------------------------
#define MCS_PURPOSE_INIT 1u
#define MCS_PURPOSE_STEP 2u
#define MCS_KILLING_SAMPLE 0xFFFFFFFFu

__device__ __forceinline__ uint4 philox4x32_10(uint4 c, uint2 k)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const unsigned hi0 = __umulhi(0xD2511F53u, c.x), lo0 = 0xD2511F53u * c.x;
        const unsigned hi1 = __umulhi(0xCD9E8D57u, c.z), lo1 = 0xCD9E8D57u * c.z;
        c = make_uint4(hi1 ^ c.y ^ k.x, lo1, hi0 ^ c.w ^ k.y, lo0);
        k.x += 0x9E3779B9u; k.y += 0xBB67AE85u;
    }
    return c;
}

// uint32 -> (0,1): ((x >> 9) + 1/2) 2^-23, exact in fp32.
__device__ __forceinline__ float u01(unsigned x) { return ((float)(x >> 9) + 0.5f) * (1.0f / 8388608.0f); }
