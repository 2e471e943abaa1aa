// traverse.cuh -- closest point on the triangle soup through the packed LBVH.
//
// The geometric query under walk-on-spheres: "the nearest boundary point"
// (PAPER.md:155), served by a BVH in the paper's own implementation
// (PAPER.md:383).  fp32 throughout; all differences are taken from the raw
// fp32 inputs relative to the query point, so the error scales with the local
// feature size and not with the absolute coordinates.
//
// Tie rule (R15): smaller fp32 squared distance, then smaller
// ORIGINAL face index.  Sub-trees are pruned only when their box distance is
// strictly larger than the best distance so far, so the result does not depend
// on the traversal order.
#pragma once
#include "common.cuh"

#define MCS_STACK 96      // >= 63 Morton bits + log2(F) index-tie levels

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
    float tt = den > 0.0f ? -dot3(a, ab) / den : 0.0f;
    tt = fminf(fmaxf(tt, 0.0f), 1.0f);
    t = tt;
    float3 c = f3(fmaf(tt, ab.x, a.x), fmaf(tt, ab.y, a.y), fmaf(tt, ab.z, a.z));
    return dot3(c, c);
}

// a*b - c*d with the rounding error of c*d compensated through an FMA (Kahan's
// difference of products): the result is within ~1.5 ulp of the exact value even under
// heavy cancellation.  Used for the face normal, so that sliver triangles (aspect
// ratio > 100, BASELINE.json config 3) keep an accurate supporting plane.
__device__ __forceinline__ float diff_of_products(float a, float b, float c, float d)
{
    const float cd = __fmul_rn(c, d);
    const float err = __fmaf_rn(-c, d, cd);
    const float r = __fmaf_rn(a, b, -cd);
    return __fadd_rn(r, err);
}

// Closest point of triangle (a, b, c) to p, computed on the triangle translated by -p
// (A, B, C = vertices seen from p, so every rounding error scales with the distance to
// the triangle, not with the absolute coordinates):
//   n = ab x ac (compensated), q = projection of p on the plane = ((A.n)/|n|^2) n,
//   edge functions w_b = ((C-q) x (A-q)).n, w_c = ((A-q) x (B-q)).n, w_a = |n|^2 - w_b - w_c
//   (|n|^2-scaled barycentrics of q).  All >= 0: the answer is q.  Otherwise the closest
//   point lies on an edge whose edge function is negative (at most two): clamp onto those.
// Removing the normal component before forming the edge functions keeps them accurate for
// far-away p; the compensated normal keeps them accurate for slivers.
// Returns the squared distance; (v, w) are the weights of b and c.
// Zero-area faces (|ab x ac|^2 <= 1e-12 max|e|^4) fall back to their three edges
// (R16).
__device__ __forceinline__ float closest_point_triangle(float3 p, float3 a, float3 b, float3 c, float& v, float& w)
{
    const float3 ab = b - a, ac = c - a;
    const float3 A = a - p, B = b - p, C = c - p;
    const float3 n = f3(diff_of_products(ab.y, ac.z, ab.z, ac.y),
                        diff_of_products(ab.z, ac.x, ab.x, ac.z),
                        diff_of_products(ab.x, ac.y, ab.y, ac.x));
    const float nn = dot3(n, n);
    const float e2 = fmaxf(dot3(ab, ab), dot3(ac, ac));
    float t, best, d;
    if (nn <= 1e-12f * e2 * e2) {
        best = origin_to_segment(A, B, t); v = t; w = 0.0f;
        d = origin_to_segment(B, C, t); if (d < best) { best = d; v = 1.0f - t; w = t; }
        d = origin_to_segment(C, A, t); if (d < best) { best = d; v = 0.0f; w = 1.0f - t; }
        return best;
    }
    const float rnn = 1.0f / nn;
    const float An = dot3(A, n);
    const float hq = An * rnn;
    const float3 q = f3(hq * n.x, hq * n.y, hq * n.z);
    const float3 Aq = A - q, Bq = B - q, Cq = C - q;
    const float wb = dot3(cross3(Cq, Aq), n);
    const float wc = dot3(cross3(Aq, Bq), n);
    const float wa = nn - wb - wc;
    if (wa >= 0.0f && wb >= 0.0f && wc >= 0.0f) {                 // face
        v = fminf(wb * rnn, 1.0f);
        w = fminf(wc * rnn, 1.0f - v);
        return An * hq;
    }
    best = CUDART_INF_F;
    if (wc < 0.0f) { best = origin_to_segment(A, B, t); v = t; w = 0.0f; }                                    // edge ab
    if (wa < 0.0f) { d = origin_to_segment(B, C, t); if (d < best) { best = d; v = 1.0f - t; w = t; } }       // edge bc
    if (wb < 0.0f) { d = origin_to_segment(C, A, t); if (d < best) { best = d; v = 0.0f; w = 1.0f - t; } }    // edge ca
    return best;
}

__device__ __forceinline__ float box_dist2(float3 p, float lx, float ly, float lz, float hx, float hy, float hz)
{
    const float dx = fmaxf(fmaxf(lx - p.x, p.x - hx), 0.0f);
    const float dy = fmaxf(fmaxf(ly - p.y, p.y - hy), 0.0f);
    const float dz = fmaxf(fmaxf(lz - p.z, p.z - hz), 0.0f);
    return fmaf(dx, dx, fmaf(dy, dy, dz * dz));
}

__device__ __forceinline__ void load_tri(const PackedTri* __restrict__ tris, int k, float3& a, float3& b, float3& c, int& orig)
{
    const float4* t = reinterpret_cast<const float4*>(tris + k);
    const float4 t0 = __ldg(t), t1 = __ldg(t + 1), t2 = __ldg(t + 2);
    a = f3(t0.x, t0.y, t0.z); b = f3(t1.x, t1.y, t1.z); c = f3(t2.x, t2.y, t2.z);
    orig = __float_as_int(t0.w);
}

__device__ __forceinline__ void test_triangle(const PackedTri* __restrict__ tris, int k, float3 p, ClosestHit& h)
{
    float3 a, b, c; int orig; float v, w;
    load_tri(tris, k, a, b, c, orig);
    const float d2 = closest_point_triangle(p, a, b, c, v, w);
    if (d2 < h.d2 || (d2 == h.d2 && orig < h.tri)) { h.d2 = d2; h.tri = orig; h.k = k; h.v = v; h.w = w; }
}

// Full closest-point traversal.  `h` carries the initial bound on entry
// (h.d2 = +inf, h.tri = INT_MAX for an unbounded query, or the result of testing
// a guessed triangle first) and the answer on exit.
// ANY = true: stop as soon as any triangle with d2 < h.d2 is found (bounded
// "is anything closer than R" probe of the tangent-ball bisection);
// the caller sets h.tri = -1 so that equal distances do not count.
template <bool COUNT, bool ANY>
__device__ __forceinline__ void bvh_closest_point(const BvhNode* __restrict__ nodes, const PackedTri* __restrict__ tris,
                                                  float3 p, ClosestHit& h, TraversalCounters& cnt)
{
    int   stack_n[MCS_STACK];
    float stack_d[MCS_STACK];
    int sp = 0;
    int node = 0;
    const float bound0 = h.d2;
    // A sub-tree is pruned when its box is farther than the best distance by more than a
    // few ulps: the fp32 box distance of a face's own leaf may round above the fp32
    // distance to the face, and an equal-distance face with a smaller index must still
    // be reached for the tie rule to hold.
    const float SLACK = 1.0f + 4e-6f;
    float lim = h.d2 * SLACK;
    for (;;) {
        const float4* nd = reinterpret_cast<const float4*>(nodes + node);
        const float4 w0 = __ldg(nd), w1 = __ldg(nd + 1), w2 = __ldg(nd + 2);
        const int4 w3 = __ldg(reinterpret_cast<const int4*>(nd + 3));
        if (COUNT) cnt.nodes++;
        const float d0 = box_dist2(p, w0.x, w0.y, w0.z, w0.w, w1.x, w1.y);
        const float d1 = box_dist2(p, w1.z, w1.w, w2.x, w2.y, w2.z, w2.w);
        const int c0 = w3.x, c1 = w3.y;
        bool go0 = d0 <= lim, go1 = d1 <= lim;
        if (go0 && c0 < 0) { test_triangle(tris, ~c0, p, h); if (COUNT) cnt.tris++; go0 = false; lim = h.d2 * SLACK; }
        if (go1 && c1 < 0) {
            if (d1 <= lim) { test_triangle(tris, ~c1, p, h); if (COUNT) cnt.tris++; lim = h.d2 * SLACK; }
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
    float3 a, b, c; int orig;
    load_tri(tris, h.k, a, b, c, orig);
    const float u = 1.0f - h.v - h.w;
    return f3(fmaf(u, a.x, fmaf(h.v, b.x, h.w * c.x)),
              fmaf(u, a.y, fmaf(h.v, b.y, h.w * c.y)),
              fmaf(u, a.z, fmaf(h.v, b.z, h.w * c.z)));
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
