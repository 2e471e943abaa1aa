/*
 * dtn_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU restatement (C99, double precision, brute
 * force geometry) of the hot path of "Monte Carlo Steklov Operators for
 * Large-Scale Geometry Processing in the Wild" (arxiv 2606.05581, PAPER.md):
 * the walk-on-spheres estimator of the discrete Dirichlet-to-Neumann matrix,
 * interior (Alg. 2, Eq. 26) and exterior (Eq. 32,
 * PAPER.md:348-353, App. C.3-C.7).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load this.  It shares no code, header, table or
 * helper with paper_2606_05581_b200/csrc.  Every function cites the passage of
 * PAPER.md it follows; where the paper is silent the reading is the one listed
 * in DESIGN.md ("Readings") and named here as [Rn].
 *
 * Pins (tests/test_oracle_*.py, all run without a GPU):
 *   philox4x32_10        cuRAND host generator (independent implementation)
 *   closest point        second formulation + invariants + brute force
 *   tangent ball         closed forms (sphere, cube face)
 *   WoS                  martingale E[t] = z, Poisson kernel of the ball (Eq. 22)
 *   interior weights     analytic unit ball: S -> diag(l) minus the cap term
 *   exterior weights     analytic sphere, centred and off-centre: l, l+1, capacity
 *   mesh estimators      symmetry, PSD, zero row sums, multiplicities 1,3,5,7
 *   Alg. 1 (naive)       unit ball: (1 - (1 - eps)^l) / eps; mesh: not PSD, variance ~ 1/eps
 *   point basis (k-NN)   numpy neighbour search, weight special cases, sphere spectrum l through the estimator
 *   winding number       closed surfaces (1 / 0), octant and rectangle closed forms, hemisphere 1/2, flipped faces found
 * Parity unpinned: nothing in this file.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_PI 3.14159265358979323846

/* ------------------------------------------------------------------------- */
/* Counter-based RNG: Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11).      */
/* The paper does not describe its RNG; BASELINE.json north_star fixes        */
/* "Philox keyed by (seed, sample, walk, step)"  [R18].                        */
/* key = (seed_lo, seed_hi); counter = (sample, walk, step, purpose).         */
/* ------------------------------------------------------------------------- */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;          /* golden-ratio Weyl increments */
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* uint32 -> uniform in (0,1): ((x >> 9) + 1/2) * 2^-23, exact in fp32 and fp64 [R18]. */
double orc_u01(uint32_t x)
{
    return ((double)(x >> 9) + 0.5) * (1.0 / 8388608.0);
}

enum { ORC_PURPOSE_INIT = 1, ORC_PURPOSE_STEP = 2 };
#define ORC_KILLING_SAMPLE 0xFFFFFFFFu

static void orc_uniform2(uint64_t seed, uint32_t sample, uint32_t walk, uint32_t step,
                         uint32_t purpose, double *u1, double *u2)
{
    uint32_t ctr[4] = { sample, walk, step, purpose };
    uint32_t key[2] = { (uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32) };
    uint32_t w[4];
    orc_philox4x32_10(ctr, key, w);
    *u1 = orc_u01(w[0]);
    *u2 = orc_u01(w[1]);
}

/* ------------------------------------------------------------------------- */
/* small vector helpers                                                       */
/* ------------------------------------------------------------------------- */
static double dot3(const double a[3], const double b[3]) { return a[0]*b[0] + a[1]*b[1] + a[2]*b[2]; }
static void sub3(const double a[3], const double b[3], double o[3]) { o[0]=a[0]-b[0]; o[1]=a[1]-b[1]; o[2]=a[2]-b[2]; }
static void cross3(const double a[3], const double b[3], double o[3])
{
    o[0] = a[1]*b[2] - a[2]*b[1];
    o[1] = a[2]*b[0] - a[0]*b[2];
    o[2] = a[0]*b[1] - a[1]*b[0];
}
static double norm3(const double a[3]) { return sqrt(dot3(a, a)); }

/* ------------------------------------------------------------------------- */
/* Closest point on a segment / triangle (the geometric query under WoS,      */
/* PAPER.md:155 "the nearest boundary point").                  */
/* ------------------------------------------------------------------------- */
static double closest_on_segment(const double p[3], const double a[3], const double b[3],
                                 double cp[3], double *t_out)
{
    double ab[3], ap[3];
    sub3(b, a, ab); sub3(p, a, ap);
    double den = dot3(ab, ab);
    double t = den > 0.0 ? dot3(ap, ab) / den : 0.0;
    if (t < 0.0) t = 0.0;
    if (t > 1.0) t = 1.0;
    for (int k = 0; k < 3; ++k) cp[k] = a[k] + t * ab[k];
    double d[3]; sub3(p, cp, d);
    *t_out = t;
    return dot3(d, d);
}

/* Closest point over the three edges; used for degenerate triangles [R16]. */
static double closest_on_edges(const double p[3], const double a[3], const double b[3],
                               const double c[3], double cp[3], double bary[3])
{
    double best = INFINITY, q[3], t;
    double d2 = closest_on_segment(p, a, b, q, &t);
    if (d2 < best) { best = d2; memcpy(cp, q, sizeof q); bary[0] = 1.0 - t; bary[1] = t; bary[2] = 0.0; }
    d2 = closest_on_segment(p, b, c, q, &t);
    if (d2 < best) { best = d2; memcpy(cp, q, sizeof q); bary[0] = 0.0; bary[1] = 1.0 - t; bary[2] = t; }
    d2 = closest_on_segment(p, c, a, q, &t);
    if (d2 < best) { best = d2; memcpy(cp, q, sizeof q); bary[0] = t; bary[1] = 0.0; bary[2] = 1.0 - t; }
    return best;
}

/*
 * Voronoi-region method (Ericson, Real-Time Collision Detection, sec. 5.1.5,
 * restated): classify p against the vertex, edge and face regions of triangle
 * abc; returns the squared distance, the closest point and its barycentric
 * coordinates (weights of a, b, c).
 */
double orc_closest_point_triangle(const double p[3], const double a[3], const double b[3],
                                  const double c[3], double cp[3], double bary[3])
{
    double ab[3], ac[3], ap[3], bp[3], cpv[3], nrm[3];
    sub3(b, a, ab); sub3(c, a, ac);
    cross3(ab, ac, nrm);
    double e2 = fmax(dot3(ab, ab), dot3(ac, ac));
    if (dot3(nrm, nrm) <= 1e-24 * e2 * e2)                /* zero-area face [R16] */
        return closest_on_edges(p, a, b, c, cp, bary);

    sub3(p, a, ap);
    double d1 = dot3(ab, ap), d2 = dot3(ac, ap);
    double v, w;
    if (d1 <= 0.0 && d2 <= 0.0) { v = 0.0; w = 0.0; goto done; }            /* vertex a */
    sub3(p, b, bp);
    double d3 = dot3(ab, bp), d4 = dot3(ac, bp);
    if (d3 >= 0.0 && d4 <= d3) { v = 1.0; w = 0.0; goto done; }              /* vertex b */
    double vc = d1 * d4 - d3 * d2;
    if (vc <= 0.0 && d1 >= 0.0 && d3 <= 0.0) { v = d1 / (d1 - d3); w = 0.0; goto done; }   /* edge ab */
    sub3(p, c, cpv);
    double d5 = dot3(ab, cpv), d6 = dot3(ac, cpv);
    if (d6 >= 0.0 && d5 <= d6) { v = 0.0; w = 1.0; goto done; }              /* vertex c */
    double vb = d5 * d2 - d1 * d6;
    if (vb <= 0.0 && d2 >= 0.0 && d6 <= 0.0) { v = 0.0; w = d2 / (d2 - d6); goto done; }   /* edge ac */
    double va = d3 * d6 - d5 * d4;
    if (va <= 0.0 && (d4 - d3) >= 0.0 && (d5 - d6) >= 0.0) {                               /* edge bc */
        w = (d4 - d3) / ((d4 - d3) + (d5 - d6)); v = 1.0 - w; goto done;
    }
    {                                                                                      /* face */
        double denom = 1.0 / (va + vb + vc);
        v = vb * denom; w = vc * denom;
    }
done:
    bary[0] = 1.0 - v - w; bary[1] = v; bary[2] = w;
    for (int k = 0; k < 3; ++k) cp[k] = a[k] + v * ab[k] + w * ac[k];
    double d[3]; sub3(p, cp, d);
    return dot3(d, d);
}

/*
 * Second, independent formulation used only to pin the first one
 * (tests/test_oracle_geometry.py): project p on the plane; if the projection
 * is inside the triangle that is the answer, otherwise the nearest point of
 * the three edges.
 */
double orc_closest_point_triangle_alt(const double p[3], const double a[3], const double b[3],
                                      const double c[3], double cp[3])
{
    double ab[3], ac[3], ap[3], n[3], bary[3];
    sub3(b, a, ab); sub3(c, a, ac); sub3(p, a, ap);
    cross3(ab, ac, n);
    double nn = dot3(n, n);
    if (nn > 0.0) {
        double h = dot3(ap, n) / nn;
        double q[3] = { p[0] - h * n[0], p[1] - h * n[1], p[2] - h * n[2] };
        /* inside test by signed sub-areas */
        double qa[3], qb[3], qc[3], c0[3], c1[3], c2[3];
        sub3(a, q, qa); sub3(b, q, qb); sub3(c, q, qc);
        cross3(qb, qc, c0); cross3(qc, qa, c1); cross3(qa, qb, c2);
        if (dot3(c0, n) >= 0.0 && dot3(c1, n) >= 0.0 && dot3(c2, n) >= 0.0) {
            memcpy(cp, q, sizeof q);
            double d[3]; sub3(p, q, d);
            return dot3(d, d);
        }
    }
    return closest_on_edges(p, a, b, c, cp, bary);
}

/* ------------------------------------------------------------------------- */
/* Geometry: a triangle soup (brute force over all faces) or, for the         */
/* closed-form pins only, an analytic sphere.                                 */
/* ------------------------------------------------------------------------- */
typedef struct {
    int32_t kind;               /* 0 = triangle mesh, 1 = analytic sphere (pins) */
    int32_t pad_;
    const float *verts;         /* [V][3] fp32, as given to the CUDA path        */
    int64_t V;
    const int32_t *faces;       /* [F][3]                                         */
    int64_t F;
    double centre[3];           /* kind 1                                         */
    double radius;
} orc_geom;

typedef struct {
    double dist;                /* unsigned distance to the surface */
    double cp[3];               /* closest point                    */
    double bary[3];             /* barycentrics of cp in face `tri` */
    int64_t tri;                /* closest face, -1 for the sphere  */
} orc_hit;

static void load_vertex(const orc_geom *g, int64_t vi, double o[3])
{
    o[0] = (double)g->verts[3*vi]; o[1] = (double)g->verts[3*vi+1]; o[2] = (double)g->verts[3*vi+2];
}

/* Brute force over ALL faces: the definition of the query.  Ties: the smaller
 * squared distance wins, on equality the smaller face index [R15] (strict <
 * while scanning in increasing index order). */
void orc_closest_point(const orc_geom *g, const double x[3], orc_hit *h)
{
    if (g->kind == 1) {
        double d[3]; sub3(x, g->centre, d);
        double rho = norm3(d);
        h->dist = fabs(g->radius - rho);
        if (rho > 0.0) for (int k = 0; k < 3; ++k) h->cp[k] = g->centre[k] + g->radius * d[k] / rho;
        else { h->cp[0] = g->centre[0] + g->radius; h->cp[1] = g->centre[1]; h->cp[2] = g->centre[2]; }
        h->bary[0] = 1.0; h->bary[1] = 0.0; h->bary[2] = 0.0;
        h->tri = -1;
        return;
    }
    double best = INFINITY;
    h->tri = -1;
    for (int64_t f = 0; f < g->F; ++f) {
        double a[3], b[3], c[3], cp[3], bary[3];
        load_vertex(g, g->faces[3*f], a); load_vertex(g, g->faces[3*f+1], b); load_vertex(g, g->faces[3*f+2], c);
        double d2 = orc_closest_point_triangle(x, a, b, c, cp, bary);
        if (d2 < best) {
            best = d2; h->tri = f;
            memcpy(h->cp, cp, sizeof cp); memcpy(h->bary, bary, sizeof bary);
        }
    }
    h->dist = sqrt(best);
}

/* ------------------------------------------------------------------------- */
/* Exact distance to the Kelvin image of a flat triangle  [DESIGN.md reading E4]. */
/*                                                                            */
/* The paper runs its exterior walks on "inverted triangle meshes with        */
/* spherical-triangular elements and ... (non-planar) distance queries"       */
/* (its stated exterior bottleneck): the     */
/* Kelvin image of a flat face is a patch of the sphere through 0 that is the */
/* image of the face's plane.  The distance from a point y of the inverted    */
/* domain to that patch needs no spherical geometry: with x = kappa(y) and    */
/* the distance identity of the inversion,                                    */
/*     |kappa(x) - kappa(p)| = |x - p| / (|x| |p|),                            */
/* it is  (1/|x|) min over p in T of |x - p| / |p|  (all coordinates about    */
/* the inversion centre).  The level sets of |x - p| / |p| = k are the        */
/* spheres of Apollonius, centre x / (1 - k^2), radius k |x| / |1 - k^2|, so  */
/* the minimum over the triangle is attained                                  */
/*   - where such a sphere touches the face's plane n.p = h:                  */
/*       (n.x - h (1 - u))^2 = u |x|^2,  u = k^2  (the smaller root), at the  */
/*       foot of the sphere's centre on the plane, if that foot lies in T, or */
/*   - on an edge a + t e: the ratio of two quadratics with the same leading  */
/*       coefficient, N(t)/D(t); N'D - ND' = 0 is a quadratic in t, or        */
/*   - at a vertex.                                                            */
/* Returns min |x - p|^2 / |p|^2 and the barycentrics of the minimiser.       */
/* ------------------------------------------------------------------------- */
static double ratio2_at(const double x[3], const double p[3])
{
    double d[3]; sub3(x, p, d);
    double pp = dot3(p, p);
    return pp > 0.0 ? dot3(d, d) / pp : INFINITY;
}

double orc_inverted_ratio2_triangle(const double x[3], const double a[3], const double b[3], const double c[3],
                                    double bary[3])
{
    const double *vtx[3] = { a, b, c };
    double best = INFINITY;
    bary[0] = 1.0; bary[1] = bary[2] = 0.0;
    /* vertices and edges */
    for (int k = 0; k < 3; ++k) {
        const double *P = vtx[k], *Q = vtx[(k + 1) % 3];
        double e[3], xp[3]; sub3(Q, P, e); sub3(x, P, xp);
        const double n0 = dot3(xp, xp), n1 = -2.0 * dot3(xp, e), n2 = dot3(e, e);
        const double d0 = dot3(P, P), d1 = 2.0 * dot3(P, e);
        double cand[4] = { 0.0, 1.0, -1.0, -1.0 };
        const double qa = n2 * (d1 - n1), qb = 2.0 * n2 * (d0 - n0), qc = n1 * d0 - n0 * d1;
        if (fabs(qa) > 1e-300) {
            const double disc = qb * qb - 4.0 * qa * qc;
            if (disc >= 0.0) {
                const double sq = sqrt(disc);
                /* numerically stable pair of roots */
                const double q = -0.5 * (qb + (qb >= 0.0 ? sq : -sq));
                cand[2] = q / qa;
                if (fabs(q) > 0.0) cand[3] = qc / q;
            }
        } else if (fabs(qb) > 1e-300) {
            cand[2] = -qc / qb;
        }
        for (int j = 0; j < 4; ++j) {
            const double t = cand[j];
            if (!(t >= 0.0 && t <= 1.0)) continue;
            const double N = n0 + t * (n1 + t * n2), D = d0 + t * (d1 + t * n2);
            const double f = D > 0.0 ? N / D : INFINITY;
            if (f < best) {
                best = f;
                bary[0] = bary[1] = bary[2] = 0.0;
                bary[k] = 1.0 - t; bary[(k + 1) % 3] = t;
            }
        }
    }
    /* interior: the Apollonius sphere that touches the plane */
    double ab[3], ac[3], n[3];
    sub3(b, a, ab); sub3(c, a, ac); cross3(ab, ac, n);
    const double nn = dot3(n, n);
    const double e2 = fmax(dot3(ab, ab), dot3(ac, ac));
    if (nn > 1e-24 * e2 * e2) {
        const double inv = 1.0 / sqrt(nn);
        const double nh[3] = { n[0] * inv, n[1] * inv, n[2] * inv };
        const double h = dot3(nh, a), hx = dot3(nh, x), xx = dot3(x, x);
        double u = -1.0;
        const double A2 = h * h, B2 = 2.0 * h * (hx - h) - xx, C2 = (hx - h) * (hx - h);
        if (A2 > 1e-30 * xx) {
            const double disc = B2 * B2 - 4.0 * A2 * C2;
            if (disc >= 0.0) {
                /* smaller root, written without cancellation: B2 < 0 whenever the roots are positive */
                const double q = -0.5 * (B2 - sqrt(disc));
                u = q > 0.0 ? C2 / q : -1.0;
            }
        } else if (xx > 0.0) {
            u = C2 / xx;                                 /* plane through the inversion centre */
        }
        if (u >= 0.0 && fabs(1.0 - u) > 1e-12) {
            double cc[3] = { x[0] / (1.0 - u), x[1] / (1.0 - u), x[2] / (1.0 - u) };
            const double off = dot3(nh, cc) - h;
            double p0[3] = { cc[0] - off * nh[0], cc[1] - off * nh[1], cc[2] - off * nh[2] };
            /* barycentrics of p0 */
            double ap[3]; sub3(p0, a, ap);
            const double d00 = dot3(ab, ab), d01 = dot3(ab, ac), d11 = dot3(ac, ac), d20 = dot3(ap, ab), d21 = dot3(ap, ac);
            const double den = d00 * d11 - d01 * d01;
            const double v = (d11 * d20 - d01 * d21) / den, w = (d00 * d21 - d01 * d20) / den;
            if (v >= 0.0 && w >= 0.0 && v + w <= 1.0) {
                const double f = ratio2_at(x, p0);
                if (f < best) { best = f; bary[0] = 1.0 - v - w; bary[1] = v; bary[2] = w; }
            }
        }
    }
    return best;
}

/* Brute force over all faces: h->dist receives the RATIO min_p |x - p| / |p - o| (dimensionless; the distance in
 * Kelvin coordinates is ratio / |x - o|), h->cp the minimiser on the primal mesh.  Ties: smaller ratio, then smaller
 * face index, as in orc_closest_point. */
void orc_closest_point_inverted(const orc_geom *g, const double x[3], const double origin[3], orc_hit *h)
{
    double xr[3]; sub3(x, origin, xr);
    double best = INFINITY;
    h->tri = -1;
    for (int64_t f = 0; f < g->F; ++f) {
        double a[3], b[3], c[3], bary[3];
        load_vertex(g, g->faces[3*f], a); load_vertex(g, g->faces[3*f+1], b); load_vertex(g, g->faces[3*f+2], c);
        double ar[3], br[3], cr[3];
        sub3(a, origin, ar); sub3(b, origin, br); sub3(c, origin, cr);
        double r2 = orc_inverted_ratio2_triangle(xr, ar, br, cr, bary);
        if (r2 < best) {
            best = r2; h->tri = f;
            memcpy(h->bary, bary, sizeof bary);
            for (int k = 0; k < 3; ++k) h->cp[k] = bary[0] * a[k] + bary[1] * b[k] + bary[2] * c[k];
        }
    }
    h->dist = sqrt(best);
}

/* Batch form for the parity tests: queries in fp32 (same numbers the GPU gets).
 * second[q] = smallest distance over faces that share no vertex with the winner
 * (for the tie filter of SURVEY.md 8(c)); may be NULL. */
void orc_closest_points(const orc_geom *g, const float *q, int64_t Q,
                        double *dist, int64_t *tri, double *cp, double *bary, double *second)
{
    #pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < Q; ++i) {
        double x[3] = { q[3*i], q[3*i+1], q[3*i+2] };
        orc_hit h;
        orc_closest_point(g, x, &h);
        dist[i] = h.dist; tri[i] = h.tri;
        if (cp)   memcpy(cp + 3*i, h.cp, sizeof h.cp);
        if (bary) memcpy(bary + 3*i, h.bary, sizeof h.bary);
        if (second && g->kind == 0) {
            const int32_t *wf = g->faces + 3*h.tri;
            double best = INFINITY;
            for (int64_t f = 0; f < g->F; ++f) {
                const int32_t *ff = g->faces + 3*f;
                int share = 0;
                for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b) share |= (ff[a] == wf[b]);
                if (share) continue;
                double a3[3], b3[3], c3[3], p3[3], bb[3];
                load_vertex(g, ff[0], a3); load_vertex(g, ff[1], b3); load_vertex(g, ff[2], c3);
                double d2 = orc_closest_point_triangle(x, a3, b3, c3, p3, bb);
                if (d2 < best) best = d2;
            }
            second[i] = sqrt(best);
        }
    }
}

/* Tie filter helper for the parity tests (no method arithmetic of its own):
 * runner_up[q] = smallest distance over all faces other than the winner tri[q]
 * that are not copies of it (same three vertex indices in any order). */
void orc_runner_up(const orc_geom *g, const float *q, int64_t Q, const int64_t *tri, double *runner_up)
{
    #pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < Q; ++i) {
        double x[3] = { q[3*i], q[3*i+1], q[3*i+2] };
        const int32_t *wf = g->faces + 3*tri[i];
        double best = INFINITY;
        for (int64_t f = 0; f < g->F; ++f) {
            const int32_t *ff = g->faces + 3*f;
            if (f == tri[i]) continue;
            int same = 0;
            for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b) same += (ff[a] == wf[b]);
            if (same >= 3) continue;
            double a3[3], b3[3], c3[3], p3[3], bb[3];
            load_vertex(g, ff[0], a3); load_vertex(g, ff[1], b3); load_vertex(g, ff[2], c3);
            double d2 = orc_closest_point_triangle(x, a3, b3, c3, p3, bb);
            if (d2 < best) best = d2;
        }
        runner_up[i] = sqrt(best);
    }
}

/* ------------------------------------------------------------------------- */
/* Mesh quantities: face normal, area, AABB, r_max.            */
/* ------------------------------------------------------------------------- */
static void face_normal_area(const orc_geom *g, int64_t f, double n[3], double *area)
{
    double a[3], b[3], c[3], ab[3], ac[3];
    load_vertex(g, g->faces[3*f], a); load_vertex(g, g->faces[3*f+1], b); load_vertex(g, g->faces[3*f+2], c);
    sub3(b, a, ab); sub3(c, a, ac);
    cross3(ab, ac, n);
    double l = norm3(n);
    *area = 0.5 * l;
    if (l > 0.0) { n[0] /= l; n[1] /= l; n[2] /= l; }
}

/* Diagonal of the AABB of the vertices referenced by faces (escape test [R10b]). */
double orc_aabb_diagonal(const orc_geom *g)
{
    if (g->kind != 0 || g->F < 1) return 0.0;
    double lo[3] = { INFINITY, INFINITY, INFINITY }, hi[3] = { -INFINITY, -INFINITY, -INFINITY };
    for (int64_t f = 0; f < g->F; ++f)
        for (int c = 0; c < 3; ++c) {
            double p[3]; load_vertex(g, g->faces[3*f + c], p);
            for (int k = 0; k < 3; ++k) { if (p[k] < lo[k]) lo[k] = p[k]; if (p[k] > hi[k]) hi[k] = p[k]; }
        }
    double d[3] = { hi[0] - lo[0], hi[1] - lo[1], hi[2] - lo[2] };
    return norm3(d);
}

/* r_max = half of the shortest AABB side ("maximum diameter ... shortest side
 * length of the mesh's axis-aligned bounding box").  For the
 * exterior the box is that of the Kelvin-inverted vertices kappa(v - origin). */
double orc_rmax(const orc_geom *g, int exterior, const double origin[3])
{
    double lo[3] = { INFINITY, INFINITY, INFINITY }, hi[3] = { -INFINITY, -INFINITY, -INFINITY };
    for (int64_t i = 0; i < g->V; ++i) {
        double v[3]; load_vertex(g, i, v);
        if (exterior) {
            double w[3]; sub3(v, origin, w);
            double s = dot3(w, w);
            for (int k = 0; k < 3; ++k) v[k] = w[k] / s;          /* kappa(x) = x/|x|^2 */
        }
        for (int k = 0; k < 3; ++k) { lo[k] = fmin(lo[k], v[k]); hi[k] = fmax(hi[k], v[k]); }
    }
    double side = fmin(hi[0] - lo[0], fmin(hi[1] - lo[1], hi[2] - lo[2]));
    return (double)(float)(0.5 * side);       /* rounded to fp32: the value both sides bisect on [R4] */
}

/* R_max = largest vertex distance from the Kelvin origin (used by E3). */
double orc_max_vertex_norm(const orc_geom *g, const double origin[3])
{
    double m = 0.0;
    for (int64_t i = 0; i < g->V; ++i) {
        double v[3], w[3]; load_vertex(g, i, v); sub3(v, origin, w);
        m = fmax(m, norm3(w));
    }
    return (double)(float)m;
}

double orc_total_area(const orc_geom *g)
{
    double tot = 0.0, n[3], a;
    for (int64_t f = 0; f < g->F; ++f) { face_normal_area(g, f, n, &a); tot += a; }
    return tot;
}

/* Consistent P1 mass matrix M_pq = sum_T area_T (1 + delta_pq) / 12  [R14]. */
void orc_mass_matrix_p1(const orc_geom *g, double *M /* [V][V], zeroed by caller */)
{
    for (int64_t f = 0; f < g->F; ++f) {
        double n[3], a; face_normal_area(g, f, n, &a);
        for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j)
            M[(int64_t)g->faces[3*f+i] * g->V + g->faces[3*f+j]] += a * (i == j ? 2.0 : 1.0) / 12.0;
    }
}

/* ------------------------------------------------------------------------- */
/* Parameters and per-sample state                                            */
/* ------------------------------------------------------------------------- */
typedef struct {
    uint64_t seed;
    int32_t walks_per_sample;       /* W                                               */
    int32_t max_steps;              /* [R10] truncated walks contribute nothing         */
    double eps;                     /* WoS shell, absolute [R8]     */
    double cap_half_angle_deg;      /* theta_0 ("~2.5 deg") [R5]           */
    double rmax;                    /* from orc_rmax() times the caller's scale         */
    int32_t bisection_iters;        /* 10                                */
    int32_t importance_sample;      /* 1: z ~ J^B; 0: z uniform          */
    int32_t antithetic;             /* [R7]                                             */
    int32_t include_killing;        /* exterior: second expectation of Eq. 32           */
    int64_t n_kill_walks;
    double origin[3];               /* Kelvin origin [R12]               */
    double Rmax_norm;               /* orc_max_vertex_norm(), exterior only             */
    double escape_radius;           /* [R10b] interior: AABB diagonal; 0 = no escape test */
    int32_t estimator;              /* 0: Alg. 2 (tangent-ball jump kernel); 1: Alg. 1 (naive finite difference), interior only */
    int32_t pad_;
    double inset;                   /* Alg. 1: inset distance of the evaluation point x = s - inset n_s */
    int32_t exterior_query;         /* 0: flat-triangle query + conservative radius [E3]; 1: exact distance to the inverted faces [E4] */
    int32_t pad2_;
} orc_params;

typedef struct {                    /* one boundary sample            */
    double s[3];                    /* surface point                                    */
    double n[3];                    /* unit normal pointing out of the solid            */
    double a;                       /* quadrature weight, sum = |dOmega|                */
    int64_t tri;                    /* its face (-1 for the analytic sphere)            */
    double bary[3];
} orc_sample;

typedef struct {                    /* tangent ball in the walk domain                  */
    double c[3];                    /* centre (interior: primal; exterior: Kelvin coords about origin) */
    double pole[3];                 /* unit vector from c to the tangent point          */
    double r;                       /* 0 => sample discarded             */
    double sstar_norm;              /* |s*| (exterior), 1 otherwise                     */
} orc_ball;

/* ------------------------------------------------------------------------- */
/* LargestTangentBall ("bisection algorithm of Yu et al. with   */
/* 10 iterations"; clamp PAPER.md:642)  [R4].                   */
/* The ball of radius r about c = s - r n is accepted when no surface point is */
/* closer to c than r - eps/2.                                                */
/* ------------------------------------------------------------------------- */
void orc_tangent_ball_interior(const orc_geom *g, const orc_params *P, const orc_sample *S, orc_ball *B)
{
    double lo = 0.0, hi = P->rmax;
    for (int it = 0; it < P->bisection_iters; ++it) {
        double r = 0.5 * (lo + hi);
        double c[3] = { S->s[0] - r * S->n[0], S->s[1] - r * S->n[1], S->s[2] - r * S->n[2] };
        orc_hit h;
        orc_closest_point(g, c, &h);
        if (h.dist >= r - 0.5 * P->eps) lo = r; else hi = r;
    }
    B->r = lo;
    for (int k = 0; k < 3; ++k) { B->c[k] = S->s[k] - lo * S->n[k]; B->pole[k] = S->n[k]; }
    B->sstar_norm = 1.0;
}

/*
 * Exterior: the tangent ball lives in the inverted domain Omega*_ext
 * (PAPER.md:348-353).  s* = kappa(s - o); the unit normal at s* pointing out of
 * Omega*_ext is n* = -H_shat n (Eq. 54).  The ball B_r(c*),
 * c* = s* - r n*, is tested through the primal image of its eps/2-shrunken copy, which is again a ball as
 * long as 0 is outside it: a Kelvin ball (c*, rho) maps to centre c* / (|c*|^2 - rho^2), radius rho / (|c*|^2 - rho^2)
 * [DESIGN.md readings E2, R4].  r is limited so that 0 stays outside
 * (r < |s*|^2 / (2 s*.n*)) and by r_max of the inverted box.
 */
void orc_tangent_ball_exterior(const orc_geom *g, const orc_params *P, const orc_sample *S, orc_ball *B)
{
    double st[3]; sub3(S->s, P->origin, st);
    double sig = dot3(st, st);
    B->r = 0.0; B->sstar_norm = 0.0;
    memset(B->c, 0, sizeof B->c); memset(B->pole, 0, sizeof B->pole);
    if (!(sig > 0.0)) return;
    double sstar[3] = { st[0] / sig, st[1] / sig, st[2] / sig };
    double sn = dot3(st, S->n) / sig;                       /* shat (shat . n) = st * sn */
    double nstar[3];
    for (int k = 0; k < 3; ++k) nstar[k] = -(S->n[k] - 2.0 * st[k] * sn);   /* -(n - 2 shat (shat.n)), Eq. 54 */
    double ss2 = dot3(sstar, sstar);
    double sdn = dot3(sstar, nstar);
    double hi = P->rmax;
    if (sdn > 0.0) hi = fmin(hi, 0.45 * ss2 / sdn);
    double lo = 0.0;
    for (int it = 0; it < P->bisection_iters; ++it) {
        double r = 0.5 * (lo + hi);
        double cs[3] = { sstar[0] - r * nstar[0], sstar[1] - r * nstar[1], sstar[2] - r * nstar[2] };
        /* [R4] the probe ball is B(c*, r - eps/2) IN KELVIN COORDINATES (the walk domain: a point of the tangent ball
         * that pokes out by < eps/2 is inside the shell); it is tested through ITS OWN primal image.  (Shrinking the
         * primal image of B(c*, r) by the relative amount eps / 2r instead moves its near side by eps / (2 (|c*|^2 - r^2))
         * in primal units, many eps when that image is large.) */
        double rk = r - 0.5 * P->eps;
        if (!(rk > 0.0)) { lo = r; continue; }
        double den = dot3(cs, cs) - rk * rk;
        double cprime[3] = { P->origin[0] + cs[0] / den, P->origin[1] + cs[1] / den, P->origin[2] + cs[2] / den };
        double rprime = rk / den;
        orc_hit h;
        orc_closest_point(g, cprime, &h);
        if (h.dist >= rprime) lo = r; else hi = r;
    }
    B->r = lo;
    for (int k = 0; k < 3; ++k) { B->c[k] = sstar[k] - lo * nstar[k]; B->pole[k] = nstar[k]; }
    B->sstar_norm = sqrt(ss2);
}

/* Orthonormal frame (e1, e2, n) from a unit vector n: the branchless
 * construction of Duff et al., "Building an Orthonormal Basis, Revisited"
 * (JCGT 2017), restated.  Both sides use the same rule so that a walk's start
 * point is the same point  [DESIGN.md reading R6b]. */
static void frame_from_normal(const double n[3], double e1[3], double e2[3])
{
    double sign = copysign(1.0, n[2]);
    double a = -1.0 / (sign + n[2]);
    double b = n[0] * n[1] * a;
    e1[0] = 1.0 + sign * n[0] * n[0] * a; e1[1] = sign * b; e1[2] = -sign * n[0];
    e2[0] = b; e2[1] = sign + n[1] * n[1] * a; e2[2] = -n[1];
}

/*
 * SampleBallSurface + BallJumpKernel (Eq. 23).
 * Polar angle theta from the pole (the tangent point), q = sin(theta/2), so
 * |s - z| = 2 r q.  The cap theta < theta_0 is excluded [R5].
 *   importance: density on the sphere proportional to J^B = 1/(2 pi |s-z|^3)
 *     => pdf(q) ~ q^-2 on [q0, 1], q = 1 / (1/q0 - u1 (1/q0 - 1)); the
 *     per-walk factor  (|dB|/2) J / pdf  is the constant (1/(4r)) (1/q0 - 1) [R6]
 *   uniform: cos(theta) = 1 - 2 u1; factor (4 pi r^2 / 2) J = 1 / (8 r q^3),
 *     zero inside the cap.
 * Returns the factor; z is written in the coordinates of the ball.
 */
static double sample_ball_surface(const orc_params *P, const orc_ball *B, uint32_t sample, uint32_t walk, double z[3])
{
    double q0 = sin(0.5 * P->cap_half_angle_deg * ORC_PI / 180.0);
    uint32_t wq = P->antithetic ? (walk >> 1) : walk;
    double u1, u2;
    orc_uniform2(P->seed, sample, wq, 0u, ORC_PURPOSE_INIT, &u1, &u2);
    double q, factor;
    if (P->importance_sample) {
        q = 1.0 / (1.0 / q0 - u1 * (1.0 / q0 - 1.0));
        factor = (1.0 / (4.0 * B->r)) * (1.0 / q0 - 1.0);
    } else {
        q = sqrt(u1);
        factor = (q < q0) ? 0.0 : 1.0 / (8.0 * B->r * q * q * q);
    }
    double ct = 1.0 - 2.0 * q * q;
    double st = 2.0 * q * sqrt(fmax(0.0, 1.0 - q * q));
    double phi = 2.0 * ORC_PI * u2;
    if (P->antithetic && (walk & 1u)) phi += ORC_PI;          /* antithetic partner [R7] */
    double e1[3], e2[3];
    frame_from_normal(B->pole, e1, e2);
    double cphi = cos(phi), sphi = sin(phi);
    for (int k = 0; k < 3; ++k)
        z[k] = B->c[k] + B->r * (ct * B->pole[k] + st * (cphi * e1[k] + sphi * e2[k]));
    return factor;
}

/* Uniform direction on S^2 from two uniforms [R19]. */
static void step_direction(uint64_t seed, uint32_t sample, uint32_t walk, uint32_t step, double w[3])
{
    double u1, u2;
    orc_uniform2(seed, sample, walk, step, ORC_PURPOSE_STEP, &u1, &u2);
    double ct = 1.0 - 2.0 * u1;
    double st = sqrt(fmax(0.0, 1.0 - ct * ct));
    double phi = 2.0 * ORC_PI * u2;
    w[0] = st * cos(phi); w[1] = st * sin(phi); w[2] = ct;
}

/*
 * WalkOnSpheres in the primal domain  [R9]:
 * repeat { closest point; stop if D < eps; jump to a uniform point of the
 * sphere of radius D }.  Returns the number of jumps, or -1 if max_steps
 * jumps did not reach the shell [R10], or -3 if the walker left the bounding box
 * of the surface [R10b]: every point of the AABB is within its diagonal of every
 * surface point, so D > diagonal proves the walker is outside the box, hence
 * outside the solid -- an "unbounded" walk of an open or mis-oriented surface
 * (PAPER.md:548, 638-640).  Such a walk contributes nothing, like a truncated one.
 */
static int walk_on_spheres(const orc_geom *g, const orc_params *P, uint32_t sample, uint32_t walk,
                           const double z[3], orc_hit *h)
{
    double x[3] = { z[0], z[1], z[2] };
    for (int k = 0; ; ++k) {
        orc_closest_point(g, x, h);
        if (h->dist < P->eps) return k;
        if (P->escape_radius > 0.0 && h->dist > P->escape_radius) return -3;
        if (k == P->max_steps) return -1;
        double w[3];
        step_direction(P->seed, sample, walk, (uint32_t)(k + 1), w);
        for (int j = 0; j < 3; ++j) x[j] += h->dist * w[j];
    }
}

/*
 * WalkOnSpheres in the inverted domain Omega*_ext, carried in Kelvin
 * coordinates y about the origin  [DESIGN.md reading E3].
 * A ball about y inside Omega*_ext is found from flat-triangle queries on the
 * PRIMAL mesh:  x = kappa(y), rho = |x|, D = dist(x), and every point p of the
 * surface satisfies |kappa(x) - kappa(p)| = |x - p| / (|x||p|) with |x-p| >= D,
 * |p| <= min(R_max, rho + |x-p|), so
 *     R* = D / (rho * min(R_max, rho + D))
 * is a valid radius.  Far field (|y| R_max <= 1/2): the ball about 0 of radius
 * 1/R_max is the image of the outside of the bounding sphere, so
 * R* = 1/R_max - |y| needs no query.  Stop when R* < eps; the exit point is
 * the primal closest point.  Returns the number of jumps, -1 (truncated, [R10]) or
 * -3 (the walker is inside the solid that holds the inversion centre, [R10c]).
 */
static int walk_on_spheres_kelvin(const orc_geom *g, const orc_params *P, uint32_t sample, uint32_t walk,
                                  const double z[3], orc_hit *h)
{
    double y[3] = { z[0], z[1], z[2] };
    for (int k = 0; ; ++k) {
        double yn = norm3(y), Rstar;
        if (yn * P->Rmax_norm <= 0.5) {
            Rstar = 1.0 / P->Rmax_norm - yn;
        } else {
            double x[3] = { P->origin[0] + y[0] / (yn * yn), P->origin[1] + y[1] / (yn * yn), P->origin[2] + y[2] / (yn * yn) };
            double rho = 1.0 / yn;
            if (P->exterior_query == 1 && g->kind == 0) {
                /* [E4] the paper's own query: exact distance from y to the Kelvin-inverted faces = ratio / |x| */
                orc_closest_point_inverted(g, x, P->origin, h);
                Rstar = h->dist / rho;
                double dd[3]; sub3(x, h->cp, dd);
                h->dist = norm3(dd);                 /* primal distance to the exit point, for the [R10c] test below */
            } else {
                orc_closest_point(g, x, h);
                Rstar = h->dist / (rho * fmin(P->Rmax_norm, rho + h->dist));
            }
            if (Rstar < P->eps) return k;
            /* [R10c] The empty ball about x holds the inversion centre (D > |x - o| = rho): x lies in the same
             * component of space as the centre, i.e. INSIDE the solid.  On a closed, consistently oriented
             * surface this cannot happen (the segment from x to the centre crosses the surface, so D <= rho);
             * on an open or mis-oriented one it is the exterior twin of [R10b]: in
             * Kelvin coordinates such a walker runs off to infinity, doubling |y| every jump.  It contributes
             * nothing, like a truncated walk. */
            if (h->dist > rho) return -3;
        }
        if (k == P->max_steps) return -1;
        double w[3];
        step_direction(P->seed, sample, walk, (uint32_t)(k + 1), w);
        for (int j = 0; j < 3; ++j) y[j] += Rstar * w[j];
    }
}

/* ------------------------------------------------------------------------- */
/* Per-walk record: what one Monte Carlo sample contributes (Alg. 2 lines     */
/* 273-285; Eq. 32).                                                          */
/* ------------------------------------------------------------------------- */
typedef struct {
    int64_t sample;             /* boundary sample index, -1 for a killing walk             */
    int64_t tri_t;              /* exit face (-1: analytic sphere)                          */
    double bary_t[3];
    double t[3];                /* exit point on the primal surface                         */
    double z[3];                /* start point of the walk (walk-domain coordinates)        */
    double weight;              /* full scalar multiplying d d^T (0 if truncated/discarded) */
    int32_t steps;              /* jumps taken; -1 truncated; -2 sample discarded           */
    int32_t pad_;
} orc_record;

static void fill_sample(const orc_geom *g, const int32_t *tri, const float *bary, const float *weight,
                        const float *normal, const double *pos, int64_t i, orc_sample *S)
{
    S->a = weight[i];
    if (g->kind == 0) {
        int64_t f = tri[i];
        double a[3], b[3], c[3], area;
        load_vertex(g, g->faces[3*f], a); load_vertex(g, g->faces[3*f+1], b); load_vertex(g, g->faces[3*f+2], c);
        for (int k = 0; k < 3; ++k) S->bary[k] = bary[3*i+k];
        for (int k = 0; k < 3; ++k) S->s[k] = S->bary[0] * a[k] + S->bary[1] * b[k] + S->bary[2] * c[k];
        face_normal_area(g, f, S->n, &area);
        S->tri = f;
    } else {                       /* analytic sphere: position given, normal radial */
        for (int k = 0; k < 3; ++k) S->s[k] = pos[3*i+k];
        double d[3]; sub3(S->s, g->centre, d);
        double l = norm3(d);
        for (int k = 0; k < 3; ++k) S->n[k] = d[k] / l;
        S->tri = -1; S->bary[0] = 1.0; S->bary[1] = S->bary[2] = 0.0;
    }
    if (normal) for (int k = 0; k < 3; ++k) S->n[k] = normal[3*i+k];
}

/* One walk (sample i, walk w) of Alg. 2 lines 273-285 / Eq. 32 from the tangent ball B of
 * sample S: start point, walk-on-spheres, exit record, weight. */
static void run_one_walk(const orc_geom *g, const orc_params *P, int exterior, const orc_sample *S,
                         const orc_ball *Bp, int64_t i, int w, orc_record *R)
{
    const int W = P->walks_per_sample;
    const orc_ball B = *Bp;
    memset(R, 0, sizeof *R);
    R->sample = i; R->tri_t = -1;
    double factor;
    if (P->estimator == 1 && !exterior) {
        /* Alg. 1 (Eq. 13-16; [G2]): the walk starts at the inset point x = s - eps n_s
         * and the update is (|dOmega| / (N eps)) b_s (b_s - b_t)^T: no tangent ball, no sampling weight. */
        for (int k = 0; k < 3; ++k) R->z[k] = S->s[k] - P->inset * S->n[k];
        factor = 1.0 / P->inset;
    } else {
        if (!(B.r > 0.0)) { R->steps = -2; return; }       /* discarded sample */
        factor = sample_ball_surface(P, &B, (uint32_t)i, (uint32_t)w, R->z);
    }
    orc_hit h;
    int steps = exterior ? walk_on_spheres_kelvin(g, P, (uint32_t)i, (uint32_t)w, R->z, &h)
                         : walk_on_spheres(g, P, (uint32_t)i, (uint32_t)w, R->z, &h);
    R->steps = steps;
    if (steps < 0) return;                                   /* truncated: contributes nothing */
    R->tri_t = h.tri;
    memcpy(R->bary_t, h.bary, sizeof h.bary);
    memcpy(R->t, h.cp, sizeof h.cp);
    double wgt = (S->a / W) * factor;                        /* |dOmega| |dB| J / (2N), Alg. 2 */
    if (exterior) {
        double tt[3]; sub3(h.cp, P->origin, tt);
        /* |s*|^3 / |t*|, Eq. 32;  1/|t*| = |t - o| */
        wgt *= B.sstar_norm * B.sstar_norm * B.sstar_norm * norm3(tt);
    }
    R->weight = wgt;
}

/*
 * Run every walk of every sample and write one record per walk at slot
 * sample*W + walk (then the killing walks).  exterior = 0: Alg. 2; 1: Eq. 32.
 * balls_out (optional) receives r, c, |s*| per sample for the A2 parity test.
 * Returns the number of records.
 */
int64_t orc_run_walks(const orc_geom *g, const orc_params *P, int exterior,
                      const int32_t *tri, const float *bary, const float *weight,
                      const float *normal, const double *pos, int64_t n_s,
                      orc_record *rec, double *balls_out /* [n_s][5] or NULL */)
{
    const int W = P->walks_per_sample;
    #pragma omp parallel for schedule(dynamic, 1)
    for (int64_t i = 0; i < n_s; ++i) {
        orc_sample S;
        orc_ball B;
        fill_sample(g, tri, bary, weight, normal, pos, i, &S);
        if (P->estimator == 1 && !exterior) { memset(&B, 0, sizeof B); B.sstar_norm = 1.0; }   /* Alg. 1 has no ball */
        else if (exterior) orc_tangent_ball_exterior(g, P, &S, &B);
        else               orc_tangent_ball_interior(g, P, &S, &B);
        if (balls_out) { balls_out[5*i] = B.r; balls_out[5*i+1] = B.c[0]; balls_out[5*i+2] = B.c[1]; balls_out[5*i+3] = B.c[2]; balls_out[5*i+4] = B.sstar_norm; }
        for (int w = 0; w < W; ++w)
            run_one_walk(g, P, exterior, &S, &B, i, w, rec + i * W + w);
    }
    int64_t n_rec = n_s * W;
    if (exterior && P->include_killing) {
        /* second expectation of Eq. 32: walks from 0 = kappa(infinity), Eq. 74 */
        #pragma omp parallel for schedule(dynamic, 16)
        for (int64_t j = 0; j < P->n_kill_walks; ++j) {
            orc_record *R = rec + n_rec + j;
            memset(R, 0, sizeof *R);
            R->sample = -1; R->tri_t = -1;
            orc_hit h;
            int steps = walk_on_spheres_kelvin(g, P, ORC_KILLING_SAMPLE, (uint32_t)j, R->z, &h);
            R->steps = steps;
            if (steps < 0) continue;
            R->tri_t = h.tri;
            memcpy(R->bary_t, h.bary, sizeof h.bary);
            memcpy(R->t, h.cp, sizeof h.cp);
            double tt[3]; sub3(h.cp, P->origin, tt);
            R->weight = 4.0 * ORC_PI * norm3(tt) / (double)P->n_kill_walks;    /* 4 pi / |t0*| */
        }
        n_rec += P->n_kill_walks;
    }
    return n_rec;
}

/*
 * Sampled outputs of the same run (parity at sizes the full oracle cannot finish): the
 * records of walks w = 0..n_w-1 of the listed samples, rec[k*n_w + w] for sample ids[k],
 * and of the first n_kill_first killing walks after them.  Same Philox counters as the
 * full run: the counter holds the sample's index in the full arrays, not k.
 */
int64_t orc_run_walks_subset(const orc_geom *g, const orc_params *P, int exterior,
                             const int32_t *tri, const float *bary, const float *weight,
                             const float *normal, const int64_t *ids, int64_t n_ids, int n_w,
                             int64_t n_kill_first, orc_record *rec)
{
    #pragma omp parallel for schedule(dynamic, 1)
    for (int64_t k = 0; k < n_ids; ++k) {
        const int64_t i = ids[k];
        orc_sample S;
        orc_ball B;
        fill_sample(g, tri, bary, weight, normal, NULL, i, &S);
        if (P->estimator == 1 && !exterior) { memset(&B, 0, sizeof B); B.sstar_norm = 1.0; }   /* Alg. 1 has no ball */
        else if (exterior) orc_tangent_ball_exterior(g, P, &S, &B);
        else               orc_tangent_ball_interior(g, P, &S, &B);
        for (int w = 0; w < n_w; ++w)
            run_one_walk(g, P, exterior, &S, &B, i, w, rec + k * n_w + w);
    }
    int64_t n_rec = n_ids * n_w;
    if (exterior && P->include_killing) {
        #pragma omp parallel for schedule(dynamic, 16)
        for (int64_t j = 0; j < n_kill_first; ++j) {
            orc_record *R = rec + n_rec + j;
            memset(R, 0, sizeof *R);
            R->sample = -1; R->tri_t = -1;
            orc_hit h;
            int steps = walk_on_spheres_kelvin(g, P, ORC_KILLING_SAMPLE, (uint32_t)j, R->z, &h);
            R->steps = steps;
            if (steps < 0) continue;
            R->tri_t = h.tri;
            memcpy(R->bary_t, h.bary, sizeof h.bary);
            memcpy(R->t, h.cp, sizeof h.cp);
            double tt[3]; sub3(h.cp, P->origin, tt);
            R->weight = 4.0 * ORC_PI * norm3(tt) / (double)P->n_kill_walks;    /* 4 pi / |t0*| */
        }
        n_rec += n_kill_first;
    }
    return n_rec;
}

/*
 * Measurement helper (bench.py, SURVEY.md 8(d) "oracle-side ideal"): the PRIMAL query points of the closest-point
 * queries that the walks w = 0..n_w-1 of the samples `ids` make (at most max_pos per walk; for the exterior the points
 * x = kappa(y) at which the flat-triangle query is taken, far-field jumps without a query left out), with the exact
 * distance found there.  The same loops as walk_on_spheres / walk_on_spheres_kelvin, recording instead of returning.
 * pos [n_ids * n_w * max_pos][3], dist [same], in blocks of max_pos per walk; count [n_ids * n_w] = points in each
 * block; returns the total.
 */
int64_t orc_walk_query_points(const orc_geom *g, const orc_params *P, int exterior,
                              const int32_t *tri, const float *bary, const float *weight, const float *normal,
                              const int64_t *ids, int64_t n_ids, int n_w, int max_pos, double *pos, double *dist,
                              int32_t *count /* [n_ids * n_w]: points written in the block of walk (k, w) */)
{
    int64_t n_total = 0;
    #pragma omp parallel for schedule(dynamic, 1) reduction(+:n_total)
    for (int64_t k = 0; k < n_ids; ++k) {
        const int64_t i = ids[k];
        orc_sample S; orc_ball B;
        fill_sample(g, tri, bary, weight, normal, NULL, i, &S);
        if (exterior) orc_tangent_ball_exterior(g, P, &S, &B); else orc_tangent_ball_interior(g, P, &S, &B);
        for (int w = 0; w < n_w; ++w) {
            const int64_t blk = (k * n_w + w) * (int64_t)max_pos;
            int n_here = 0;
            count[k * n_w + w] = 0;
            if (!(B.r > 0.0)) continue;
            double z[3];
            sample_ball_surface(P, &B, (uint32_t)i, (uint32_t)w, z);
            double x[3] = { z[0], z[1], z[2] };
            for (int step = 0; step <= P->max_steps && n_here < max_pos; ++step) {
                orc_hit h;
                double radius;
                if (exterior) {
                    double yn = norm3(x);
                    if (yn * P->Rmax_norm <= 0.5) radius = 1.0 / P->Rmax_norm - yn;
                    else {
                        double q[3] = { P->origin[0] + x[0] / (yn * yn), P->origin[1] + x[1] / (yn * yn), P->origin[2] + x[2] / (yn * yn) };
                        double rho = 1.0 / yn;
                        orc_closest_point(g, q, &h);
                        memcpy(pos + 3 * (blk + n_here), q, sizeof q); dist[blk + n_here] = h.dist; ++n_here;
                        radius = h.dist / (rho * fmin(P->Rmax_norm, rho + h.dist));
                        if (radius < P->eps || h.dist > rho) break;
                    }
                } else {
                    orc_closest_point(g, x, &h);
                    memcpy(pos + 3 * (blk + n_here), x, sizeof x); dist[blk + n_here] = h.dist; ++n_here;
                    radius = h.dist;
                    if (radius < P->eps || (P->escape_radius > 0.0 && radius > P->escape_radius)) break;
                }
                double wdir[3];
                step_direction(P->seed, (uint32_t)i, (uint32_t)w, (uint32_t)(step + 1), wdir);
                for (int j = 0; j < 3; ++j) x[j] += radius * wdir[j];
            }
            count[k * n_w + w] = n_here;
            n_total += n_here;
        }
    }
    return n_total;
}

/*
 * Accumulate S = sum_w weight_w d d^T in the hat basis (PAPER.md:177-190,
 * 277-285): d = b(s) - b(t) has the barycentric coordinates of s on the
 * vertices of tri_s and minus those of t on the vertices of tri_t; a killing
 * record contributes weight * b(t0) b(t0)^T.  Records are visited in slot
 * order.  S2 (optional) receives an estimate of the variance of every entry:
 * for each sample, W/(W-1) * (sum x^2 - (sum x)^2 / W) over its walks' entry
 * contributions x (killing walks form one group).
 */
typedef struct { int64_t key; double val; } orc_entry;
static int entry_cmp(const void *a, const void *b)
{
    int64_t ka = ((const orc_entry *)a)->key, kb = ((const orc_entry *)b)->key;
    return (ka > kb) - (ka < kb);
}

static int build_d(const orc_geom *g, const orc_record *R, const int32_t *tri, const float *bary,
                   int64_t idx[6], double val[6])
{
    int n = 0;
    if (R->sample >= 0) {
        const int32_t *fs = g->faces + 3 * (int64_t)tri[R->sample];
        for (int k = 0; k < 3; ++k) { idx[n] = fs[k]; val[n] = (double)bary[3*R->sample + k]; ++n; }
    }
    const int32_t *ft = g->faces + 3 * R->tri_t;
    double sign = (R->sample >= 0) ? -1.0 : 1.0;
    for (int k = 0; k < 3; ++k) {
        int found = -1;
        for (int m = 0; m < n; ++m) if (idx[m] == ft[k]) found = m;
        if (found >= 0) val[found] += sign * R->bary_t[k];
        else { idx[n] = ft[k]; val[n] = sign * R->bary_t[k]; ++n; }
    }
    return n;
}

static void accumulate_hat_impl(const orc_geom *g, const orc_record *rec, int64_t n_rec,
                                const int32_t *tri, const float *bary, int64_t K,
                                double *S, double *S2, int naive)
{
    orc_entry *buf = NULL;
    int64_t cap = 0;
    for (int64_t g0 = 0; g0 < n_rec; ) {
        /* one group = the walks of one sample (or all killing walks) */
        int64_t g1 = g0;
        int64_t sample = rec[g0].sample;
        while (g1 < n_rec && rec[g1].sample == sample) ++g1;
        int64_t n_e = 0;
        if (S2 && 36 * (g1 - g0) > cap) { cap = 36 * (g1 - g0); buf = (orc_entry *)realloc(buf, cap * sizeof *buf); }
        for (int64_t r = g0; r < g1; ++r) {
            const orc_record *R = rec + r;
            if (R->steps < 0 || R->weight == 0.0) continue;
            int64_t idx[6]; double val[6];
            int n = build_d(g, R, tri, bary, idx, val);
            double bsv[6] = { 0, 0, 0, 0, 0, 0 };              /* b_s on the merged vertex list (Alg. 1) */
            if (naive && R->sample >= 0) {
                const int32_t *fs = g->faces + 3 * (int64_t)tri[R->sample];
                for (int m = 0; m < n; ++m) for (int k = 0; k < 3; ++k)
                    if (idx[m] == fs[k]) bsv[m] += (double)bary[3 * R->sample + k];
            }
            for (int p = 0; p < n; ++p) for (int q = 0; q < n; ++q) {
                /* Alg. 2: w d d^T.  Alg. 1: w b_s d^T, symmetrised as in its last line: (S + S^T)/2 */
                double x = naive ? R->weight * 0.5 * (bsv[p] * val[q] + bsv[q] * val[p])
                                 : R->weight * val[p] * val[q];
                S[idx[p] * K + idx[q]] += x;
                if (S2) { buf[n_e].key = idx[p] * K + idx[q]; buf[n_e].val = x; ++n_e; }
            }
        }
        if (S2 && n_e > 0) {
            double Wg = (double)(g1 - g0);
            qsort(buf, (size_t)n_e, sizeof *buf, entry_cmp);
            for (int64_t e0 = 0; e0 < n_e; ) {
                int64_t e1 = e0; double s1 = 0.0, s2 = 0.0;
                while (e1 < n_e && buf[e1].key == buf[e0].key) { s1 += buf[e1].val; s2 += buf[e1].val * buf[e1].val; ++e1; }
                double var = (Wg > 1.0) ? Wg / (Wg - 1.0) * (s2 - s1 * s1 / Wg) : s2;
                S2[buf[e0].key] += var > 0.0 ? var : 0.0;
                e0 = e1;
            }
        }
        g0 = g1;
    }
    free(buf);
}

void orc_accumulate_hat(const orc_geom *g, const orc_record *rec, int64_t n_rec,
                        const int32_t *tri, const float *bary, int64_t K,
                        double *S /* [K][K] zeroed by caller */, double *S2 /* [K][K] or NULL */)
{
    accumulate_hat_impl(g, rec, n_rec, tri, bary, K, S, S2, 0);
}

/* Alg. 1's update  S += w b_s (b_s - b_t)^T  followed by its symmetrisation. */
void orc_accumulate_hat_naive(const orc_geom *g, const orc_record *rec, int64_t n_rec,
                              const int32_t *tri, const float *bary, int64_t K, double *S, double *S2)
{
    accumulate_hat_impl(g, rec, n_rec, tri, bary, K, S, S2, 1);
}

/* ------------------------------------------------------------------------- */
/* Point-based function space: k-NN bilateral interpolator (PAPER.md:373-379;  */
/* App. B, Eq. 44-45).  The basis functions live on a point  */
/* cloud (x_i, n_i), i < K; the value of a boundary function at a query point  */
/* q with normal n_q is  sum_{i in N_k(q)} w_i(q) phi(x_i),                     */
/*   w~_i = exp(-|q - x_i|^2 / (2 sigma^2)) exp(-(1 - <n_q, n_i>) / tau_n),    */
/*   w_i = w~_i / sum_j w~_j,                                                  */
/* so the vector b(q) of Alg. 2 has the k non-zeros w_i(q).                    */
/* Readings: [Rk1] the w~ are formed relative to the largest       */
/* exponent (identical after normalisation; no 0/0 when q is many sigma away   */
/* from every point); [Rk2] neighbours by squared distance, ties by smaller    */
/* index; [Rk3] k is clamped to K; [Rk4] n_q is the sample's normal at s and    */
/* the normal of the exit face at t.                                           */
/* ------------------------------------------------------------------------- */
typedef struct {
    const float *points;        /* [K][3] */
    const float *normals;       /* [K][3] unit */
    int64_t K;
    int32_t k;                  /* neighbours (paper: 8) */
    int32_t pad_;
    double sigma, tau_n;        /* paper: 0.025, 0.8 */
} orc_point_basis;

#define ORC_KNN_MAX 32

void orc_knn_weights(const orc_point_basis *PB, const double q[3], const double nq[3],
                     int64_t *idx /* [k] */, double *w /* [k] */)
{
    int k = PB->k < PB->K ? PB->k : (int)PB->K;
    if (k > ORC_KNN_MAX) k = ORC_KNN_MAX;
    double bd[ORC_KNN_MAX]; int64_t bi[ORC_KNN_MAX];
    int n = 0;
    for (int64_t i = 0; i < PB->K; ++i) {                      /* brute force over all points */
        double d[3] = { q[0] - (double)PB->points[3*i], q[1] - (double)PB->points[3*i+1], q[2] - (double)PB->points[3*i+2] };
        double d2 = dot3(d, d);
        if (n == k && !(d2 < bd[k-1])) continue;                /* strict <: on a tie the smaller index stays */
        int pos = n < k ? n : k - 1;
        while (pos > 0 && d2 < bd[pos-1]) { bd[pos] = bd[pos-1]; bi[pos] = bi[pos-1]; --pos; }
        bd[pos] = d2; bi[pos] = i;
        if (n < k) ++n;
    }
    double lg[ORC_KNN_MAX], lmax = -INFINITY, sum = 0.0;
    for (int j = 0; j < k; ++j) {
        const float *ni = PB->normals + 3 * bi[j];
        double c = nq[0] * (double)ni[0] + nq[1] * (double)ni[1] + nq[2] * (double)ni[2];
        lg[j] = -bd[j] / (2.0 * PB->sigma * PB->sigma) - (1.0 - c) / PB->tau_n;     /* Eq. 45 */
        if (lg[j] > lmax) lmax = lg[j];
    }
    for (int j = 0; j < k; ++j) { w[j] = exp(lg[j] - lmax); sum += w[j]; }          /* [Rk1] */
    for (int j = 0; j < k; ++j) { w[j] /= sum; idx[j] = bi[j]; }
    for (int j = k; j < PB->k; ++j) { idx[j] = -1; w[j] = 0.0; }
}

/* S += weight d d^T with d = b(s) - b(t) in the point basis (killing: weight b(t) b(t)^T), plus the
 * per-entry variance estimate of orc_accumulate_hat.  s and n_s come from the sample arrays (mesh:
 * tri/bary, sphere: pos), t from the record, n_t from the exit face (sphere: radial)  [Rk4]. */
void orc_accumulate_points(const orc_geom *g, const orc_point_basis *PB, const orc_record *rec, int64_t n_rec,
                           const int32_t *tri, const float *bary, const float *weight, const float *normal,
                           const double *pos, double *S /* [K][K] zeroed */, double *S2 /* or NULL */)
{
    const int64_t K = PB->K;
    const int k = PB->k;
    orc_entry *buf = NULL;
    int64_t cap = 0;
    for (int64_t g0 = 0; g0 < n_rec; ) {
        int64_t g1 = g0, sample = rec[g0].sample;
        while (g1 < n_rec && rec[g1].sample == sample) ++g1;
        int64_t is[ORC_KNN_MAX]; double ws[ORC_KNN_MAX];
        if (sample >= 0) {
            orc_sample SS;
            fill_sample(g, tri, bary, weight, normal, pos, sample, &SS);
            orc_knn_weights(PB, SS.s, SS.n, is, ws);
        }
        int64_t n_e = 0;
        const int64_t per = (int64_t)(2 * k) * (2 * k);
        if (S2 && per * (g1 - g0) > cap) { cap = per * (g1 - g0); buf = (orc_entry *)realloc(buf, cap * sizeof *buf); }
        for (int64_t r = g0; r < g1; ++r) {
            const orc_record *R = rec + r;
            if (R->steps < 0 || R->weight == 0.0) continue;
            double nt[3], area;
            if (g->kind == 0) face_normal_area(g, R->tri_t, nt, &area);
            else { double d[3]; sub3(R->t, g->centre, d); double l = norm3(d); for (int c = 0; c < 3; ++c) nt[c] = d[c] / l; }
            int64_t it[ORC_KNN_MAX]; double wt[ORC_KNN_MAX];
            orc_knn_weights(PB, R->t, nt, it, wt);
            int64_t idx[2 * ORC_KNN_MAX]; double val[2 * ORC_KNN_MAX];
            int n = 0;
            if (sample >= 0) for (int j = 0; j < k; ++j) if (is[j] >= 0) { idx[n] = is[j]; val[n] = ws[j]; ++n; }
            const double sign = sample >= 0 ? -1.0 : 1.0;
            for (int j = 0; j < k; ++j) {
                if (it[j] < 0) continue;
                int found = -1;
                for (int m = 0; m < n; ++m) if (idx[m] == it[j]) found = m;
                if (found >= 0) val[found] += sign * wt[j];
                else { idx[n] = it[j]; val[n] = sign * wt[j]; ++n; }
            }
            for (int p = 0; p < n; ++p) for (int q = 0; q < n; ++q) {
                double x = R->weight * val[p] * val[q];
                S[idx[p] * K + idx[q]] += x;
                if (S2) { buf[n_e].key = idx[p] * K + idx[q]; buf[n_e].val = x; ++n_e; }
            }
        }
        if (S2 && n_e > 0) {
            double Wg = (double)(g1 - g0);
            qsort(buf, (size_t)n_e, sizeof *buf, entry_cmp);
            for (int64_t e0 = 0; e0 < n_e; ) {
                int64_t e1 = e0; double s1 = 0.0, s2 = 0.0;
                while (e1 < n_e && buf[e1].key == buf[e0].key) { s1 += buf[e1].val; s2 += buf[e1].val * buf[e1].val; ++e1; }
                double var = (Wg > 1.0) ? Wg / (Wg - 1.0) * (s2 - s1 * s1 / Wg) : s2;
                S2[buf[e0].key] += var > 0.0 ? var : 0.0;
                e0 = e1;
            }
        }
        g0 = g1;
    }
    free(buf);
}

/* ------------------------------------------------------------------------- */
/* Generalised winding number and sidedness ("we repair     */
/* normals using generalized winding numbers"; Jacobson et al. 2013).         */
/* ------------------------------------------------------------------------- */
/*
 * w(p) = (1/4 pi) sum_f Omega_f(p): Omega_f = signed solid angle of face f seen from p, by the formula of
 * Van Oosterom & Strackee (1983):  tan(Omega/2) = a.(b x c) / (|a||b||c| + (a.b)|c| + (b.c)|a| + (c.a)|b|),
 * a, b, c = the vertices minus p.  Faces wound counter-clockwise seen from outside give w = 1 inside a closed
 * surface and 0 outside.  exclude[i] >= 0: that face is left out of the sum for point i (NULL: none).
 */
void orc_winding_number(const orc_geom *g, const double *p, int64_t n, const int64_t *exclude, double *w)
{
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t i = 0; i < n; ++i) {
        double sum = 0.0;
        for (int64_t f = 0; f < g->F; ++f) {
            if (exclude && exclude[i] == f) continue;
            double v[3][3], len[3];
            for (int k = 0; k < 3; ++k) {
                load_vertex(g, g->faces[3*f+k], v[k]);
                for (int d = 0; d < 3; ++d) v[k][d] -= p[3*i+d];
                len[k] = sqrt(v[k][0]*v[k][0] + v[k][1]*v[k][1] + v[k][2]*v[k][2]);
            }
            const double *a = v[0], *b = v[1], *c = v[2];
            double det = a[0] * (b[1]*c[2] - b[2]*c[1]) - a[1] * (b[0]*c[2] - b[2]*c[0]) + a[2] * (b[0]*c[1] - b[1]*c[0]);
            double ab = a[0]*b[0] + a[1]*b[1] + a[2]*b[2], bc = b[0]*c[0] + b[1]*c[1] + b[2]*c[2], ca = c[0]*a[0] + c[1]*a[1] + c[2]*a[2];
            double den = len[0]*len[1]*len[2] + ab*len[2] + bc*len[0] + ca*len[1];
            sum += 2.0 * atan2(det, den);
        }
        w[i] = sum / (4.0 * ORC_PI);
    }
}

/*
 * Sidedness of boundary samples  [DESIGN.md reading G-R1; the paper names the tool, not the rule].
 * For sample i on face f with face normal n_f (winding order) and h = h_scale * sqrt(area_f):
 *     d_i = w_{-f}(s - h n_f) - w_{-f}(s + h n_f),
 * w_{-f} = the winding number of the surface WITHOUT face f (its own jump of exactly 1 across itself carries no
 * information).  On a closed, outward-oriented surface w falls from 1 to 0 going out, so d > 0: n_f points out.
 * d < 0: the face is wound the wrong way round with respect to the surface about it; the outward normal is -n_f.
 * out_normal [n][3] = sign(d) n_f (d = 0 keeps n_f), d_out [n] = d.
 */
void orc_orient_samples(const orc_geom *g, const int32_t *tri, const float *bary, int64_t n, double h_scale,
                        double *out_normal, double *d_out)
{
    double *pts = (double *)malloc((size_t)n * 6 * sizeof(double));
    int64_t *excl = (int64_t *)malloc((size_t)n * 2 * sizeof(int64_t));
    double *w = (double *)malloc((size_t)n * 2 * sizeof(double));
    for (int64_t i = 0; i < n; ++i) {
        int64_t f = tri[i];
        double a[3], b[3], c[3], nrm[3], area, s[3];
        load_vertex(g, g->faces[3*f], a); load_vertex(g, g->faces[3*f+1], b); load_vertex(g, g->faces[3*f+2], c);
        face_normal_area(g, f, nrm, &area);
        double h = h_scale * sqrt(area);
        for (int k = 0; k < 3; ++k) {
            s[k] = (double)bary[3*i] * a[k] + (double)bary[3*i+1] * b[k] + (double)bary[3*i+2] * c[k];
            pts[6*i+k] = s[k] - h * nrm[k];          /* back  */
            pts[6*i+3+k] = s[k] + h * nrm[k];        /* front */
            out_normal[3*i+k] = nrm[k];
        }
        excl[2*i] = excl[2*i+1] = f;
    }
    orc_winding_number(g, pts, 2 * n, excl, w);
    for (int64_t i = 0; i < n; ++i) {
        double d = w[2*i] - w[2*i+1];
        d_out[i] = d;
        if (d < 0.0) for (int k = 0; k < 3; ++k) out_normal[3*i+k] = -out_normal[3*i+k];
    }
    free(pts); free(excl); free(w);
}

size_t orc_sizeof_point_basis(void) { return sizeof(orc_point_basis); }

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

size_t orc_sizeof_record(void) { return sizeof(orc_record); }
size_t orc_sizeof_params(void) { return sizeof(orc_params); }
size_t orc_sizeof_geom(void)   { return sizeof(orc_geom); }
