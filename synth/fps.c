/* fps.c -- greedy farthest-point sampling over a candidate point set (input generator only:
 * BASELINE.json configs 3-4 choose their boundary samples "by farthest-point sampling").
 * Holds none of the method's arithmetic.  Plain C, single thread, deterministic.
 *
 * Same picks as the textbook loop  d2[i] = min(d2[i], |p_i - p|^2); next = first argmax(d2)  with
 * |.|^2 = (dx*dx + dy*dy) + dz*dz in fp32 without contraction (the numpy loop this replaces, which took
 * minutes on 1 M candidates).  The candidates arrive sorted along a space-filling curve (by the caller) and
 * are cut into buckets of consecutive points, each with its bounding box and its current maximum of d2: a
 * bucket whose box is at least as far from the new point p as that maximum cannot change (every point of the
 * box is at least the box distance from p, in fp32 too: rounding is monotone) and is skipped, so late
 * iterations touch a handful of buckets.
 *
 *   pts    [n][3] fp32 candidates (curve order)
 *   orig   [n]    index of each candidate before the sort (ties: smallest original index wins, as argmax does)
 *   first  position (in curve order) of the first chosen point
 *   chosen [m]    out: ORIGINAL indices in the order they were picked
 * returns 0, or -1 on bad arguments / allocation failure.
 */
#include <stdint.h>
#include <stdlib.h>

#define BUCKET 256

static float box_d2(const float* lo, const float* hi, float px, float py, float pz)
{
    float dx = lo[0] - px > px - hi[0] ? lo[0] - px : px - hi[0]; dx = dx > 0.0f ? dx : 0.0f;
    float dy = lo[1] - py > py - hi[1] ? lo[1] - py : py - hi[1]; dy = dy > 0.0f ? dy : 0.0f;
    float dz = lo[2] - pz > pz - hi[2] ? lo[2] - pz : pz - hi[2]; dz = dz > 0.0f ? dz : 0.0f;
    return (dx * dx + dy * dy) + dz * dz;
}

/* d2[i] = min(d2[i], |p_i - p|^2) over one bucket; returns the bucket's maximum (branch-free: vectorised). */
__attribute__((target_clones("avx2", "default")))
static float update_bucket(const float* restrict x, const float* restrict y, const float* restrict z,
                           float* restrict d2, int64_t n, float px, float py, float pz)
{
    float best = -1.0f;
    for (int64_t i = 0; i < n; ++i) {
        const float dx = x[i] - px, dy = y[i] - py, dz = z[i] - pz;
        const float d = (dx * dx + dy * dy) + dz * dz;
        const float v = d < d2[i] ? d : d2[i];
        d2[i] = v;
        best = v > best ? v : best;
    }
    return best;
}

int synth_fps(const float* pts, const int64_t* orig, int64_t n, int64_t first, int64_t m, int64_t* chosen)
{
    if (!pts || !orig || !chosen || n < 1 || m < 1 || m > n || first < 0 || first >= n) return -1;
    const int64_t nb = (n + BUCKET - 1) / BUCKET;
    float* x = (float*)malloc(sizeof(float) * (size_t)n * 4);
    float* box = (float*)malloc(sizeof(float) * (size_t)nb * 7);       /* lo[3], hi[3], max d2 */
    int64_t* barg = (int64_t*)malloc(sizeof(int64_t) * (size_t)nb);    /* position of the bucket's maximum (smallest orig) */
    if (!x || !box || !barg) { free(x); free(box); free(barg); return -1; }
    float *y = x + n, *z = y + n, *d2 = z + n;
    for (int64_t i = 0; i < n; ++i) { x[i] = pts[3 * i]; y[i] = pts[3 * i + 1]; z[i] = pts[3 * i + 2]; d2[i] = 3.0e38f; }
    for (int64_t b = 0; b < nb; ++b) {
        const int64_t lo = b * BUCKET, hi = lo + BUCKET < n ? lo + BUCKET : n;
        float* q = box + 7 * b;
        q[0] = q[3] = x[lo]; q[1] = q[4] = y[lo]; q[2] = q[5] = z[lo];
        for (int64_t i = lo + 1; i < hi; ++i) {
            if (x[i] < q[0]) q[0] = x[i];
            if (x[i] > q[3]) q[3] = x[i];
            if (y[i] < q[1]) q[1] = y[i];
            if (y[i] > q[4]) q[4] = y[i];
            if (z[i] < q[2]) q[2] = z[i];
            if (z[i] > q[5]) q[5] = z[i];
        }
        q[6] = 3.0e38f; barg[b] = lo;
    }
    int64_t cur = first;
    chosen[0] = orig[first];
    for (int64_t it = 1; it < m; ++it) {
        const float px = x[cur], py = y[cur], pz = z[cur];
        float gbest = -1.0f; int64_t garg = 0;
        for (int64_t b = 0; b < nb; ++b) {
            float* q = box + 7 * b;
            if (box_d2(q, q + 3, px, py, pz) < q[6]) {
                const int64_t lo = b * BUCKET, hi = lo + BUCKET < n ? lo + BUCKET : n;
                const float best = update_bucket(x + lo, y + lo, z + lo, d2 + lo, hi - lo, px, py, pz);
                int64_t arg = -1;
                for (int64_t i = lo; i < hi; ++i) if (d2[i] == best && (arg < 0 || orig[i] < orig[arg])) arg = i;
                q[6] = best; barg[b] = arg;
            }
            if (q[6] > gbest || (q[6] == gbest && orig[barg[b]] < orig[garg])) { gbest = q[6]; garg = barg[b]; }
        }
        cur = garg;
        chosen[it] = orig[cur];
    }
    free(x); free(box); free(barg);
    return 0;
}
