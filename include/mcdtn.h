/*
 * mcdtn.h -- C ABI of the B200-native Monte Carlo Dirichlet-to-Neumann estimator.
 *
 * Hot path of "Monte Carlo Steklov Operators for Large-Scale Geometry Processing
 * in the Wild" (arxiv 2606.05581; citations are PAPER.md:<line>): the
 * walk-on-spheres estimator that fills the discrete DtN matrix of a triangle
 * mesh, interior (Alg. 2 / Eq. 26) and exterior (Eq. 32,
 * PAPER.md:348-353, App. C.3-C.7).
 *
 * Conventions
 *   - Every pointer is a DEVICE pointer unless its comment says "host".
 *   - The caller owns every buffer it passes in; the library owns only the
 *     opaque mcs_bvh handle (packed triangles + nodes in device memory).
 *   - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).
 *     Work is enqueued on it; a call blocks the host only where stated.
 *   - Return value: MCS_OK (0) or a negative MCS_E* code.  No exceptions, no
 *     aborts.  mcs_error_string() names a code.
 *   - All floating point on this path is fp32 (the paper states no precision);
 *     statistics counters are 64-bit integers.
 *   - There is no CPU fallback: every entry point needs a CUDA device.
 */
#ifndef MCDTN_H
#define MCDTN_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define MCS_OK            0
#define MCS_EINVAL      (-1)   /* null / negative size / index out of range / eps <= 0 / K mismatch */
#define MCS_EDEGENERATE (-2)   /* zero total area, non-finite vertex, Kelvin origin on a vertex      */
#define MCS_ENOMEM      (-3)   /* workspace too small or device allocation failed                     */
#define MCS_ECUDA       (-4)   /* CUDA runtime error (code in mcs_stats.cuda_error when available)    */
#define MCS_ETOOLARGE   (-5)   /* size beyond a fixed maximum of the entry point (mcs_sort_pairs_u64_static)     */
#define MCS_WNOTCONVERGED 1    /* warning (results written): an iteration stopped at its cap, see mcs_steklov_eigs */

typedef struct mcs_bvh mcs_bvh;

/* ------------------------------------------------------------------------ */
/* (1) LBVH over the triangle soup -- subsystem "A0 mesh pack" + "A1 LBVH     */
/* build" of SURVEY.md 8(a).  The paper uses a BVH for its distance queries   */
/* and treats every triangle as absorbing, so   */
/* the build assumes nothing about manifoldness, orientation, area or the     */
/* number of components.                                                       */
/* ------------------------------------------------------------------------ */
typedef struct {                 /* all zero = defaults */
    int32_t no_split;            /* 1: one leaf per face.  0: long thin faces enter the tree as several leaf references,
                                    one per slab across their longest edge (sliver-heavy CAD meshes;
                                    the box of a rotated sliver is almost all empty space).  Query results are the same
                                    either way: every reference carries the whole triangle                              */
    int32_t max_pieces;          /* references per face at most (0: 64)                                                 */
    float   split_length;        /* a face is cut when its longest edge exceeds this many mean edge lengths and its
                                    aspect L^2 / 2A exceeds 8; pieces are about this long (0: 4)                         */
    float   split_budget;        /* extra references per face on average at most; the piece length is raised until
                                    this holds (0: 1)                                                                    */
} mcs_build_opts;

typedef struct {
    int64_t V, F;                /* vertices, faces                                  */
    int64_t n_nodes;             /* internal nodes of the packed tree (n_leaves - 1) */
    int32_t max_depth;           /* deepest leaf (root = 0)                          */
    int32_t n_degenerate;        /* zero-area faces (kept: they absorb as segments)  */
    float   aabb_lo[3], aabb_hi[3];   /* box of the vertices referenced by faces     */
    double  area;                /* total surface area |dOmega|                      */
    size_t  device_bytes;        /* device memory owned by the handle                */
    int64_t n_leaves;            /* leaf references: F plus the extra slabs of split faces */
    double  sah_cost;            /* surface-area cost of the tree: sum over child boxes of area x (1 inner, 80/18 leaf)
                                    / area of the root box -- expected box tests + weighted triangle tests of a random
                                    line; a quality readout, lower is better                                             */
} mcs_bvh_info_t;

/*
 * Build.  verts [V][3] fp32 and faces [F][3] int32 are read on `stream`; the
 * handle keeps its own copies, so the caller may free them after the call.
 * Blocks the host until the build has finished (it reads back error flags).
 * The handle's device memory comes from the device's stream-ordered pool
 * (cudaMallocAsync on `stream`; the pool's release threshold is raised so that
 * build/free cycles reuse memory).  mcs_free_bvh returns it in the order of the
 * legacy default stream after making that stream wait for the last call that used the handle (the handle
 * records an event on the stream of every call that reads the tree), so kernels still queued on a non-blocking
 * stream finish first; it does not block the host.  A handle used on several streams at once must be
 * synchronised by the caller before it is freed (only the last call's stream is tracked).
 * Errors: MCS_EINVAL (null pointer, V < 1, F < 1, face index outside [0,V)),
 * MCS_EDEGENERATE (non-finite vertex, zero total area), MCS_ENOMEM, MCS_ECUDA.
 */
int  mcs_build_bvh(const float* verts, int64_t V, const int32_t* faces, int64_t F,
                   const mcs_build_opts* opts /* host, may be NULL */,
                   void* stream, mcs_bvh** out /* host */);
void mcs_free_bvh(mcs_bvh* bvh);
int  mcs_bvh_info(const mcs_bvh* bvh, mcs_bvh_info_t* out /* host */);

/*
 * Structure dump for the invariant tests (SURVEY.md 8(c) "LBVH (GPU)").
 * Each output may be NULL.  nodes: [n_nodes][16] 32-bit words, the packed node
 * (see DESIGN.md "BVH node"); leaf_tri: [n_leaves] original face index of the k-th
 * leaf in Morton order; morton: [n_leaves] sorted 63-bit keys.  Blocks the host.
 */
int  mcs_bvh_dump(const mcs_bvh* bvh, uint32_t* nodes, int32_t* leaf_tri, uint64_t* morton,
                  void* stream);

/* ------------------------------------------------------------------------ */
/* (2) Closest point on the triangle soup -- the geometric query under WoS    */
/* ("nearest boundary point").                      */
/* q [Q][3] -> dist [Q] (unsigned distance), tri [Q] (original face index;    */
/* ties: smaller fp32 squared distance, then smaller index), bary [Q][3]       */
/* (barycentrics of the closest point in that face).  Outputs may be NULL.    */
/* Asynchronous on `stream`.                                                   */
/* ------------------------------------------------------------------------ */
int  mcs_closest_point(const mcs_bvh* bvh, const float* q, int64_t Q,
                       float* dist, int32_t* tri, float* bary, void* stream);

/* Same query by exhaustive scan over all faces on the device (cross-check of
 * the tree; thread per query, faces tiled through shared memory).            */
int  mcs_closest_point_bruteforce(const mcs_bvh* bvh, const float* q, int64_t Q,
                                  float* dist, int32_t* tri, float* bary, void* stream);

/* ------------------------------------------------------------------------ */
/* (3)-(4) Estimators.                                                         */
/* ------------------------------------------------------------------------ */
typedef struct {                 /* boundary samples: point s with its face */
    const int32_t* tri;          /* [n_s] face of each sample                              */
    const float*   bary;         /* [n_s][3] barycentrics of s in that face                */
    const float*   weight;       /* [n_s] quadrature weight a_i, sum = |dOmega| (Eq. 26)   */
    const float*   normal;       /* [n_s][3] unit normal pointing out of the solid, or NULL
                                    (then the face normal (v1-v0)x(v2-v0) is used)         */
    int64_t n_s;
} mcs_samples;

typedef struct {                 /* boundary basis functions b(.) of Alg. 2 */
    int32_t kind;                /* 0 = hat functions on the mesh vertices (K = V);
                                    1 = point-based k-NN bilateral interpolator (App. B
                                        Eq. 44-45): K = number of points, b(q) has the k weights w_i(q)   */
    int32_t pad_;
    int64_t K;
    /* kind 1 only (ignored for kind 0) */
    const float* points;         /* [K][3] positions x_i                                                */
    const float* normals;        /* [K][3] unit normals n_i                                             */
    int32_t k;                   /* neighbours, 1..16 (paper: 8); clamped to K                          */
    float   sigma;               /* spatial falloff (paper: 0.025)                                      */
    float   tau_n;               /* normal falloff (paper: 0.8)                                         */
    int32_t pad2_;
} mcs_basis;

typedef struct {
    uint64_t seed;               /* Philox4x32-10 key; counter = (sample, walk, step, purpose) */
    int32_t  walks_per_sample;   /* W >= 1                                                     */
    int32_t  max_steps;          /* walks longer than this contribute nothing (counted)        */
    float    eps;                /* WoS shell, absolute                    */
    float    cap_half_angle_deg; /* excluded cap about s, PAPER.md:395 ("~2.5 deg")            */
    float    rmax_scale;         /* r_max = rmax_scale * (shortest AABB side)/2  */
    float    rmax_override;      /* > 0: use this r_max instead of the AABB rule               */
    int32_t  bisection_iters;    /* LargestTangentBall iterations, PAPER.md:383 (10); 1..24    */
    int32_t  importance_sample;  /* 1: z ~ J^B; 0: z uniform on the ball        */
    int32_t  antithetic;         /* 1: walks 2j, 2j+1 are antipodal in azimuth  */
    int32_t  include_killing;    /* exterior only: second expectation of Eq. 32                */
    int64_t  n_kill_walks;       /* exterior only                                              */
    float    kelvin_origin[3];   /* exterior only: a point strictly inside the solid */
    int32_t  output_kind;        /* 0: dense row-major fp32 [K][K] (K <= 65535);
                                    1: sparse COO, upper triangle (any K < 2^31)                */
    int64_t  coo_capacity;       /* output_kind 1: entries mcs_matrix.coo_* can hold (sizes the workspace) */
    int32_t  estimator;          /* 0: Alg. 2, the tangent-ball jump-kernel estimator;
                                    1: Alg. 1, the naive finite-difference estimator (Eq. 16),
                                       interior only: walks start at s - inset * n_s, update
                                       (a_i / (W inset)) b_s (b_s - b_t)^T, symmetrised; NOT PSD at finite N */
    float    inset;              /* estimator 1: inset distance (the paper's epsilon of Eq. 13), > 0 */
    float    far_alpha;          /* 0: every closest-point query is exact (default).  > 0: far-field queries return a LOWER
                                    BOUND of the distance: a sub-tree whose box diagonal is <= far_alpha x its box distance
                                    is not descended, its box distance stands for its faces.  The walker then jumps with a
                                    radius between D / (1 + far_alpha) and D.  WoS only needs a ball inside the domain
                                    (PAPER.md:155), so the estimator is unchanged in expectation; single walks differ from
                                    the exact run.  The shell test and the exit point always come from an exact query.
                                    Deterministic (independent of the schedule).  Measured best on a 2 M-face in-the-
                                    wild mesh: 1 (interior), 2 (exterior) with far_near_factor 2; at most 4             */
    float    far_near_factor;    /* far_alpha > 0: boxes closer than this many eps are always descended (0: 16; >= 2)  */
    int32_t  exterior_query;     /* exterior only.  0 (default): flat-triangle query at x = kappa(y) on the primal tree with
                                    the conservative radius D / (rho min(R_max, rho + D)) (E3).  1: the paper's own
                                    query, the EXACT distance from y to the Kelvin-inverted faces = (1/|x|) min
                                    over the mesh of |x - p| / |p - o| (E4): larger balls, fewer jumps, a dearer
                                    query; same estimator.  Not combinable with far_alpha                              */
    int32_t  nonblocking;        /* mcs_estimate_dtn_interior / _exterior / _both (there: in both blocks); ignored elsewhere.  0 (default): the call blocks the host for small
                                    read-backs (below) and returns device-side input errors.  1: the call ONLY ENQUEUES work on
                                    `stream` -- no read-back, no allocation, no copy from host memory -- so it returns at once and
                                    may be captured in a CUDA graph.  Needs output_kind 0, basis kind 0 and host_stats == NULL
                                    (MCS_EINVAL otherwise).  Same kernels, same bits.  Input errors only the device can see (a
                                    sample's face index out of range, a vertex at the Kelvin origin) cannot be returned then:
                                    such a call skips its walks and fills `out` with NaN                                 */
} mcs_params;

typedef struct {
    int32_t kind;                /* must equal params.output_kind                    */
    int32_t pad_;
    int64_t K;
    float*  dense;               /* kind 0: [K][K] row-major, overwritten             */
    /* kind 1: the UPPER triangle (row <= col) of the symmetric matrix in coordinate form,
     * sorted by (row, col), one entry per (row, col); S[col][row] = S[row][col] is implied. */
    int64_t  coo_capacity;       /* entries each of the three arrays can hold (= params.coo_capacity) */
    int32_t* coo_row;
    int32_t* coo_col;
    float*   coo_val;
    int64_t* coo_nnz;            /* device scalar: entries written.  MCS_ENOMEM when more than
                                    coo_capacity are needed; then it holds a lower bound of the need */
} mcs_matrix;

typedef struct {                 /* host; filled when passed non-NULL (forces a stream sync) */
    int64_t n_samples, n_discarded;       /* samples whose tangent ball degenerated */
    int64_t n_walks, n_truncated;         /* walks started / cut at max_steps or outside the AABB */
    int64_t n_steps;                      /* position updates x += d*omega                         */
    int64_t n_queries;                    /* closest-point queries: every WoS iteration + one tangent-ball traversal per sample */
    int64_t n_nodes_visited, n_tris_tested;   /* traversal work actually done (flop/byte model)    */
    int64_t n_prep_queries, n_prep_nodes, n_prep_tris;  /* of which: the tangent-ball traversals (A2) */
    int64_t n_entries, n_unique;          /* (row,col,value) records expanded / after reduction    */
    int64_t workspace_needed;             /* bytes; set on MCS_ENOMEM too                           */
    int64_t n_far_queries;                /* walk-kernel queries answered by a lower bound (far_alpha > 0; counter build) */
    int64_t nodes_hist[16];               /* walk-kernel queries by floor(log2(nodes visited)), bin 15 = rest */
    int32_t cuda_error;                   /* cudaError_t on MCS_ECUDA                               */
    int32_t pad_;
} mcs_stats;

/*
 * Workspace (bytes) the estimators need for these arguments; `exterior` selects
 * the operator.  Pointers inside samples are not dereferenced.
 */
size_t mcs_workspace_bytes(const mcs_bvh* bvh, const mcs_samples* samples, const mcs_basis* basis,
                           const mcs_params* params, int exterior);

/*
 * Interior DtN estimate (Alg. 2):
 *   S = sum over samples i, walks w of  (a_i / W) * (|dB_r(c)| / 2) J / pdf * d d^T,
 *   d = b(s_i) - b(t_iw), t_iw the WoS exit point of a walk started on the
 *   largest tangent ball at s_i.  S is symmetric PSD by construction.
 * samples/basis/params/out are host structs holding device pointers.  The
 * library never allocates here: all scratch lives in `workspace`.
 * Work is enqueued on `stream`.  With params.nonblocking = 1 (dense output, hat basis, host_stats == NULL) that is all
 * the call does: it returns at once and may be captured in a CUDA graph; workspace, out, the samples' arrays and the
 * bvh handle must stay alive until the work has run (every time the graph runs).  Otherwise the call blocks the host:
 * once after the preparation (one 16-byte read-back of the device-side input checks, so that MCS_EINVAL /
 * MCS_EDEGENERATE come back before the walks start); COO output and the point basis once more per accumulation chunk
 * (entry count); with host_stats != NULL it returns when everything is done.
 * Errors: MCS_EINVAL, MCS_ENOMEM (workspace_bytes too small), MCS_ECUDA.
 */
int mcs_estimate_dtn_interior(const mcs_bvh* bvh, const mcs_samples* samples, const mcs_basis* basis,
                              const mcs_params* params, void* workspace, size_t workspace_bytes,
                              const mcs_matrix* out, mcs_stats* host_stats, void* stream);

/*
 * Exterior DtN estimate (Eq. 32): the same estimator in the
 * Kelvin-inverted domain about params.kelvin_origin with the factor
 * |s*|^3 / |t*|, plus (include_killing) n_kill_walks walks from kappa(infinity)
 * adding (4 pi / |t0*|) b(t0) b(t0)^T / n_kill_walks.
 * Walks end with steps >= 0 (landed), -1 (max_steps jumps, R10), -2 (sample discarded)
 * or -3: interior, the jump radius exceeds the AABB diagonal (the walker is outside the box, R10b); exterior,
 * the distance to the surface exceeds the distance to kelvin_origin (the walker is inside the solid, R10c).
 * -1 and -3 contribute nothing and are counted in mcs_stats.n_truncated.
 */
int mcs_estimate_dtn_exterior(const mcs_bvh* bvh, const mcs_samples* samples, const mcs_basis* basis,
                              const mcs_params* params, void* workspace, size_t workspace_bytes,
                              const mcs_matrix* out, mcs_stats* host_stats, void* stream);

/*
 * Both operators of one mesh in one call (the unit BASELINE configs 1-4 ask for: "interior and exterior DtN"):
 * the same two estimates as mcs_estimate_dtn_interior(params_interior) and mcs_estimate_dtn_exterior(params_exterior),
 * bit for bit (walks are keyed by (seed, sample, walk, step) and accumulated in a fixed order, so the result does
 * not depend on the schedule), with the two persistent walk kernels overlapped: all preparation runs on `stream`,
 * then the interior's walk + accumulation go to a library-owned high-priority stream and the exterior's to a
 * low-priority one (the interior's blocks are dispatched first; the exterior's fill the SM slots its tail gives up),
 * both waiting for the preparation; `stream` waits for both before the call's work is complete, so the caller sees
 * ordinary stream semantics.  out_interior and out_exterior must be different buffers;
 * workspace >= mcs_workspace_bytes_both (the two operators' workspaces side by side).
 * Asynchronous on `stream` up to the exterior's read-back of its Kelvin bounds (a few microseconds of device
 * work) unless a stats pointer is given.  Errors: as mcs_estimate_dtn_*.
 */
size_t mcs_workspace_bytes_both(const mcs_bvh* bvh, const mcs_samples* samples, const mcs_basis* basis,
                                const mcs_params* params_interior, const mcs_params* params_exterior);
int mcs_estimate_dtn_both(const mcs_bvh* bvh, const mcs_samples* samples, const mcs_basis* basis,
                          const mcs_params* params_interior, const mcs_params* params_exterior,
                          void* workspace, size_t workspace_bytes,
                          const mcs_matrix* out_interior, const mcs_matrix* out_exterior,
                          mcs_stats* host_stats_interior, mcs_stats* host_stats_exterior, void* stream);

/*
 * The whole path from HOST buffers, for callers that keep their data on the CPU
 * (and for the end-to-end measurement): uploads the mesh and the samples,
 * builds the LBVH, runs the requested estimators (operators: bit 0 = interior,
 * bit 1 = exterior) and downloads the dense K x K matrices (K = V, hat basis).
 * EVERY pointer here is a HOST pointer, including those inside `samples`
 * (pinned memory makes the copies asynchronous but is not required);
 * out_interior / out_exterior are [V][V] fp32 and may be NULL when their bit is
 * clear.  Device memory is allocated and freed inside the call (stream-ordered);
 * with both bits set the two operators run as in mcs_estimate_dtn_both;
 * the call blocks until the results are in the host buffers.  `stats` (host,
 * may be NULL) receives the counters of the LAST operator run.
 * Errors: as mcs_build_bvh and mcs_estimate_dtn_*.
 */
int mcs_estimate_dtn_host(const float* verts, int64_t V, const int32_t* faces, int64_t F,
                          const mcs_samples* samples, const mcs_params* params, int operators,
                          float* out_interior, float* out_exterior, mcs_stats* stats, void* stream);

/*
 * The same from HOST buffers with the SPARSE output, for meshes whose V x V matrix cannot be dense (BASELINE
 * config 3: 2 M faces): upload of the mesh and the samples, LBVH build, optionally the sidedness
 * pre-pass (orient_h_scale > 0: mcs_orient_samples with that h_scale -- or, with orient_beta > 0,
 * mcs_orient_samples_fast with that beta -- decides the side of every sample and replaces samples->normal;
 * PAPER.md:638-640), BOTH estimators as in mcs_estimate_dtn_both with output_kind 1, download.
 * EVERY pointer is a HOST pointer.  out_*: capacity = entries the three arrays can hold; on return nnz = entries
 * written (upper triangle, sorted by (row, col)).  MCS_ENOMEM when a capacity is too small: nnz then holds a lower
 * bound of the need and nothing is copied.  params_*->output_kind / coo_capacity are ignored (taken from out_*).
 * Device memory is allocated and freed inside the call (stream-ordered pool); blocks until the results are in the
 * host buffers.  Errors: as mcs_build_bvh, mcs_orient_samples and mcs_estimate_dtn_*.
 */
typedef struct {
    int64_t  capacity;           /* in: entries row/col/val can hold                          */
    int32_t* row;                /* host [capacity]                                           */
    int32_t* col;
    float*   val;
    int64_t  nnz;                /* out                                                       */
} mcs_host_coo;
int mcs_estimate_dtn_host_coo(const float* verts, int64_t V, const int32_t* faces, int64_t F,
                              const mcs_samples* samples, const mcs_params* params_interior, const mcs_params* params_exterior,
                              float orient_h_scale, float orient_beta, mcs_host_coo* out_interior, mcs_host_coo* out_exterior,
                              mcs_stats* stats_interior, mcs_stats* stats_exterior, void* stream);

/*
 * Many meshes in one call (BASELINE config 4: "1024 seeded synthetic meshes ... interior and exterior DtN ... meshes/s
 * end to end"; dataset-scale runs, one shape after another).  For every item: LBVH build, optional
 * sidedness pre-pass (orient_h_scale > 0: mcs_orient_samples, or mcs_orient_samples_fast when orient_beta > 0; the
 * normals are written to item.normal_out and used as the samples' normals), then both estimators as in
 * mcs_estimate_dtn_both with DENSE outputs (item.basis.K squared each; params_*->output_kind must be 0;
 * params_exterior->kelvin_origin is replaced by item.kelvin_origin).  `n_workers` (0: 4, at most 16) host threads, each
 * with its own stream and workspace, take the items in turn, so that the small launches, the host read-backs and the
 * tail of one mesh's walks overlap with the bulk of another's; every item is computed exactly as by the single calls
 * (results do not depend on n_workers).  items is a HOST array whose pointers are DEVICE pointers; item.rc receives the
 * item's return code.  Work starts after what `stream` holds at the call (uploads) and `stream` continues after all
 * of it; the call blocks until everything is done.  Returns the first non-zero item code.
 */
typedef struct {
    const float*   verts;        /* [V][3] device */
    int64_t        V;
    const int32_t* faces;        /* [F][3] device */
    int64_t        F;
    mcs_samples    samples;      /* device pointers; samples.normal is replaced by normal_out when orient_h_scale > 0 */
    mcs_basis      basis;        /* kind 0: K = V; kind 1: the point basis of this mesh */
    float          kelvin_origin[3];
    int32_t        rc;           /* out */
    float*         out_interior; /* [K][K] device */
    float*         out_exterior; /* [K][K] device */
    float*         normal_out;   /* [n_s][3] device, or NULL when orient_h_scale <= 0 */
} mcs_batch_item;
int mcs_estimate_dtn_batch(mcs_batch_item* items /* host */, int64_t n_items, const mcs_params* params_interior,
                           const mcs_params* params_exterior, float orient_h_scale, float orient_beta, int32_t n_workers,
                           void* stream);

/* ------------------------------------------------------------------------ */
/* Test / benchmark hooks for the individual steps of SURVEY.md 8(a).         */
/* ------------------------------------------------------------------------ */
typedef struct {                 /* one termination record per walk, slot = sample*W + walk, */
    int32_t tri_t;               /* then the killing walks.  tri_t < 0: no contribution      */
    float   b1, b2;              /* barycentrics of t on vertices 1, 2 of tri_t (b0 = 1-b1-b2) */
    float   weight;              /* full scalar multiplying d d^T                             */
} mcs_record;

/* A2: tangent balls.  balls [n_s][8] = (c.x, c.y, c.z, r, pole.x, pole.y, pole.z, |s*|) in
 * the walk domain's coordinates (exterior: Kelvin coordinates about the origin). */
int mcs_tangent_balls(const mcs_bvh* bvh, const mcs_samples* samples, const mcs_params* params,
                      int exterior, float* balls, void* stream);

/* Workspace (bytes) of mcs_run_walks and of mcs_accumulate. */
size_t mcs_walk_workspace_bytes(const mcs_samples* samples);
size_t mcs_accumulate_workspace_bytes(const mcs_bvh* bvh, const mcs_samples* samples, const mcs_basis* basis,
                                      const mcs_params* params, int64_t n_records);

/* A2-A6: run every walk and write records [n_s*W (+ n_kill_walks)] and, if non-NULL,
 * steps [same length] (jumps taken; -1 truncated at max_steps; -2 sample discarded; -3 interior
 * walker left the bounding box of the mesh, cut and counted as truncated: DESIGN.md R10b). */
int mcs_run_walks(const mcs_bvh* bvh, const mcs_samples* samples, const mcs_params* params,
                  int exterior, void* workspace, size_t workspace_bytes,
                  mcs_record* records, int32_t* steps, mcs_stats* host_stats, void* stream);

/* A7: deterministic accumulation of records into the matrix (sort by key +
 * segmented sum; no float atomics). */
int mcs_accumulate(const mcs_bvh* bvh, const mcs_samples* samples, const mcs_basis* basis,
                   const mcs_params* params, const mcs_record* records, int64_t n_records,
                   void* workspace, size_t workspace_bytes, const mcs_matrix* out,
                   mcs_stats* host_stats, void* stream);

/* k-NN bilateral weights of a kind-1 basis at Q query points q [Q][3] with unit normals nq [Q][3]
 * (Eq. 44-45): idx [Q][k] (neighbours by increasing distance, ties by smaller index; -1 beyond K),
 * w [Q][k] (sum 1).  Exhaustive search over the K points.  Asynchronous on `stream`. */
int mcs_knn_weights(const mcs_basis* basis, const float* q, const float* nq, int64_t Q,
                    int32_t* idx, float* w, void* stream);

/* Philox4x32-10 words for counters [n][4] and one key [2] (host): out [n][4].
 * Lets the tests pin the device generator against the known answers. */
int mcs_philox4x32_10(const uint32_t* counters, int64_t n, const uint32_t* key /* host */,
                      uint32_t* out, void* stream);

/* Stable LSD radix sort of (key, value) pairs, test hook for the sort used by
 * the LBVH build and by the accumulation.  keys/vals are sorted in place;
 * workspace must hold mcs_sort_workspace_bytes(n) bytes. */
size_t mcs_sort_workspace_bytes(int64_t n);
int mcs_sort_pairs_u64(uint64_t* keys, uint32_t* vals, int64_t n, int32_t key_bits,
                       void* workspace, size_t workspace_bytes, void* stream);

/* The same sort for callers that may not allocate and have no workspace to hand in (code under CUDA graph
 * capture, tight serving loops, harnesses that forbid cudaMalloc): the workspace is a file-scope device array
 * inside the library (sort.cu), 12.25 MiB that every GPU which loads the library holds until the process exits.
 * keys [n] / vals [n]: device pointers, sorted in place (stable, low `key_bits` bits of the key), as above.
 * Limit: n <= mcs_sort_static_max_n() = 2^20 pairs; beyond it the call returns MCS_ETOOLARGE and does nothing.
 * The call allocates nothing and frees nothing (no cudaMalloc / cudaFree / allocating library routine) and is
 * asynchronous on `stream`.  All calls on one device share the one array and it keeps the last call's contents
 * (nothing in it needs to start at zero): calls that OVERLAP on the GPU -- different streams with no ordering
 * between them, or two host threads -- race on it; order them on one stream or with events.
 * Errors: MCS_EINVAL (null pointer, n < 0, key_bits outside [0, 64]), MCS_ETOOLARGE, MCS_ECUDA. */
int64_t mcs_sort_static_max_n(void);
int mcs_sort_pairs_u64_static(uint64_t* keys, uint32_t* vals, int64_t n, int32_t key_bits, void* stream);

/* Measurement hooks (bench.py).  mcs_launch_count: kernels this library has launched in
 * this process.  mcs_profile_enable(1): estimate_* calls record CUDA events on their stream
 * around their phases; mcs_profile_last blocks on the last call's events and returns the
 * elapsed device time of each phase in milliseconds (MCS_EINVAL if nothing was recorded).
 * Not thread safe: one profiled call at a time. */
typedef struct {
    float prep_ms;               /* A2: Z-order sort + tangent balls            */
    float walk_ms;               /* A3-A6: the persistent walk kernel           */
    float accumulate_ms;         /* A7                                          */
    float total_ms;
    /* mcs_estimate_dtn_both only (else 0): start of the interior walk kernel to the end of the interior / exterior
     * kernel; walk_ms is the larger, accumulate_ms what follows it */
    float walk_interior_ms, walk_exterior_ms;
} mcs_phase_times;
unsigned long long mcs_launch_count(void);
int mcs_profile_enable(int on);
int mcs_profile_last(mcs_phase_times* out /* host */);

/* Generalised winding number of the mesh (Jacobson et al. 2013):
 *     w(p) = (1 / 4 pi) sum_f Omega_f(p),  Omega_f = signed solid angle of face f seen from p (Van Oosterom-Strackee),
 * 1 inside a closed surface wound counter-clockwise seen from outside, 0 outside.  Exhaustive over all faces.
 * points [n][3] device fp32; exclude [n] device int32 or NULL: original index of a face left out for that point
 * (-1: none); w_out [n] device.  workspace >= mcs_winding_workspace_bytes(bvh, n).  Asynchronous on `stream`.
 *
 * mcs_orient_samples: sidedness of boundary samples by rule G-R1 of DESIGN.md.  For sample i on face f with face
 * normal n_f (winding order) and h = h_scale * sqrt(area_f):  d_i = w_-f(s - h n_f) - w_-f(s + h n_f), w_-f = the
 * winding number without face f.  d > 0: n_f points out of the solid.  normal_out [n_s][3] device = sign(d) n_f,
 * usable as mcs_samples.normal; d_out [n_s] device or NULL.  samples->weight and ->normal are not read.
 * workspace >= mcs_winding_workspace_bytes(bvh, n_s).  Blocks the host (it reads back an error flag).
 * Errors: MCS_EINVAL (null pointer, n < 1, h_scale <= 0, sample face out of range), MCS_ENOMEM, MCS_ECUDA. */
size_t mcs_winding_workspace_bytes(const mcs_bvh* bvh, int64_t n);
int mcs_winding_number(const mcs_bvh* bvh, const float* points, const int32_t* exclude /* may be NULL */, int64_t n,
                       float* w_out, void* workspace, size_t workspace_bytes, void* stream);
int mcs_orient_samples(const mcs_bvh* bvh, const mcs_samples* samples, float h_scale, float* normal_out,
                       float* d_out /* may be NULL */, void* workspace, size_t workspace_bytes, void* stream);

/* mcs_orient_samples_fast: the same decision from a hierarchical evaluation.  d_i is a difference of the winding number
 * at two points 2h apart, so only the surface near the sample decides it: faces are grouped along a Z-order curve in a
 * binary tree of (area vector, centroid, radius); a node farther than beta radii from the sample is replaced by its
 * dipole term for BOTH probes (same cut, so the truncation error largely cancels in d), nearer nodes are opened and their
 * faces summed exactly; the sample's own face is left out as above.  beta >= 1.5 (typical 2-3: |d - exact| of a few 1e-3
 * on unit-sized meshes; the decision differs from the exact one only where |d| is that small).  The hierarchy is built on
 * the first call and kept in the handle.  No workspace.  Blocks the host (error flag).  About F / (few thousand) times
 * less work than the exhaustive sum: BASELINE config 3 (20 000 samples, 2 M faces) 455 ms -> a few ms. */
int mcs_orient_samples_fast(const mcs_bvh* bvh, const mcs_samples* samples, float h_scale, float beta, float* normal_out,
                            float* d_out /* may be NULL */, void* stream);

/* Reduced Ritz-Galerkin DtN matrix: for basis functions
 * phi_k = sum_v Phi[v][k] hat_v (Phi [V][K] device fp32, row-major: e.g. low-frequency Laplacian eigenmodes at the
 * vertices) the matrix the paper accumulates from dense vectors b(p) = Phi^T iota(p) equals Phi^T S Phi for the
 * nodal matrix S [V][V] of mcs_estimate_dtn_* (dense output).  out [K][K] device, exactly symmetric.
 * workspace >= mcs_project_workspace_bytes(V, K).  Asynchronous on `stream`.  V, K <= 65535.
 * Errors: MCS_EINVAL, MCS_ENOMEM, MCS_ECUDA. */
size_t mcs_project_workspace_bytes(int64_t V, int64_t K);
int mcs_project_galerkin(const float* S, const float* Phi, int64_t V, int64_t K, float* out,
                         void* workspace, size_t workspace_bytes, void* stream);
/* The same from the sparse output (mcs_matrix kind 1): row, col, val [nnz] device, the upper triangle sorted by
 * (row, col) with one entry per position, as mcs_estimate_dtn_* writes it; any V < 2^31 (the reduced basis is how a
 * K x K operator is obtained on meshes whose V x V matrix cannot be dense).  Deterministic (no atomics).
 * workspace >= mcs_project_coo_workspace_bytes(V, K).  Blocks the host (it reads back an error flag).
 * Errors: MCS_EINVAL (also: an entry below the diagonal or out of range, rows not sorted), MCS_ENOMEM, MCS_ECUDA. */
size_t mcs_project_coo_workspace_bytes(int64_t V, int64_t K);
int mcs_project_galerkin_coo(const int32_t* row, const int32_t* col, const float* val, int64_t nnz,
                             const float* Phi, int64_t V, int64_t K, float* out,
                             void* workspace, size_t workspace_bytes, void* stream);

/* Smallest Steklov eigenpairs of estimated DtN matrices:
 *     S psi = lambda M psi,  M = diag(mass)  (lumped boundary mass),
 * for a batch of `batch` dense symmetric matrices S [batch][K][K] (symmetrised inside) with mass [batch][K] > 0.
 * evals [batch][n_eig] ascending; evecs [batch][n_eig][K] (may be NULL), M-orthonormal: psi_i^T M psi_j = delta_ij.
 * Two solvers, both fp32 on A = M^-1/2 S M^-1/2.  (1) One-sided Jacobi: all eigenpairs are computed, the n_eig smallest
 * returned; the only choice for K < 1024.  (2) Chebyshev-filtered subspace iteration for FEW eigenpairs of a LARGE matrix
 * (K >= 1024, n_eig <= 256, block of n_eig + max(16, n_eig / 4) columns rounded up to 64, at most K / 2): products A X only,
 * 2 K^2 m flops each, so the lowest 64 modes at K = 2562 take 28 ms instead of 0.52 s and K = 16384 (the paper's 2^14
 * points) is within reach; residuals |A x - theta x| <= 2e-5 x (Gershgorin bound of A) on exit.
 * mcs_steklov_eigs chooses: (2) where it applies, and (1) after all if (2) did not converge within its 40 iterations (a
 * spectrum crowded at its low end).  mcs_steklov_eigs_method: method 0 = that choice, 1 = Jacobi, 2 = subspace iteration
 * (MCS_EINVAL where it does not apply; MCS_WNOTCONVERGED instead of the fall-back).
 * sweeps_out (host, may be NULL): Jacobi sweeps or subspace iterations used.  Blocks the host once per sweep / iteration.
 * The solver is made for the symmetric POSITIVE SEMI-DEFINITE matrices of Alg. 2 / Eq. 32: one-sided Jacobi diagonalises
 * A^2, so an indefinite input (Alg. 1, estimator = 1) with eigenvalues +l and -l of equal magnitude can leave mixed
 * vectors.  Returns MCS_WNOTCONVERGED (> 0, results written) when the sweep cap (30) was reached with rotations still
 * being applied.  K <= 16384.  Errors: MCS_EINVAL, MCS_ENOMEM (workspace), MCS_ECUDA. */
size_t mcs_steklov_eigs_workspace_bytes(int64_t K, int64_t batch);
int mcs_steklov_eigs(const float* S, const float* mass, int64_t K, int64_t batch, int32_t n_eig,
                     float* evals, float* evecs, void* workspace, size_t workspace_bytes,
                     int32_t* sweeps_out /* host */, void* stream);
int mcs_steklov_eigs_method(const float* S, const float* mass, int64_t K, int64_t batch, int32_t n_eig, int32_t method,
                            float* evals, float* evecs, void* workspace, size_t workspace_bytes,
                            int32_t* sweeps_out /* host */, void* stream);

/* Roofline denominators measured on this device (bench.py): FP32
 * CUDA-core throughput of independent FMA chains (TFLOP/s, 2 flop per FMA) and the read
 * bandwidth of a 24 MiB L2-resident buffer with 16-byte loads (GB/s).  Each allocates a
 * scratch buffer, times 6 launches with CUDA events on `stream`, returns the best, blocks. */
int mcs_measure_fp32_tflops(double* tflops /* host */, void* stream);
int mcs_measure_l2_gbs(double* gbs /* host */, void* stream);

const char* mcs_error_string(int code);
const char* mcs_version(void);
/* sizeof of the ABI structs, for bindings to check their mirrors against:
 * 0 mcs_samples, 1 mcs_basis, 2 mcs_params, 3 mcs_matrix, 4 mcs_stats, 5 mcs_bvh_info_t,
 * 6 mcs_record, 7 mcs_host_coo, 8 mcs_batch_item; anything else: 0. */
size_t mcs_abi_sizeof(int which);

#ifdef __cplusplus
}
#endif
#endif /* MCDTN_H */
