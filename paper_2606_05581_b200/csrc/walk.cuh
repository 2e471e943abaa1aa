// walk.cuh -- internal interface between walk.cu, accumulate.cu and capi.cu.
#pragma once
#include "common.cuh"

enum {
    ST_WORK = 0,        // work-queue head of the persistent walk kernel
    ST_STEPS, ST_QUERIES, ST_TRUNCATED, ST_DISCARDED, ST_NODES, ST_TRIS,
    ST_ENTRIES, ST_UNIQUE,
    ST_PREP_QUERIES, ST_PREP_NODES, ST_PREP_TRIS,   // tangent-ball share of ST_QUERIES / ST_NODES / ST_TRIS
    ST_FAR,             // queries answered by a lower bound (far_alpha > 0)
    ST_HIST = 16,       // 16 bins: queries of the walk kernel by floor(log2(nodes visited))
    ST_COUNT = 32
};

struct WalkGeom {
    const BvhNode*   nodes;
    const WideNode*  wide;         // 4-wide collapse of `nodes` (walk kernel)
    const PackedTri* tris;
    const float*     verts;
    const int32_t*   faces;
};

// Values of one call that are computed ON THE DEVICE (so that no call has to read them back before it can go on):
// r_max of the tangent balls (exterior: from the AABB of the Kelvin-inverted vertices), R_max = max |v - o|
// (E3), and the input errors only the device can see.  Lives behind the counters of the walk workspace.
struct WalkDyn {
    float rmax, Rmax;
    int   err;                     // WALK_ERR_* bits; non-zero poisons the call: every record is written as discarded
    int   pad_;
};
enum { WALK_ERR_SAMPLE_FACE = 1,   // a sample's face index is outside [0, F)            -> MCS_EINVAL
       WALK_ERR_DEGENERATE = 2 };  // a vertex at the Kelvin origin, or R_max not > 0     -> MCS_EDEGENERATE

struct WalkArgs {
    const float4*   balls;         // [n_s][2]: (c.xyz, r), (pole.xyz, |s*|)
    const uint32_t* order;         // Z-order permutation of the samples
    const float*    weight;        // [n_s] quadrature weights a_i
    const int32_t*  sample_slot;   // [n_s] sorted triangle slot of each sample's face
    long long n_s, n_kill;
    int   W, max_steps, chunk;
    int   importance, antithetic;
    int   naive;                   // Alg. 1: balls hold the start point, no ball sampling
    float inv_inset;
    float eps, q0, inv_q0;
    float ox, oy, oz;
    const WalkDyn* dyn;            // R_max (exterior) and the poison flag, device-resident
    float mesh_scale;              // |coordinates|_1 bound of the mesh (prune_limit)
    float escape;                  // interior: AABB diagonal (R10b); exterior: +inf
    float far_alpha2, far_near;    // far-field lower-bound queries: alpha^2 (0: exact queries only), near threshold k eps
    uint32_t key0, key1;
    float4* records;               // mcs_record viewed as float4
    int32_t* steps;
    int*     coop_scratch;         // [grid][warps][COOP_NCAP + COOP_LCAP] warp lists of the cooperative path
    unsigned long long* work_counter;
    unsigned long long* stats;
};

int64_t walk_num_records(const mcs_samples* s, const mcs_params* p, int exterior);
size_t  walk_workspace_bytes(const mcs_samples* s);
int walk_run(const mcs_bvh* b, const mcs_samples* s, const mcs_params* p, int exterior,
             void* ws, size_t ws_bytes, float4* records, int32_t* steps, bool balls_only, float* balls_out,
             bool count, unsigned long long** stats_dev_out, cudaStream_t st, struct WalkLaunch* defer = nullptr,
             bool check_now = true);
// check_now = true: walk_run blocks once, after the preparation, and returns the device-side input errors (MCS_EINVAL for a
// sample face out of range, MCS_EDEGENERATE for a vertex at the Kelvin origin) before the walk kernel is launched.
// check_now = false: nothing is read back; a call with such an error is poisoned (all records discarded) and the caller
// reads the flags later with walk_error_code / from the copy of the counters (walk_dyn_of).
const WalkDyn* walk_dyn_of(const unsigned long long* stats_dev);
int walk_error_code(int err_bits);

// A prepared launch of the walk kernel (walk_run with `defer`): everything before the kernel has been
// enqueued on walk_run's stream; walk_launch may enqueue the kernel on another stream that waits for it.
struct WalkLaunch {
    void (*fn)(WalkGeom, WalkArgs);
    unsigned grid, block;
    bool coop;                     // the variant with the warp-cooperative path was chosen
    WalkGeom g;
    WalkArgs a;
};
int walk_launch(const WalkLaunch* w, cudaStream_t st);

// Batched launch (mcs_estimate_dtn_batch): the prepared launches of many (mesh, operator) pairs run as ONE persistent
// kernel over the concatenation of their walks.  ctx / counter / scratch: device memory of the caller
// (walk_batch_scratch_bytes); blocks the host only for the upload of the contexts (pageable source).
struct WalkCtx {
    WalkGeom g;
    WalkArgs a;
    long long begin;               // first global walk index of the segment (a multiple of the chunk)
    int ext, far;                  // exterior operator; far-field cut on
};
struct WalkBatch {
    long long total;               // padded walk count of all segments
    int n_ctx, chunk;
    unsigned long long* work_counter;
    int* coop_scratch;
};
size_t walk_batch_scratch_bytes(int n_launches);
int walk_launch_batch(const WalkLaunch* launches, const int* exterior, const int* far, int n_launches,
                      void* scratch, size_t scratch_bytes, cudaStream_t st);

size_t accumulate_workspace_bytes(const mcs_bvh* b, const mcs_basis* basis, int64_t n_records);
size_t accumulate_coo_workspace_bytes(const mcs_bvh* b, int64_t n_records, int64_t coo_capacity);
int accumulate_coo_run(const mcs_bvh* b, const mcs_samples* s, const mcs_basis* basis, int W, int naive,
                       const float4* records, int64_t n_records, void* ws, size_t ws_bytes,
                       const mcs_matrix* out, unsigned long long* stats_dev, cudaStream_t st);
int accumulate_run(const mcs_bvh* b, const mcs_samples* s, const mcs_basis* basis, int W, int naive,
                   const float4* records, int64_t n_records, void* ws, size_t ws_bytes,
                   const mcs_matrix* out, unsigned long long* stats_dev, cudaStream_t st);

// point-based k-NN basis (mcs_basis.kind 1), accumulate.cu
size_t accumulate_points_workspace_bytes(const mcs_samples* s, const mcs_basis* basis, int64_t n_records);
int accumulate_points_run(const mcs_bvh* b, const mcs_samples* s, const mcs_basis* basis, int W,
                          const float4* records, int64_t n_records, void* ws, size_t ws_bytes,
                          const mcs_matrix* out, unsigned long long* stats_dev, cudaStream_t st);
int knn_weights_run(const mcs_basis* basis, const float* q, const float* nq, int64_t Q, int32_t* idx, float* w, cudaStream_t st);
