// common.cuh -- shared declarations of the CUDA path (sm_100a only).
// Nothing here is shared with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <mutex>
#include <math_constants.h>
#include <stdint.h>
#include <stddef.h>

#include "../../include/mcdtn.h"

#define MCS_CUDA_TRY(expr)                                     \
    do {                                                       \
        cudaError_t e__ = (expr);                              \
        if (e__ != cudaSuccess) { mcs_set_last_cuda_error((int)e__); return MCS_ECUDA; } \
    } while (0)

// Launch counter (bench.py's gpu_launches) and phase marks (CUDA events on the
// caller's stream, recorded only while mcs_profile_enable(1) is in effect).
void mcs_note_launch();
enum { MCS_MARK_BEGIN = 0, MCS_MARK_WALK_BEGIN, MCS_MARK_WALK_END, MCS_MARK_END, MCS_MARK_WALK_END2 /* optional: second walk kernel */, MCS_MARK_COUNT };
void mcs_prof_mark(int which, cudaStream_t st);

void mcs_set_last_cuda_error(int e);
int  mcs_get_last_cuda_error();

static inline int64_t ceil_div64(int64_t a, int64_t b) { return (a + b - 1) / b; }
static inline size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

// ---------------------------------------------------------------------------
// Packed geometry owned by the handle.
// ---------------------------------------------------------------------------
// One internal node = 64 bytes = 4 x 16-byte loads:
//   w0 = (lo0.x, lo0.y, lo0.z, hi0.x)
//   w1 = (hi0.y, hi0.z, lo1.x, lo1.y)
//   w2 = (lo1.z, hi1.x, hi1.y, hi1.z)
//   w3 = (child0, child1, parent, unused) as int32
// child >= 0: internal node index; child < 0: leaf, sorted triangle k = ~child.
struct __align__(16) BvhNode {
    float4 w0, w1, w2;
    int4   w3;
};

// One packed triangle = 64 bytes = 4 x 16-byte loads, in Morton order:
//   t0 = (v0.x, v0.y, v0.z, original face index as int bits)
//   t1 = (v1.x, v1.y, v1.z, |n|^2)   t2 = (v2.x, v2.y, v2.z, 1/|n|^2)
//   t3 = (n.x, n.y, n.z, flags as int bits: bit 0 = zero-area face, bit 1 = not the first leaf reference of its face),
//        n = (v1-v0) x (v2-v0)
// The vertices are the caller's fp32 numbers; n, |n|^2 are computed in fp64 by the build
// and rounded once.
struct __align__(16) PackedTri {
    float4 t0, t1, t2, t3;
};

// One 4-wide node of the walk kernel = 128 bytes = 4 x 32-byte loads: every second level of the
// binary tree collapsed (a binary node at even depth with its grandchildren, or a leaf child where
// the tree ends earlier).
//   f[6k .. 6k+5] = box of child k (lo.xyz, hi.xyz), k = 0..3;  an empty slot has lo = +inf
//   c[k]          = child k: >= 0 wide node index, < 0 leaf ~c = sorted triangle slot
//   pad[4]        = squared diagonal of the box of child k as float bits (+inf for an empty slot)
struct __align__(32) WideNode {
    float f[24];
    int   c[4];
    int   pad[4];
};

struct mcs_bvh {
    int64_t V, F, n_nodes;
    int64_t n_leaves;      // leaf references: F, plus the extra slabs of split slivers (bvh.cu)
    float*     verts;      // [V][3] copy of the input
    int32_t*   faces;      // [F][3] copy of the input
    BvhNode*   nodes;      // [max(F-1,1)]
    WideNode*  wide;       // [n_wide] 4-wide collapse of `nodes` (walk kernel); root = 0
    int64_t    n_wide;
    PackedTri* tris;       // [n_leaves] Morton order; leaf k holds the whole triangle of its face
    int32_t*   leaf_tri;   // [n_leaves] original face index of sorted leaf k
    int32_t*   face_slot;  // [F] first sorted leaf of original face f
    uint64_t*  morton;     // [n_leaves] sorted keys
    int32_t    root;       // index of the root node (0)
    int32_t    max_depth;
    int32_t    n_degenerate;
    float      aabb_lo[3], aabb_hi[3];
    double     area;
    double     sah_cost;   // surface-area cost of the packed tree (bvh.cu sah_partial_kernel)
    size_t     device_bytes;
    int        device;
    mutable cudaEvent_t last_use;   // recorded on the stream of every call that reads the tree (mcs_free_bvh waits for it)
    // face hierarchy of mcs_orient_samples_fast (winding.cu), built on first use
    mutable std::mutex wn_mutex;
    mutable void*      wn_nodes;    // float4 [2 G][2]: (centroid, radius), (area vector, area); heap order, root = 1
    mutable uint32_t*  wn_order;    // [F] faces along the Z-order curve
    mutable int32_t*   wn_face_pos; // [F] position of a face in wn_order
    mutable long long  wn_G;        // leaf groups, padded to a power of two
    mutable int        wn_levels;   // level of the leaf groups (root = 0)
};

// Every entry point that enqueues work reading the tree calls this with its stream when it is done enqueuing.
void mcs_bvh_touch(const mcs_bvh* b, cudaStream_t st);
void mcs_free_bvh_on(mcs_bvh* b, cudaStream_t st);

// ---------------------------------------------------------------------------
// radix sort / scan (sort.cu)
// ---------------------------------------------------------------------------
size_t sort_workspace_bytes(int64_t n, int key_bytes);
// Stable LSD radix sort, 8 bits per pass over bits [0, key_bits).  keys/vals are
// sorted in place (the workspace holds the ping-pong copies).
int sort_pairs_u64(uint64_t* keys, uint32_t* vals, int64_t n, int key_bits,
                   void* ws, size_t ws_bytes, cudaStream_t st);
int sort_pairs_u32(uint32_t* keys, uint32_t* vals, int64_t n, int key_bits,
                   void* ws, size_t ws_bytes, cudaStream_t st);
// The same with the number of pairs known on the device only: *n_dev <= n_cap pairs are sorted; n_cap sizes the grids and the
// workspace (sort_workspace_bytes(n_cap, 4)).  Never blocks the host.
int sort_pairs_u32_devn(uint32_t* keys, uint32_t* vals, int64_t n_cap, const uint32_t* n_dev, int key_bits,
                        void* ws, size_t ws_bytes, cudaStream_t st);
size_t scan_workspace_bytes(int64_t n);
// Exclusive prefix sum of uint32 counts into uint64-safe? No: totals fit in
// int64 on the host side; device array is uint32 (n_entries per chunk < 2^32).
int exclusive_scan_u32(const uint32_t* in, uint32_t* out, int64_t n, uint32_t* total_out /* device, may be NULL */,
                       void* ws, size_t ws_bytes, cudaStream_t st);
