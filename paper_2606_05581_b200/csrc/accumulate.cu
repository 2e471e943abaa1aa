// accumulate.cu -- deterministic accumulation of per-walk records into the DtN
// matrix:   S = sum_walks  weight * d d^T,
// d = b(s) - b(t) in the hat basis (Eq. 26), a
// killing record contributing weight * b(t0) b(t0)^T (Eq. 32, second term).
//
// The paper defers the outer products "to be computed in batches to avoid shared
// memory contention".  Here the accumulation is a two-level
// sort-by-key segmented reduction, with no float atomics anywhere:
//
//  level 1 (on chip)  A block takes 256 consecutive record slots, sorts them in shared
//      memory by (sample, exit face) and reduces every run to ONE pair record: the
//      moments  w = sum wgt,  A_k = sum wgt eta_k,  M_kl = sum wgt eta_k eta_l  of the
//      exit-point barycentrics about a reference r (the pair's first exit point),
//      eta = b(t) - r.  All walks of a pair share b(s) and the six vertices involved, so
//      sum wgt d d^T  over the pair, d = (b(s) - r) - eta, is a function of (w, A, M, r) alone.
//      With W walks per sample this shrinks the stream that has to be sorted globally by the
//      number of walks per (sample, exit face) pair.
//  level 2 (global)   Pair records are expanded to upper-triangular (row*K+col, value)
//      entries in slot order, stable-radix-sorted by key, every run of equal keys is
//      summed by a segmented scan of fixed shape, and the run sums are added to the
//      dense matrix (one writer per entry); runs that cross a tile are completed in
//      tile order by a second small kernel.  The upper triangle is mirrored at the end.
//
// Every sum has a fixed association order (the position of an item after a stable
// sort, the shape of the scan), so the result is bit-identical from run to run and
// exactly symmetric.
#include "walk.cuh"

namespace {

constexpr int AT = 256;
constexpr int CH = 256;                               // record slots per level-1 block
#ifndef MCS_DENSE_CHUNK_LOG2
#define MCS_DENSE_CHUNK_LOG2 22
#endif
constexpr int64_t MAX_CHUNK_WALKS = (int64_t)1 << MCS_DENSE_CHUNK_LOG2;
// Sparse output: the running list of unique entries is re-sorted with every chunk's new entries, so fewer, larger chunks
// pay (B200: 180 GB; a 16 Mi-walk chunk takes about 17 GB of workspace per operator at BASELINE config 3's sizes).
#ifndef MCS_COO_CHUNK_LOG2
#define MCS_COO_CHUNK_LOG2 24
#endif
constexpr int64_t MAX_CHUNK_WALKS_COO = (int64_t)1 << MCS_COO_CHUNK_LOG2;
constexpr int MAX_ENTRIES_PER_PAIR = 21;              // upper triangle of a 6 x 6 block
constexpr int RT = 1024;                              // entries per tile of the run reduction

// Moments of a pair are taken about a reference exit point (the barycentrics r of the pair's first walk):
// eta = b(t) - r.  Most of the weight sits in walks that land close to their sample, where d = b(s) - b(t)
// is small; sums of raw b b^T would lose three digits to cancellation there, sums of eta eta^T do not.
struct __align__(16) PairRec {
    int   sample;            // -1: killing walk (no b(s) part)
    int   tri_t;
    float w;                 // sum wgt
    float A[3];              // sum wgt eta_k
    float M[6];              // sum wgt eta_k eta_l : 00 01 02 11 12 22
    float ref1, ref2;        // reference barycentrics r_1, r_2 (r_0 = 1 - r_1 - r_2); killing: 0, 0, eta = b
    float pad_[2];
};

struct AccArgs {
    const float4*  records;
    const int32_t* faces;
    const int32_t* s_tri;
    const float*   s_bary;
    long long n_main;       // records below this index belong to sample (index / W)
    int W;
    int naive;              // Alg. 1: entries of (1/2)(b_s d^T + d b_s^T) instead of d d^T
    long long K;
};

// ---------------------------------------------------------------------------
// Segmented inclusive scan over the CH (or RT) threads of a block, NV values per
// thread, fixed shape: Hillis-Steele inside a warp restricted to the lane's segment,
// then the warps' trailing partial sums are chained in warp order.
// head: this thread starts a new segment.  On return v[] holds the inclusive sum of
// the thread's segment up to and including itself, as far as the segment lies inside
// the block.  Returns true when the thread's segment has its head inside the block.
// ---------------------------------------------------------------------------
template <int NV, int NWARPS>
__device__ __forceinline__ bool block_segmented_scan(float (&v)[NV], bool head, float (*s_tail)[NV], int* s_has_head)
{
    const unsigned FULL = 0xFFFFFFFFu;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned heads = __ballot_sync(FULL, head);
    const unsigned upto = heads & (0xFFFFFFFFu >> (31 - lane));          // heads at lanes <= lane
    const int seg_start = upto ? 31 - __clz(upto) : 0;                    // first lane of my segment inside the warp
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
#pragma unroll
        for (int q = 0; q < NV; ++q) {
            const float t = __shfl_up_sync(FULL, v[q], o);
            if (lane - o >= seg_start) v[q] += t;
        }
    }
    if (lane == 31) {
#pragma unroll
        for (int q = 0; q < NV; ++q) s_tail[warp][q] = v[q];
        s_has_head[warp] = heads != 0;
    }
    __syncthreads();
    bool headed = upto != 0;
    if (!headed && warp > 0) {                                            // my segment started in an earlier warp
        float carry[NV];
#pragma unroll
        for (int q = 0; q < NV; ++q) carry[q] = 0.0f;
        int first = warp - 1;
        while (first > 0 && !s_has_head[first]) --first;                  // warp holding the segment's head (or warp 0)
        headed = s_has_head[first] != 0;
        for (int w = first; w < warp; ++w)                                // chained left to right
#pragma unroll
            for (int q = 0; q < NV; ++q) carry[q] += s_tail[w][q];
#pragma unroll
        for (int q = 0; q < NV; ++q) v[q] = carry[q] + v[q];
    }
    __syncthreads();
    return headed;
}

// ---------------------------------------------------------------------------
// Level 1.
// ---------------------------------------------------------------------------
__global__ void __launch_bounds__(CH)
pair_reduce_kernel(AccArgs a, long long j0, long long n, PairRec* __restrict__ pairs, uint32_t* __restrict__ pair_counts)
{
    __shared__ unsigned long long s_key[CH];
    __shared__ float4 s_rec[CH];
    __shared__ float s_tail[CH / 32][10];
    __shared__ float s_tail2[CH / 32][2];
    __shared__ int s_has_head[CH / 32];
    __shared__ int s_warp_runs[CH / 32];
    const int tid = threadIdx.x;
    const long long base = j0 + (long long)blockIdx.x * CH;
    const long long slot = base + tid;
    const long long first_sample = base < a.n_main ? base / a.W : 0;
    unsigned long long key = ~0ull;
    if (slot < j0 + n) {
        const float4 rec = a.records[slot];
        s_rec[tid] = rec;
        const int tri_t = __float_as_int(rec.x);
        if (tri_t >= 0 && rec.w != 0.0f) {
            const unsigned long long sl = slot < a.n_main ? (unsigned long long)(slot / a.W - first_sample) : 0x1FFull;
            key = (sl << 40) | ((unsigned long long)(unsigned)tri_t << 8) | (unsigned long long)tid;
        }
    }
    s_key[tid] = key;
    __syncthreads();
    // bitonic sort of CH unique 64-bit keys (the low byte is the slot: ties keep slot order)
    for (int k = 2; k <= CH; k <<= 1) {
        for (int j = k >> 1; j > 0; j >>= 1) {
            const int partner = tid ^ j;
            if (partner > tid) {
                const unsigned long long x = s_key[tid], y = s_key[partner];
                const bool up = (tid & k) == 0;
                if ((x > y) == up) { s_key[tid] = y; s_key[partner] = x; }
            }
            __syncthreads();
        }
    }
    key = s_key[tid];
    const bool valid = key != ~0ull;
    const unsigned long long gid = key >> 8;
    const bool head = valid && (tid == 0 || (s_key[tid - 1] >> 8) != gid);
    const bool tail = valid && (tid == CH - 1 || (s_key[tid + 1] >> 8) != gid);     // invalid keys sort last
    float v[10], ref[2];
    {
        const float4 rec = s_rec[valid ? (int)(key & 0xFF) : 0];
        const float wgt = valid ? rec.w : 0.0f;
        const bool killing = (gid >> 32) == 0x1FFull;
        // reference of the run = barycentrics of its first walk, broadcast by a segmented sum of (r at the head, 0 elsewhere)
        ref[0] = (head && !killing) ? rec.y : 0.0f; ref[1] = (head && !killing) ? rec.z : 0.0f;
        block_segmented_scan<2, CH / 32>(ref, head || !valid, s_tail2, s_has_head);
        const float e1 = rec.y - ref[0], e2 = rec.z - ref[1];
        const float e0 = killing ? 1.0f - rec.y - rec.z : -(e1 + e2);
        v[0] = wgt; v[1] = wgt * e0; v[2] = wgt * e1; v[3] = wgt * e2;
        v[4] = v[1] * e0; v[5] = v[1] * e1; v[6] = v[1] * e2; v[7] = v[2] * e1; v[8] = v[2] * e2; v[9] = v[3] * e2;
    }
    block_segmented_scan<10, CH / 32>(v, head || !valid, s_tail, s_has_head);
    // rank of my run among the block's runs (runs are counted at their tails)
    const unsigned tails = __ballot_sync(0xFFFFFFFFu, tail);
    const int lane = tid & 31, warp = tid >> 5;
    if (lane == 0) s_warp_runs[warp] = __popc(tails);
    __syncthreads();
    int before = 0, total = 0;
    for (int w = 0; w < CH / 32; ++w) { const int c = s_warp_runs[w]; if (w < warp) before += c; total += c; }
    if (tail) {
        const int rank = before + __popc(tails & ((1u << lane) - 1u));
        PairRec r;
        const unsigned sl = (unsigned)(gid >> 32);
        r.sample = sl == 0x1FFu ? -1 : (int)(first_sample + sl);
        r.tri_t = (int)(gid & 0xFFFFFFFFu);
        r.w = v[0]; r.A[0] = v[1]; r.A[1] = v[2]; r.A[2] = v[3];
        for (int q = 0; q < 6; ++q) r.M[q] = v[4 + q];
        r.ref1 = ref[0]; r.ref2 = ref[1]; r.pad_[0] = r.pad_[1] = 0.0f;
        pairs[(long long)blockIdx.x * CH + rank] = r;
    }
    if (tid == 0) pair_counts[blockIdx.x] = (uint32_t)total;
}

// ---------------------------------------------------------------------------
// Level 1b: pairs of one chunk that share (sample, exit face) are merged.  A sample's W walks span W / 256 level-1
// blocks, and most of them land on the same few hundred faces, so the same pair comes out of many blocks (BASELINE
// config 3, W = 4096: 5 pair records per distinct pair).  The chunk's pair records are stable-sorted by (sample, face)
// and every run is folded into its first record, in slot order, after moving the moments to that record's reference
// point: with delta = r_j - r_0,  A' = A + w delta,  M' = M + A delta^T + delta A^T + w delta delta^T.
// ---------------------------------------------------------------------------
__global__ void __launch_bounds__(AT)
pair_keys_kernel(const PairRec* __restrict__ pairs, const uint32_t* __restrict__ pair_counts, long long n_slots,
                 long long first_sample, int face_bits, unsigned long long* __restrict__ keys, uint32_t* __restrict__ vals)
{
    const long long i = (long long)blockIdx.x * AT + threadIdx.x;
    if (i >= n_slots) return;
    unsigned long long key = ~0ull >> 1;                                    // invalid slots sort last (63-bit keys)
    if ((uint32_t)(i % CH) < pair_counts[i / CH]) {
        const int sample = pairs[i].sample, tri = pairs[i].tri_t;
        if (tri >= 0 && sample >= 0)
            key = ((unsigned long long)((long long)sample - first_sample) << face_bits) | (unsigned long long)(unsigned)tri;
    }
    keys[i] = key;
    vals[i] = (uint32_t)i;
}

__global__ void __launch_bounds__(AT)
pair_merge_kernel(const PairRec* __restrict__ pairs, const unsigned long long* __restrict__ keys, const uint32_t* __restrict__ vals,
                  long long n_slots, PairRec* __restrict__ merged, uint32_t* __restrict__ merged_counts)
{
    const long long i = (long long)blockIdx.x * AT + threadIdx.x;
    if (i >= n_slots) return;
    if (i % CH == 0) merged_counts[i / CH] = CH;                            // every slot is looked at; tri_t = -1 marks the empty ones
    const unsigned long long key = keys[i];
    PairRec r;
    r.sample = -1; r.tri_t = -1; r.w = 0.0f; r.A[0] = r.A[1] = r.A[2] = 0.0f;
    for (int q = 0; q < 6; ++q) r.M[q] = 0.0f;
    r.ref1 = r.ref2 = 0.0f; r.pad_[0] = r.pad_[1] = 0.0f;
    if (key != (~0ull >> 1) && (i == 0 || keys[i - 1] != key)) {            // head of a run: fold the run into it
        r = pairs[vals[i]];
        for (long long j = i + 1; j < n_slots && keys[j] == key; ++j) {
            const PairRec o = pairs[vals[j]];
            const float d1 = o.ref1 - r.ref1, d2 = o.ref2 - r.ref2;
            const float dl[3] = { -(d1 + d2), d1, d2 };
            // moments of o about r's reference
            float A[3], M[6];
            for (int k = 0; k < 3; ++k) A[k] = fmaf(o.w, dl[k], o.A[k]);
            int q = 0;
            for (int k = 0; k < 3; ++k)
                for (int l = k; l < 3; ++l, ++q)
                    M[q] = o.M[q] + o.A[k] * dl[l] + dl[k] * o.A[l] + o.w * dl[k] * dl[l];
            r.w += o.w;
            for (int k = 0; k < 3; ++k) r.A[k] += A[k];
            for (int k = 0; k < 6; ++k) r.M[k] += M[k];
        }
    }
    merged[i] = r;
}

// ---------------------------------------------------------------------------
// Killing walks (Eq. 32, second term) carry no sample: their key is the exit face alone, and
// 256 consecutive ones rarely share a face.  They are reduced globally instead: sort the
// walks by exit face (stable: slot order inside a face), segmented-sum the six moments
// per face into M_face, and hand one pair record per face to level 2.
// ---------------------------------------------------------------------------
__global__ void __launch_bounds__(AT)
kill_keys_kernel(const float4* __restrict__ records, long long j0, long long n, uint32_t invalid_key,
                 uint32_t* __restrict__ keys, uint32_t* __restrict__ vals)
{
    const long long i = (long long)blockIdx.x * AT + threadIdx.x;
    if (i >= n) return;
    const float4 rec = records[j0 + i];
    const int tri_t = __float_as_int(rec.x);
    keys[i] = (tri_t >= 0 && rec.w != 0.0f) ? (uint32_t)tri_t : invalid_key;
    vals[i] = (uint32_t)i;
}

__global__ void __launch_bounds__(RT)
kill_reduce_kernel(const float4* __restrict__ records, long long j0, const uint32_t* __restrict__ keys,
                   const uint32_t* __restrict__ vals, long long n, uint32_t invalid_key,
                   float* __restrict__ mface, uint32_t* __restrict__ carry_key, float* __restrict__ carry_sum)
{
    __shared__ float s_tail[RT / 32][6];
    __shared__ int s_has_head[RT / 32];
    const long long i = (long long)blockIdx.x * RT + threadIdx.x;
    const uint32_t key = i < n ? keys[i] : invalid_key;
    const bool valid = key != invalid_key;                       // invalid keys sort last
    const bool head = valid && (i == 0 || keys[i - 1] != key);
    const bool last = valid && (threadIdx.x == RT - 1 || i + 1 >= n || keys[i + 1] != key);
    float v[6] = { 0.f, 0.f, 0.f, 0.f, 0.f, 0.f };
    if (valid) {
        const float4 rec = records[j0 + vals[i]];
        const float b1 = rec.y, b2 = rec.z, b0 = 1.0f - b1 - b2;
        const float w0 = rec.w * b0, w1 = rec.w * b1, w2 = rec.w * b2;
        v[0] = w0 * b0; v[1] = w0 * b1; v[2] = w0 * b2; v[3] = w1 * b1; v[4] = w1 * b2; v[5] = w2 * b2;
    }
    const bool headed = block_segmented_scan<6, RT / 32>(v, head || !valid, s_tail, s_has_head);
    if (threadIdx.x == 0) carry_key[blockIdx.x] = 0xFFFFFFFFu;
    __syncthreads();
    if (last) {
        if (headed) { for (int q = 0; q < 6; ++q) mface[6 * (long long)key + q] += v[q]; }
        else { carry_key[blockIdx.x] = key; for (int q = 0; q < 6; ++q) carry_sum[6 * (long long)blockIdx.x + q] = v[q]; }
    }
}

__global__ void __launch_bounds__(AT)
kill_carry_fixup_kernel(const uint32_t* __restrict__ carry_key, const float* __restrict__ carry_sum, long long n_tiles,
                        float* __restrict__ mface)
{
    const long long b = (long long)blockIdx.x * AT + threadIdx.x;
    if (b >= n_tiles) return;
    const uint32_t key = carry_key[b];
    if (key == 0xFFFFFFFFu) return;
    if (b > 0 && carry_key[b - 1] == key) return;
    float total[6];
    for (int q = 0; q < 6; ++q) total[q] = carry_sum[6 * b + q];
    for (long long j = b + 1; j < n_tiles && carry_key[j] == key; ++j)
        for (int q = 0; q < 6; ++q) total[q] += carry_sum[6 * j + q];
    for (int q = 0; q < 6; ++q) mface[6 * (long long)key + q] += total[q];
}

// faces [f0, f0 + n) -> pair records (sample = -1); a face no killing walk reached gets tri_t = -1
__global__ void __launch_bounds__(AT)
kill_pairs_kernel(const float* __restrict__ mface, long long f0, long long n, long long n_slots,
                  PairRec* __restrict__ pairs, uint32_t* __restrict__ pair_counts)
{
    const long long i = (long long)blockIdx.x * AT + threadIdx.x;
    if (i >= n_slots) return;
    PairRec r;
    r.sample = -1; r.tri_t = -1; r.w = 0.0f; r.A[0] = r.A[1] = r.A[2] = 0.0f;
    r.ref1 = r.ref2 = 0.0f; r.pad_[0] = r.pad_[1] = 0.0f;
    bool any = false;
    for (int q = 0; q < 6; ++q) { r.M[q] = i < n ? mface[6 * (f0 + i) + q] : 0.0f; any = any || r.M[q] != 0.0f; }
    if (any) r.tri_t = (int)(f0 + i);
    pairs[i] = r;
    if (i % CH == 0) pair_counts[i / CH] = CH;
}

// ---------------------------------------------------------------------------
// Level 2: pair record -> upper-triangular entries.
// The merged vertex list holds the (<= 3) vertices of the sample's face and the
// (<= 3) vertices of the exit face, shared vertices once.
// ---------------------------------------------------------------------------
struct PairBlock {
    int   idx[6];
    float bs[6];          // b_v(s)
    float ds[6];          // D_v = b_v(s) - r_v(t): the pair's d at the reference exit point
    float At[6];          // sum wgt eta_v(t)
    int   tmask[6];       // corners of the exit face that are this vertex (bit k)
    int   m;
};

__device__ __forceinline__ int pair_block_slot(PairBlock& B, int vtx)
{
    for (int q = 0; q < B.m; ++q) if (B.idx[q] == vtx) return q;
    B.idx[B.m] = vtx; B.bs[B.m] = 0.0f; B.ds[B.m] = 0.0f; B.At[B.m] = 0.0f; B.tmask[B.m] = 0;
    return B.m++;
}

__device__ __forceinline__ void build_pair_block(const AccArgs& a, const PairRec& r, PairBlock& B)
{
    B.m = 0;
    if (r.sample >= 0) {
        const long long fs = a.s_tri[r.sample];
        for (int k = 0; k < 3; ++k) {
            const int q = pair_block_slot(B, a.faces[3 * fs + k]);
            const float bk = a.s_bary[3 * (long long)r.sample + k];
            B.bs[q] += bk; B.ds[q] += bk;
        }
    }
    const long long ft = r.tri_t;
    const bool killing = r.sample < 0;
    const float rb[3] = { killing ? 0.0f : 1.0f - r.ref1 - r.ref2, r.ref1, r.ref2 };
    for (int k = 0; k < 3; ++k) {
        const int q = pair_block_slot(B, a.faces[3 * ft + k]);
        B.ds[q] -= rb[k];
        B.At[q] += r.A[k];
        B.tmask[q] |= 1 << k;
    }
}

__device__ __forceinline__ float moment(const PairRec& r, int k, int l)
{
    if (k > l) { const int t = k; k = l; l = t; }
    return r.M[k == 0 ? l : (k == 1 ? 2 + l : 5)];
}

// sum wgt b_p(t) b_q(t) for merged vertices p, q
__device__ __forceinline__ float moment_block(const PairRec& r, int maskp, int maskq)
{
    float e = 0.0f;
    for (int k = 0; k < 3; ++k)
        if (maskp & (1 << k))
            for (int l = 0; l < 3; ++l)
                if (maskq & (1 << l)) e += moment(r, k, l);
    return e;
}

__global__ void __launch_bounds__(AT)
count_entries_kernel(AccArgs a, const PairRec* __restrict__ pairs, const uint32_t* __restrict__ pair_counts,
                     long long n_slots, uint32_t* __restrict__ counts)
{
    const long long i = (long long)blockIdx.x * AT + threadIdx.x;
    if (i >= n_slots) return;
    uint32_t c = 0;
    if ((uint32_t)(i % CH) < pair_counts[i / CH] && pairs[i].tri_t >= 0) {
        PairBlock B;
        build_pair_block(a, pairs[i], B);
        for (int p = 0; p < B.m; ++p) for (int q = 0; q < B.m; ++q) c += (B.idx[p] <= B.idx[q]) ? 1u : 0u;
    }
    counts[i] = c;
}

template <typename KeyT>
__global__ void __launch_bounds__(AT)
expand_entries_kernel(AccArgs a, const PairRec* __restrict__ pairs, const uint32_t* __restrict__ pair_counts,
                      long long n_slots, const uint32_t* __restrict__ offsets,
                      KeyT* __restrict__ keys, uint32_t* __restrict__ vals)
{
    const long long i = (long long)blockIdx.x * AT + threadIdx.x;
    if (i >= n_slots) return;
    if ((uint32_t)(i % CH) >= pair_counts[i / CH]) return;
    const PairRec r = pairs[i];
    if (r.tri_t < 0) return;
    PairBlock B;
    build_pair_block(a, r, B);
    uint32_t o = offsets[i];
    for (int p = 0; p < B.m; ++p)
        for (int q = 0; q < B.m; ++q)
            if (B.idx[p] <= B.idx[q]) {
                // sum over the pair's walks of wgt * d_p d_q,  d = b(s) - b(t) = D - eta
                float e;
                if (a.naive) {
                    // Alg. 1: sum wgt (1/2)(b_s,p d_q + b_s,q d_p),  sum wgt d = w D - A
                    e = 0.5f * (B.bs[p] * (r.w * B.ds[q] - B.At[q]) + B.bs[q] * (r.w * B.ds[p] - B.At[p]));
                } else {
                    e = r.w * B.ds[p] * B.ds[q] - B.ds[p] * B.At[q] - B.At[p] * B.ds[q];
                    if (B.tmask[p] && B.tmask[q]) e += moment_block(r, B.tmask[p], B.tmask[q]);
                }
                keys[o] = (KeyT)((long long)B.idx[p] * a.K + B.idx[q]);
                vals[o] = __float_as_uint(e);
                ++o;
            }
}

// ---------------------------------------------------------------------------
// Run sums of the sorted entries.  A run whose head lies in this tile is added to the
// matrix by its last thread in the tile; the leading part of a run that began in an
// earlier tile goes to carry[tile] and is added by carry_fixup_kernel in tile order.
// ---------------------------------------------------------------------------
__global__ void __launch_bounds__(RT)
reduce_runs_dense_kernel(const uint32_t* __restrict__ keys, const uint32_t* __restrict__ vals, long long n,
                         float* __restrict__ S, uint32_t* __restrict__ carry_key, float* __restrict__ carry_sum,
                         unsigned long long* __restrict__ n_unique, const uint32_t* __restrict__ n_dev)
{
    __shared__ float s_tail[RT / 32][1];
    __shared__ int s_has_head[RT / 32];
    if (n_dev) {                                        // length known on the device only: the grid covers the capacity
        n = (long long)*n_dev;
        if ((long long)blockIdx.x * RT >= n) { if (threadIdx.x == 0) carry_key[blockIdx.x] = 0xFFFFFFFFu; return; }
    }
    const long long i = (long long)blockIdx.x * RT + threadIdx.x;
    const bool valid = i < n;
    const uint32_t key = valid ? keys[i] : 0xFFFFFFFFu;
    const bool head = valid && (i == 0 || keys[i - 1] != key);
    const bool last = valid && (threadIdx.x == RT - 1 || i + 1 >= n || keys[i + 1] != key);
    float v[1] = { valid ? __uint_as_float(vals[i]) : 0.0f };
    const bool headed = block_segmented_scan<1, RT / 32>(v, head || !valid, s_tail, s_has_head);
    if (threadIdx.x == 0) carry_key[blockIdx.x] = 0xFFFFFFFFu;
    __syncthreads();
    if (last) {
        if (headed) S[key] += v[0];
        else { carry_key[blockIdx.x] = key; carry_sum[blockIdx.x] = v[0]; }
    }
    const unsigned m = __ballot_sync(0xFFFFFFFFu, head);
    if (n_unique && (threadIdx.x & 31) == 0 && m) atomicAdd(n_unique, (unsigned long long)__popc(m));
}

__global__ void add_count_kernel(unsigned long long* __restrict__ total, const uint32_t* __restrict__ n) { *total += *n; }

__global__ void __launch_bounds__(AT)
carry_fixup_kernel(const uint32_t* __restrict__ carry_key, const float* __restrict__ carry_sum, long long n_tiles,
                   float* __restrict__ S)
{
    const long long b = (long long)blockIdx.x * AT + threadIdx.x;
    if (b >= n_tiles) return;
    const uint32_t key = carry_key[b];
    if (key == 0xFFFFFFFFu) return;
    if (b > 0 && carry_key[b - 1] == key) return;                        // not the first carry of this run
    float total = carry_sum[b];
    for (long long j = b + 1; j < n_tiles && carry_key[j] == key; ++j) total += carry_sum[j];
    S[key] += total;
}

// ---------------------------------------------------------------------------
// Sparse output (output_kind 1): the same run sums, written compactly.  Pass 1 counts the
// run heads of every tile; after an exclusive scan a run's output slot is
// (heads before its tile) + (heads in the tile up to its own) - 1.
// ---------------------------------------------------------------------------
__global__ void __launch_bounds__(RT)
count_heads_kernel(const unsigned long long* __restrict__ keys, long long n, uint32_t* __restrict__ tile_heads)
{
    __shared__ int s_cnt[RT / 32];
    const long long i = (long long)blockIdx.x * RT + threadIdx.x;
    const bool head = i < n && (i == 0 || keys[i - 1] != keys[i]);
    const unsigned m = __ballot_sync(0xFFFFFFFFu, head);
    if ((threadIdx.x & 31) == 0) s_cnt[threadIdx.x >> 5] = __popc(m);
    __syncthreads();
    if (threadIdx.x == 0) {
        int t = 0;
        for (int w = 0; w < RT / 32; ++w) t += s_cnt[w];
        tile_heads[blockIdx.x] = (uint32_t)t;
    }
}

__global__ void __launch_bounds__(RT)
reduce_runs_compact_kernel(const unsigned long long* __restrict__ keys, const uint32_t* __restrict__ vals, long long n,
                           const uint32_t* __restrict__ tile_offset,
                           unsigned long long* __restrict__ out_keys, float* __restrict__ out_vals,
                           unsigned long long* __restrict__ carry_key, float* __restrict__ carry_sum)
{
    __shared__ float s_tail[RT / 32][1];
    __shared__ int s_has_head[RT / 32];
    __shared__ int s_cnt[RT / 32];
    const long long i = (long long)blockIdx.x * RT + threadIdx.x;
    const bool valid = i < n;
    const unsigned long long key = valid ? keys[i] : ~0ull;
    const bool head = valid && (i == 0 || keys[i - 1] != key);
    const bool last = valid && (threadIdx.x == RT - 1 || i + 1 >= n || keys[i + 1] != key);
    float v[1] = { valid ? __uint_as_float(vals[i]) : 0.0f };
    const bool headed = block_segmented_scan<1, RT / 32>(v, head || !valid, s_tail, s_has_head);
    const unsigned m = __ballot_sync(0xFFFFFFFFu, head);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (lane == 0) s_cnt[warp] = __popc(m);
    if (threadIdx.x == 0) carry_key[blockIdx.x] = ~0ull;
    __syncthreads();
    if (last) {
        if (headed) {
            int heads_upto = __popc(m & (0xFFFFFFFFu >> (31 - lane)));           // heads at or before me: my run's head is the last
            for (int w = 0; w < warp; ++w) heads_upto += s_cnt[w];
            const long long slot = (long long)tile_offset[blockIdx.x] + heads_upto - 1;
            out_keys[slot] = key; out_vals[slot] = v[0];
        } else {
            carry_key[blockIdx.x] = key; carry_sum[blockIdx.x] = v[0];
        }
    }
}

// Leading parts of runs that began in an earlier tile, added in tile order.  The run's slot is
// the last one opened before the tile: tile_offset[tile] - 1.
__global__ void __launch_bounds__(AT)
carry_fixup_compact_kernel(const unsigned long long* __restrict__ carry_key, const float* __restrict__ carry_sum,
                           long long n_tiles, const uint32_t* __restrict__ tile_offset, float* __restrict__ out_vals)
{
    const long long b = (long long)blockIdx.x * AT + threadIdx.x;
    if (b >= n_tiles) return;
    const unsigned long long key = carry_key[b];
    if (key == ~0ull) return;
    if (b > 0 && carry_key[b - 1] == key) return;
    float total = carry_sum[b];
    for (long long j = b + 1; j < n_tiles && carry_key[j] == key; ++j) total += carry_sum[j];
    out_vals[(long long)tile_offset[b] - 1] += total;
}

__global__ void __launch_bounds__(AT)
coo_write_kernel(const unsigned long long* __restrict__ keys, const float* __restrict__ vals, long long n, long long K,
                 int32_t* __restrict__ row, int32_t* __restrict__ col, float* __restrict__ val)
{
    const long long i = (long long)blockIdx.x * AT + threadIdx.x;
    if (i >= n) return;
    const unsigned long long k = keys[i];
    row[i] = (int32_t)(k / (unsigned long long)K);
    col[i] = (int32_t)(k % (unsigned long long)K);
    val[i] = vals[i];
}

__global__ void __launch_bounds__(AT)
mirror_kernel(float* __restrict__ S, long long K)
{
    const long long i = (long long)blockIdx.x * AT + threadIdx.x;
    if (i >= K * K) return;
    const long long row = i / K, col = i - row * K;
    if (row > col) S[i] = S[col * K + row];
}

int key_bits_for(long long K)
{
    unsigned long long m = (unsigned long long)K * (unsigned long long)K - 1ull;
    int bits = 0;
    while (m) { ++bits; m >>= 1; }
    return bits < 1 ? 1 : bits;
}

int bits_for_count(unsigned long long m)     // bits needed for values 0..m
{
    int bits = 0;
    while (m) { ++bits; m >>= 1; }
    return bits < 1 ? 1 : bits;
}

// slots per chunk: walks of one chunk, or faces of one chunk of the killing pass
int64_t chunk_slots(int64_t n_records, int64_t F, int64_t max_walks = MAX_CHUNK_WALKS)
{
    int64_t c = n_records < max_walks ? n_records : max_walks;
    const int64_t f = F < max_walks ? F : max_walks;
    if (f > c) c = f;
    return c < 1 ? 1 : c;
}

// Killing records [n_main, n_main + n_kill) -> mface[F][6], in pieces of at most `cap` walks.
int kill_prereduce(const float4* records, long long n_main, long long n_kill, long long F, float* mface,
                   uint32_t* keys, uint32_t* vals, long long cap, uint32_t* carry_key, float* carry_sum6,
                   void* sort_ws, size_t sort_bytes, cudaStream_t st)
{
    MCS_CUDA_TRY(cudaMemsetAsync(mface, 0, (size_t)F * 6 * sizeof(float), st));
    const uint32_t invalid = (uint32_t)F;
    const int bits = bits_for_count((unsigned long long)F);
    for (long long k0 = 0; k0 < n_kill; k0 += cap) {
        const long long n = (n_kill - k0) < cap ? (n_kill - k0) : cap;
        mcs_note_launch(), kill_keys_kernel<<<(unsigned)ceil_div64(n, AT), AT, 0, st>>>(records, n_main + k0, n, invalid, keys, vals);
        int rc = sort_pairs_u32(keys, vals, n, bits, sort_ws, sort_bytes, st);
        if (rc != MCS_OK) return rc;
        const long long n_tiles = ceil_div64(n, RT);
        mcs_note_launch(), kill_reduce_kernel<<<(unsigned)n_tiles, RT, 0, st>>>(records, n_main + k0, keys, vals, n, invalid,
                                                                               mface, carry_key, carry_sum6);
        mcs_note_launch(), kill_carry_fixup_kernel<<<(unsigned)ceil_div64(n_tiles, AT), AT, 0, st>>>(carry_key, carry_sum6, n_tiles, mface);
    }
    MCS_CUDA_TRY(cudaGetLastError());
    return MCS_OK;
}

// Level 1b on the host side: sort the chunk's pair records by (sample, exit face) and fold the runs (see pair_merge_kernel).
// key_buf / val_buf: scratch for n_slots 64-bit keys and 32-bit indices (the entry buffers, not in use yet).
int merge_pairs(const PairRec* pairs, const uint32_t* pair_counts, long long n_slots, long long first_sample, long long n_samples,
                long long F, unsigned long long* key_buf, uint32_t* val_buf, void* sort_ws, size_t sort_bytes,
                PairRec* merged, uint32_t* merged_counts, cudaStream_t st)
{
    const int face_bits = bits_for_count((unsigned long long)F);
    const int bits = face_bits + bits_for_count((unsigned long long)n_samples) + 1;    // + 1: the invalid key
    const unsigned nblk = (unsigned)ceil_div64(n_slots, AT);
    mcs_note_launch(), pair_keys_kernel<<<nblk, AT, 0, st>>>(pairs, pair_counts, n_slots, first_sample, face_bits, key_buf, val_buf);
    int rc = sort_pairs_u64((uint64_t*)key_buf, val_buf, n_slots, bits > 63 ? 63 : bits, sort_ws, sort_bytes, st);
    if (rc != MCS_OK) return rc;
    mcs_note_launch(), pair_merge_kernel<<<nblk, AT, 0, st>>>(pairs, key_buf, val_buf, n_slots, merged, merged_counts);
    return MCS_OK;
}

struct AccLayout {
    size_t pairs, pairs2, pair_counts, pair_counts2, counts, keys, vals, carry_key, carry_sum, mface, scan, sort, total;
    int64_t C, E, n_blocks, n_tiles;
};

AccLayout acc_layout(int64_t n_records, int64_t F)
{
    AccLayout L;
    L.C = chunk_slots(n_records, F);
    L.n_blocks = ceil_div64(L.C, CH);
    const int64_t slots = L.n_blocks * CH;
    L.E = slots * MAX_ENTRIES_PER_PAIR;
    L.n_tiles = ceil_div64(L.E, RT);
    size_t off = 0;
    L.pairs = off;       off += align_up((size_t)slots * sizeof(PairRec));
    L.pairs2 = off;      off += align_up((size_t)slots * sizeof(PairRec));
    L.pair_counts = off; off += align_up((size_t)L.n_blocks * 4);
    L.pair_counts2 = off; off += align_up((size_t)L.n_blocks * 4);
    L.counts = off;      off += align_up((size_t)(slots + 1) * 4);
    L.keys = off;        off += align_up((size_t)L.E * 4);
    L.vals = off;        off += align_up((size_t)L.E * 4);
    L.carry_key = off;   off += align_up((size_t)L.n_tiles * 4);
    L.carry_sum = off;   off += align_up((size_t)L.n_tiles * 24);
    L.mface = off;       off += align_up((size_t)F * 24);
    L.scan = off;        off += align_up(scan_workspace_bytes(slots) + 256);
    L.sort = off;        off += align_up(sort_workspace_bytes(L.E, 4));
    L.total = off + 1024;
    return L;
}

}  // namespace

size_t accumulate_workspace_bytes(const mcs_bvh* b, const mcs_basis* basis, int64_t n_records)
{
    (void)basis;
    return acc_layout(n_records, b->F).total;
}

int accumulate_run(const mcs_bvh* b, const mcs_samples* s, const mcs_basis* basis, int W, int naive,
                   const float4* records, int64_t n_records, void* ws, size_t ws_bytes,
                   const mcs_matrix* out, unsigned long long* stats_dev, cudaStream_t st)
{
    if (!b || !s || !basis || !out || !records || n_records < 0) return MCS_EINVAL;
    if (basis->kind != 0 || basis->K != b->V) return MCS_EINVAL;
    if (out->kind != 0 || out->K != basis->K || !out->dense) return MCS_EINVAL;
    const long long K = basis->K;
    if (K > 65535) return MCS_EINVAL;                 // dense keys are 32-bit (row*K + col)
    const AccLayout L = acc_layout(n_records, b->F);
    if (!ws || ws_bytes < L.total) return MCS_ENOMEM;

    char* base = (char*)ws;
    PairRec* pairs = (PairRec*)(base + L.pairs);
    PairRec* pairs2 = (PairRec*)(base + L.pairs2);
    uint32_t* pair_counts = (uint32_t*)(base + L.pair_counts);
    uint32_t* pair_counts2 = (uint32_t*)(base + L.pair_counts2);
    uint32_t* counts = (uint32_t*)(base + L.counts);
    uint32_t* keys = (uint32_t*)(base + L.keys);
    uint32_t* vals = (uint32_t*)(base + L.vals);
    uint32_t* carry_key = (uint32_t*)(base + L.carry_key);
    float* carry_sum = (float*)(base + L.carry_sum);
    float* mface = (float*)(base + L.mface);
    void* scan_ws = base + L.scan;
    void* sort_ws = base + L.sort;
    const size_t scan_bytes = L.sort - L.scan, sort_bytes = L.total - L.sort;

    AccArgs a;
    a.records = records; a.faces = b->faces; a.s_tri = s->tri; a.s_bary = s->bary;
    a.n_main = (long long)s->n_s * W; a.W = W; a.naive = naive; a.K = K;
    const int bits = key_bits_for(K);
    const long long n_main = a.n_main < n_records ? a.n_main : n_records, n_kill = n_records - n_main;

    MCS_CUDA_TRY(cudaMemsetAsync(out->dense, 0, (size_t)K * K * sizeof(float), st));
    if (n_kill > 0) {
        int rc = kill_prereduce(records, n_main, n_kill, b->F, mface, keys, vals, L.E, carry_key, carry_sum, sort_ws, sort_bytes, st);
        if (rc != MCS_OK) return rc;
    }
    if (stats_dev) MCS_CUDA_TRY(cudaMemsetAsync(stats_dev + ST_ENTRIES, 0, 8, st));
    // phase 0: the walks of the samples, chunk by chunk; phase 1: one pair record per face from the killing walks
    for (int phase = 0; phase < 2; ++phase)
    for (int64_t j0 = 0, total = phase == 0 ? n_main : (n_kill > 0 ? b->F : 0); j0 < total; j0 += L.C) {
        const long long n = (total - j0) < L.C ? (total - j0) : L.C;
        const long long nblk1 = ceil_div64(n, CH), slots = nblk1 * CH;
        const PairRec* pp = pairs; const uint32_t* pc = pair_counts;
        if (phase == 0) {
            mcs_note_launch(), pair_reduce_kernel<<<(unsigned)nblk1, CH, 0, st>>>(a, j0, n, pairs, pair_counts);
            if (a.W > CH) {                            // a sample spans several level-1 blocks: fold its repeated pairs (level 1b)
                int rcm = merge_pairs(pairs, pair_counts, slots, j0 / a.W, n / a.W + 2, b->F, (unsigned long long*)keys, vals,
                                      sort_ws, sort_bytes, pairs2, pair_counts2, st);
                if (rcm != MCS_OK) return rcm;
                pp = pairs2; pc = pair_counts2;
            }
        } else mcs_note_launch(), kill_pairs_kernel<<<(unsigned)ceil_div64(slots, AT), AT, 0, st>>>(mface, j0, n, slots, pairs, pair_counts);
        const unsigned nblk = (unsigned)ceil_div64(slots, AT);
        mcs_note_launch(), count_entries_kernel<<<nblk, AT, 0, st>>>(a, pp, pc, slots, counts);
        int rc = exclusive_scan_u32(counts, counts, slots, counts + slots, scan_ws, scan_bytes, st);
        if (rc != MCS_OK) return rc;
        // The number of entries of the chunk stays on the device (counts[slots]): the sort and the run reduction take
        // it from there and their grids cover the chunk's capacity (tiles beyond the length exit at once), so the loop
        // never blocks the host and a call can be captured in a CUDA graph.
        const uint32_t* n_entries_dev = counts + slots;
        const long long cap = slots * MAX_ENTRIES_PER_PAIR;
        if (stats_dev) mcs_note_launch(), add_count_kernel<<<1, 1, 0, st>>>(stats_dev + ST_ENTRIES, n_entries_dev);
        mcs_note_launch(), expand_entries_kernel<uint32_t><<<nblk, AT, 0, st>>>(a, pp, pc, slots, counts, keys, vals);
        rc = sort_pairs_u32_devn(keys, vals, cap, n_entries_dev, bits, sort_ws, sort_bytes, st);
        if (rc != MCS_OK) return rc;
        const long long n_tiles = ceil_div64(cap, RT);
        mcs_note_launch(), reduce_runs_dense_kernel<<<(unsigned)n_tiles, RT, 0, st>>>(
            keys, vals, 0, out->dense, carry_key, carry_sum, stats_dev ? stats_dev + ST_UNIQUE : nullptr, n_entries_dev);
        mcs_note_launch(), carry_fixup_kernel<<<(unsigned)ceil_div64(n_tiles, AT), AT, 0, st>>>(carry_key, carry_sum, n_tiles, out->dense);
    }
    mcs_note_launch(), mirror_kernel<<<(unsigned)ceil_div64(K * K, AT), AT, 0, st>>>(out->dense, K);
    MCS_CUDA_TRY(cudaGetLastError());
    return MCS_OK;
}

// ---------------------------------------------------------------------------
// Sparse (COO) accumulation, any K < 2^31: 64-bit keys.  The list of unique entries found
// so far sits at the front of the key buffer; every chunk appends its entries behind it,
// the whole is stable-sorted and reduced into the other buffer.  The running list comes
// first in the buffer, so the order of every sum is fixed.
// ---------------------------------------------------------------------------
namespace {

// ---------------------------------------------------------------------------
// Stable merge of two sorted (key, value) lists, A before B on equal keys: out = the sequence a stable sort of the
// concatenation A | B would give.  The running list of unique entries (A) is already sorted, so only a chunk's new
// entries (B) go through the radix sort and one merge pass replaces five radix passes over the running list.
// Merge path: a block finds where its tile of MG_TILE outputs starts and ends in A and B (two binary searches in global
// memory), stages both pieces in shared memory, every thread finds its own start (binary search in shared memory) and
// merges MG_V outputs; the tile leaves through shared memory, coalesced.
// ---------------------------------------------------------------------------
constexpr int MG_T = 256, MG_V = 7, MG_TILE = MG_T * MG_V;

template <typename Ptr>
__device__ __forceinline__ long long merge_path_split(Ptr A, long long na, Ptr B, long long nb, long long diag)
{
    long long lo = diag > nb ? diag - nb : 0, hi = diag < na ? diag : na;
    while (lo < hi) {
        const long long mid = (lo + hi) >> 1;
        if (A[mid] <= B[diag - 1 - mid]) lo = mid + 1; else hi = mid;      // A[mid] precedes B[diag-1-mid] (ties: A first)
    }
    return lo;                                                           // elements of A among the first `diag` outputs
}

__global__ void __launch_bounds__(MG_T)
merge_sorted_kernel(const unsigned long long* __restrict__ ka, const uint32_t* __restrict__ va, long long na,
                    const unsigned long long* __restrict__ kb, const uint32_t* __restrict__ vb, long long nb,
                    unsigned long long* __restrict__ ko, uint32_t* __restrict__ vo)
{
    __shared__ unsigned long long s_k[MG_TILE], s_ok[MG_TILE];
    __shared__ uint32_t s_v[MG_TILE], s_ov[MG_TILE];
    __shared__ long long s_split[2];
    const long long n = na + nb;
    const long long d0 = (long long)blockIdx.x * MG_TILE;
    const long long d1 = d0 + MG_TILE < n ? d0 + MG_TILE : n;
    if (threadIdx.x < 2) s_split[threadIdx.x] = merge_path_split(ka, na, kb, nb, threadIdx.x == 0 ? d0 : d1);
    __syncthreads();
    const long long a0 = s_split[0], a1 = s_split[1], b0 = d0 - a0, b1 = d1 - a1;
    const int ca = (int)(a1 - a0), cb = (int)(b1 - b0);
    for (int i = threadIdx.x; i < ca; i += MG_T) { s_k[i] = ka[a0 + i]; s_v[i] = va[a0 + i]; }
    for (int i = threadIdx.x; i < cb; i += MG_T) { s_k[ca + i] = kb[b0 + i]; s_v[ca + i] = vb[b0 + i]; }
    __syncthreads();
    const unsigned long long* A = s_k;
    const unsigned long long* B = s_k + ca;
    const int total = ca + cb;
    int diag = threadIdx.x * MG_V;
    if (diag > total) diag = total;
    int ia = (int)merge_path_split(A, (long long)ca, B, (long long)cb, (long long)diag);
    int ib = diag - ia;
#pragma unroll
    for (int i = 0; i < MG_V; ++i) {
        const int o = diag + i;
        if (o < total) {
            const bool take_a = ib >= cb || (ia < ca && A[ia] <= B[ib]);
            const int src = take_a ? ia : ca + ib;
            s_ok[o] = s_k[src]; s_ov[o] = s_v[src];
            ia += take_a ? 1 : 0; ib += take_a ? 0 : 1;
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < total; i += MG_T) { ko[d0 + i] = s_ok[i]; vo[d0 + i] = s_ov[i]; }
}

struct CooLayout {
    size_t pairs, pairs2, pair_counts, pair_counts2, counts, keys[2], vals[2], tile_heads, carry_key, carry_sum, mface, scan, sort, total;
    int64_t C, E, cap, n_blocks, n_tiles;
};

CooLayout coo_layout(int64_t n_records, int64_t coo_capacity, int64_t F)
{
    CooLayout L;
    L.C = chunk_slots(n_records, F, MAX_CHUNK_WALKS_COO);
    L.n_blocks = ceil_div64(L.C, CH);
    const int64_t slots = L.n_blocks * CH;
    L.E = slots * MAX_ENTRIES_PER_PAIR;
    L.cap = L.E + (coo_capacity > 0 ? coo_capacity : 0);
    L.n_tiles = ceil_div64(L.cap, RT);
    size_t off = 0;
    L.pairs = off;       off += align_up((size_t)slots * sizeof(PairRec));
    L.pairs2 = off;      off += align_up((size_t)slots * sizeof(PairRec));
    L.pair_counts = off; off += align_up((size_t)L.n_blocks * 4);
    L.pair_counts2 = off; off += align_up((size_t)L.n_blocks * 4);
    L.counts = off;      off += align_up((size_t)(slots + 1) * 4);
    for (int q = 0; q < 2; ++q) {
        L.keys[q] = off; off += align_up((size_t)L.cap * 8);
        L.vals[q] = off; off += align_up((size_t)L.cap * 4);
    }
    L.tile_heads = off;  off += align_up((size_t)(L.n_tiles + 1) * 4);
    L.carry_key = off;   off += align_up((size_t)L.n_tiles * 8);
    L.carry_sum = off;   off += align_up((size_t)L.n_tiles * 24);
    L.mface = off;       off += align_up((size_t)F * 24);
    const int64_t scan_n = slots > L.n_tiles ? slots : L.n_tiles;
    L.scan = off;        off += align_up(scan_workspace_bytes(scan_n) + 256);
    L.sort = off;        off += align_up(sort_workspace_bytes(L.cap, 8));
    L.total = off + 1024;
    return L;
}

int key_bits_for64(long long K)
{
    unsigned long long m = (unsigned long long)K * (unsigned long long)K - 1ull;
    int bits = 0;
    while (m) { ++bits; m >>= 1; }
    return bits < 1 ? 1 : bits;
}

}  // namespace

size_t accumulate_coo_workspace_bytes(const mcs_bvh* b, int64_t n_records, int64_t coo_capacity)
{
    return coo_layout(n_records, coo_capacity, b->F).total;
}

int accumulate_coo_run(const mcs_bvh* b, const mcs_samples* s, const mcs_basis* basis, int W, int naive,
                       const float4* records, int64_t n_records, void* ws, size_t ws_bytes,
                       const mcs_matrix* out, unsigned long long* stats_dev, cudaStream_t st)
{
    if (!b || !s || !basis || !out || !records || n_records < 0) return MCS_EINVAL;
    if (basis->kind != 0 || basis->K != b->V) return MCS_EINVAL;
    if (out->kind != 1 || out->K != basis->K || out->coo_capacity < 1) return MCS_EINVAL;
    if (!out->coo_row || !out->coo_col || !out->coo_val || !out->coo_nnz) return MCS_EINVAL;
    const long long K = basis->K;
    const CooLayout L = coo_layout(n_records, out->coo_capacity, b->F);
    if (!ws || ws_bytes < L.total) return MCS_ENOMEM;
    if (L.cap >= ((int64_t)1 << 32)) return MCS_EINVAL;

    char* base = (char*)ws;
    PairRec* pairs = (PairRec*)(base + L.pairs);
    PairRec* pairs2 = (PairRec*)(base + L.pairs2);
    uint32_t* pair_counts = (uint32_t*)(base + L.pair_counts);
    uint32_t* pair_counts2 = (uint32_t*)(base + L.pair_counts2);
    uint32_t* counts = (uint32_t*)(base + L.counts);
    unsigned long long* keys[2] = { (unsigned long long*)(base + L.keys[0]), (unsigned long long*)(base + L.keys[1]) };
    uint32_t* vals[2] = { (uint32_t*)(base + L.vals[0]), (uint32_t*)(base + L.vals[1]) };
    uint32_t* tile_heads = (uint32_t*)(base + L.tile_heads);
    unsigned long long* carry_key = (unsigned long long*)(base + L.carry_key);
    float* carry_sum = (float*)(base + L.carry_sum);
    void* scan_ws = base + L.scan;
    void* sort_ws = base + L.sort;
    const size_t scan_bytes = L.sort - L.scan, sort_bytes = L.total - L.sort;

    AccArgs a;
    a.records = records; a.faces = b->faces; a.s_tri = s->tri; a.s_bary = s->bary;
    a.n_main = (long long)s->n_s * W; a.W = W; a.naive = naive; a.K = K;
    const int bits = key_bits_for64(K);

    float* mface = (float*)(base + L.mface);
    const long long n_main = a.n_main < n_records ? a.n_main : n_records, n_kill = n_records - n_main;
    if (n_kill > 0) {
        int rc = kill_prereduce(records, n_main, n_kill, b->F, mface, (uint32_t*)keys[0], vals[0], L.cap,
                                (uint32_t*)carry_key, carry_sum, sort_ws, sort_bytes, st);
        if (rc != MCS_OK) return rc;
    }
    unsigned long long entries_total = 0;
    long long n_u = 0;
    int cur = 0;
    for (int phase = 0; phase < 2; ++phase)
    for (int64_t j0 = 0, total = phase == 0 ? n_main : (n_kill > 0 ? b->F : 0); j0 < total; j0 += L.C) {
        const long long n = (total - j0) < L.C ? (total - j0) : L.C;
        const long long nblk1 = ceil_div64(n, CH), slots = nblk1 * CH;
        const PairRec* pp = pairs; const uint32_t* pc = pair_counts;
        if (phase == 0) {
            mcs_note_launch(), pair_reduce_kernel<<<(unsigned)nblk1, CH, 0, st>>>(a, j0, n, pairs, pair_counts);
            if (a.W > CH) {                            // level 1b: fold the pairs a sample repeats over its level-1 blocks
                int rcm = merge_pairs(pairs, pair_counts, slots, j0 / a.W, n / a.W + 2, b->F, keys[cur] + n_u, vals[cur] + n_u,
                                      sort_ws, sort_bytes, pairs2, pair_counts2, st);
                if (rcm != MCS_OK) return rcm;
                pp = pairs2; pc = pair_counts2;
            }
        } else mcs_note_launch(), kill_pairs_kernel<<<(unsigned)ceil_div64(slots, AT), AT, 0, st>>>(mface, j0, n, slots, pairs, pair_counts);
        const unsigned nblk = (unsigned)ceil_div64(slots, AT);
        mcs_note_launch(), count_entries_kernel<<<nblk, AT, 0, st>>>(a, pp, pc, slots, counts);
        int rc = exclusive_scan_u32(counts, counts, slots, counts + slots, scan_ws, scan_bytes, st);
        if (rc != MCS_OK) return rc;
        uint32_t n_entries = 0;
        MCS_CUDA_TRY(cudaMemcpyAsync(&n_entries, counts + slots, 4, cudaMemcpyDeviceToHost, st));
        MCS_CUDA_TRY(cudaStreamSynchronize(st));
        if (n_entries == 0) continue;
        entries_total += n_entries;
        mcs_note_launch(), expand_entries_kernel<unsigned long long><<<nblk, AT, 0, st>>>(
            a, pp, pc, slots, counts, keys[cur] + n_u, vals[cur] + n_u);
        const long long n_tot = n_u + n_entries;
        // the chunk's new entries are sorted on their own; the running list (sorted, unique) joins by one stable merge
        // pass, running entry first on equal keys: the same sequence a stable sort of the whole would give
        rc = sort_pairs_u64((uint64_t*)(keys[cur] + n_u), vals[cur] + n_u, n_entries, bits, sort_ws, sort_bytes, st);
        if (rc != MCS_OK) return rc;
        int src = cur;                                // buffer that holds the sorted sequence
        if (n_u > 0) {
            mcs_note_launch(), merge_sorted_kernel<<<(unsigned)ceil_div64(n_tot, MG_TILE), MG_T, 0, st>>>(
                keys[cur], vals[cur], n_u, keys[cur] + n_u, vals[cur] + n_u, (long long)n_entries, keys[1 - cur], vals[1 - cur]);
            src = 1 - cur;
        }
        const long long n_tiles = ceil_div64(n_tot, RT);
        mcs_note_launch(), count_heads_kernel<<<(unsigned)n_tiles, RT, 0, st>>>(keys[src], n_tot, tile_heads);
        rc = exclusive_scan_u32(tile_heads, tile_heads, n_tiles, tile_heads + n_tiles, scan_ws, scan_bytes, st);
        if (rc != MCS_OK) return rc;
        uint32_t n_heads = 0;
        MCS_CUDA_TRY(cudaMemcpyAsync(&n_heads, tile_heads + n_tiles, 4, cudaMemcpyDeviceToHost, st));
        MCS_CUDA_TRY(cudaStreamSynchronize(st));
        if ((long long)n_heads > out->coo_capacity) {
            const long long need = n_heads;                                 // a lower bound on the final count
            MCS_CUDA_TRY(cudaMemcpyAsync(out->coo_nnz, &need, 8, cudaMemcpyHostToDevice, st));
            MCS_CUDA_TRY(cudaStreamSynchronize(st));
            return MCS_ENOMEM;
        }
        mcs_note_launch(), reduce_runs_compact_kernel<<<(unsigned)n_tiles, RT, 0, st>>>(
            keys[src], vals[src], n_tot, tile_heads, keys[1 - src], (float*)vals[1 - src], carry_key, carry_sum);
        mcs_note_launch(), carry_fixup_compact_kernel<<<(unsigned)ceil_div64(n_tiles, AT), AT, 0, st>>>(
            carry_key, carry_sum, n_tiles, tile_heads, (float*)vals[1 - src]);
        cur = 1 - src;
        n_u = n_heads;
    }
    if (n_u > 0)
        mcs_note_launch(), coo_write_kernel<<<(unsigned)ceil_div64(n_u, AT), AT, 0, st>>>(
            keys[cur], (const float*)vals[cur], n_u, K, out->coo_row, out->coo_col, out->coo_val);
    const unsigned long long h2[2] = { entries_total, (unsigned long long)n_u };
    MCS_CUDA_TRY(cudaMemcpyAsync(out->coo_nnz, &n_u, 8, cudaMemcpyHostToDevice, st));
    if (stats_dev) {
        MCS_CUDA_TRY(cudaMemcpyAsync(stats_dev + ST_ENTRIES, &h2[0], 8, cudaMemcpyHostToDevice, st));
        MCS_CUDA_TRY(cudaMemcpyAsync(stats_dev + ST_UNIQUE, &h2[1], 8, cudaMemcpyHostToDevice, st));
    }
    MCS_CUDA_TRY(cudaGetLastError());
    MCS_CUDA_TRY(cudaStreamSynchronize(st));                               // host scalars above live on this frame
    return MCS_OK;
}

// ===========================================================================
// Point-based function space (mcs_basis.kind 1): k-NN bilateral interpolator of
// PAPER.md App. B (Eq. 44-45).  b(q) has the k weights
//   w_i(q) ~ exp(-|q - x_i|^2 / (2 sigma^2)) exp(-(1 - <n_q, n_i>) / tau_n)
// over the k nearest points, normalised; d = b(s) - b(t) has up to 2k non-zeros, so
// a walk expands to up to 2k(2k+1)/2 upper-triangular entries, which go through the
// same stable sort + fixed-shape run sums as the hat basis.
// Readings (DESIGN.md Rk1-Rk4): weights formed relative to the largest exponent;
// neighbours by fp32 squared distance, ties by smaller index; k clamped to K;
// n_q = sample normal at s, normal of the exit face at t.
// ===========================================================================
namespace {

constexpr int KNN_MAX = 16;
constexpr int KNN_TILE = 256;
constexpr int64_t PB_CHUNK_WALKS = (int64_t)1 << 19;

// Uniform grid over the points (used when K > KNN_GRID_MIN): points sorted by cell, start/count per cell.
struct PointGrid {
    const uint32_t* cell_start;
    const uint32_t* cell_count;
    const uint32_t* sorted_idx;     // point index at sorted position
    float lox, loy, loz, h, inv_h;
    int nx, ny, nz;
};

struct PointBasisDev {
    const float* points;
    const float* normals;
    long long K;
    int k;
    float inv2s2, inv_tau;
    int use_grid;
    PointGrid grid;
};

constexpr int KNN_GRID_MIN = 1024;

// Insert candidate (d2, idx) into the sorted list of the KL best: order by d2, then by smaller index [Rk2].
// KL = 8 for k <= 8, else KNN_MAX: the list only has to hold the k nearest, and its length is what an insertion costs -- in
// a warp some lane inserts at almost every candidate, so all 32 pay for it (ncu, config-4 sample, k = 8 with a 16-entry
// list: 41 000 warp instructions per record warp = 80 per candidate, 200 registers, one block per SM).
template <int KL>
__device__ __forceinline__ void knn_insert(float (&bd)[KL], int (&bi)[KL], float d2, int idx)
{
    if (d2 < bd[KL - 1] || (d2 == bd[KL - 1] && idx < bi[KL - 1])) {
        bd[KL - 1] = d2; bi[KL - 1] = idx;
#pragma unroll
        for (int m = KL - 1; m > 0; --m)
            if (bd[m] < bd[m - 1] || (bd[m] == bd[m - 1] && bi[m] < bi[m - 1])) {
                const float td = bd[m]; bd[m] = bd[m - 1]; bd[m - 1] = td;
                const int ti = bi[m]; bi[m] = bi[m - 1]; bi[m - 1] = ti;
            }
    }
}

// Grid search: rings of cells about the query's cell.  After ring r every point within r*h - off of q has been
// seen (off = distance from q to its clamped cell), so the search stops when the k-th best is closer than that.
template <int KL>
__device__ __forceinline__ void knn_gather_grid(const PointBasisDev& pb, float3 q, float (&bd)[KL], int (&bi)[KL])
{
    const PointGrid& G = pb.grid;
    const float fx = (q.x - G.lox) * G.inv_h, fy = (q.y - G.loy) * G.inv_h, fz = (q.z - G.loz) * G.inv_h;
    const int cx = min(max((int)floorf(fx), 0), G.nx - 1), cy = min(max((int)floorf(fy), 0), G.ny - 1), cz = min(max((int)floorf(fz), 0), G.nz - 1);
    // distance from q to its (clamped) cell box, 0 when inside
    const float ox = fmaxf(fmaxf((float)cx - fx, fx - (float)(cx + 1)), 0.0f), oy = fmaxf(fmaxf((float)cy - fy, fy - (float)(cy + 1)), 0.0f),
                oz = fmaxf(fmaxf((float)cz - fz, fz - (float)(cz + 1)), 0.0f);
    const float off = sqrtf(ox * ox + oy * oy + oz * oz) * G.h;
    const int kk = pb.k < pb.K ? pb.k : (int)pb.K;
    const int rmax = max(G.nx, max(G.ny, G.nz));
    for (int r = 0; r <= rmax; ++r) {
        for (int dz = -r; dz <= r; ++dz) {
            const int z = cz + dz;
            if (z < 0 || z >= G.nz) continue;
            for (int dy = -r; dy <= r; ++dy) {
                const int y = cy + dy;
                if (y < 0 || y >= G.ny) continue;
                const bool face = (dz == -r || dz == r || dy == -r || dy == r);
                for (int dx = -r; dx <= r; dx += (face || r == 0) ? 1 : 2 * r) {     // only the shell of the cube
                    const int x = cx + dx;
                    if (x < 0 || x >= G.nx) continue;
                    const long long c = ((long long)z * G.ny + y) * G.nx + x;
                    const uint32_t s0 = G.cell_start[c], n = G.cell_count[c];
                    for (uint32_t j = 0; j < n; ++j) {
                        const int i = (int)G.sorted_idx[s0 + j];
                        const float dxp = q.x - pb.points[3 * (long long)i], dyp = q.y - pb.points[3 * (long long)i + 1],
                                    dzp = q.z - pb.points[3 * (long long)i + 2];
                        knn_insert<KL>(bd, bi, fmaf(dxp, dxp, fmaf(dyp, dyp, dzp * dzp)), i);
                    }
                }
            }
        }
        const float reach = fmaxf((float)r * G.h - off, 0.0f);
        if (bi[kk - 1] >= 0 && bd[kk - 1] < reach * reach) break;
    }
}

// k-NN of one query per thread: exhaustive (points staged through shared memory; every thread of the block must
// call this) or through the grid; the k best are kept sorted in registers (static indices only).
template <int KL>
__device__ __forceinline__ void knn_weights_device(const PointBasisDev& pb, bool active, float3 q, float3 nq,
                                                   float4* s_pts, int* idx_out, float* w_out)
{
    float bd[KL]; int bi[KL];
#pragma unroll
    for (int j = 0; j < KL; ++j) { bd[j] = CUDART_INF_F; bi[j] = -1; }
    const int k = pb.k;
    if (pb.use_grid) {
        if (active) knn_gather_grid<KL>(pb, q, bd, bi);
    } else {
        for (long long base = 0; base < pb.K; base += KNN_TILE) {
            const int n = (int)((pb.K - base) < KNN_TILE ? (pb.K - base) : KNN_TILE);
            __syncthreads();
            for (int j = threadIdx.x; j < n; j += blockDim.x)
                s_pts[j] = make_float4(pb.points[3 * (base + j)], pb.points[3 * (base + j) + 1], pb.points[3 * (base + j) + 2], 0.0f);
            __syncthreads();
            if (active) {
                for (int j = 0; j < n; ++j) {
                    const float4 p = s_pts[j];
                    const float dx = q.x - p.x, dy = q.y - p.y, dz = q.z - p.z;
                    knn_insert<KL>(bd, bi, fmaf(dx, dx, fmaf(dy, dy, dz * dz)), (int)(base + j));
                }
            }
        }
    }
    if (!active) return;
    // only the first k count: the list holds the KL >= k nearest in order
    float lg[KL], lmax = -CUDART_INF_F;
#pragma unroll
    for (int j = 0; j < KL; ++j) {
        const bool use = j < k && bi[j] >= 0;
        float c = 0.0f;
        if (use) {
            const float* ni = pb.normals + 3 * (long long)bi[j];
            c = fmaf(nq.x, ni[0], fmaf(nq.y, ni[1], nq.z * ni[2]));
        }
        lg[j] = use ? -bd[j] * pb.inv2s2 - (1.0f - c) * pb.inv_tau : -CUDART_INF_F;
        lmax = fmaxf(lmax, lg[j]);
    }
    float sum = 0.0f;
#pragma unroll
    for (int j = 0; j < KL; ++j) { lg[j] = (j < k && bi[j] >= 0) ? expf(lg[j] - lmax) : 0.0f; sum += lg[j]; }
    const float inv = 1.0f / sum;
#pragma unroll
    for (int j = 0; j < KL; ++j)
        if (j < k) { idx_out[j] = bi[j]; w_out[j] = lg[j] * inv; }
}

// ---- grid build ------------------------------------------------------------
__device__ __forceinline__ int pg_float_to_ordered(float f) { int i = __float_as_int(f); return i >= 0 ? i : i ^ 0x7FFFFFFF; }

__global__ void __launch_bounds__(AT)
points_bbox_kernel(const float* __restrict__ pts, long long K, int* __restrict__ out /* lo[3], hi[3] ordered */)
{
    const long long i = (long long)blockIdx.x * AT + threadIdx.x;
    if (i >= K) return;
    for (int d = 0; d < 3; ++d) {
        const int v = pg_float_to_ordered(pts[3 * i + d]);
        atomicMin(&out[d], v); atomicMax(&out[3 + d], v);
    }
}

__global__ void __launch_bounds__(AT)
points_cell_kernel(const float* __restrict__ pts, long long K, PointGrid G, uint32_t* __restrict__ keys, uint32_t* __restrict__ vals)
{
    const long long i = (long long)blockIdx.x * AT + threadIdx.x;
    if (i >= K) return;
    const int x = min(max((int)floorf((pts[3 * i] - G.lox) * G.inv_h), 0), G.nx - 1);
    const int y = min(max((int)floorf((pts[3 * i + 1] - G.loy) * G.inv_h), 0), G.ny - 1);
    const int z = min(max((int)floorf((pts[3 * i + 2] - G.loz) * G.inv_h), 0), G.nz - 1);
    keys[i] = (uint32_t)(((long long)z * G.ny + y) * G.nx + x);
    vals[i] = (uint32_t)i;
}

__global__ void __launch_bounds__(AT)
points_ranges_kernel(const uint32_t* __restrict__ keys, long long K, uint32_t* __restrict__ cell_start, uint32_t* __restrict__ cell_count)
{
    const long long i = (long long)blockIdx.x * AT + threadIdx.x;
    if (i >= K) return;
    const uint32_t c = keys[i];
    if (i == 0 || keys[i - 1] != c) {
        long long j = i + 1;
        while (j < K && keys[j] == c) ++j;            // cells hold a handful of points
        cell_start[c] = (uint32_t)i; cell_count[c] = (uint32_t)(j - i);
    }
}

template <int KL>
__global__ void __launch_bounds__(AT)
knn_queries_kernel(PointBasisDev pb, const float* __restrict__ q, const float* __restrict__ nq, long long Q,
                   int32_t* __restrict__ idx, float* __restrict__ w)
{
    __shared__ float4 s_pts[KNN_TILE];
    const long long i = (long long)blockIdx.x * AT + threadIdx.x;
    const bool active = i < Q;
    float3 qq = make_float3(0.f, 0.f, 0.f), nn = make_float3(0.f, 0.f, 1.f);
    if (active) { qq = make_float3(q[3 * i], q[3 * i + 1], q[3 * i + 2]); nn = make_float3(nq[3 * i], nq[3 * i + 1], nq[3 * i + 2]); }
    int io[KL]; float wo[KL];
    knn_weights_device<KL>(pb, active, qq, nn, s_pts, io, wo);
    if (active)
        for (int j = 0; j < pb.k; ++j) { idx[i * pb.k + j] = io[j]; w[i * pb.k + j] = wo[j]; }
}

__device__ __forceinline__ void face_point_normal(const float* __restrict__ verts, const int32_t* __restrict__ faces,
                                                  long long f, float b0, float b1, float b2, float3& p, float3& n)
{
    const long long i0 = faces[3 * f], i1 = faces[3 * f + 1], i2 = faces[3 * f + 2];
    const float3 a = make_float3(verts[3 * i0], verts[3 * i0 + 1], verts[3 * i0 + 2]);
    const float3 b = make_float3(verts[3 * i1], verts[3 * i1 + 1], verts[3 * i1 + 2]);
    const float3 c = make_float3(verts[3 * i2], verts[3 * i2 + 1], verts[3 * i2 + 2]);
    p = make_float3(fmaf(b0, a.x, fmaf(b1, b.x, b2 * c.x)), fmaf(b0, a.y, fmaf(b1, b.y, b2 * c.y)), fmaf(b0, a.z, fmaf(b1, b.z, b2 * c.z)));
    const float ux = b.x - a.x, uy = b.y - a.y, uz = b.z - a.z, vx = c.x - a.x, vy = c.y - a.y, vz = c.z - a.z;
    n = make_float3(uy * vz - uz * vy, uz * vx - ux * vz, ux * vy - uy * vx);
    const float l = sqrtf(fmaf(n.x, n.x, fmaf(n.y, n.y, n.z * n.z)));
    if (l > 0.0f) { n.x /= l; n.y /= l; n.z /= l; }
}

// b(s) of every sample
template <int KL>
__global__ void __launch_bounds__(AT)
knn_samples_kernel(PointBasisDev pb, const float* __restrict__ verts, const int32_t* __restrict__ faces,
                   const int32_t* __restrict__ s_tri, const float* __restrict__ s_bary, const float* __restrict__ s_normal,
                   long long n_s, int32_t* __restrict__ idx, float* __restrict__ w)
{
    __shared__ float4 s_pts[KNN_TILE];
    const long long i = (long long)blockIdx.x * AT + threadIdx.x;
    const bool active = i < n_s;
    float3 p = make_float3(0.f, 0.f, 0.f), n = make_float3(0.f, 0.f, 1.f);
    if (active) {
        face_point_normal(verts, faces, s_tri[i], s_bary[3 * i], s_bary[3 * i + 1], s_bary[3 * i + 2], p, n);
        if (s_normal) n = make_float3(s_normal[3 * i], s_normal[3 * i + 1], s_normal[3 * i + 2]);
    }
    int io[KL]; float wo[KL];
    knn_weights_device<KL>(pb, active, p, n, s_pts, io, wo);
    if (active)
        for (int j = 0; j < pb.k; ++j) { idx[i * pb.k + j] = io[j]; w[i * pb.k + j] = wo[j]; }
}

// b(t) of the records [j0, j0 + n): idx = -1 everywhere for a record without contribution
// Blocks per SM: the kernel compiles to ~195 registers unbounded (one block of 256 threads per SM, 12 % of the warp slots); held
// to 85 registers (three blocks) with the 8-entry list the config-4 sample goes 78.7 -> 83.8 meshes/s (two blocks: 83.1; four
// blocks spill: 73.9).
template <int KL>
__global__ void __launch_bounds__(AT, KL <= 8 ? 3 : 2)
knn_records_kernel(PointBasisDev pb, const float* __restrict__ verts, const int32_t* __restrict__ faces,
                   const float4* __restrict__ records, long long j0, long long n,
                   int32_t* __restrict__ idx, float* __restrict__ w)
{
    __shared__ float4 s_pts[KNN_TILE];
    const long long i = (long long)blockIdx.x * AT + threadIdx.x;
    bool active = i < n;
    float3 p = make_float3(0.f, 0.f, 0.f), nrm = make_float3(0.f, 0.f, 1.f);
    if (active) {
        const float4 rec = records[j0 + i];
        const int tri_t = __float_as_int(rec.x);
        if (tri_t >= 0 && rec.w != 0.0f) face_point_normal(verts, faces, tri_t, 1.0f - rec.y - rec.z, rec.y, rec.z, p, nrm);
        else { active = false; for (int j = 0; j < pb.k; ++j) { idx[i * pb.k + j] = -1; w[i * pb.k + j] = 0.0f; } }
    }
    int io[KL]; float wo[KL];
    knn_weights_device<KL>(pb, active, p, nrm, s_pts, io, wo);
    if (active)
        for (int j = 0; j < pb.k; ++j) { idx[i * pb.k + j] = io[j]; w[i * pb.k + j] = wo[j]; }
}

}  // namespace

namespace {

// d = b(s) - b(t) of record i as a merged list (shared points once); killing walks: d = b(t).
__device__ __forceinline__ int build_d_points(int k, bool has_s, const int32_t* __restrict__ is, const float* __restrict__ ws,
                                              const int32_t* __restrict__ it, const float* __restrict__ wt,
                                              int* idx, float* val)
{
    int m = 0;
    if (has_s)
        for (int j = 0; j < k; ++j) if (is[j] >= 0) { idx[m] = is[j]; val[m] = ws[j]; ++m; }
    const float sign = has_s ? -1.0f : 1.0f;
    for (int j = 0; j < k; ++j) {
        if (it[j] < 0) continue;
        int found = -1;
        for (int q = 0; q < m; ++q) if (idx[q] == it[j]) found = q;
        if (found >= 0) val[found] += sign * wt[j];
        else { idx[m] = it[j]; val[m] = sign * wt[j]; ++m; }
    }
    return m;
}

__global__ void __launch_bounds__(AT)
count_entries_points_kernel(int k, long long j0, long long n, long long n_main, int W,
                            const int32_t* __restrict__ is, const float* __restrict__ ws,
                            const int32_t* __restrict__ it, const float* __restrict__ wt, uint32_t* __restrict__ counts)
{
    const long long i = (long long)blockIdx.x * AT + threadIdx.x;
    if (i >= n) return;
    uint32_t c = 0;
    if (it[i * k] >= 0) {
        const bool has_s = j0 + i < n_main;
        const long long smp = has_s ? (j0 + i) / W : 0;
        int idx[2 * KNN_MAX]; float val[2 * KNN_MAX];
        const int m = build_d_points(k, has_s, is + smp * k, ws + smp * k, it + i * k, wt + i * k, idx, val);
        c = (uint32_t)(m * (m + 1) / 2);
    }
    counts[i] = c;
}

__global__ void __launch_bounds__(AT)
expand_entries_points_kernel(int k, long long j0, long long n, long long n_main, int W, long long K,
                             const float4* __restrict__ records,
                             const int32_t* __restrict__ is, const float* __restrict__ ws,
                             const int32_t* __restrict__ it, const float* __restrict__ wt,
                             const uint32_t* __restrict__ offsets, uint32_t* __restrict__ keys, uint32_t* __restrict__ vals)
{
    const long long i = (long long)blockIdx.x * AT + threadIdx.x;
    if (i >= n || it[i * k] < 0) return;
    const bool has_s = j0 + i < n_main;
    const long long smp = has_s ? (j0 + i) / W : 0;
    int idx[2 * KNN_MAX]; float val[2 * KNN_MAX];
    const int m = build_d_points(k, has_s, is + smp * k, ws + smp * k, it + i * k, wt + i * k, idx, val);
    const float wgt = records[j0 + i].w;
    uint32_t o = offsets[i];
    for (int p = 0; p < m; ++p)
        for (int q = p; q < m; ++q) {
            const int r = idx[p] < idx[q] ? idx[p] : idx[q], c = idx[p] < idx[q] ? idx[q] : idx[p];
            keys[o] = (uint32_t)((long long)r * K + c);
            vals[o] = __float_as_uint(wgt * val[p] * val[q]);
            ++o;
        }
}

struct PbLayout {
    size_t is, ws, it, wt, counts, keys, vals, carry_key, carry_sum, scan, sort, grid, total;
    int64_t C, E, n_tiles;
};

// scratch of the point grid: keys[K] | vals[K] | cell_start[cells] | cell_count[cells] | bbox ints | sort workspace
int64_t grid_max_cells(int64_t K) { return 16 * K + 64; }
size_t grid_scratch_bytes(int64_t K)
{
    return 2 * align_up((size_t)K * 4) + 2 * align_up((size_t)grid_max_cells(K) * 4) + 256 + align_up(sort_workspace_bytes(K, 4));
}

// Builds the grid over the points in `scratch` (blocks the host once, to read the bounding box).
int build_point_grid(const mcs_basis* basis, void* scratch, PointGrid* G, cudaStream_t st)
{
    const int64_t K = basis->K;
    char* p = (char*)scratch;
    uint32_t* keys = (uint32_t*)p;  p += align_up((size_t)K * 4);
    uint32_t* vals = (uint32_t*)p;  p += align_up((size_t)K * 4);
    uint32_t* start = (uint32_t*)p; p += align_up((size_t)grid_max_cells(K) * 4);
    uint32_t* count = (uint32_t*)p; p += align_up((size_t)grid_max_cells(K) * 4);
    int* box = (int*)p;             p += 256;
    void* sort_ws = p;
    int h[6] = { 0x7FFFFFFF, 0x7FFFFFFF, 0x7FFFFFFF, (int)0x80000000, (int)0x80000000, (int)0x80000000 };
    MCS_CUDA_TRY(cudaMemcpyAsync(box, h, sizeof h, cudaMemcpyHostToDevice, st));
    mcs_note_launch(), points_bbox_kernel<<<(unsigned)ceil_div64(K, AT), AT, 0, st>>>(basis->points, K, box);
    MCS_CUDA_TRY(cudaMemcpyAsync(h, box, sizeof h, cudaMemcpyDeviceToHost, st));
    MCS_CUDA_TRY(cudaStreamSynchronize(st));
    float lo[3], hi[3];
    for (int d = 0; d < 6; ++d) { int v = h[d] >= 0 ? h[d] : h[d] ^ 0x7FFFFFFF; memcpy(d < 3 ? &lo[d] : &hi[d - 3], &v, 4); }
    const float ex = hi[0] - lo[0], ey = hi[1] - lo[1], ez = hi[2] - lo[2];
    if (!(ex >= 0.0f) || !(ey >= 0.0f) || !(ez >= 0.0f)) return MCS_EDEGENERATE;          // non-finite point
    const float diag = sqrtf(ex * ex + ey * ey + ez * ez);
    float cell = diag > 0.0f ? diag / sqrtf((float)K) : 1.0f;                             // ~ one point spacing on a surface
    int nx, ny, nz;
    for (;;) {
        nx = (int)(ex / cell) + 1; ny = (int)(ey / cell) + 1; nz = (int)(ez / cell) + 1;
        if ((int64_t)nx * ny * nz <= grid_max_cells(K) - 64) break;
        cell *= 1.25f;
    }
    G->cell_start = start; G->cell_count = count; G->sorted_idx = vals;
    G->lox = lo[0]; G->loy = lo[1]; G->loz = lo[2]; G->h = cell; G->inv_h = 1.0f / cell;
    G->nx = nx; G->ny = ny; G->nz = nz;
    const int64_t cells = (int64_t)nx * ny * nz;
    MCS_CUDA_TRY(cudaMemsetAsync(start, 0, (size_t)cells * 4, st));
    MCS_CUDA_TRY(cudaMemsetAsync(count, 0, (size_t)cells * 4, st));
    mcs_note_launch(), points_cell_kernel<<<(unsigned)ceil_div64(K, AT), AT, 0, st>>>(basis->points, K, *G, keys, vals);
    int bits = 1;
    while (((int64_t)1 << bits) < cells) ++bits;
    int rc = sort_pairs_u32(keys, vals, K, bits, sort_ws, sort_workspace_bytes(K, 4), st);
    if (rc != MCS_OK) return rc;
    mcs_note_launch(), points_ranges_kernel<<<(unsigned)ceil_div64(K, AT), AT, 0, st>>>(keys, K, start, count);
    MCS_CUDA_TRY(cudaGetLastError());
    return MCS_OK;
}

PbLayout pb_layout(int64_t n_s, int64_t n_records, int k, int64_t K)
{
    PbLayout L;
    L.C = n_records < PB_CHUNK_WALKS ? (n_records < 1 ? 1 : n_records) : PB_CHUNK_WALKS;
    L.E = L.C * (int64_t)(2 * k) * (2 * k + 1) / 2;
    L.n_tiles = ceil_div64(L.E, RT);
    size_t off = 0;
    L.is = off;        off += align_up((size_t)n_s * k * 4);
    L.ws = off;        off += align_up((size_t)n_s * k * 4);
    L.it = off;        off += align_up((size_t)L.C * k * 4);
    L.wt = off;        off += align_up((size_t)L.C * k * 4);
    L.counts = off;    off += align_up((size_t)(L.C + 1) * 4);
    L.keys = off;      off += align_up((size_t)L.E * 4);
    L.vals = off;      off += align_up((size_t)L.E * 4);
    L.carry_key = off; off += align_up((size_t)L.n_tiles * 4);
    L.carry_sum = off; off += align_up((size_t)L.n_tiles * 4);
    L.scan = off;      off += align_up(scan_workspace_bytes(L.C) + 256);
    L.sort = off;      off += align_up(sort_workspace_bytes(L.E, 4));
    L.grid = off;      off += K > KNN_GRID_MIN ? align_up(grid_scratch_bytes(K)) : 0;
    L.total = off + 1024;
    return L;
}

int check_point_basis(const mcs_basis* basis)
{
    if (!basis || basis->kind != 1 || basis->K < 1 || !basis->points || !basis->normals) return MCS_EINVAL;
    if (basis->k < 1 || basis->k > KNN_MAX || !(basis->sigma > 0.0f) || !(basis->tau_n > 0.0f)) return MCS_EINVAL;
    return MCS_OK;
}

PointBasisDev point_basis_dev(const mcs_basis* basis)
{
    PointBasisDev pb;
    pb.points = basis->points; pb.normals = basis->normals; pb.K = basis->K;
    pb.k = basis->k < basis->K ? basis->k : (int)basis->K;
    pb.inv2s2 = 1.0f / (2.0f * basis->sigma * basis->sigma);
    pb.inv_tau = 1.0f / basis->tau_n;
    pb.use_grid = 0;
    memset(&pb.grid, 0, sizeof pb.grid);
    return pb;
}

}  // namespace

size_t accumulate_points_workspace_bytes(const mcs_samples* s, const mcs_basis* basis, int64_t n_records)
{
    const int k = basis->k < 1 ? 1 : (basis->k > KNN_MAX ? KNN_MAX : basis->k);
    return pb_layout(s->n_s, n_records, k, basis->K).total;
}

int knn_weights_run(const mcs_basis* basis, const float* q, const float* nq, int64_t Q, int32_t* idx, float* w, cudaStream_t st)
{
    int rc = check_point_basis(basis);
    if (rc != MCS_OK) return rc;
    if (Q < 0 || (Q > 0 && (!q || !nq || !idx || !w))) return MCS_EINVAL;
    if (Q == 0) return MCS_OK;
    PointBasisDev pb = point_basis_dev(basis);
    pb.k = basis->k;                                  // output stride is the caller's k; slots beyond K hold -1 / 0
    void* scratch = nullptr;
    if (basis->K > KNN_GRID_MIN) {                    // test hook: its own scratch for the grid
        cudaError_t e = cudaMalloc(&scratch, grid_scratch_bytes(basis->K));
        if (e != cudaSuccess) { mcs_set_last_cuda_error((int)e); return MCS_ENOMEM; }
        rc = build_point_grid(basis, scratch, &pb.grid, st);
        if (rc != MCS_OK) { cudaFree(scratch); return rc; }
        pb.use_grid = 1;
    }
    if (pb.k <= 8) mcs_note_launch(), knn_queries_kernel<8><<<(unsigned)ceil_div64(Q, AT), AT, 0, st>>>(pb, q, nq, Q, idx, w);
    else mcs_note_launch(), knn_queries_kernel<KNN_MAX><<<(unsigned)ceil_div64(Q, AT), AT, 0, st>>>(pb, q, nq, Q, idx, w);
    cudaError_t e = cudaGetLastError();
    if (scratch) { cudaStreamSynchronize(st); cudaFree(scratch); }
    if (e != cudaSuccess) { mcs_set_last_cuda_error((int)e); return MCS_ECUDA; }
    return MCS_OK;
}

int accumulate_points_run(const mcs_bvh* b, const mcs_samples* s, const mcs_basis* basis, int W,
                          const float4* records, int64_t n_records, void* ws, size_t ws_bytes,
                          const mcs_matrix* out, unsigned long long* stats_dev, cudaStream_t st)
{
    if (!b || !s || !out || !records || n_records < 0) return MCS_EINVAL;
    int rc = check_point_basis(basis);
    if (rc != MCS_OK) return rc;
    if (out->kind != 0 || out->K != basis->K || !out->dense) return MCS_EINVAL;      // dense output only for now
    const long long K = basis->K;
    if (K > 65535) return MCS_EINVAL;
    const int k = basis->k;
    const PbLayout L = pb_layout(s->n_s, n_records, k, basis->K);
    if (!ws || ws_bytes < L.total) return MCS_ENOMEM;
    char* base = (char*)ws;
    int32_t* is = (int32_t*)(base + L.is);  float* wsm = (float*)(base + L.ws);
    int32_t* it = (int32_t*)(base + L.it);  float* wt = (float*)(base + L.wt);
    uint32_t* counts = (uint32_t*)(base + L.counts);
    uint32_t* keys = (uint32_t*)(base + L.keys);
    uint32_t* vals = (uint32_t*)(base + L.vals);
    uint32_t* carry_key = (uint32_t*)(base + L.carry_key);
    float* carry_sum = (float*)(base + L.carry_sum);
    void* scan_ws = base + L.scan;
    void* sort_ws = base + L.sort;
    const size_t scan_bytes = L.sort - L.scan, sort_bytes = L.total - L.sort;
    PointBasisDev pb = point_basis_dev(basis);
    pb.k = k;
    if (basis->K > KNN_GRID_MIN) {
        rc = build_point_grid(basis, base + L.grid, &pb.grid, st);
        if (rc != MCS_OK) return rc;
        pb.use_grid = 1;
    }
    const long long n_main = (long long)s->n_s * W < n_records ? (long long)s->n_s * W : n_records;
    const int bits = key_bits_for(K);

    MCS_CUDA_TRY(cudaMemsetAsync(out->dense, 0, (size_t)K * K * sizeof(float), st));
    if (k <= 8) mcs_note_launch(), knn_samples_kernel<8><<<(unsigned)ceil_div64(s->n_s, AT), AT, 0, st>>>(
        pb, b->verts, b->faces, s->tri, s->bary, s->normal, s->n_s, is, wsm);
    else mcs_note_launch(), knn_samples_kernel<KNN_MAX><<<(unsigned)ceil_div64(s->n_s, AT), AT, 0, st>>>(
        pb, b->verts, b->faces, s->tri, s->bary, s->normal, s->n_s, is, wsm);
    unsigned long long entries_total = 0;
    for (int64_t j0 = 0; j0 < n_records; j0 += L.C) {
        const long long n = (n_records - j0) < L.C ? (n_records - j0) : L.C;
        const unsigned nblk = (unsigned)ceil_div64(n, AT);
        if (k <= 8) mcs_note_launch(), knn_records_kernel<8><<<nblk, AT, 0, st>>>(pb, b->verts, b->faces, records, j0, n, it, wt);
        else mcs_note_launch(), knn_records_kernel<KNN_MAX><<<nblk, AT, 0, st>>>(pb, b->verts, b->faces, records, j0, n, it, wt);
        mcs_note_launch(), count_entries_points_kernel<<<nblk, AT, 0, st>>>(k, j0, n, n_main, W, is, wsm, it, wt, counts);
        rc = exclusive_scan_u32(counts, counts, n, counts + n, scan_ws, scan_bytes, st);
        if (rc != MCS_OK) return rc;
        uint32_t n_entries = 0;
        MCS_CUDA_TRY(cudaMemcpyAsync(&n_entries, counts + n, 4, cudaMemcpyDeviceToHost, st));
        MCS_CUDA_TRY(cudaStreamSynchronize(st));
        if (n_entries == 0) continue;
        entries_total += n_entries;
        mcs_note_launch(), expand_entries_points_kernel<<<nblk, AT, 0, st>>>(k, j0, n, n_main, W, K, records, is, wsm, it, wt,
                                                                            counts, keys, vals);
        rc = sort_pairs_u32(keys, vals, n_entries, bits, sort_ws, sort_bytes, st);
        if (rc != MCS_OK) return rc;
        const long long n_tiles = ceil_div64(n_entries, RT);
        mcs_note_launch(), reduce_runs_dense_kernel<<<(unsigned)n_tiles, RT, 0, st>>>(
            keys, vals, n_entries, out->dense, carry_key, carry_sum, stats_dev ? stats_dev + ST_UNIQUE : nullptr, nullptr);
        mcs_note_launch(), carry_fixup_kernel<<<(unsigned)ceil_div64(n_tiles, AT), AT, 0, st>>>(carry_key, carry_sum, n_tiles, out->dense);
    }
    mcs_note_launch(), mirror_kernel<<<(unsigned)ceil_div64(K * K, AT), AT, 0, st>>>(out->dense, K);
    if (stats_dev)
        MCS_CUDA_TRY(cudaMemcpyAsync(stats_dev + ST_ENTRIES, &entries_total, 8, cudaMemcpyHostToDevice, st));
    MCS_CUDA_TRY(cudaGetLastError());
    if (stats_dev) MCS_CUDA_TRY(cudaStreamSynchronize(st));
    return MCS_OK;
}
