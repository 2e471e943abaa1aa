// accumulate.cu -- deterministic accumulation of per-walk records into the DtN
// matrix:   S = sum_walks  weight * d d^T,
// d = b(s) - b(t) in the hat basis (Eq. 26), a
// killing record contributing weight * b(t0) b(t0)^T (Eq. 32, second term).
//
// The paper defers the outer products "to be computed in batches to avoid shared
// memory contention".  Here: expand every walk into its
// upper-triangular (row, col, value) entries in slot order, stable radix sort by
// key = row*K + col, sum each run of equal keys left to right, add the run sums
// to the dense matrix (one writer per entry, so no atomics), and mirror the
// upper triangle at the end.  The result is bit-identical from run to run and
// exactly symmetric.
#include "walk.cuh"

namespace {

constexpr int AT = 256;
constexpr int64_t MAX_CHUNK_WALKS = (int64_t)1 << 22;
constexpr int MAX_ENTRIES_PER_WALK = 21;          // upper triangle of a 6 x 6 block

struct AccArgs {
    const float4*  records;
    const int32_t* faces;
    const int32_t* s_tri;
    const float*   s_bary;
    long long n_main;       // records below this index belong to sample (index / W)
    int W;
    long long K;
};

// d = b(s) - b(t): up to 6 (vertex, value) pairs; shared vertices are merged.
__device__ __forceinline__ int build_d(const AccArgs& a, long long j, const float4 rec, int idx[6], float val[6])
{
    int n = 0;
    float sign = 1.0f;
    if (j < a.n_main) {
        const long long smp = j / a.W;
        const long long fs = a.s_tri[smp];
        for (int k = 0; k < 3; ++k) { idx[n] = a.faces[3 * fs + k]; val[n] = a.s_bary[3 * smp + k]; ++n; }
        sign = -1.0f;
    }
    const long long ft = __float_as_int(rec.x);
    const float bt[3] = { 1.0f - rec.y - rec.z, rec.y, rec.z };
    for (int k = 0; k < 3; ++k) {
        const int v = a.faces[3 * ft + k];
        int found = -1;
        for (int m = 0; m < n; ++m) if (idx[m] == v) found = m;
        if (found >= 0) val[found] += sign * bt[k];
        else { idx[n] = v; val[n] = sign * bt[k]; ++n; }
    }
    return n;
}

__global__ void __launch_bounds__(AT)
count_entries_kernel(AccArgs a, long long j0, long long n, uint32_t* __restrict__ counts)
{
    const long long i = (long long)blockIdx.x * AT + threadIdx.x;
    if (i >= n) return;
    const float4 rec = a.records[j0 + i];
    uint32_t c = 0;
    if (__float_as_int(rec.x) >= 0 && rec.w != 0.0f) {
        int idx[6]; float val[6];
        const int m = build_d(a, j0 + i, rec, idx, val);
        for (int p = 0; p < m; ++p) for (int q = 0; q < m; ++q) c += (idx[p] <= idx[q]) ? 1u : 0u;
    }
    counts[i] = c;
}

__global__ void __launch_bounds__(AT)
expand_entries_kernel(AccArgs a, long long j0, long long n, const uint32_t* __restrict__ offsets,
                      uint32_t* __restrict__ keys, uint32_t* __restrict__ vals)
{
    const long long i = (long long)blockIdx.x * AT + threadIdx.x;
    if (i >= n) return;
    const float4 rec = a.records[j0 + i];
    if (__float_as_int(rec.x) < 0 || rec.w == 0.0f) return;
    int idx[6]; float val[6];
    const int m = build_d(a, j0 + i, rec, idx, val);
    uint32_t o = offsets[i];
    for (int p = 0; p < m; ++p)
        for (int q = 0; q < m; ++q)
            if (idx[p] <= idx[q]) {
                keys[o] = (uint32_t)((long long)idx[p] * a.K + idx[q]);
                vals[o] = __float_as_uint(rec.w * val[p] * val[q]);
                ++o;
            }
}

// One thread per run of equal keys: sum left to right, add to the dense matrix.
__global__ void __launch_bounds__(AT)
reduce_runs_dense_kernel(const uint32_t* __restrict__ keys, const uint32_t* __restrict__ vals, long long n,
                         float* __restrict__ S, unsigned long long* __restrict__ n_unique)
{
    const long long i = (long long)blockIdx.x * AT + threadIdx.x;
    bool head = false;
    if (i < n) {
        const uint32_t key = keys[i];
        head = (i == 0) || (keys[i - 1] != key);
        if (head) {
            float sum = __uint_as_float(vals[i]);
            for (long long j = i + 1; j < n && keys[j] == key; ++j) sum += __uint_as_float(vals[j]);
            S[key] += sum;
        }
    }
    const unsigned m = __ballot_sync(0xFFFFFFFFu, head);
    if (n_unique && (threadIdx.x & 31) == 0 && m) atomicAdd(n_unique, (unsigned long long)__popc(m));
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

}  // namespace

size_t accumulate_workspace_bytes(const mcs_bvh* b, const mcs_basis* basis, int64_t n_records)
{
    (void)b; (void)basis;
    const int64_t C = n_records < MAX_CHUNK_WALKS ? (n_records < 1 ? 1 : n_records) : MAX_CHUNK_WALKS;
    const int64_t E = C * MAX_ENTRIES_PER_WALK;
    return align_up((size_t)(C + 1) * 4) + 2 * align_up((size_t)E * 4) + sort_workspace_bytes(E, 4) +
           scan_workspace_bytes(C) + 1024;
}

int accumulate_run(const mcs_bvh* b, const mcs_samples* s, const mcs_basis* basis, int W,
                   const float4* records, int64_t n_records, void* ws, size_t ws_bytes,
                   const mcs_matrix* out, unsigned long long* stats_dev, cudaStream_t st)
{
    if (!b || !s || !basis || !out || !records || n_records < 0) return MCS_EINVAL;
    if (basis->kind != 0 || basis->K != b->V) return MCS_EINVAL;
    if (out->kind != 0 || out->K != basis->K || !out->dense) return MCS_EINVAL;
    const long long K = basis->K;
    if (K > 65535) return MCS_EINVAL;                 // dense keys are 32-bit (row*K + col)
    if (!ws || ws_bytes < accumulate_workspace_bytes(b, basis, n_records)) return MCS_ENOMEM;

    const int64_t C = n_records < MAX_CHUNK_WALKS ? (n_records < 1 ? 1 : n_records) : MAX_CHUNK_WALKS;
    const int64_t E = C * MAX_ENTRIES_PER_WALK;
    char* ptr = (char*)ws;
    uint32_t* counts = (uint32_t*)ptr;  ptr += align_up((size_t)(C + 1) * 4);
    uint32_t* keys = (uint32_t*)ptr;    ptr += align_up((size_t)E * 4);
    uint32_t* vals = (uint32_t*)ptr;    ptr += align_up((size_t)E * 4);
    void* scan_ws = ptr;                ptr += scan_workspace_bytes(C) + 256;
    ptr = (char*)align_up((size_t)ptr);
    void* sort_ws = ptr;
    const size_t sort_bytes = ws_bytes - (size_t)(ptr - (char*)ws);

    AccArgs a;
    a.records = records; a.faces = b->faces; a.s_tri = s->tri; a.s_bary = s->bary;
    a.n_main = (long long)s->n_s * W; a.W = W; a.K = K;
    const int bits = key_bits_for(K);

    MCS_CUDA_TRY(cudaMemsetAsync(out->dense, 0, (size_t)K * K * sizeof(float), st));
    unsigned long long entries_total = 0;
    for (int64_t j0 = 0; j0 < n_records; j0 += C) {
        const long long n = (n_records - j0) < C ? (n_records - j0) : C;
        const unsigned nblk = (unsigned)ceil_div64(n, AT);
        mcs_note_launch(), count_entries_kernel<<<nblk, AT, 0, st>>>(a, j0, n, counts);
        int rc = exclusive_scan_u32(counts, counts, n, counts + n, scan_ws, scan_workspace_bytes(C) + 256, st);
        if (rc != MCS_OK) return rc;
        uint32_t n_entries = 0;
        MCS_CUDA_TRY(cudaMemcpyAsync(&n_entries, counts + n, 4, cudaMemcpyDeviceToHost, st));
        MCS_CUDA_TRY(cudaStreamSynchronize(st));
        if (n_entries == 0) continue;
        entries_total += n_entries;
        mcs_note_launch(), expand_entries_kernel<<<nblk, AT, 0, st>>>(a, j0, n, counts, keys, vals);
        rc = sort_pairs_u32(keys, vals, n_entries, bits, sort_ws, sort_bytes, st);
        if (rc != MCS_OK) return rc;
        mcs_note_launch(), reduce_runs_dense_kernel<<<(unsigned)ceil_div64(n_entries, AT), AT, 0, st>>>(
            keys, vals, n_entries, out->dense, stats_dev ? stats_dev + ST_UNIQUE : nullptr);
    }
    mcs_note_launch(), mirror_kernel<<<(unsigned)ceil_div64(K * K, AT), AT, 0, st>>>(out->dense, K);
    if (stats_dev)
        MCS_CUDA_TRY(cudaMemcpyAsync(stats_dev + ST_ENTRIES, &entries_total, 8, cudaMemcpyHostToDevice, st));
    MCS_CUDA_TRY(cudaGetLastError());
    if (stats_dev) MCS_CUDA_TRY(cudaStreamSynchronize(st));     // entries_total lives on this stack frame
    return MCS_OK;
}
