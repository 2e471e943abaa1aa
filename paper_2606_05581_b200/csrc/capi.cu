// capi.cu -- the C ABI entry points of include/mcdtn.h that tie the steps together.
#include "walk.cuh"

#include <string.h>

static thread_local int g_last_cuda_error = 0;
void mcs_set_last_cuda_error(int e) { g_last_cuda_error = e; }
int  mcs_get_last_cuda_error() { return g_last_cuda_error; }

#include <atomic>
static std::atomic<unsigned long long> g_launches{0};
void mcs_note_launch() { g_launches.fetch_add(1, std::memory_order_relaxed); }

static int g_prof_on = 0;
static cudaEvent_t g_prof_ev[MCS_MARK_COUNT];
static bool g_prof_have = false, g_prof_marked[MCS_MARK_COUNT];
void mcs_prof_mark(int which, cudaStream_t st)
{
    if (!g_prof_on || which < 0 || which >= MCS_MARK_COUNT) return;
    if (!g_prof_have) {
        for (int i = 0; i < MCS_MARK_COUNT; ++i) cudaEventCreate(&g_prof_ev[i]);
        g_prof_have = true;
    }
    if (which == MCS_MARK_BEGIN) for (int i = 0; i < MCS_MARK_COUNT; ++i) g_prof_marked[i] = false;
    cudaEventRecord(g_prof_ev[which], st);
    g_prof_marked[which] = true;
}

namespace {

struct Layout {
    size_t records_off, walk_off, acc_off, total;
    int64_t n_records;
};

Layout make_layout(const mcs_bvh* b, const mcs_samples* s, const mcs_basis* basis, const mcs_params* p, int exterior,
                   bool with_records, bool with_acc)
{
    Layout L;
    L.n_records = walk_num_records(s, p, exterior);
    size_t off = 0;
    L.records_off = off; if (with_records) off += align_up((size_t)L.n_records * sizeof(mcs_record));
    L.walk_off = off;    off += align_up(walk_workspace_bytes(s));
    L.acc_off = off;     if (with_acc) off += align_up(accumulate_workspace_bytes(b, basis, L.n_records));
    L.total = off + 256;
    return L;
}

void fill_stats(mcs_stats* hs, const unsigned long long* h, const mcs_samples* s, int64_t n_records)
{
    hs->n_samples = s->n_s;
    hs->n_discarded = (int64_t)h[ST_DISCARDED];
    hs->n_walks = n_records;
    hs->n_truncated = (int64_t)h[ST_TRUNCATED];
    hs->n_steps = (int64_t)h[ST_STEPS];
    hs->n_queries = (int64_t)h[ST_QUERIES];
    hs->n_nodes_visited = (int64_t)h[ST_NODES];
    hs->n_tris_tested = (int64_t)h[ST_TRIS];
    hs->n_entries = (int64_t)h[ST_ENTRIES];
    hs->n_unique = (int64_t)h[ST_UNIQUE];
}

int fail(int rc, mcs_stats* hs)
{
    if (hs && rc == MCS_ECUDA) hs->cuda_error = mcs_get_last_cuda_error();
    return rc;
}

int estimate(const mcs_bvh* b, const mcs_samples* s, const mcs_basis* basis, const mcs_params* p, int exterior,
             void* ws, size_t ws_bytes, const mcs_matrix* out, mcs_stats* hs, void* stream)
{
    if (hs) memset(hs, 0, sizeof *hs);
    if (!b || !s || !basis || !p || !out) return MCS_EINVAL;
    if (p->output_kind != 0 || out->kind != p->output_kind) return MCS_EINVAL;
    if (p->walks_per_sample < 1 || s->n_s < 1) return MCS_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    const Layout L = make_layout(b, s, basis, p, exterior, true, true);
    if (hs) hs->workspace_needed = (int64_t)L.total;
    if (!ws || ws_bytes < L.total) return MCS_ENOMEM;
    char* base = (char*)ws;
    float4* records = (float4*)(base + L.records_off);
    unsigned long long* stats_dev = nullptr;
    mcs_prof_mark(MCS_MARK_BEGIN, st);
    int rc = walk_run(b, s, p, exterior, base + L.walk_off, align_up(walk_workspace_bytes(s)), records, nullptr,
                      false, nullptr, hs != nullptr, &stats_dev, st);
    if (rc != MCS_OK) return fail(rc, hs);
    rc = accumulate_run(b, s, basis, p->walks_per_sample, records, L.n_records, base + L.acc_off,
                        align_up(accumulate_workspace_bytes(b, basis, L.n_records)), out, stats_dev, st);
    if (rc != MCS_OK) return fail(rc, hs);
    mcs_prof_mark(MCS_MARK_END, st);
    if (hs) {
        unsigned long long h[ST_COUNT];
        cudaError_t e = cudaMemcpyAsync(h, stats_dev, sizeof h, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) { mcs_set_last_cuda_error((int)e); return fail(MCS_ECUDA, hs); }
        fill_stats(hs, h, s, L.n_records);
    }
    return MCS_OK;
}

}  // namespace

extern "C" unsigned long long mcs_launch_count(void) { return g_launches.load(); }

extern "C" int mcs_profile_enable(int on) { g_prof_on = on ? 1 : 0; return MCS_OK; }

extern "C" int mcs_profile_last(mcs_phase_times* out)
{
    if (!out) return MCS_EINVAL;
    memset(out, 0, sizeof *out);
    if (!g_prof_have) return MCS_EINVAL;
    for (int i = 0; i < MCS_MARK_COUNT; ++i) if (!g_prof_marked[i]) return MCS_EINVAL;
    MCS_CUDA_TRY(cudaEventSynchronize(g_prof_ev[MCS_MARK_END]));
    MCS_CUDA_TRY(cudaEventElapsedTime(&out->prep_ms, g_prof_ev[MCS_MARK_BEGIN], g_prof_ev[MCS_MARK_WALK_BEGIN]));
    MCS_CUDA_TRY(cudaEventElapsedTime(&out->walk_ms, g_prof_ev[MCS_MARK_WALK_BEGIN], g_prof_ev[MCS_MARK_WALK_END]));
    MCS_CUDA_TRY(cudaEventElapsedTime(&out->accumulate_ms, g_prof_ev[MCS_MARK_WALK_END], g_prof_ev[MCS_MARK_END]));
    MCS_CUDA_TRY(cudaEventElapsedTime(&out->total_ms, g_prof_ev[MCS_MARK_BEGIN], g_prof_ev[MCS_MARK_END]));
    return MCS_OK;
}

extern "C" size_t mcs_workspace_bytes(const mcs_bvh* b, const mcs_samples* s, const mcs_basis* basis,
                                      const mcs_params* p, int exterior)
{
    if (!b || !s || !basis || !p || s->n_s < 1 || p->walks_per_sample < 1) return 0;
    return make_layout(b, s, basis, p, exterior, true, true).total;
}

extern "C" int mcs_estimate_dtn_interior(const mcs_bvh* b, const mcs_samples* s, const mcs_basis* basis,
                                         const mcs_params* p, void* ws, size_t ws_bytes,
                                         const mcs_matrix* out, mcs_stats* hs, void* stream)
{
    return estimate(b, s, basis, p, 0, ws, ws_bytes, out, hs, stream);
}

extern "C" int mcs_estimate_dtn_exterior(const mcs_bvh* b, const mcs_samples* s, const mcs_basis* basis,
                                         const mcs_params* p, void* ws, size_t ws_bytes,
                                         const mcs_matrix* out, mcs_stats* hs, void* stream)
{
    return estimate(b, s, basis, p, 1, ws, ws_bytes, out, hs, stream);
}

extern "C" int mcs_tangent_balls(const mcs_bvh* b, const mcs_samples* s, const mcs_params* p, int exterior,
                                 float* balls, void* stream)
{
    if (!b || !s || !p || !balls || s->n_s < 1) return MCS_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    void* ws = nullptr;
    const size_t bytes = align_up(walk_workspace_bytes(s));
    cudaError_t e = cudaMalloc(&ws, bytes);            // test hook: not on the estimator path
    if (e != cudaSuccess) { mcs_set_last_cuda_error((int)e); return MCS_ENOMEM; }
    int rc = walk_run(b, s, p, exterior, ws, bytes, nullptr, nullptr, true, balls, false, nullptr, st);
    cudaStreamSynchronize(st);
    cudaFree(ws);
    return rc;
}

extern "C" int mcs_run_walks(const mcs_bvh* b, const mcs_samples* s, const mcs_params* p, int exterior,
                             void* ws, size_t ws_bytes, mcs_record* records, int32_t* steps,
                             mcs_stats* hs, void* stream)
{
    if (hs) memset(hs, 0, sizeof *hs);
    if (!b || !s || !p || !records || s->n_s < 1 || p->walks_per_sample < 1) return MCS_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t need = align_up(walk_workspace_bytes(s));
    if (hs) hs->workspace_needed = (int64_t)need;
    if (!ws || ws_bytes < need) return MCS_ENOMEM;
    unsigned long long* stats_dev = nullptr;
    int rc = walk_run(b, s, p, exterior, ws, ws_bytes, (float4*)records, steps, false, nullptr, hs != nullptr, &stats_dev, st);
    if (rc != MCS_OK) return fail(rc, hs);
    if (hs) {
        unsigned long long h[ST_COUNT];
        cudaError_t e = cudaMemcpyAsync(h, stats_dev, sizeof h, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) { mcs_set_last_cuda_error((int)e); return fail(MCS_ECUDA, hs); }
        fill_stats(hs, h, s, walk_num_records(s, p, exterior));
    }
    return MCS_OK;
}

extern "C" int mcs_accumulate(const mcs_bvh* b, const mcs_samples* s, const mcs_basis* basis, const mcs_params* p,
                              const mcs_record* records, int64_t n_records, void* ws, size_t ws_bytes,
                              const mcs_matrix* out, mcs_stats* hs, void* stream)
{
    if (hs) memset(hs, 0, sizeof *hs);
    if (!b || !s || !basis || !p || !records || !out) return MCS_EINVAL;
    if (n_records < s->n_s * (int64_t)p->walks_per_sample) return MCS_EINVAL;
    const size_t need = align_up(accumulate_workspace_bytes(b, basis, n_records)) + 512;
    if (hs) hs->workspace_needed = (int64_t)need;
    if (!ws || ws_bytes < need) return MCS_ENOMEM;
    cudaStream_t st = (cudaStream_t)stream;
    unsigned long long* stats_dev = (unsigned long long*)ws;       // first 512 bytes: counters
    MCS_CUDA_TRY(cudaMemsetAsync(stats_dev, 0, ST_COUNT * 8, st));
    int rc = accumulate_run(b, s, basis, p->walks_per_sample, (const float4*)records, n_records,
                            (char*)ws + 512, ws_bytes - 512, out, stats_dev, st);
    if (rc != MCS_OK) return fail(rc, hs);
    if (hs) {
        unsigned long long h[ST_COUNT];
        cudaError_t e = cudaMemcpyAsync(h, stats_dev, sizeof h, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) { mcs_set_last_cuda_error((int)e); return fail(MCS_ECUDA, hs); }
        fill_stats(hs, h, s, n_records);
    }
    return MCS_OK;
}

extern "C" size_t mcs_accumulate_workspace_bytes(const mcs_bvh* b, const mcs_basis* basis, int64_t n_records)
{
    if (!b || !basis) return 0;
    return align_up(accumulate_workspace_bytes(b, basis, n_records)) + 512;
}

extern "C" size_t mcs_walk_workspace_bytes(const mcs_samples* s)
{
    if (!s || s->n_s < 1) return 0;
    return align_up(walk_workspace_bytes(s));
}

extern "C" size_t mcs_sort_workspace_bytes(int64_t n) { return sort_workspace_bytes(n, 8); }

extern "C" int mcs_sort_pairs_u64(uint64_t* keys, uint32_t* vals, int64_t n, int32_t key_bits,
                                  void* ws, size_t ws_bytes, void* stream)
{
    if (n < 0 || (n > 0 && (!keys || !vals || !ws))) return MCS_EINVAL;
    return sort_pairs_u64(keys, vals, n, key_bits, ws, ws_bytes, (cudaStream_t)stream);
}

extern "C" const char* mcs_error_string(int code)
{
    switch (code) {
        case MCS_OK: return "ok";
        case MCS_EINVAL: return "invalid argument";
        case MCS_EDEGENERATE: return "degenerate input (zero area, non-finite vertex, or Kelvin origin on a vertex)";
        case MCS_ENOMEM: return "workspace too small or device allocation failed";
        case MCS_ECUDA: return "CUDA runtime error";
        default: return "unknown error";
    }
}

extern "C" size_t mcs_abi_sizeof(int which)
{
    switch (which) {
        case 0: return sizeof(mcs_samples);
        case 1: return sizeof(mcs_basis);
        case 2: return sizeof(mcs_params);
        case 3: return sizeof(mcs_matrix);
        case 4: return sizeof(mcs_stats);
        case 5: return sizeof(mcs_bvh_info_t);
        case 6: return sizeof(mcs_record);
        default: return 0;
    }
}

extern "C" const char* mcs_version(void) { return "mcdtn 0.1 (sm_100a)"; }
