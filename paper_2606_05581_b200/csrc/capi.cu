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

size_t acc_ws_bytes(const mcs_bvh* b, const mcs_samples* s, const mcs_basis* basis, const mcs_params* p, int64_t n_records)
{
    if (basis->kind == 1) return accumulate_points_workspace_bytes(s, basis, n_records);
    return p->output_kind == 1 ? accumulate_coo_workspace_bytes(b, n_records, p->coo_capacity)
                               : accumulate_workspace_bytes(b, basis, n_records);
}

int acc_run(const mcs_bvh* b, const mcs_samples* s, const mcs_basis* basis, const mcs_params* p,
            const float4* records, int64_t n_records, void* ws, size_t ws_bytes,
            const mcs_matrix* out, unsigned long long* stats_dev, cudaStream_t st)
{
    if (basis->kind == 1) {                    // point basis: Alg. 2 / Eq. 32, dense output
        if (p->output_kind != 0 || p->estimator != 0) return MCS_EINVAL;
        return accumulate_points_run(b, s, basis, p->walks_per_sample, records, n_records, ws, ws_bytes, out, stats_dev, st);
    }
    if (p->output_kind == 1)
        return accumulate_coo_run(b, s, basis, p->walks_per_sample, p->estimator == 1, records, n_records, ws, ws_bytes, out, stats_dev, st);
    return accumulate_run(b, s, basis, p->walks_per_sample, p->estimator == 1, records, n_records, ws, ws_bytes, out, stats_dev, st);
}

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
    L.acc_off = off;     if (with_acc) off += align_up(acc_ws_bytes(b, s, basis, p, L.n_records));
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
    hs->n_prep_queries = (int64_t)h[ST_PREP_QUERIES];
    hs->n_prep_nodes = (int64_t)h[ST_PREP_NODES];
    hs->n_prep_tris = (int64_t)h[ST_PREP_TRIS];
    hs->n_entries = (int64_t)h[ST_ENTRIES];
    hs->n_unique = (int64_t)h[ST_UNIQUE];
    hs->n_far_queries = (int64_t)h[ST_FAR];
    for (int b = 0; b < 16; ++b) hs->nodes_hist[b] = (int64_t)h[ST_HIST + b];
}

int fail(int rc, mcs_stats* hs)
{
    if (hs && rc == MCS_ECUDA) hs->cuda_error = mcs_get_last_cuda_error();
    return rc;
}

// A poisoned call (WalkDyn.err, asynchronous path only: nothing is read back, so no error code can be returned) does not
// leave a plausible matrix behind: the output is filled with NaN.
__global__ void poison_output_kernel(const WalkDyn* __restrict__ dyn, float* __restrict__ out, long long n)
{
    if (!dyn->err) return;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        out[i] = __int_as_float(0x7FC00000);
}

int estimate(const mcs_bvh* b, const mcs_samples* s, const mcs_basis* basis, const mcs_params* p, int exterior,
             void* ws, size_t ws_bytes, const mcs_matrix* out, mcs_stats* hs, void* stream)
{
    if (hs) memset(hs, 0, sizeof *hs);
    if (!b || !s || !basis || !p || !out) return MCS_EINVAL;
    if ((p->output_kind != 0 && p->output_kind != 1) || out->kind != p->output_kind) return MCS_EINVAL;
    if (p->output_kind == 1 && (p->coo_capacity < 1 || out->coo_capacity != p->coo_capacity)) return MCS_EINVAL;
    if (p->walks_per_sample < 1 || s->n_s < 1) return MCS_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    const Layout L = make_layout(b, s, basis, p, exterior, true, true);
    if (hs) hs->workspace_needed = (int64_t)L.total;
    if (!ws || ws_bytes < L.total) return MCS_ENOMEM;
    char* base = (char*)ws;
    float4* records = (float4*)(base + L.records_off);
    unsigned long long* stats_dev = nullptr;
    mcs_prof_mark(MCS_MARK_BEGIN, st);
    // params.nonblocking (dense output in the hat basis, no host_stats): the call only enqueues work -- nothing is read back, nothing is
    // allocated, no host memory is copied -- so it returns at once and may be captured in a CUDA graph.
    // Every other combination blocks (statistics and COO sizes are read back) and reports input errors early.
    if (p->nonblocking != 0 && (p->nonblocking != 1 || hs || p->output_kind != 0 || basis->kind != 0)) return MCS_EINVAL;
    const bool async_path = p->nonblocking == 1;
    int rc = walk_run(b, s, p, exterior, base + L.walk_off, align_up(walk_workspace_bytes(s)), records, nullptr,
                      false, nullptr, hs != nullptr, &stats_dev, st, nullptr, !async_path);
    if (rc != MCS_OK) return fail(rc, hs);
    rc = acc_run(b, s, basis, p, records, L.n_records, base + L.acc_off,
                 align_up(acc_ws_bytes(b, s, basis, p, L.n_records)), out, async_path ? nullptr : stats_dev, st);
    if (rc == MCS_OK && async_path) {
        mcs_note_launch(), poison_output_kernel<<<64, 256, 0, st>>>(walk_dyn_of(stats_dev), out->dense, (long long)out->K * out->K);
        if (cudaGetLastError() != cudaSuccess) rc = MCS_ECUDA;
    }
    mcs_bvh_touch(b, st);
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

__global__ void stream_delay_kernel(unsigned long long ns)
{
    unsigned long long t0, t;
    asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t0));
    do { asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t)); } while (t - t0 < ns);
}

// Both operators of one mesh with their walk kernels overlapped ("The tail"): everything that
// precedes the two walk kernels runs on `st` (the exterior's preparation reads back its Kelvin bounds), then the
// interior walk and its accumulation go to a library-owned high-priority stream and the exterior's to a low-priority
// one, both waiting for the preparation; `st` waits for both at the end.  The exterior's blocks take the SM slots the interior
// launch gives up in its tail, and the interior's accumulation fills the exterior's tail.
// which: 0 = the interior's stream (highest priority: its blocks are dispatched first, so the exterior's bulk runs
// beside the interior's long tail and not the other way round), 1 = the exterior's stream (lowest priority).
// Per host thread: the two side streams (interior: highest priority, exterior: lowest) and the three events of
// estimate_both, created for the thread's current device, recreated when that changes, destroyed with the thread
// (mcs_estimate_dtn_batch runs estimate_both on short-lived worker threads).
struct BothCtx {
    cudaStream_t ss[2] = { nullptr, nullptr };
    cudaEvent_t ev[3] = { nullptr, nullptr, nullptr };
    int dev = -1;
    void release()
    {
        if (dev < 0) return;
        int cur = -1;
        cudaGetDevice(&cur);
        if (cur != dev) cudaSetDevice(dev);
        for (auto& x : ss) { if (x) cudaStreamDestroy(x); x = nullptr; }
        for (auto& x : ev) { if (x) cudaEventDestroy(x); x = nullptr; }
        if (cur >= 0 && cur != dev) cudaSetDevice(cur);
        dev = -1;
    }
    bool ensure()
    {
        int cur = 0;
        if (cudaGetDevice(&cur) != cudaSuccess) return false;
        if (dev == cur) return true;
        release();
        int least = 0, greatest = 0;
        if (cudaDeviceGetStreamPriorityRange(&least, &greatest) != cudaSuccess) return false;
        bool ok = cudaStreamCreateWithPriority(&ss[0], cudaStreamNonBlocking, greatest) == cudaSuccess &&
                  cudaStreamCreateWithPriority(&ss[1], cudaStreamNonBlocking, least) == cudaSuccess;
        for (auto& x : ev) ok = ok && cudaEventCreateWithFlags(&x, cudaEventDisableTiming) == cudaSuccess;
        dev = cur;
        if (!ok) { release(); return false; }
        return true;
    }
    ~BothCtx() { release(); }
};
thread_local BothCtx g_both;

int estimate_both(const mcs_bvh* b, const mcs_samples* s, const mcs_basis* basis,
                  const mcs_params* p_int, const mcs_params* p_ext, void* ws, size_t ws_bytes,
                  const mcs_matrix* out_int, const mcs_matrix* out_ext, mcs_stats* hs_int, mcs_stats* hs_ext, void* stream,
                  float* host_int = nullptr, float* host_ext = nullptr)   // host copies of dense outputs, each on its operator's stream
{
    if (hs_int) memset(hs_int, 0, sizeof *hs_int);
    if (hs_ext) memset(hs_ext, 0, sizeof *hs_ext);
    if (!b || !s || !basis || !p_int || !p_ext || !out_int || !out_ext) return MCS_EINVAL;
    const mcs_params* pp[2] = { p_int, p_ext };
    const mcs_matrix* oo[2] = { out_int, out_ext };
    mcs_stats* hh[2] = { hs_int, hs_ext };
    for (int x = 0; x < 2; ++x) {
        const mcs_params* p = pp[x];
        if ((p->output_kind != 0 && p->output_kind != 1) || oo[x]->kind != p->output_kind) return MCS_EINVAL;
        if (p->output_kind == 1 && (p->coo_capacity < 1 || oo[x]->coo_capacity != p->coo_capacity)) return MCS_EINVAL;
        if (p->walks_per_sample < 1) return MCS_EINVAL;
    }
    if (s->n_s < 1) return MCS_EINVAL;
    if (out_int->kind == out_ext->kind && (out_int->kind == 0 ? out_int->dense == out_ext->dense : out_int->coo_val == out_ext->coo_val))
        return MCS_EINVAL;                            // the two operators run concurrently: separate outputs
    // params.nonblocking (set in BOTH parameter blocks; dense output, hat basis, no host_stats): enqueue only, as in the
    // single calls.  The side streams fork from `stream` by an event and join it again, so the whole call can be captured.
    const bool nb = p_int->nonblocking != 0 || p_ext->nonblocking != 0;
    if (nb && (p_int->nonblocking != 1 || p_ext->nonblocking != 1 || hs_int || hs_ext || host_int || host_ext ||
               p_int->output_kind != 0 || p_ext->output_kind != 0 || basis->kind != 0)) return MCS_EINVAL;
    if (!g_both.ensure()) return MCS_ECUDA;
    cudaStream_t st = (cudaStream_t)stream, st1 = g_both.ss[0], st2 = g_both.ss[1];

    Layout L[2];
    for (int x = 0; x < 2; ++x) L[x] = make_layout(b, s, basis, pp[x], x, true, true);
    const size_t total = L[0].total + L[1].total;
    for (int x = 0; x < 2; ++x) if (hh[x]) hh[x]->workspace_needed = (int64_t)total;
    if (!ws || ws_bytes < total) return MCS_ENOMEM;
    char* base[2] = { (char*)ws, (char*)ws + L[0].total };
    cudaEvent_t ev_prep = g_both.ev[0], ev_done = g_both.ev[1], ev_done1 = g_both.ev[2];
    unsigned long long* stats_dev[2] = { nullptr, nullptr };
    WalkLaunch wl[2];
    mcs_prof_mark(MCS_MARK_BEGIN, st);
    for (int x = 1; x >= 0; --x) {                    // exterior first: its host read-back happens before anything long runs
        int rc = walk_run(b, s, pp[x], x, base[x] + L[x].walk_off, align_up(walk_workspace_bytes(s)),
                          (float4*)(base[x] + L[x].records_off), nullptr, false, nullptr, hh[x] != nullptr, &stats_dev[x], st, &wl[x], !nb);
        if (rc != MCS_OK) return fail(rc, hh[x]);
    }
    // Measured and not kept: both operators' walks as two segments of ONE launch of the batched kernel (no delay kernel, no
    // priorities).  Bit-identical results, but slower: configs[1] 47.6 -> 57.4 ms per call (the per-lane context costs the
    // lean 64-register variant 184 bytes of spills), config 3 walk span 891 -> 1191 ms (interior and exterior lanes, exact
    // and far-field queries share warps and diverge).  The two specialised kernels on two streams stay.
    MCS_CUDA_TRY(cudaEventRecord(ev_prep, st));
    MCS_CUDA_TRY(cudaStreamWaitEvent(st1, ev_prep, 0));
    MCS_CUDA_TRY(cudaStreamWaitEvent(st2, ev_prep, 0));
    mcs_prof_mark(MCS_MARK_WALK_BEGIN, st);
    // Both streams are released by the same event, and which kernel the hardware then dispatches first is a race
    // that the priorities do not settle (measured: 48.4 or 51.6 ms per call at random).  The exterior's stream
    // therefore first runs a one-thread kernel that spins for 30 us: the interior's blocks are all resident by then.
    int rc = walk_launch(&wl[0], st1);
    mcs_prof_mark(MCS_MARK_WALK_END2, st1);
    mcs_note_launch(), stream_delay_kernel<<<1, 1, 0, st2>>>(30000ull);
    if (rc == MCS_OK) rc = walk_launch(&wl[1], st2);
    mcs_prof_mark(MCS_MARK_WALK_END, st2);            // walk_ms: both walk kernels, from the first block to the last
    cudaStream_t ss[2] = { st1, st2 };
    for (int x = 0; x < 2 && rc == MCS_OK; ++x)
        rc = acc_run(b, s, basis, pp[x], (const float4*)(base[x] + L[x].records_off), L[x].n_records, base[x] + L[x].acc_off,
                     align_up(acc_ws_bytes(b, s, basis, pp[x], L[x].n_records)), oo[x], nb ? nullptr : stats_dev[x], ss[x]);
    for (int x = 0; x < 2 && rc == MCS_OK && nb; ++x) {
        mcs_note_launch(), poison_output_kernel<<<64, 256, 0, ss[x]>>>(walk_dyn_of(stats_dev[x]), oo[x]->dense, (long long)oo[x]->K * oo[x]->K);
        if (cudaGetLastError() != cudaSuccess) rc = MCS_ECUDA;
    }
    float* host_out[2] = { host_int, host_ext };
    for (int x = 0; x < 2 && rc == MCS_OK; ++x)
        if (host_out[x] && oo[x]->kind == 0) {        // the interior's download runs beside the exterior's accumulation
            cudaError_t ec = cudaMemcpyAsync(host_out[x], oo[x]->dense, (size_t)oo[x]->K * oo[x]->K * 4, cudaMemcpyDeviceToHost, ss[x]);
            if (ec != cudaSuccess) { mcs_set_last_cuda_error((int)ec); rc = MCS_ECUDA; }
        }
    // join even after an error: the caller's stream must not run ahead of work queued on the second one
    cudaError_t e = cudaEventRecord(ev_done, st2);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(st, ev_done, 0);
    if (e == cudaSuccess) e = cudaEventRecord(ev_done1, st1);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(st, ev_done1, 0);
    mcs_bvh_touch(b, st);                             // after the join: covers both side streams
    if (rc != MCS_OK) return fail(rc, hs_ext);
    if (e != cudaSuccess) { mcs_set_last_cuda_error((int)e); return fail(MCS_ECUDA, hs_ext); }
    mcs_prof_mark(MCS_MARK_END, st);
    for (int x = 0; x < 2; ++x) {
        if (!hh[x]) continue;
        unsigned long long h[ST_COUNT];
        e = cudaMemcpyAsync(h, stats_dev[x], sizeof h, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) { mcs_set_last_cuda_error((int)e); return fail(MCS_ECUDA, hh[x]); }
        fill_stats(hh[x], h, s, L[x].n_records);
        hh[x]->workspace_needed = (int64_t)total;
    }
    return MCS_OK;
}

}  // namespace

extern "C" size_t mcs_workspace_bytes_both(const mcs_bvh* b, const mcs_samples* s, const mcs_basis* basis,
                                           const mcs_params* p_int, const mcs_params* p_ext)
{
    if (!b || !s || !basis || !p_int || !p_ext || s->n_s < 1 || p_int->walks_per_sample < 1 || p_ext->walks_per_sample < 1) return 0;
    return make_layout(b, s, basis, p_int, 0, true, true).total + make_layout(b, s, basis, p_ext, 1, true, true).total;
}

extern "C" int mcs_estimate_dtn_both(const mcs_bvh* b, const mcs_samples* s, const mcs_basis* basis,
                                     const mcs_params* p_int, const mcs_params* p_ext, void* ws, size_t ws_bytes,
                                     const mcs_matrix* out_int, const mcs_matrix* out_ext,
                                     mcs_stats* hs_int, mcs_stats* hs_ext, void* stream)
{
    return estimate_both(b, s, basis, p_int, p_ext, ws, ws_bytes, out_int, out_ext, hs_int, hs_ext, stream);
}

extern "C" unsigned long long mcs_launch_count(void) { return g_launches.load(); }

extern "C" int mcs_profile_enable(int on) { g_prof_on = on ? 1 : 0; return MCS_OK; }

extern "C" int mcs_profile_last(mcs_phase_times* out)
{
    if (!out) return MCS_EINVAL;
    memset(out, 0, sizeof *out);
    if (!g_prof_have) return MCS_EINVAL;
    for (int i = 0; i < MCS_MARK_COUNT; ++i) if (!g_prof_marked[i] && i != MCS_MARK_WALK_END2) return MCS_EINVAL;
    MCS_CUDA_TRY(cudaEventSynchronize(g_prof_ev[MCS_MARK_END]));
    MCS_CUDA_TRY(cudaEventElapsedTime(&out->prep_ms, g_prof_ev[MCS_MARK_BEGIN], g_prof_ev[MCS_MARK_WALK_BEGIN]));
    MCS_CUDA_TRY(cudaEventElapsedTime(&out->walk_ms, g_prof_ev[MCS_MARK_WALK_BEGIN], g_prof_ev[MCS_MARK_WALK_END]));
    MCS_CUDA_TRY(cudaEventElapsedTime(&out->accumulate_ms, g_prof_ev[MCS_MARK_WALK_END], g_prof_ev[MCS_MARK_END]));
    MCS_CUDA_TRY(cudaEventElapsedTime(&out->total_ms, g_prof_ev[MCS_MARK_BEGIN], g_prof_ev[MCS_MARK_END]));
    if (g_prof_marked[MCS_MARK_WALK_END2]) {          // two overlapped walk kernels: the span up to the later end
        float w2 = 0.0f;
        MCS_CUDA_TRY(cudaEventElapsedTime(&w2, g_prof_ev[MCS_MARK_WALK_BEGIN], g_prof_ev[MCS_MARK_WALK_END2]));
        out->walk_interior_ms = w2; out->walk_exterior_ms = out->walk_ms;
        if (w2 > out->walk_ms) out->walk_ms = w2;
        out->accumulate_ms = out->total_ms - out->prep_ms - out->walk_ms;
    }
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

extern "C" int mcs_estimate_dtn_host(const float* verts, int64_t V, const int32_t* faces, int64_t F,
                                     const mcs_samples* hs, const mcs_params* p, int operators,
                                     float* out_interior, float* out_exterior, mcs_stats* stats, void* stream)
{
    if (stats) memset(stats, 0, sizeof *stats);
    if (!verts || !faces || !hs || !p || V < 1 || F < 1 || hs->n_s < 1) return MCS_EINVAL;
    if (!hs->tri || !hs->bary || !hs->weight) return MCS_EINVAL;
    if ((operators & 3) == 0 || (operators & ~3) || p->output_kind != 0) return MCS_EINVAL;
    if (((operators & 1) && !out_interior) || ((operators & 2) && !out_exterior)) return MCS_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    const int64_t n_s = hs->n_s;
    const size_t nb_v = (size_t)V * 12, nb_f = (size_t)F * 12, nb_m = (size_t)V * V * 4;
    const size_t nb_tri = (size_t)n_s * 4, nb_bary = (size_t)n_s * 12, nb_w = (size_t)n_s * 4;
    const size_t nb_n = hs->normal ? (size_t)n_s * 12 : 0;
    // one staging block: verts | faces | tri | bary | weight | normal
    size_t off_v = 0, off_f = align_up(off_v + nb_v), off_t = align_up(off_f + nb_f), off_b = align_up(off_t + nb_tri),
           off_w = align_up(off_b + nb_bary), off_n = align_up(off_w + nb_w), in_total = align_up(off_n + nb_n) + 256;
    {   // keep the stream-ordered pool's memory across calls (default: released at every synchronisation)
        int dev = 0; cudaMemPool_t pool;
        if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetDefaultMemPool(&pool, dev) == cudaSuccess) {
            unsigned long long keep = ~0ull;
            cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
        }
    }
    char* d_in = nullptr; float* d_out = nullptr; void* d_ws = nullptr;
    mcs_bvh* bvh = nullptr;
    int rc = MCS_OK;
    cudaError_t e = cudaMallocAsync((void**)&d_in, in_total, st);
    if (e == cudaSuccess) e = cudaMallocAsync((void**)&d_out, operators == 3 ? 2 * nb_m : nb_m, st);
    if (e != cudaSuccess) { mcs_set_last_cuda_error((int)e); rc = MCS_ENOMEM; goto done; }
    e = cudaMemcpyAsync(d_in + off_v, verts, nb_v, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_in + off_f, faces, nb_f, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_in + off_t, hs->tri, nb_tri, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_in + off_b, hs->bary, nb_bary, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_in + off_w, hs->weight, nb_w, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess && nb_n) e = cudaMemcpyAsync(d_in + off_n, hs->normal, nb_n, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) { mcs_set_last_cuda_error((int)e); rc = MCS_ECUDA; goto done; }
    rc = mcs_build_bvh((const float*)(d_in + off_v), V, (const int32_t*)(d_in + off_f), F, nullptr, stream, &bvh);
    if (rc != MCS_OK) goto done;
    {
        mcs_samples ds;
        ds.tri = (const int32_t*)(d_in + off_t); ds.bary = (const float*)(d_in + off_b);
        ds.weight = (const float*)(d_in + off_w); ds.normal = nb_n ? (const float*)(d_in + off_n) : nullptr;
        ds.n_s = n_s;
        mcs_basis basis; basis.kind = 0; basis.pad_ = 0; basis.K = V;
        mcs_matrix m; memset(&m, 0, sizeof m); m.kind = 0; m.K = V; m.dense = d_out;
        size_t need = 0;
        for (int ext = 0; ext < 2; ++ext)
            if (operators & (1 << ext)) {
                const size_t b = make_layout(bvh, &ds, &basis, p, ext, true, true).total;
                need = b > need ? b : need;
            }
        if (operators == 3) {                         // both: walk kernels overlapped on two streams
            mcs_matrix m2 = m; m2.dense = d_out + (size_t)V * V;
            need = make_layout(bvh, &ds, &basis, p, 0, true, true).total + make_layout(bvh, &ds, &basis, p, 1, true, true).total;
            e = cudaMallocAsync(&d_ws, need, st);
            if (e != cudaSuccess) { mcs_set_last_cuda_error((int)e); rc = MCS_ENOMEM; goto done; }
            rc = estimate_both(bvh, &ds, &basis, p, p, d_ws, need, &m, &m2, nullptr, stats, stream, out_interior, out_exterior);
            goto done;
        }
        e = cudaMallocAsync(&d_ws, need, st);
        if (e != cudaSuccess) { mcs_set_last_cuda_error((int)e); rc = MCS_ENOMEM; goto done; }
        for (int ext = 0; ext < 2 && rc == MCS_OK; ++ext) {
            if (!(operators & (1 << ext))) continue;
            rc = estimate(bvh, &ds, &basis, p, ext, d_ws, need, &m, stats, stream);
            if (rc != MCS_OK) break;
            e = cudaMemcpyAsync(ext ? out_exterior : out_interior, d_out, nb_m, cudaMemcpyDeviceToHost, st);
            if (e != cudaSuccess) { mcs_set_last_cuda_error((int)e); rc = MCS_ECUDA; }
        }
    }
done:
    if (d_ws) cudaFreeAsync(d_ws, st);
    if (d_out) cudaFreeAsync(d_out, st);
    if (d_in) cudaFreeAsync(d_in, st);
    e = cudaStreamSynchronize(st);
    if (rc == MCS_OK && e != cudaSuccess) { mcs_set_last_cuda_error((int)e); rc = MCS_ECUDA; }
    if (bvh) mcs_free_bvh(bvh);
    return fail(rc, stats);
}

// The same from host buffers with the SPARSE output (any V: BASELINE config 3, 2 M faces, ~1 M vertices): upload,
// LBVH build, optional sidedness pre-pass (G-R1), both estimators into device COO buffers of the caller's capacity,
// download of the entries that were written.
extern "C" int mcs_estimate_dtn_host_coo(const float* verts, int64_t V, const int32_t* faces, int64_t F,
                                         const mcs_samples* hs, const mcs_params* p_int, const mcs_params* p_ext,
                                         float orient_h_scale, float orient_beta, mcs_host_coo* out_interior, mcs_host_coo* out_exterior,
                                         mcs_stats* stats_interior, mcs_stats* stats_exterior, void* stream)
{
    if (stats_interior) memset(stats_interior, 0, sizeof *stats_interior);
    if (stats_exterior) memset(stats_exterior, 0, sizeof *stats_exterior);
    if (!verts || !faces || !hs || !p_int || !p_ext || !out_interior || !out_exterior || V < 1 || F < 1 || hs->n_s < 1) return MCS_EINVAL;
    if (!hs->tri || !hs->bary || !hs->weight) return MCS_EINVAL;
    mcs_host_coo* ho[2] = { out_interior, out_exterior };
    for (int x = 0; x < 2; ++x) {
        if (ho[x]->capacity < 1 || !ho[x]->row || !ho[x]->col || !ho[x]->val) return MCS_EINVAL;
        ho[x]->nnz = 0;
    }
    cudaStream_t st = (cudaStream_t)stream;
    const int64_t n_s = hs->n_s;
    const size_t nb_v = (size_t)V * 12, nb_f = (size_t)F * 12;
    const size_t nb_tri = (size_t)n_s * 4, nb_bary = (size_t)n_s * 12, nb_w = (size_t)n_s * 4, nb_n = (size_t)n_s * 12;
    const bool orient = orient_h_scale > 0.0f;
    const bool have_n = orient || hs->normal;
    size_t off_v = 0, off_f = align_up(off_v + nb_v), off_t = align_up(off_f + nb_f), off_b = align_up(off_t + nb_tri),
           off_w = align_up(off_b + nb_bary), off_n = align_up(off_w + nb_w), in_total = align_up(off_n + nb_n) + 256;
    {
        int dev = 0; cudaMemPool_t pool;
        if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetDefaultMemPool(&pool, dev) == cudaSuccess) {
            unsigned long long keep = ~0ull;
            cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
        }
    }
    char* d_in = nullptr; char* d_out = nullptr; void* d_ws = nullptr; void* d_wws = nullptr;
    mcs_bvh* bvh = nullptr;
    int rc = MCS_OK;
    size_t out_off[2], out_total = 0;
    for (int x = 0; x < 2; ++x) { out_off[x] = out_total; out_total += align_up((size_t)ho[x]->capacity * 12 + 64); }
    cudaError_t e = cudaMallocAsync((void**)&d_in, in_total, st);
    if (e == cudaSuccess) e = cudaMallocAsync((void**)&d_out, out_total, st);
    if (e != cudaSuccess) { mcs_set_last_cuda_error((int)e); rc = MCS_ENOMEM; goto done; }
    e = cudaMemcpyAsync(d_in + off_v, verts, nb_v, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_in + off_f, faces, nb_f, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_in + off_t, hs->tri, nb_tri, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_in + off_b, hs->bary, nb_bary, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_in + off_w, hs->weight, nb_w, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess && hs->normal && !orient) e = cudaMemcpyAsync(d_in + off_n, hs->normal, nb_n, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) { mcs_set_last_cuda_error((int)e); rc = MCS_ECUDA; goto done; }
    rc = mcs_build_bvh((const float*)(d_in + off_v), V, (const int32_t*)(d_in + off_f), F, nullptr, stream, &bvh);
    if (rc != MCS_OK) goto done;
    {
        mcs_samples ds;
        ds.tri = (const int32_t*)(d_in + off_t); ds.bary = (const float*)(d_in + off_b);
        ds.weight = (const float*)(d_in + off_w); ds.normal = nullptr; ds.n_s = n_s;
        if (orient && orient_beta > 0.0f) {           // sidedness from the hierarchical evaluation
            rc = mcs_orient_samples_fast(bvh, &ds, orient_h_scale, orient_beta, (float*)(d_in + off_n), nullptr, stream);
            if (rc != MCS_OK) goto done;
        } else if (orient) {                          // sidedness by the winding number (DESIGN.md G-R1)
            const size_t wb = mcs_winding_workspace_bytes(bvh, n_s);
            e = cudaMallocAsync(&d_wws, wb, st);
            if (e != cudaSuccess) { mcs_set_last_cuda_error((int)e); rc = MCS_ENOMEM; goto done; }
            rc = mcs_orient_samples(bvh, &ds, orient_h_scale, (float*)(d_in + off_n), nullptr, d_wws, wb, stream);
            if (rc != MCS_OK) goto done;
        }
        if (have_n) ds.normal = (const float*)(d_in + off_n);
        mcs_basis basis; memset(&basis, 0, sizeof basis); basis.kind = 0; basis.K = V;
        mcs_params pp[2] = { *p_int, *p_ext };
        mcs_matrix mm[2];
        for (int x = 0; x < 2; ++x) {
            pp[x].output_kind = 1; pp[x].coo_capacity = ho[x]->capacity;
            memset(&mm[x], 0, sizeof mm[x]);
            char* o = d_out + out_off[x];
            mm[x].kind = 1; mm[x].K = V; mm[x].coo_capacity = ho[x]->capacity;
            mm[x].coo_nnz = (int64_t*)o;
            mm[x].coo_row = (int32_t*)(o + 64); mm[x].coo_col = mm[x].coo_row + ho[x]->capacity;
            mm[x].coo_val = (float*)(mm[x].coo_col + ho[x]->capacity);
        }
        const size_t need = make_layout(bvh, &ds, &basis, &pp[0], 0, true, true).total + make_layout(bvh, &ds, &basis, &pp[1], 1, true, true).total;
        e = cudaMallocAsync(&d_ws, need, st);
        if (e != cudaSuccess) { mcs_set_last_cuda_error((int)e); rc = MCS_ENOMEM; goto done; }
        rc = estimate_both(bvh, &ds, &basis, &pp[0], &pp[1], d_ws, need, &mm[0], &mm[1], stats_interior, stats_exterior, stream);
        // entry counts first (on MCS_ENOMEM they hold a lower bound of the need), then the entries that were written
        int64_t nnz[2] = { 0, 0 };
        for (int x = 0; x < 2; ++x) {
            cudaError_t ec = cudaMemcpyAsync(&nnz[x], mm[x].coo_nnz, 8, cudaMemcpyDeviceToHost, st);
            if (ec != cudaSuccess && rc == MCS_OK) { mcs_set_last_cuda_error((int)ec); rc = MCS_ECUDA; }
        }
        e = cudaStreamSynchronize(st);
        if (e != cudaSuccess && rc == MCS_OK) { mcs_set_last_cuda_error((int)e); rc = MCS_ECUDA; }
        for (int x = 0; x < 2; ++x) ho[x]->nnz = nnz[x];
        if (rc != MCS_OK) goto done;
        for (int x = 0; x < 2 && e == cudaSuccess; ++x) {
            const size_t nb = (size_t)nnz[x] * 4;
            e = cudaMemcpyAsync(ho[x]->row, mm[x].coo_row, nb, cudaMemcpyDeviceToHost, st);
            if (e == cudaSuccess) e = cudaMemcpyAsync(ho[x]->col, mm[x].coo_col, nb, cudaMemcpyDeviceToHost, st);
            if (e == cudaSuccess) e = cudaMemcpyAsync(ho[x]->val, mm[x].coo_val, nb, cudaMemcpyDeviceToHost, st);
        }
        if (e != cudaSuccess) { mcs_set_last_cuda_error((int)e); rc = MCS_ECUDA; }
    }
done:
    if (d_ws) cudaFreeAsync(d_ws, st);
    if (d_wws) cudaFreeAsync(d_wws, st);
    if (d_out) cudaFreeAsync(d_out, st);
    if (d_in) cudaFreeAsync(d_in, st);
    e = cudaStreamSynchronize(st);
    if (rc == MCS_OK && e != cudaSuccess) { mcs_set_last_cuda_error((int)e); rc = MCS_ECUDA; }
    if (bvh) mcs_free_bvh(bvh);
    return fail(rc, stats_exterior);
}

// ---------------------------------------------------------------------------
// Batch entry point (BASELINE config 4: "1024 seeded synthetic meshes ... interior and exterior DtN ... meshes/s end
// to end"; ~450 k shapes, one shape after another per GPU).  A small mesh cannot keep the device busy: its
// 0.5 M walks are over almost as soon as they start and 90 % of the run is the tail of its longest walks (a 400-jump
// exterior walk is 10 000 dependent node visits).  Running several meshes' kernels side by side on worker streams does
// not help much either (measured 1.4x for 4 streams: every warp of every kernel holds some long walk to the end, so the
// block slots stay taken).  The batch call therefore owns the schedule (see the body): worker threads prepare the
// meshes, ONE persistent launch walks them all, worker threads accumulate.  Every mesh is computed exactly as by the
// single calls (fixed record slots, ordered accumulation): the results do not depend on the workers or the grouping.
// ---------------------------------------------------------------------------
#include <stdlib.h>
#include <thread>
#include <vector>

namespace {

struct BatchMeshState {                     // one item between the phases of the single-launch batch path
    mcs_bvh* bvh = nullptr;
    mcs_samples smp;
    mcs_params p[2];
    Layout L[2];
    char* ws = nullptr;
    size_t ws_bytes = 0;
    WalkLaunch wl[2];
    unsigned long long* stats_dev[2] = { nullptr, nullptr };
    int rc = MCS_OK;
};

}  // namespace

extern "C" int mcs_estimate_dtn_batch(mcs_batch_item* items, int64_t n_items, const mcs_params* p_int, const mcs_params* p_ext,
                                      float orient_h_scale, float orient_beta, int32_t n_workers, void* stream)
{
    if (!items || n_items < 1 || !p_int || !p_ext) return MCS_EINVAL;
    if (p_int->output_kind != 0 || p_ext->output_kind != 0) return MCS_EINVAL;      // dense [K][K] outputs
    if (p_ext->exterior_query != 0) return MCS_EINVAL;                              // the batched launch runs the E3 query
    for (int64_t i = 0; i < n_items; ++i) {
        const mcs_batch_item& it = items[i];
        if (!it.verts || !it.faces || it.V < 1 || it.F < 1 || it.samples.n_s < 1 || !it.samples.tri || !it.samples.bary ||
            !it.samples.weight || !it.out_interior || !it.out_exterior || it.out_interior == it.out_exterior) return MCS_EINVAL;
        if (orient_h_scale > 0.0f && !it.normal_out) return MCS_EINVAL;
        items[i].rc = MCS_OK;
    }
    int dev = 0;
    MCS_CUDA_TRY(cudaGetDevice(&dev));
    int nw = n_workers > 0 ? n_workers : 4;
    if (nw > 16) nw = 16;
    if ((int64_t)nw > n_items) nw = (int)n_items;
    cudaStream_t st = (cudaStream_t)stream;
    cudaEvent_t ev_start = nullptr, ev_walk = nullptr;
    MCS_CUDA_TRY(cudaEventCreateWithFlags(&ev_start, cudaEventDisableTiming));
    MCS_CUDA_TRY(cudaEventCreateWithFlags(&ev_walk, cudaEventDisableTiming));
    MCS_CUDA_TRY(cudaEventRecord(ev_start, st));                 // the workers' streams start after what the caller has queued (uploads)
    std::vector<cudaStream_t> ws(nw, nullptr);
    std::vector<cudaEvent_t> ev_done(nw, nullptr);
    for (int w = 0; w < nw; ++w) {
        if (cudaStreamCreateWithFlags(&ws[w], cudaStreamNonBlocking) != cudaSuccess ||
            cudaEventCreateWithFlags(&ev_done[w], cudaEventDisableTiming) != cudaSuccess) return MCS_ECUDA;
        cudaStreamWaitEvent(ws[w], ev_start, 0);
    }
    int rc_all = MCS_OK;
    // Groups of at most GROUP meshes: within a group (1) the workers build the trees, decide the sides and prepare the
    // walks of their meshes (tangent balls, Z-order), (2) ONE persistent launch runs the walks of both operators of all
    // the group's meshes -- a small mesh alone leaves the device in the tail of its longest walks almost from the
    // start; together the meshes are one job of the size the throughput kernel is made for -- and (3) the workers
    // accumulate their meshes' records into the caller's matrices and free the trees.
    const int64_t GROUP = 64;
    void* batch_scratch = nullptr;
    const size_t batch_scratch_bytes = walk_batch_scratch_bytes((int)(2 * (n_items < GROUP ? n_items : GROUP)));
    if (cudaMallocAsync(&batch_scratch, batch_scratch_bytes, st) != cudaSuccess) return MCS_ENOMEM;
    for (int64_t g0 = 0; g0 < n_items; g0 += GROUP) {
        const int64_t gn = (n_items - g0) < GROUP ? (n_items - g0) : GROUP;
        std::vector<BatchMeshState> state((size_t)gn);
        auto phase1 = [&](int w) {
            cudaSetDevice(dev);
            cudaStream_t s = ws[w];
            for (int64_t k = w; k < gn; k += nw) {
                mcs_batch_item& it = items[g0 + k];
                BatchMeshState& M = state[(size_t)k];
                int rc = mcs_build_bvh(it.verts, it.V, it.faces, it.F, nullptr, s, &M.bvh);
                M.smp = it.samples;
                if (rc == MCS_OK && orient_h_scale > 0.0f) {
                    if (orient_beta > 0.0f) rc = mcs_orient_samples_fast(M.bvh, &M.smp, orient_h_scale, orient_beta, it.normal_out, nullptr, s);
                    else {
                        const size_t wb = mcs_winding_workspace_bytes(M.bvh, M.smp.n_s);
                        void* wws = nullptr;
                        if (cudaMallocAsync(&wws, wb, s) != cudaSuccess) rc = MCS_ENOMEM;
                        else { rc = mcs_orient_samples(M.bvh, &M.smp, orient_h_scale, it.normal_out, nullptr, wws, wb, s); cudaFreeAsync(wws, s); }
                    }
                    M.smp.normal = it.normal_out;
                }
                if (rc == MCS_OK) {
                    M.p[0] = *p_int; M.p[1] = *p_ext;
                    for (int d = 0; d < 3; ++d) M.p[1].kelvin_origin[d] = it.kelvin_origin[d];
                    if (M.p[0].walks_per_sample < 1 || M.p[1].walks_per_sample < 1) rc = MCS_EINVAL;
                }
                if (rc == MCS_OK) {
                    for (int x = 0; x < 2; ++x) M.L[x] = make_layout(M.bvh, &M.smp, &it.basis, &M.p[x], x, true, true);
                    M.ws_bytes = M.L[0].total + M.L[1].total;
                    if (cudaMallocAsync((void**)&M.ws, M.ws_bytes, s) != cudaSuccess) rc = MCS_ENOMEM;
                }
                for (int x = 1; x >= 0 && rc == MCS_OK; --x) {
                    char* base = M.ws + (x ? M.L[0].total : 0);
                    rc = walk_run(M.bvh, &M.smp, &M.p[x], x, base + M.L[x].walk_off, align_up(walk_workspace_bytes(&M.smp)),
                                  (float4*)(base + M.L[x].records_off), nullptr, false, nullptr, false, &M.stats_dev[x], s, &M.wl[x]);
                }
                M.rc = rc;
            }
            cudaEventRecord(ev_done[w], s);
        };
        {
            std::vector<std::thread> threads;
            for (int w = 1; w < nw; ++w) threads.emplace_back(phase1, w);
            phase1(0);
            for (auto& t : threads) t.join();
        }
        // (2) one launch for the walks of every mesh that got this far
        std::vector<WalkLaunch> launches; std::vector<int> ext, far;
        for (int64_t k = 0; k < gn; ++k) {
            const BatchMeshState& M = state[(size_t)k];
            if (M.rc != MCS_OK) continue;
            for (int x = 0; x < 2; ++x) { launches.push_back(M.wl[x]); ext.push_back(x); far.push_back(M.p[x].far_alpha > 0.0f ? 1 : 0); }
        }
        for (int w = 0; w < nw; ++w) cudaStreamWaitEvent(st, ev_done[w], 0);
        int rc2 = MCS_OK;
        if (!launches.empty())
            rc2 = walk_launch_batch(launches.data(), ext.data(), far.data(), (int)launches.size(), batch_scratch, batch_scratch_bytes, st);
        cudaEventRecord(ev_walk, st);
        // (3) accumulation per mesh on the workers' streams
        auto phase3 = [&](int w) {
            cudaSetDevice(dev);
            cudaStream_t s = ws[w];
            cudaStreamWaitEvent(s, ev_walk, 0);
            for (int64_t k = w; k < gn; k += nw) {
                mcs_batch_item& it = items[g0 + k];
                BatchMeshState& M = state[(size_t)k];
                int rc = M.rc != MCS_OK ? M.rc : rc2;
                for (int x = 0; x < 2 && rc == MCS_OK; ++x) {
                    char* base = M.ws + (x ? M.L[0].total : 0);
                    mcs_matrix m; memset(&m, 0, sizeof m);
                    m.kind = 0; m.K = it.basis.K; m.dense = x ? it.out_exterior : it.out_interior;
                    rc = acc_run(M.bvh, &M.smp, &it.basis, &M.p[x], (const float4*)(base + M.L[x].records_off), M.L[x].n_records,
                                 base + M.L[x].acc_off, align_up(acc_ws_bytes(M.bvh, &M.smp, &it.basis, &M.p[x], M.L[x].n_records)),
                                 &m, M.stats_dev[x], s);
                }
                if (M.bvh) { mcs_bvh_touch(M.bvh, s); mcs_free_bvh_on(M.bvh, s); M.bvh = nullptr; }
                if (M.ws) { cudaFreeAsync(M.ws, s); M.ws = nullptr; }
                it.rc = rc;
            }
            cudaEventRecord(ev_done[w], s);
        };
        {
            std::vector<std::thread> threads;
            for (int w = 1; w < nw; ++w) threads.emplace_back(phase3, w);
            phase3(0);
            for (auto& t : threads) t.join();
        }
        for (int w = 0; w < nw; ++w) cudaStreamWaitEvent(st, ev_done[w], 0);
        for (int64_t k = 0; k < gn; ++k) if (items[g0 + k].rc != MCS_OK && rc_all == MCS_OK) rc_all = items[g0 + k].rc;
    }
    cudaFreeAsync(batch_scratch, st);
    cudaError_t e = cudaStreamSynchronize(st);                   // streams and events are destroyed below: wait for them
    for (int w = 0; w < nw; ++w) { cudaStreamSynchronize(ws[w]); cudaStreamDestroy(ws[w]); cudaEventDestroy(ev_done[w]); }
    cudaEventDestroy(ev_start); cudaEventDestroy(ev_walk);
    if (rc_all == MCS_OK && e != cudaSuccess) { mcs_set_last_cuda_error((int)e); rc_all = MCS_ECUDA; }
    return rc_all;
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
    mcs_bvh_touch(b, st);
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
    if ((p->output_kind != 0 && p->output_kind != 1) || out->kind != p->output_kind) return MCS_EINVAL;
    if (p->output_kind == 1 && (p->coo_capacity < 1 || out->coo_capacity != p->coo_capacity)) return MCS_EINVAL;
    const size_t need = align_up(acc_ws_bytes(b, s, basis, p, n_records)) + 512;
    if (hs) hs->workspace_needed = (int64_t)need;
    if (!ws || ws_bytes < need) return MCS_ENOMEM;
    cudaStream_t st = (cudaStream_t)stream;
    unsigned long long* stats_dev = (unsigned long long*)ws;       // first 512 bytes: counters
    MCS_CUDA_TRY(cudaMemsetAsync(stats_dev, 0, ST_COUNT * 8, st));
    int rc = acc_run(b, s, basis, p, (const float4*)records, n_records, (char*)ws + 512, ws_bytes - 512, out, stats_dev, st);
    mcs_bvh_touch(b, st);
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

extern "C" int mcs_knn_weights(const mcs_basis* basis, const float* q, const float* nq, int64_t Q,
                               int32_t* idx, float* w, void* stream)
{
    return knn_weights_run(basis, q, nq, Q, idx, w, (cudaStream_t)stream);
}

extern "C" size_t mcs_accumulate_workspace_bytes(const mcs_bvh* b, const mcs_samples* s, const mcs_basis* basis,
                                                 const mcs_params* p, int64_t n_records)
{
    if (!b || !s || !basis || !p) return 0;
    return align_up(acc_ws_bytes(b, s, basis, p, n_records)) + 512;
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
        case MCS_WNOTCONVERGED: return "warning: iteration stopped at its cap before converging (results written)";
        case MCS_EINVAL: return "invalid argument";
        case MCS_EDEGENERATE: return "degenerate input (zero area, non-finite vertex, or Kelvin origin on a vertex)";
        case MCS_ENOMEM: return "workspace too small or device allocation failed";
        case MCS_ECUDA: return "CUDA runtime error";
        case MCS_ETOOLARGE: return "size beyond the fixed maximum of this entry point";
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
        case 7: return sizeof(mcs_host_coo);
        case 8: return sizeof(mcs_batch_item);
        default: return 0;
    }
}

extern "C" const char* mcs_version(void) { return "mcdtn 0.1 (sm_100a)"; }
