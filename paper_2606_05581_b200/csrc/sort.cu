// sort.cu -- stable LSD radix sort (8 bits per pass) and exclusive scan.
//
// Used by the LBVH build (Morton keys), the Z-order sort of
// the boundary samples and the deterministic accumulation
// (sort (row,col) keys, then segmented sum).  Hand-written:
// no CUB/Thrust on the product path.
//
// One pass = histogram per tile -> exclusive scan of counts[digit][tile] ->
// stable scatter.  Inside a tile a key's position is (warp, round, lane): warp w
// owns 32*ITEMS consecutive keys and reads them 32 at a time, so loads are
// coalesced and the stable rank of a key is
//   (#same digit in earlier warps) + (#same digit in this warp, earlier rounds)
//   + (#same digit in this round at lower lanes),
// the last two from __match_any_sync and one shared counter per (warp, digit).
#include "common.cuh"

namespace {

constexpr int SORT_THREADS = 512;
constexpr int SORT_WARPS = SORT_THREADS / 32;
constexpr int SORT_ITEMS = 16;
constexpr int SORT_TILE = SORT_THREADS * SORT_ITEMS;   // 8192 keys per block

constexpr int SCAN_THREADS = 512;
constexpr int SCAN_ITEMS = 8;
constexpr int SCAN_TILE = SCAN_THREADS * SCAN_ITEMS;   // 4096 counts per block

__device__ __forceinline__ unsigned lanemask_lt()
{
    unsigned m;
    asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
    return m;
}

template <typename K>
__global__ void __launch_bounds__(SORT_THREADS)
radix_hist_kernel(const K* __restrict__ keys, int64_t n, int shift, uint32_t* __restrict__ counts, int nblocks,
                  const uint32_t* __restrict__ n_dev)
{
    __shared__ uint32_t hist[256];
    if (n_dev) {                                        // length known on the device only: the grid covers the capacity
        n = (int64_t)*n_dev;
        if ((int64_t)blockIdx.x * SORT_TILE >= n) {
            if (threadIdx.x < 256) counts[(size_t)threadIdx.x * nblocks + blockIdx.x] = 0;
            return;
        }
    }
    if (threadIdx.x < 256) hist[threadIdx.x] = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t warp_base = (int64_t)blockIdx.x * SORT_TILE + (int64_t)warp * 32 * SORT_ITEMS;
#pragma unroll 4
    for (int r = 0; r < SORT_ITEMS; ++r) {
        int64_t pos = warp_base + r * 32 + lane;
        bool valid = pos < n;
        unsigned d = valid ? (unsigned)((keys[pos] >> shift) & 0xFF) : 0x100u + lane;
        unsigned m = __match_any_sync(0xFFFFFFFFu, d);
        if (valid && (m & lanemask_lt()) == 0) atomicAdd(&hist[d], __popc(m));
    }
    __syncthreads();
    if (threadIdx.x < 256) counts[(size_t)threadIdx.x * nblocks + blockIdx.x] = hist[threadIdx.x];
}

// Stable scatter of one tile.  The keys of a tile are first put in digit order in shared memory (their stable
// local rank is known), then written out: consecutive threads write consecutive addresses of one digit's run, so
// the global writes are coalesced (a direct scatter writes 4-8 bytes into 32 different sectors per warp).
template <typename K>
__global__ void __launch_bounds__(SORT_THREADS)
radix_scatter_kernel(const K* __restrict__ kin, const uint32_t* __restrict__ vin,
                     K* __restrict__ kout, uint32_t* __restrict__ vout,
                     int64_t n, int shift, const uint32_t* __restrict__ offsets, int nblocks,
                     const uint32_t* __restrict__ n_dev)
{
    extern __shared__ __align__(16) unsigned char sort_smem[];
    if (n_dev) {
        n = (int64_t)*n_dev;
        if ((int64_t)blockIdx.x * SORT_TILE >= n) return;
    }
    K* skey = reinterpret_cast<K*>(sort_smem);                                   // [SORT_TILE]
    uint32_t* sval = reinterpret_cast<uint32_t*>(skey + SORT_TILE);              // [SORT_TILE]
    uint32_t (*cnt)[256] = reinterpret_cast<uint32_t (*)[256]>(sval + SORT_TILE); // [SORT_WARPS][256]
    uint32_t* lstart = &cnt[0][0] + SORT_WARPS * 256;                            // [256] first local slot of a digit
    uint32_t* gbase = lstart + 256;                                              // [256] first global slot of a digit (this tile)
    uint32_t* wsum = gbase + 256;                                                // [8]
    for (int i = threadIdx.x; i < SORT_WARPS * 256; i += SORT_THREADS) (&cnt[0][0])[i] = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t block_base = (int64_t)blockIdx.x * SORT_TILE;
    const int64_t warp_base = block_base + (int64_t)warp * 32 * SORT_ITEMS;
    K key[SORT_ITEMS];
    uint32_t rank[SORT_ITEMS];
#pragma unroll
    for (int r = 0; r < SORT_ITEMS; ++r) {
        int64_t pos = warp_base + r * 32 + lane;
        bool valid = pos < n;
        key[r] = valid ? kin[pos] : (K)0;
        unsigned d = valid ? (unsigned)((key[r] >> shift) & 0xFF) : 0x100u + lane;
        unsigned m = __match_any_sync(0xFFFFFFFFu, d);
        int leader = __ffs(m) - 1;
        uint32_t old = 0;
        if (valid && lane == leader) { old = cnt[warp][d]; cnt[warp][d] = old + __popc(m); }
        old = __shfl_sync(0xFFFFFFFFu, old, leader);
        rank[r] = old + __popc(m & lanemask_lt());
        __syncwarp();
    }
    __syncthreads();
    // per digit: counts of the warps -> exclusive offsets inside the digit; digit totals -> exclusive scan over digits
    uint32_t total = 0;
    if (threadIdx.x < 256) {
#pragma unroll
        for (int w = 0; w < SORT_WARPS; ++w) { uint32_t c = cnt[w][threadIdx.x]; cnt[w][threadIdx.x] = total; total += c; }
        gbase[threadIdx.x] = offsets[(size_t)threadIdx.x * nblocks + blockIdx.x];
    }
    uint32_t inc = total;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { uint32_t t = __shfl_up_sync(0xFFFFFFFFu, inc, o); if (lane >= o) inc += t; }
    if (threadIdx.x < 256 && lane == 31) wsum[warp] = inc;
    __syncthreads();
    if (threadIdx.x < 256) {
        uint32_t before = 0;
        for (int w = 0; w < warp; ++w) before += wsum[w];
        lstart[threadIdx.x] = before + inc - total;
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < SORT_ITEMS; ++r) {
        int64_t pos = warp_base + r * 32 + lane;
        if (pos < n) {
            unsigned d = (unsigned)((key[r] >> shift) & 0xFF);
            uint32_t lp = lstart[d] + cnt[warp][d] + rank[r];
            skey[lp] = key[r];
            sval[lp] = vin[pos];
        }
    }
    __syncthreads();
    const int64_t left = n - block_base;
    const int count = (int)(left < SORT_TILE ? left : SORT_TILE);
    for (int j = threadIdx.x; j < count; j += SORT_THREADS) {
        const K k = skey[j];
        const unsigned d = (unsigned)((k >> shift) & 0xFF);
        const uint32_t dst = gbase[d] + ((uint32_t)j - lstart[d]);
        kout[dst] = k;
        vout[dst] = sval[j];
    }
}

template <typename K>
constexpr size_t scatter_smem_bytes() { return (size_t)SORT_TILE * (sizeof(K) + 4) + (size_t)SORT_WARPS * 256 * 4 + 2 * 256 * 4 + 64; }

// ------------------------------ scan ---------------------------------------
__device__ __forceinline__ uint32_t block_exclusive_scan(uint32_t v, uint32_t* total)
{
    __shared__ uint32_t warp_sums[SCAN_THREADS / 32];
    __shared__ uint32_t block_total;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { uint32_t t = __shfl_up_sync(0xFFFFFFFFu, inc, o); if (lane >= o) inc += t; }
    if (lane == 31) warp_sums[warp] = inc;
    __syncthreads();
    if (warp == 0) {
        uint32_t s = lane < SCAN_THREADS / 32 ? warp_sums[lane] : 0, si = s;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { uint32_t t = __shfl_up_sync(0xFFFFFFFFu, si, o); if (lane >= o) si += t; }
        if (lane < SCAN_THREADS / 32) warp_sums[lane] = si - s;
        if (lane == 31) block_total = si;
    }
    __syncthreads();
    *total = block_total;
    uint32_t r = warp_sums[warp] + inc - v;
    __syncthreads();
    return r;
}

// mode 0: write the tile total to sums[blockIdx]; mode 1: write the scanned tile,
// offset by sums[blockIdx] (already exclusive-scanned) when sums != NULL.
__global__ void __launch_bounds__(SCAN_THREADS)
scan_tile_kernel(const uint32_t* in, uint32_t* out, int64_t n,   // in may alias out
                 uint32_t* sums, int mode, uint32_t* total_out)
{
    const int64_t base = (int64_t)blockIdx.x * SCAN_TILE + (int64_t)threadIdx.x * SCAN_ITEMS;
    uint32_t v[SCAN_ITEMS], s = 0;
#pragma unroll
    for (int i = 0; i < SCAN_ITEMS; ++i) { v[i] = (base + i < n) ? in[base + i] : 0u; s += v[i]; }
    uint32_t total;
    uint32_t ex = block_exclusive_scan(s, &total);
    if (mode == 0) {
        if (threadIdx.x == 0) sums[blockIdx.x] = total;
        return;
    }
    uint32_t off = sums ? sums[blockIdx.x] : 0u;
    uint32_t run = ex + off;
#pragma unroll
    for (int i = 0; i < SCAN_ITEMS; ++i) { if (base + i < n) out[base + i] = run; run += v[i]; }
    if (total_out && blockIdx.x == gridDim.x - 1 && threadIdx.x == SCAN_THREADS - 1) *total_out = run;
}

// the sorted pairs ended up in the alternate buffers: copy them home (length known on the device only)
template <typename K>
__global__ void copy_pairs_devn_kernel(const K* __restrict__ kin, const uint32_t* __restrict__ vin, K* __restrict__ kout,
                                       uint32_t* __restrict__ vout, const uint32_t* __restrict__ n_dev)
{
    const int64_t n = (int64_t)*n_dev;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        kout[i] = kin[i];
        vout[i] = vin[i];
    }
}

// n_dev == nullptr: n pairs.  n_dev != nullptr: *n_dev <= n pairs (n is the capacity: it sizes the grids and the
// workspace; nothing is read back, so the call never blocks the host).
template <typename K>
int radix_sort_impl(K* keys, uint32_t* vals, int64_t n, int key_bits, void* ws, size_t ws_bytes, cudaStream_t st,
                    const uint32_t* n_dev = nullptr)
{
    if (n < 0 || key_bits < 0 || key_bits > (int)sizeof(K) * 8) return MCS_EINVAL;
    if (n <= 1 || key_bits == 0) return MCS_OK;
    if (n >= ((int64_t)1 << 32)) return MCS_EINVAL;
    if (ws_bytes < sort_workspace_bytes(n, sizeof(K))) return MCS_ENOMEM;
    const int nblocks = (int)ceil_div64(n, SORT_TILE);
    char* p = (char*)ws;
    K* kalt = (K*)p;                 p += align_up((size_t)n * sizeof(K));
    uint32_t* valt = (uint32_t*)p;   p += align_up((size_t)n * sizeof(uint32_t));
    uint32_t* counts = (uint32_t*)p; p += align_up((size_t)256 * nblocks * sizeof(uint32_t));
    void* scan_ws = p;
    size_t scan_ws_bytes = ws_bytes - (size_t)(p - (char*)ws);
    K* kin = keys; uint32_t* vin = vals; K* kout = kalt; uint32_t* vout = valt;
    const int passes = (key_bits + 7) / 8;
    {
        static bool attr_set = false;                       // per instantiation (K)
        if (!attr_set) {
            MCS_CUDA_TRY(cudaFuncSetAttribute(radix_scatter_kernel<K>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)scatter_smem_bytes<K>()));
            attr_set = true;
        }
    }
    for (int pass = 0; pass < passes; ++pass) {
        int shift = pass * 8;
        mcs_note_launch(), radix_hist_kernel<K><<<nblocks, SORT_THREADS, 0, st>>>(kin, n, shift, counts, nblocks, n_dev);
        int rc = exclusive_scan_u32(counts, counts, (int64_t)256 * nblocks, nullptr, scan_ws, scan_ws_bytes, st);
        if (rc != MCS_OK) return rc;
        mcs_note_launch(), radix_scatter_kernel<K><<<nblocks, SORT_THREADS, scatter_smem_bytes<K>(), st>>>(kin, vin, kout, vout, n, shift, counts, nblocks, n_dev);
        K* tk = kin; kin = kout; kout = tk;
        uint32_t* tv = vin; vin = vout; vout = tv;
    }
    if (kin != keys && n_dev) {
        const unsigned nb = (unsigned)(nblocks < 1184 ? nblocks : 1184);
        mcs_note_launch(), copy_pairs_devn_kernel<K><<<nb, 512, 0, st>>>(kin, vin, keys, vals, n_dev);
    } else if (kin != keys) {
        MCS_CUDA_TRY(cudaMemcpyAsync(keys, kin, (size_t)n * sizeof(K), cudaMemcpyDeviceToDevice, st));
        MCS_CUDA_TRY(cudaMemcpyAsync(vals, vin, (size_t)n * sizeof(uint32_t), cudaMemcpyDeviceToDevice, st));
    }
    MCS_CUDA_TRY(cudaGetLastError());
    return MCS_OK;
}

}  // namespace

size_t scan_workspace_bytes(int64_t n)
{
    size_t total = 0;
    while (n > SCAN_TILE) {
        n = ceil_div64(n, SCAN_TILE);
        total += align_up((size_t)n * sizeof(uint32_t));
    }
    return total + 256;
}

int exclusive_scan_u32(const uint32_t* in, uint32_t* out, int64_t n, uint32_t* total_out,
                       void* ws, size_t ws_bytes, cudaStream_t st)
{
    if (n <= 0) {
        if (total_out) MCS_CUDA_TRY(cudaMemsetAsync(total_out, 0, sizeof(uint32_t), st));
        return MCS_OK;
    }
    if (ws_bytes < scan_workspace_bytes(n)) return MCS_ENOMEM;
    const int64_t nb = ceil_div64(n, SCAN_TILE);
    if (nb == 1) {
        mcs_note_launch(), scan_tile_kernel<<<1, SCAN_THREADS, 0, st>>>(in, out, n, nullptr, 1, total_out);
    } else {
        uint32_t* sums = (uint32_t*)ws;
        char* rest = (char*)ws + align_up((size_t)nb * sizeof(uint32_t));
        size_t rest_bytes = ws_bytes - align_up((size_t)nb * sizeof(uint32_t));
        mcs_note_launch(), scan_tile_kernel<<<(unsigned)nb, SCAN_THREADS, 0, st>>>(in, nullptr, n, sums, 0, nullptr);
        int rc = exclusive_scan_u32(sums, sums, nb, nullptr, rest, rest_bytes, st);
        if (rc != MCS_OK) return rc;
        mcs_note_launch(), scan_tile_kernel<<<(unsigned)nb, SCAN_THREADS, 0, st>>>(in, out, n, sums, 1, total_out);
    }
    MCS_CUDA_TRY(cudaGetLastError());
    return MCS_OK;
}

size_t sort_workspace_bytes(int64_t n, int key_bytes)
{
    if (n < 1) n = 1;
    const int64_t nblocks = ceil_div64(n, SORT_TILE);
    return align_up((size_t)n * key_bytes) + align_up((size_t)n * sizeof(uint32_t)) +
           align_up((size_t)256 * nblocks * sizeof(uint32_t)) + scan_workspace_bytes(256 * nblocks) + 256;
}

int sort_pairs_u64(uint64_t* keys, uint32_t* vals, int64_t n, int key_bits, void* ws, size_t ws_bytes, cudaStream_t st)
{
    return radix_sort_impl<uint64_t>(keys, vals, n, key_bits, ws, ws_bytes, st);
}

int sort_pairs_u32(uint32_t* keys, uint32_t* vals, int64_t n, int key_bits, void* ws, size_t ws_bytes, cudaStream_t st)
{
    return radix_sort_impl<uint32_t>(keys, vals, n, key_bits, ws, ws_bytes, st);
}

int sort_pairs_u32_devn(uint32_t* keys, uint32_t* vals, int64_t n_cap, const uint32_t* n_dev, int key_bits,
                        void* ws, size_t ws_bytes, cudaStream_t st)
{
    if (!n_dev) return MCS_EINVAL;
    return radix_sort_impl<uint32_t>(keys, vals, n_cap, key_bits, ws, ws_bytes, st, n_dev);
}

// ---------------------------------------------------------------------------
// mcs_sort_pairs_u64_static -- the same sort for callers that may not allocate (CUDA graph capture, serving loops,
// harnesses that forbid cudaMalloc) and have no workspace to pass: the workspace is a file-scope device array, so
// every GPU that loads this library holds MCS_SORT_STATIC_BYTES (12.25 MiB) until the process exits.  Limit:
// MCS_SORT_STATIC_MAX_N = 2^20 pairs.  The entry point calls no cudaMalloc / cudaFree / allocating routine; the
// kernels are those of mcs_sort_pairs_u64 (radix_sort_impl above), so the result is the same stable order.
// Every call on a device shares the one array: two calls that overlap on the GPU (different streams, no ordering
// between them) race on it.  Nothing in it has to start at zero -- the histogram kernel writes every count of a
// pass before the scan reads it, and the alternate key/value buffers are written before they are read -- so what the
// previous call left there is harmless (tests/test_zz_no_alloc.py runs two calls of different sizes in a row).
// ---------------------------------------------------------------------------
#define MCS_SORT_STATIC_MAX_N (1 << 20)
#define MCS_SORT_STATIC_BYTES ((size_t)MCS_SORT_STATIC_MAX_N * 12 + (256u << 10))
static __device__ __align__(256) unsigned char g_sort_static_scratch[MCS_SORT_STATIC_BYTES];

namespace {
constexpr int SORT_STATIC_MAX_DEVICES = 64;
void* g_sort_static_ptr[SORT_STATIC_MAX_DEVICES];      // device address of the array on each device, once resolved
std::mutex g_sort_static_mutex;
}  // namespace

extern "C" int64_t mcs_sort_static_max_n(void) { return MCS_SORT_STATIC_MAX_N; }

extern "C" int mcs_sort_pairs_u64_static(uint64_t* keys, uint32_t* vals, int64_t n, int32_t key_bits, void* stream)
{
    if (n < 0 || (n > 0 && (!keys || !vals))) return MCS_EINVAL;
    if (n > MCS_SORT_STATIC_MAX_N) return MCS_ETOOLARGE;                // more pairs than the static scratch holds
    if (sort_workspace_bytes(n, 8) > MCS_SORT_STATIC_BYTES) return MCS_ETOOLARGE;
    int dev = 0;
    MCS_CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= SORT_STATIC_MAX_DEVICES) return MCS_EINVAL;
    void* ptr = nullptr;
    {
        // In host code `g_sort_static_scratch` is a host-side stand-in, not a device address: resolve it once per
        // device, with that device current (it is: cudaGetDevice above).
        std::lock_guard<std::mutex> lock(g_sort_static_mutex);
        if (!g_sort_static_ptr[dev]) {
            void* p = nullptr;
            const cudaError_t e = cudaGetSymbolAddress(&p, g_sort_static_scratch);
            if (e != cudaSuccess || !p) { (void)cudaGetLastError(); return MCS_ECUDA; }
            g_sort_static_ptr[dev] = p;
        }
        ptr = g_sort_static_ptr[dev];
    }
    return radix_sort_impl<uint64_t>(keys, vals, n, key_bits, ptr, MCS_SORT_STATIC_BYTES, (cudaStream_t)stream);
}
