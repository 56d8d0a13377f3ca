// scan.cu -- exclusive prefix sums (integer; used for CSR row pointers and compaction offsets).
// Three-kernel hierarchical scan: per-block inclusive scan + block totals, recursive scan of the
// totals, uniform add. Integer arithmetic only, so the result is exact and order-independent.
#include "common.cuh"

namespace {
constexpr int SCAN_THREADS = 256;
constexpr int SCAN_ITEMS = 8;
constexpr int SCAN_BLOCK = SCAN_THREADS * SCAN_ITEMS; // 2048 items per block

template <typename TIn>
__global__ void __launch_bounds__(SCAN_THREADS) k_scan_block(const TIn *__restrict__ in, int64_t *__restrict__ out,
                                                             int64_t n, int64_t *__restrict__ block_sums) {
    __shared__ int64_t warp_tot[SCAN_THREADS / 32];
    const int64_t base = (int64_t)blockIdx.x * SCAN_BLOCK + (int64_t)threadIdx.x * SCAN_ITEMS;
    int64_t v[SCAN_ITEMS];
    int64_t run = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        int64_t idx = base + k;
        run += (idx < n) ? (int64_t)in[idx] : 0;
        v[k] = run;
    }
    // inclusive scan of per-thread totals across the block
    int64_t x = run;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        int64_t y = __shfl_up_sync(0xffffffffu, x, d);
        if (lane >= d) x += y;
    }
    if (lane == 31) warp_tot[warp] = x;
    __syncthreads();
    if (warp == 0) {
        int64_t w = (lane < SCAN_THREADS / 32) ? warp_tot[lane] : 0;
#pragma unroll
        for (int d = 1; d < SCAN_THREADS / 32; d <<= 1) {
            int64_t y = __shfl_up_sync(0xffffffffu, w, d);
            if (lane >= d) w += y;
        }
        if (lane < SCAN_THREADS / 32) warp_tot[lane] = w;
    }
    __syncthreads();
    const int64_t thread_excl = (x - run) + (warp > 0 ? warp_tot[warp - 1] : 0);
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        int64_t idx = base + k;
        if (idx < n) out[idx + 1] = thread_excl + v[k];
    }
    if (threadIdx.x == SCAN_THREADS - 1) block_sums[blockIdx.x] = thread_excl + run;
    if (blockIdx.x == 0 && threadIdx.x == 0) out[0] = 0;
}

__global__ void __launch_bounds__(SCAN_THREADS) k_scan_add(int64_t *__restrict__ out, int64_t n,
                                                           const int64_t *__restrict__ block_offs) {
    const int64_t off = block_offs[blockIdx.x]; // exclusive offsets: block_offs[b] = sum of blocks < b
    if (off == 0) return;
    const int64_t base = (int64_t)blockIdx.x * SCAN_BLOCK;
    for (int k = threadIdx.x; k < SCAN_BLOCK; k += SCAN_THREADS) {
        int64_t idx = base + k;
        if (idx < n) out[idx + 1] += off;
    }
}

template <typename TIn>
void scan_rec(const LaunchCtx &ctx, const TIn *in, int64_t *out, int64_t n, int64_t *ws) {
    const int64_t nb = (n + SCAN_BLOCK - 1) / SCAN_BLOCK;
    int64_t *sums = ws;            // [nb]
    int64_t *offs = ws + nb;       // [nb + 1] exclusive scan of sums
    LAUNCH(ctx, k_scan_block<TIn>, (unsigned)nb, SCAN_THREADS, 0, in, out, n, sums);
    if (nb > 1) {
        scan_rec<int64_t>(ctx, sums, offs, nb, offs + nb + 1);
        LAUNCH(ctx, k_scan_add, (unsigned)nb, SCAN_THREADS, 0, out, n, offs);
    }
}
} // namespace

size_t scan_workspace_bytes(int64_t n) {
    size_t tot = 0;
    while (true) {
        int64_t nb = (n + SCAN_BLOCK - 1) / SCAN_BLOCK;
        tot += (size_t)(2 * nb + 1);
        if (nb <= 1) break;
        n = nb;
    }
    return (tot + 8) * sizeof(int64_t);
}

void exclusive_scan_i32_to_i64(const LaunchCtx &ctx, const int32_t *in, int64_t *out, int64_t n, void *workspace) {
    if (n <= 0) {
        cudaMemsetAsync(out, 0, sizeof(int64_t), ctx.stream);
        return;
    }
    scan_rec<int32_t>(ctx, in, out, n, (int64_t *)workspace);
}

// ---------------------------------------------------------------------------------------------------------------
// reann_row_ptr_noalloc (include/reann.h): the same three-kernel scan for callers that must not allocate (code
// under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc). The block totals and their scanned
// offsets -- the workspace the handle path takes from a cudaMalloc'ed buffer -- live in a file-scope device array
// of fixed size. Every GPU that loads the library holds these 130 KB until the process exits.
//
// In host code `g_scan_scratch` is a host-side stand-in, not a device address: the kernels are given the pointer
// that cudaGetSymbolAddress returns, looked up once per device with that device current.
// ---------------------------------------------------------------------------------------------------------------
#include <mutex>

#include "../../include/reann.h"

struct reann;
int set_err(reann *h, int code, const char *fmt, ...);   // api.cu; h == nullptr: text read by reann_last_error(NULL)

namespace {
// words of workspace scan_rec() touches for n = REANN_NOALLOC_MAX_ROWS (2^24): level 1 has 8192 blocks
// (2*8192 + 1 words), level 2 four (9), level 3 one (3); scan_workspace_bytes(2^24) = 131 240 B. Rounded up to a
// multiple of 256 B.
constexpr int64_t NOALLOC_WORDS = 16640;
static __device__ __align__(256) int64_t g_scan_scratch[NOALLOC_WORDS];

constexpr int NOALLOC_MAX_DEV = 64;
std::mutex g_noalloc_mu;
int64_t *g_noalloc_ptr[NOALLOC_MAX_DEV] = {};   // device address of g_scan_scratch on device d (nullptr: not looked up)
} // namespace

extern "C" int reann_row_ptr_noalloc(const int32_t *counts, int64_t n_rows, int64_t *row_ptr, void *cuda_stream) {
    if (n_rows < 0 || !row_ptr || (n_rows > 0 && !counts))
        return set_err(nullptr, REANN_ERR_ARG, "reann_row_ptr_noalloc: NULL pointer or negative n_rows");
    if (n_rows > (int64_t)REANN_NOALLOC_MAX_ROWS)
        return set_err(nullptr, REANN_ERR_UNSUPPORTED,
                       "reann_row_ptr_noalloc: n_rows = %lld exceeds the static scratch (REANN_NOALLOC_MAX_ROWS = %lld); "
                       "use the handle path",
                       (long long)n_rows, (long long)REANN_NOALLOC_MAX_ROWS);
    if (scan_workspace_bytes(n_rows) > sizeof(int64_t) * (size_t)NOALLOC_WORDS)
        return set_err(nullptr, REANN_ERR_UNSUPPORTED, "reann_row_ptr_noalloc: scratch too small for n_rows = %lld",
                       (long long)n_rows);
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess)
        return set_err(nullptr, REANN_ERR_CUDA, "reann_row_ptr_noalloc: cudaGetDevice failed: %s", cudaGetErrorString(e));
    if (dev < 0 || dev >= NOALLOC_MAX_DEV)
        return set_err(nullptr, REANN_ERR_UNSUPPORTED, "reann_row_ptr_noalloc: device ordinal %d >= %d", dev, NOALLOC_MAX_DEV);
    int64_t *ws = nullptr;
    {
        std::lock_guard<std::mutex> lk(g_noalloc_mu);
        if (!g_noalloc_ptr[dev]) {
            void *p = nullptr;
            e = cudaGetSymbolAddress(&p, g_scan_scratch);   // the current device's copy
            if (e != cudaSuccess || !p)
                return set_err(nullptr, REANN_ERR_CUDA, "reann_row_ptr_noalloc: cudaGetSymbolAddress failed: %s",
                               cudaGetErrorString(e));
            g_noalloc_ptr[dev] = (int64_t *)p;
        }
        ws = g_noalloc_ptr[dev];
    }
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    if (n_rows == 0) {
        e = cudaMemsetAsync(row_ptr, 0, sizeof(int64_t), stream);
    } else {
        // Nothing in the scratch has to start at zero: k_scan_block writes every block total, the recursive scan
        // writes every offset (including offs[0] = 0) before k_scan_add reads it, all in stream order within this
        // call. What the previous call left behind is never read.
        int64_t launches = 0;
        LaunchCtx ctx{stream, &launches, nullptr};
        scan_rec<int32_t>(ctx, counts, row_ptr, n_rows, ws);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess)
        return set_err(nullptr, REANN_ERR_CUDA, "reann_row_ptr_noalloc: launch failed: %s", cudaGetErrorString(e));
    return REANN_OK;
}
