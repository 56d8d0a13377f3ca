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
