// dense_tc.cu -- rows A6+A7 / A9 of SURVEY.md section 8(a) on the 5th-generation tensor cores:
// the per-species GEMM chain of the folded contraction + atomic NN (Eq. 1 outer sums + Eq. 2,
// PAPER.md:35-43) and of its reverse pass (Eq. 5 / Appendix B steps 1-2), as tcgen05.mma
// kind::tf32 with FP32 accumulators in tensor memory (TMEM).
//
// FP32-class accuracy from TF32 operands ("3xTF32"): every operand x is split into
//   x_hi = x rounded to 10 mantissa bits,   x_lo = x - x_hi   (exact in FP32, then rounded to TF32)
// and each product is issued as  A_lo B_hi + A_hi B_lo  (first, while the accumulator is small)
// followed by  A_hi B_hi;  the dropped A_lo B_lo term is 2^-22 relative.
// The tensor core adds into its FP32 accumulator with truncation (measured on B200: one
// accumulator over K = 576 carries a -6e-6 relative bias, 10x the error of an FP32 FMA loop), so
// K is cut into groups of 32 (64 in the last reverse GEMM, whose result only feeds the forces): every group
// accumulates into a fresh TMEM buffer (three buffers in rotation) which the compute threads then add into
// FP32 registers with round-to-nearest.
//
// One CTA = one tile of 128 atoms of one species (UMMA M = 128, cta_group::1):
//   forward   z1 = Q U + b1;  h1 = SiLU(z1);  z2 = h1 W2 + b2;  h2 = SiLU(z2);  out = h2 W3 + b3
//   reverse   h2bar = outbar W3^T; z2bar = h2bar SiLU'(z2); h1bar = z2bar W2^T; z1bar = h1bar SiLU'(z1);
//             Qbar = z1bar U^T
// (Q = radial-pair products of the neighbour sums b, U = folded contraction x first layer; see
// dense.cu for the algebra.) The two GEMMs with K or N = n_out <= 16 (W3) are done in FP32 on the
// plain ALUs by the compute threads: they are < 3 % of the flops and carry the output precision.
//
// Threads: 8 compute warps + 1 control warp. Compute thread (w, lane) owns tile row
// m = 32 (w % 4) + lane (= its TMEM lane) and the column half w / 4 of every accumulator; it
// converts raw operands to hi/lo images, drains group accumulators into registers, applies
// bias / SiLU / stash and produces the next GEMM's A operand. One lane of the control warp streams
// operands with cp.async.bulk (pre-split weight chunk images; raw Q chunks), issues the MMAs and
// commits them to mbarriers. K is processed in chunks of 32 floats.
//
// Global "tile-quad" layout of Q, Qbar and the z stash (shared with gram.cu):
//   element (tile, column q, row r) at float offset  (tile * ncol/4 + q/4) * 512 + r * 4 + q % 4
// i.e. [tile][q/4][128 rows][4]: a K chunk of 32 columns is one contiguous 16 KB block already in
// the order of the shared-memory operand, and a warp (32 rows) reads / writes 512 contiguous bytes.
//
// Shared-memory operand layout (no swizzle, K-major "core matrices" of 8 rows x 16 bytes):
//   element (row r, k) of a [R][32] chunk lives at byte  (k/4)*(R*16) + r*16 + (k%4)*4,
//   i.e. LBO (K direction) = R*16 bytes, SBO (row-group direction) = 128 bytes; the lo image
//   follows the hi image. Weight chunks are stored in global memory in exactly this image
//   (built once in reann_create), so one bulk copy per chunk brings hi and lo.
#include "common.cuh"
#include "tc_common.cuh"

namespace {
using namespace tc;

constexpr int TM = DENSE_TC_TM;        // 128 rows (atoms) per tile
constexpr int KC = 32;                 // floats per K chunk
constexpr int NSTAGE = 3;              // ring depth (A slot + B slot per stage)
constexpr int NASLOT = 4;              // A slots: 0-2 ring / resident operands, 3 = raw-Q staging (forward)
constexpr int A_HALF = TM * KC * 4;    // bytes of one A image (hi or lo) = one raw Q chunk
constexpr int A_SLOT = 2 * A_HALF;     // 32 KB
constexpr int B_SLOT = 2 * 128 * KC * 4; // 32 KB (N <= 128)
constexpr int SM_A = 0, SM_B = NASLOT * A_SLOT, SM_BAR = SM_B + NSTAGE * B_SLOT;
constexpr int SM_TOTAL = SM_BAR + 256;
constexpr uint32_t A_LBO = TM * 16;
constexpr int NCOMPUTE = 256, NTHREADS = NCOMPUTE + 64, CTL_WARP = 8, COPY_WARP = 9;   // warp 8 issues the MMAs, warp 9 the bulk copies
constexpr uint32_t COL_BUF = 128;      // TMEM columns per group buffer
constexpr int NBUF = 3;                // group buffers: one filling, one complete, one being drained
constexpr uint32_t TMEM_COLS = 512;    // allocation (power of two >= NBUF * COL_BUF)
constexpr uint32_t COL_A = NBUF * COL_BUF; // forward GEMM 1: A operand (hi | lo images of a Q chunk) in TMEM, two slots of 64 columns
constexpr uint32_t A_TSLOT = 2 * KC;

// barrier slots (8 bytes each) in the barrier area
enum { BAR_BFULL = 0, BAR_MMA = 3, BAR_AFULL = 6, BAR_AH = 9, BAR_QFULL = 13, BAR_QEMPTY = 15, BAR_DFULL = 17,
       BAR_DEMPTY = 20, BAR_ARES = 23, BAR_TDONE = 24, BAR_COUNT = 25 };

// Optional timeline trace of one CTA (development aid, compiled only with -DREANN_TC_TRACE):
// role 0 = control thread, 1 = compute thread 0; slot k = clock64().
#ifdef REANN_TC_TRACE
__device__ long long g_tc_trace[2 * 2 * 128];
#define TC_TRACE(kern, role, k)                                                                      \
    do {                                                                                             \
        if (blockIdx.x == 5 && (k) < 128) g_tc_trace[((kern) * 2 + (role)) * 128 + (k)] = clock64(); \
    } while (0)
#else
#define TC_TRACE(kern, role, k) ((void)0)
#endif

__device__ __forceinline__ void compute_sync() { asm volatile("bar.sync 1, 256;" ::: "memory"); } // the 8 compute warps
__device__ __forceinline__ void store_split4(unsigned char *a_slot, int k4, int row, const float *x) {
    float4 h, l;
    split_tf32(x[0], h.x, l.x); split_tf32(x[1], h.y, l.y); split_tf32(x[2], h.z, l.z); split_tf32(x[3], h.w, l.w);
    float4 *p = reinterpret_cast<float4 *>(a_slot + k4 * (int)A_LBO + row * 16);
    p[0] = h;
    p[A_HALF / 16] = l;
}

__device__ __forceinline__ float silu_f(float z) { return __fdividef(z, 1.0f + __expf(-z)); }
__device__ __forceinline__ float dsilu_f(float z) {
    const float s = __fdividef(1.0f, 1.0f + __expf(-z));
    return s * (1.0f + z * (1.0f - s));
}

// ---- common prologue / epilogue of both kernels ----
__device__ __forceinline__ uint32_t tc_prologue(unsigned char *smem, uint32_t *tmem_base_s, uint32_t ah_count) {
    const int tid = threadIdx.x, warp = tid >> 5;
    const uint32_t bar0 = smem_u32(smem + SM_BAR);
    if (tid == 0) {
        for (int s = 0; s < NSTAGE; ++s) {
            mbar_init(bar0 + 8 * (BAR_BFULL + s), 1);
            mbar_init(bar0 + 8 * (BAR_MMA + s), 1);
            mbar_init(bar0 + 8 * (BAR_AFULL + s), NCOMPUTE);
        }
        for (int k = 0; k < 4; ++k) mbar_init(bar0 + 8 * (BAR_AH + k), ah_count);
        for (int d = 0; d < 2; ++d) {
            mbar_init(bar0 + 8 * (BAR_QFULL + d), 1);
            mbar_init(bar0 + 8 * (BAR_QEMPTY + d), NCOMPUTE);
        }
        for (int d = 0; d < NBUF; ++d) {
            mbar_init(bar0 + 8 * (BAR_DFULL + d), 1);
            mbar_init(bar0 + 8 * (BAR_DEMPTY + d), NCOMPUTE);
        }
        mbar_init(bar0 + 8 * BAR_ARES, NCOMPUTE);
        mbar_init(bar0 + 8 * BAR_TDONE, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == CTL_WARP) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_base_s)), "r"(TMEM_COLS)
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    return *tmem_base_s;
}
__device__ __forceinline__ void tc_epilogue(uint32_t tmem) {
    tc_fence_before();
    __syncthreads();
    if ((int)(threadIdx.x >> 5) == CTL_WARP)
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(TMEM_COLS) : "memory");
}

// ---- control-thread helpers ----
// The kernels are persistent (a CTA walks over tiles): `sb` / `gb` are the steps / accumulator groups issued for
// earlier tiles, so that ring slots and mbarrier parities run on over tile boundaries; i and g are tile-local.
struct Ctl {
    uint32_t bar0, a0, b0, tmem;
    int sb, gb;
    bool tf32;   // REANN_MLP_MODE=tf32: hi images only, one accumulator per GEMM (see mma_chunk_1x)
    __device__ __forceinline__ uint32_t bar(int k) const { return bar0 + 8u * (uint32_t)k; }
    // stream the weight chunk of step i into its B slot (after the MMAs of step i-3 released it)
    __device__ __forceinline__ void copy_b(int i_loc, const float *src, int n_rows) const {
        const int i = sb + i_loc;
        const int s = i % NSTAGE;
        if (i >= NSTAGE) mbar_wait(bar(BAR_MMA + s), (uint32_t)(((i / NSTAGE) - 1) & 1));
        const uint32_t bytes = (uint32_t)n_rows * KC * 4 * (tf32 ? 1 : 2);     // the lo image follows the hi image
        if (elect_one()) {
            mbar_expect_tx(bar(BAR_BFULL + s), bytes);
            bulk_g2s(b0 + (uint32_t)s * B_SLOT, src, bytes, bar(BAR_BFULL + s));
        }
        __syncwarp();
    }
    // One K chunk = one accumulation group (step i, group buffer i % NBUF):
    //   D[:, 0:n) = A_lo B_hi^T + A_hi B_lo^T  (4 x K = 8),  then  D += A_hi B_hi^T  (4 x K = 8)
    __device__ __forceinline__ void mma_chunk(int i_loc, int a_slot, int n_rows, int g_loc) const {
        const int i = sb + i_loc, g = gb + g_loc;
        const int s = i % NSTAGE, d = g % NBUF;
        if (g >= NBUF) mbar_wait(bar(BAR_DEMPTY + d), (uint32_t)(((g / NBUF) - 1) & 1));
        mbar_wait(bar(BAR_BFULL + s), (uint32_t)((i / NSTAGE) & 1));
        tc_fence_after();
        const uint32_t dm = tmem + COL_BUF * (uint32_t)d;
        if (elect_one()) {
            issue(i, a_slot, n_rows, dm, true, false, true);
            issue(i, a_slot, n_rows, dm, false, true, false);
            tc_commit(bar(BAR_MMA + s));
            tc_commit(bar(BAR_DFULL + d));
        }
        __syncwarp();
    }
    // Plain TF32 (the fast mode with a restated tolerance): D (+)= A_hi B_hi^T only, the chunks of one GEMM accumulate
    // in ONE buffer (first: overwrite; last: hand the buffer to the compute threads) -- one TMEM drain per GEMM
    __device__ __forceinline__ void mma_chunk_1x(int i_loc, int a_slot, int n_rows, int g_loc, bool first, bool last) const {
        const int i = sb + i_loc, g = gb + g_loc;
        const int s = i % NSTAGE, d = g % NBUF;
        if (first && g >= NBUF) mbar_wait(bar(BAR_DEMPTY + d), (uint32_t)(((g / NBUF) - 1) & 1));
        mbar_wait(bar(BAR_BFULL + s), (uint32_t)((i / NSTAGE) & 1));
        tc_fence_after();
        const uint32_t dm = tmem + COL_BUF * (uint32_t)d;
        if (elect_one()) {
            issue(i, a_slot, n_rows, dm, false, true, first);
            tc_commit(bar(BAR_MMA + s));
            if (last) tc_commit(bar(BAR_DFULL + d));
        }
        __syncwarp();
    }
    // The same two with the A operand in tensor memory (TS form: `a_col` = first column of the hi image, lo image KC
    // columns further): the MMAs then read only B from shared memory
    __device__ __forceinline__ void mma_chunk_ts(int i_loc, uint32_t a_col, int n_rows, int g_loc) const {
        const int i = sb + i_loc, g = gb + g_loc;
        const int s = i % NSTAGE, d = g % NBUF;
        if (g >= NBUF) mbar_wait(bar(BAR_DEMPTY + d), (uint32_t)(((g / NBUF) - 1) & 1));
        mbar_wait(bar(BAR_BFULL + s), (uint32_t)((i / NSTAGE) & 1));
        tc_fence_after();
        const uint32_t dm = tmem + COL_BUF * (uint32_t)d;
        if (elect_one()) {
            issue_ts(i, a_col, n_rows, dm, true, false, true);
            issue_ts(i, a_col, n_rows, dm, false, true, false);
            tc_commit(bar(BAR_MMA + s));
            tc_commit(bar(BAR_DFULL + d));
        }
        __syncwarp();
    }
    __device__ __forceinline__ void mma_chunk_1x_ts(int i_loc, uint32_t a_col, int n_rows, int g_loc, bool first, bool last) const {
        const int i = sb + i_loc, g = gb + g_loc;
        const int s = i % NSTAGE, d = g % NBUF;
        if (first && g >= NBUF) mbar_wait(bar(BAR_DEMPTY + d), (uint32_t)(((g / NBUF) - 1) & 1));
        mbar_wait(bar(BAR_BFULL + s), (uint32_t)((i / NSTAGE) & 1));
        tc_fence_after();
        const uint32_t dm = tmem + COL_BUF * (uint32_t)d;
        if (elect_one()) {
            issue_ts(i, a_col, n_rows, dm, false, true, first);
            tc_commit(bar(BAR_MMA + s));
            if (last) tc_commit(bar(BAR_DFULL + d));
        }
        __syncwarp();
    }
    __device__ __forceinline__ void issue_ts(int i, uint32_t a_col, int n_rows, uint32_t dm, bool corr, bool main, bool fresh) const {
        const int s = i % NSTAGE;
        const uint32_t idesc = make_idesc(n_rows);
        const uint32_t a_hi = tmem + a_col, a_lo = a_hi + KC;
        const uint32_t b_lbo = (uint32_t)n_rows * 16;
        const uint32_t b_hi = b0 + (uint32_t)s * B_SLOT, b_lo = b_hi + (uint32_t)n_rows * KC * 4;
#pragma unroll
        for (int kk = 0; kk < KC / 8; ++kk) {
            const uint64_t bh = make_desc(b_hi + kk * 2 * b_lbo, b_lbo), bl = make_desc(b_lo + kk * 2 * b_lbo, b_lbo);
            if (corr) {
                umma_tf32_ts(dm, a_lo + kk * 8, bh, idesc, (fresh && kk == 0) ? 0u : 1u);
                umma_tf32_ts(dm, a_hi + kk * 8, bl, idesc, 1u);
            }
            if (main) umma_tf32_ts(dm, a_hi + kk * 8, bh, idesc, (fresh && !corr && kk == 0) ? 0u : 1u);
        }
    }
    // Two K chunks (steps i, i+1) = one accumulation group of K = 64: all corrections first, then hi.hi of both
    __device__ __forceinline__ void mma_pair(int i_loc, int a_slot0, int a_slot1, int n_rows, int g_loc) const {
        const int i = sb + i_loc, g = gb + g_loc;
        const int d = g % NBUF;
        if (g >= NBUF) mbar_wait(bar(BAR_DEMPTY + d), (uint32_t)(((g / NBUF) - 1) & 1));
        mbar_wait(bar(BAR_BFULL + i % NSTAGE), (uint32_t)((i / NSTAGE) & 1));
        mbar_wait(bar(BAR_BFULL + (i + 1) % NSTAGE), (uint32_t)(((i + 1) / NSTAGE) & 1));
        tc_fence_after();
        const uint32_t dm = tmem + COL_BUF * (uint32_t)d;
        if (elect_one()) {
            issue(i, a_slot0, n_rows, dm, true, false, true);
            issue(i + 1, a_slot1, n_rows, dm, true, false, false);
            issue(i, a_slot0, n_rows, dm, false, true, false);
            tc_commit(bar(BAR_MMA + i % NSTAGE));
            issue(i + 1, a_slot1, n_rows, dm, false, true, false);
            tc_commit(bar(BAR_MMA + (i + 1) % NSTAGE));
            tc_commit(bar(BAR_DFULL + d));
        }
        __syncwarp();
    }
    // mma_pair with the hi image of the A operand in tensor memory (columns a_col0 / a_col1) and the lo image in the
    // shared-memory slots: two of the three products per K step then read only B from shared memory
    __device__ __forceinline__ void mma_pair_mixed(int i_loc, int a_slot0, int a_slot1, uint32_t a_col0, uint32_t a_col1, int n_rows,
                                                   int g_loc) const {
        const int i = sb + i_loc, g = gb + g_loc;
        const int d = g % NBUF;
        if (g >= NBUF) mbar_wait(bar(BAR_DEMPTY + d), (uint32_t)(((g / NBUF) - 1) & 1));
        mbar_wait(bar(BAR_BFULL + i % NSTAGE), (uint32_t)((i / NSTAGE) & 1));
        mbar_wait(bar(BAR_BFULL + (i + 1) % NSTAGE), (uint32_t)(((i + 1) / NSTAGE) & 1));
        tc_fence_after();
        const uint32_t dm = tmem + COL_BUF * (uint32_t)d;
        if (elect_one()) {
            issue_mixed(i, a_slot0, a_col0, n_rows, dm, true, false, true);
            issue_mixed(i + 1, a_slot1, a_col1, n_rows, dm, true, false, false);
            issue_mixed(i, a_slot0, a_col0, n_rows, dm, false, true, false);
            tc_commit(bar(BAR_MMA + i % NSTAGE));
            issue_mixed(i + 1, a_slot1, a_col1, n_rows, dm, false, true, false);
            tc_commit(bar(BAR_MMA + (i + 1) % NSTAGE));
            tc_commit(bar(BAR_DFULL + d));
        }
        __syncwarp();
    }
    __device__ __forceinline__ void issue_mixed(int i, int a_slot, uint32_t a_col, int n_rows, uint32_t dm, bool corr, bool main,
                                                bool fresh) const {
        const int s = i % NSTAGE;
        const uint32_t idesc = make_idesc(n_rows);
        const uint32_t a_lo = a0 + (uint32_t)a_slot * A_SLOT + A_HALF, a_hi = tmem + a_col;
        const uint32_t b_lbo = (uint32_t)n_rows * 16;
        const uint32_t b_hi = b0 + (uint32_t)s * B_SLOT, b_lo = b_hi + (uint32_t)n_rows * KC * 4;
#pragma unroll
        for (int kk = 0; kk < KC / 8; ++kk) {
            const uint64_t al = make_desc(a_lo + kk * 2 * A_LBO, A_LBO);
            const uint64_t bh = make_desc(b_hi + kk * 2 * b_lbo, b_lbo), bl = make_desc(b_lo + kk * 2 * b_lbo, b_lbo);
            if (corr) {
                umma_tf32(dm, al, bh, idesc, (fresh && kk == 0) ? 0u : 1u);
                umma_tf32_ts(dm, a_hi + kk * 8, bl, idesc, 1u);
            }
            if (main) umma_tf32_ts(dm, a_hi + kk * 8, bh, idesc, (fresh && !corr && kk == 0) ? 0u : 1u);
        }
    }
    // the MMAs of one chunk: corrections (A_lo B_hi + A_hi B_lo) and / or main (A_hi B_hi); fresh: overwrite D first
    __device__ __forceinline__ void issue(int i, int a_slot, int n_rows, uint32_t dm, bool corr, bool main, bool fresh) const {
        const int s = i % NSTAGE;
        const uint32_t idesc = make_idesc(n_rows);
        const uint32_t a_hi = a0 + (uint32_t)a_slot * A_SLOT, a_lo = a_hi + A_HALF;
        const uint32_t b_lbo = (uint32_t)n_rows * 16;
        const uint32_t b_hi = b0 + (uint32_t)s * B_SLOT, b_lo = b_hi + (uint32_t)n_rows * KC * 4;
#pragma unroll
        for (int kk = 0; kk < KC / 8; ++kk) {
            const uint64_t ah = make_desc(a_hi + kk * 2 * A_LBO, A_LBO), al = make_desc(a_lo + kk * 2 * A_LBO, A_LBO);
            const uint64_t bh = make_desc(b_hi + kk * 2 * b_lbo, b_lbo), bl = make_desc(b_lo + kk * 2 * b_lbo, b_lbo);
            if (corr) {
                umma_tf32(dm, al, bh, idesc, (fresh && kk == 0) ? 0u : 1u);
                umma_tf32(dm, ah, bl, idesc, 1u);
            }
            if (main) umma_tf32(dm, ah, bh, idesc, (fresh && !corr && kk == 0) ? 0u : 1u);
        }
    }
};

// ---- compute-thread helpers ----
// acc[0..CW) += group buffer of step g, columns [col0, col0 + CW) of this thread's TMEM lane
template <int CW>
__device__ __forceinline__ void drain_group(float *acc, uint32_t bar0, uint32_t tl, int g, int col0, bool read) {
    const int d = g % NBUF;
    mbar_wait(bar0 + 8 * (BAR_DFULL + d), (uint32_t)((g / NBUF) & 1));
    tc_fence_after();
    if (read) {
        const uint32_t ta = tl + COL_BUF * (uint32_t)d + (uint32_t)col0;
        if constexpr (CW == 16) {
            uint32_t v[16];
            tmem_ld16(ta, v);
            tmem_wait_ld();
#pragma unroll
            for (int k = 0; k < 16; ++k) acc[k] += __uint_as_float(v[k]);
        } else {
            uint32_t v[CW];
#pragma unroll
            for (int c = 0; c < CW / 32; ++c) tmem_ld32(ta + c * 32, v + c * 32);
            tmem_wait_ld();
#pragma unroll
            for (int k = 0; k < CW; ++k) acc[k] += __uint_as_float(v[k]);
        }
    }
    tc_fence_before();
    mbar_arrive(bar0 + 8 * (BAR_DEMPTY + d));
}
// wait until the MMAs that last read stage (i % NSTAGE) are complete
__device__ __forceinline__ void wait_stage_free(uint32_t bar0, int i) {
    if (i >= NSTAGE) mbar_wait(bar0 + 8 * (BAR_MMA + i % NSTAGE), (uint32_t)(((i / NSTAGE) - 1) & 1));
}
// x[0..CW) (columns col0 .. of row m) -> hi/lo images in A slots col/32; arrives on the chunk barriers
template <int CW>
__device__ __forceinline__ void store_operand(const float *x, unsigned char *a_base, uint32_t bar0, int col0, int m) {
#pragma unroll
    for (int k4 = 0; k4 < CW / 4; ++k4) {
        const int col = col0 + k4 * 4;
        store_split4(a_base + (col >> 5) * A_SLOT, (col & 31) >> 2, m, x + k4 * 4);
    }
    fence_async_smem();
#pragma unroll
    for (int c = 0; c < (CW + 31) / 32; ++c) mbar_arrive(bar0 + 8 * (BAR_AH + (col0 >> 5) + c));
}
// The same, four columns at a time from inside the activation loop: x4 = columns [col0 + 4 k4, + 4) of row m. A 32-column
// chunk is published as soon as this thread's share of it is written, so that the next GEMM starts on the first chunks
// while the threads are still working on the later ones.
template <int CW>
__device__ __forceinline__ void store4_publish(const float *x4, unsigned char *a_base, uint32_t bar0, int col0, int k4, int m) {
    const int col = col0 + 4 * k4;
    store_split4(a_base + (col >> 5) * A_SLOT, (col & 31) >> 2, m, x4);
    if (((col + 4) & 31) == 0 || k4 == CW / 4 - 1) {
        fence_async_smem();
        mbar_arrive(bar0 + 8 * (BAR_AH + (col >> 5)));
    }
}
// Order in which the K chunks of a GEMM whose A operand comes out of an activation phase are consumed: the two column
// halves of the compute threads finish their chunks in parallel (0 and NCH/2 first), so the chunks are taken alternately
__host__ __device__ constexpr int chunk_order(int k, int nch) { return nch >= 4 ? ((k & 1) ? nch / 2 + k / 2 : k / 2) : k; }
__host__ __device__ constexpr int cdiv(int a, int b) { return (a + b - 1) / b; }

// ============================================================================ forward
struct TcFwdArgs {
    const DenseWT *w;       // [S]
    const DenseTile *tiles; // 128-atom tiles
    const int32_t *sp_list;
    const float *Q;         // tile-quad layout, K1 columns
    float *z_stash;         // tile-quad layout, zs columns (z1 | z2)
    float *out;             // rows of stride out_stride, atom order
    int out_stride, K1, nout, zs, n_tiles, tf32;
    const int32_t *skip;    // see LaunchCtx
};

template <int NCH1, int NCH2>
__global__ void __launch_bounds__(NTHREADS, 1) k_dense_tc_fwd(TcFwdArgs A) {
    SKIP_GUARD(A.skip);
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ uint32_t tmem_base_s;
    constexpr int H1p = NCH1 * 32, H2p = NCH2 * 32, CW1 = H1p / 2, CW2 = H2p / 2;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int warp_u = __shfl_sync(0xffffffffu, warp, 0);           // warp-uniform for the compiler
    const uint32_t bar0 = smem_u32(smem + SM_BAR);
    const uint32_t tmem = tc_prologue(smem, &tmem_base_s, CW1 >= 32 ? 128u : 256u);
    const int n1 = A.K1 / KC, total = n1 + NCH1;
    // running counters over the tiles of this CTA: steps (B ring, MMA barriers), groups (TMEM buffers), Q chunks (A ring)
    int sb = 0, gb = 0, qb = 0, it = 0;

    // Two control warps, each walking its own warp-uniform control flow with one elected lane acting: the MMA warp only
    // waits for operands / a free accumulator and issues (a tcgen05.mma is accepted at the pace of the tensor pipe, so
    // anything else this warp did between two chunks would leave the pipe idle); the copy warp streams the weight
    // chunks and the raw Q chunks ahead of it, paced by the ring barriers alone.
    if (warp_u == CTL_WARP) {
        Ctl c{bar0, smem_u32(smem + SM_A), smem_u32(smem + SM_B), tmem, 0, 0, A.tf32 != 0};
        for (int tile_idx = blockIdx.x; tile_idx < A.n_tiles; tile_idx += gridDim.x, ++it) {
            c.sb = sb; c.gb = gb;
            for (int i = 0; i < total; ++i) {
                if (i < n1) {
                    const int j = qb + i, sa = j % NSTAGE;
                    mbar_wait(c.bar(BAR_AFULL + sa), (uint32_t)((j / NSTAGE) & 1));
                    TC_TRACE(0, 0, 2 * i);
                    const uint32_t a_col = COL_A + A_TSLOT * (uint32_t)(i & 1);
                    if (A.tf32) c.mma_chunk_1x_ts(i, a_col, H1p, 0, i == 0, i == n1 - 1);
                    else c.mma_chunk_ts(i, a_col, H1p, i);
                } else {
                    const int kq = chunk_order(i - n1, NCH1);
                    mbar_wait(c.bar(BAR_AH + kq), (uint32_t)(it & 1));
                    TC_TRACE(0, 0, 2 * i);
                    if (A.tf32) c.mma_chunk_1x(i, kq, H2p, 1, i == n1, i == total - 1);
                    else c.mma_chunk(i, kq, H2p, i);
                }
                TC_TRACE(0, 0, 2 * i + 1);
            }
            sb += total; gb += A.tf32 ? 2 : total; qb += n1;
        }
    } else if (warp_u == COPY_WARP) {
        Ctl c{bar0, smem_u32(smem + SM_A), smem_u32(smem + SM_B), tmem, 0, 0, A.tf32 != 0};
        const uint32_t stg = c.a0 + 3u * A_SLOT;
        for (int tile_idx = blockIdx.x; tile_idx < A.n_tiles; tile_idx += gridDim.x, ++it) {
            const DenseTile tile = A.tiles[tile_idx];
            const DenseWT W = A.w[tile.species];
            const float *Qt = A.Q + (size_t)tile_idx * A.K1 * TM;
            c.sb = sb; c.gb = gb;
            auto issue_q = [&](int j_loc) {   // raw Q chunk -> staging buffer (J & 1)
                const int j = qb + j_loc, qs = j & 1;
                if (j >= 2) mbar_wait(c.bar(BAR_QEMPTY + qs), (uint32_t)(((j >> 1) - 1) & 1));
                if (elect_one()) {
                    mbar_expect_tx(c.bar(BAR_QFULL + qs), A_HALF);
                    bulk_g2s(stg + (uint32_t)qs * A_HALF, Qt + (size_t)j_loc * (KC * TM), A_HALF, c.bar(BAR_QFULL + qs));
                }
                __syncwarp();
            };
            auto copy_b = [&](int i) {
                if (i < n1) c.copy_b(i, W.g1 + (size_t)i * (2 * H1p * KC), H1p);
                else c.copy_b(i, W.g2 + (size_t)chunk_order(i - n1, NCH1) * (2 * H2p * KC), H2p);
            };
            copy_b(0);
            if (total > 1) copy_b(1);
            // the staging area doubles as the fourth operand slot of GEMM 2: wait for the previous tile to be done
            if (it > 0) mbar_wait(c.bar(BAR_TDONE), (uint32_t)((it - 1) & 1));
            issue_q(0);
            if (n1 > 1) issue_q(1);
            for (int i = 0; i < total; ++i) {
                if (i + 2 < n1) issue_q(i + 2);       // waits for the conversion of chunk i (its staging half)
                if (i + 2 < total) copy_b(i + 2);     // waits for the MMAs of step i - 1 (its ring slot)
            }
            sb += total; gb += A.tf32 ? 2 : total; qb += n1;
        }
    } else {
        const int m = (warp & 3) * 32 + lane, hf = warp >> 2;
        const uint32_t tl = tmem + ((uint32_t)((warp & 3) * 32) << 16);
        unsigned char *a_base = smem + SM_A;
        for (int tile_idx = blockIdx.x; tile_idx < A.n_tiles; tile_idx += gridDim.x, ++it) {
            const DenseTile tile = A.tiles[tile_idx];
            const DenseWT W = A.w[tile.species];
            const bool valid = m < tile.count;
            float *zt = A.z_stash + (size_t)tile_idx * A.zs * TM + m * 4;   // + (col/4) * 512
            if (tid == 0) TC_TRACE(0, 1, 100);
            // ---- GEMM 1: z1 = Q U.  Convert raw Q chunk i (staging -> hi/lo A slot), drain group i-1 ----
            float acc1[CW1];
#pragma unroll
            for (int c = 0; c < CW1; ++c) acc1[c] = 0.f;
#pragma unroll 1
            for (int i = 0; i < n1; ++i) {
                const int j = qb + i, sa = j % NSTAGE, qs = j & 1;
                mbar_wait(bar0 + 8 * (BAR_QFULL + qs), (uint32_t)((j >> 1) & 1));
                // TMEM operand slot i & 1: the MMAs of chunk i - 2 (this tile) must have read it
                if (i >= 2) { const int st = sb + i - 2; mbar_wait(bar0 + 8 * (BAR_MMA + st % NSTAGE), (uint32_t)((st / NSTAGE) & 1)); }
                tc_fence_after();
                // my row of the raw chunk, K columns [16 hf, 16 hf + 16): hi / lo images straight into tensor memory
                const unsigned char *stg = smem + SM_A + 3 * A_SLOT + qs * A_HALF;
                uint32_t hi[16], lo[16];
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const float4 v = *reinterpret_cast<const float4 *>(stg + (4 * hf + q) * (int)A_LBO + m * 16);
                    const float x[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        float h, l;
                        split_tf32(x[u], h, l);
                        hi[4 * q + u] = __float_as_uint(h); lo[4 * q + u] = __float_as_uint(l);
                    }
                }
                const uint32_t ta = tl + COL_A + A_TSLOT * (uint32_t)(i & 1) + 16u * (uint32_t)hf;
                tmem_st16(ta, hi);
                if (!A.tf32) tmem_st16(ta + KC, lo);
                tmem_wait_st();
                tc_fence_before();
                mbar_arrive(bar0 + 8 * (BAR_AFULL + sa));
                mbar_arrive(bar0 + 8 * (BAR_QEMPTY + qs));
                if (tid == 0) TC_TRACE(0, 1, 2 * i);
                if (i >= 1 && !A.tf32) drain_group<CW1>(acc1, bar0, tl, gb + i - 1, hf * CW1, true);
                if (tid == 0) TC_TRACE(0, 1, 2 * i + 1);
            }
            drain_group<CW1>(acc1, bar0, tl, A.tf32 ? gb : gb + n1 - 1, hf * CW1, true);
            if (tid == 0) TC_TRACE(0, 1, 101);
            // ---- z1 = acc + b1 (stash), h1 = SiLU(z1) -> A operand of GEMM 2 ----
#pragma unroll
            for (int k4 = 0; k4 < CW1 / 4; ++k4) {
                const int col = hf * CW1 + k4 * 4;
                const float4 b4 = __ldg(reinterpret_cast<const float4 *>(W.b1 + col));
                const float4 z = make_float4(acc1[k4 * 4] + b4.x, acc1[k4 * 4 + 1] + b4.y, acc1[k4 * 4 + 2] + b4.z,
                                             acc1[k4 * 4 + 3] + b4.w);
                if (valid) *reinterpret_cast<float4 *>(zt + (size_t)(col >> 2) * (TM * 4)) = z;
                const float h4[4] = {silu_f(z.x), silu_f(z.y), silu_f(z.z), silu_f(z.w)};
                store4_publish<CW1>(h4, a_base, bar0, hf * CW1, k4, m);
            }
            if (tid == 0) TC_TRACE(0, 1, 102);
            // ---- GEMM 2: z2 = h1 W2 ----
            float acc2[CW2];
#pragma unroll
            for (int c = 0; c < CW2; ++c) acc2[c] = 0.f;
            if (A.tf32) drain_group<CW2>(acc2, bar0, tl, gb + 1, hf * CW2, true);
            else {
#pragma unroll 1
                for (int kc = 0; kc < NCH1; ++kc) drain_group<CW2>(acc2, bar0, tl, gb + n1 + kc, hf * CW2, true);
            }
            if (tid == 0) TC_TRACE(0, 1, 103);
            // every MMA of the tile has completed (its last group is drained): the staging area may take the next tile's
            // first Q chunks while this tile's second activation phase runs
            if (tid == 0) mbar_arrive(bar0 + 8 * BAR_TDONE);
            // ---- z2 (stash), h2 = SiLU(z2), out = h2 W3 + b3 in FP32 (partial over this column half) ----
            float o[16];
#pragma unroll
            for (int c = 0; c < 16; ++c) o[c] = 0.f;
            // z2 = acc + b2 (stash), h2 = SiLU(z2) in place
#pragma unroll
            for (int k4 = 0; k4 < CW2 / 4; ++k4) {
                const int col = hf * CW2 + k4 * 4;
                const float4 b4 = __ldg(reinterpret_cast<const float4 *>(W.b2 + col));
                const float4 z = make_float4(acc2[k4 * 4] + b4.x, acc2[k4 * 4 + 1] + b4.y, acc2[k4 * 4 + 2] + b4.z,
                                             acc2[k4 * 4 + 3] + b4.w);
                if (valid) *reinterpret_cast<float4 *>(zt + (size_t)((H1p + col) >> 2) * (TM * 4)) = z;
                acc2[k4 * 4] = silu_f(z.x); acc2[k4 * 4 + 1] = silu_f(z.y);
                acc2[k4 * 4 + 2] = silu_f(z.z); acc2[k4 * 4 + 3] = silu_f(z.w);
            }
            if (A.nout == 1) {          // energy layer: one column of W3, four partial sums
                float o4[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
                for (int k4 = 0; k4 < CW2 / 4; ++k4) {
                    const float4 w4 = __ldg(reinterpret_cast<const float4 *>(W.w3c0 + hf * CW2 + k4 * 4));
                    o4[0] = fmaf(acc2[k4 * 4], w4.x, o4[0]); o4[1] = fmaf(acc2[k4 * 4 + 1], w4.y, o4[1]);
                    o4[2] = fmaf(acc2[k4 * 4 + 2], w4.z, o4[2]); o4[3] = fmaf(acc2[k4 * 4 + 3], w4.w, o4[3]);
                }
                o[0] = (o4[0] + o4[1]) + (o4[2] + o4[3]);
            } else {
#pragma unroll
                for (int c = 0; c < CW2; ++c) {
                    const float4 *wr = reinterpret_cast<const float4 *>(W.w3p + (size_t)(hf * CW2 + c) * 16);
                    const float hvc = acc2[c];
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        const float4 w4 = __ldg(wr + q);
                        o[q * 4] = fmaf(hvc, w4.x, o[q * 4]); o[q * 4 + 1] = fmaf(hvc, w4.y, o[q * 4 + 1]);
                        o[q * 4 + 2] = fmaf(hvc, w4.z, o[q * 4 + 2]); o[q * 4 + 3] = fmaf(hvc, w4.w, o[q * 4 + 3]);
                    }
                }
            }
            // combine the two column halves through shared memory (A slot 0 is free: every MMA has completed)
            float *xch = reinterpret_cast<float *>(smem + SM_A);
            if (hf == 1) {
#pragma unroll
                for (int q = 0; q < 4; ++q)
                    *reinterpret_cast<float4 *>(xch + (q * TM + m) * 4) = make_float4(o[q * 4], o[q * 4 + 1], o[q * 4 + 2], o[q * 4 + 3]);
            }
            compute_sync();
            if (hf == 0 && valid) {
                float *dst = A.out + (size_t)A.sp_list[tile.start + m] * A.out_stride;
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const float4 p4 = *reinterpret_cast<const float4 *>(xch + (q * TM + m) * 4);
                    const float pv[4] = {p4.x, p4.y, p4.z, p4.w};
#pragma unroll
                    for (int u = 0; u < 4; ++u)
                        if (q * 4 + u < A.nout) dst[q * 4 + u] = (o[q * 4 + u] + pv[u]) + __ldg(W.b3 + q * 4 + u);
                }
            }
            if (tid == 0) TC_TRACE(0, 1, 104);
            // tile done: the exchange area (operand slot 0) is next written in the first activation phase of the next
            // tile, which every thread reaches only through that tile's GEMM 1 barriers
            compute_sync();
            sb += total; gb += A.tf32 ? 2 : total; qb += n1;
        }
    }
    tc_epilogue(tmem);
}

// ============================================================================ reverse
struct TcBwdArgs {
    const DenseWT *w;
    const DenseTile *tiles;
    const int32_t *sp_list;
    const float *z_stash, *outbar; // outbar == nullptr: energy layer (outbar = 1)
    float *Qbar;                   // tile-quad layout, K1 columns
    int outbar_stride, K1, nout, zs, n_tiles, tf32;
    const int32_t *skip;
};

template <int NCH1, int NCH2>
__global__ void __launch_bounds__(NTHREADS, 1) k_dense_tc_bwd(TcBwdArgs A) {
    SKIP_GUARD(A.skip);
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ uint32_t tmem_base_s;
    constexpr int H1p = NCH1 * 32, H2p = NCH2 * 32, CW1 = H1p / 2, CW2 = H2p / 2;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int warp_u = __shfl_sync(0xffffffffu, warp, 0);           // warp-uniform for the compiler
    const uint32_t bar0 = smem_u32(smem + SM_BAR);
    const uint32_t tmem = tc_prologue(smem, &tmem_base_s, CW2 >= 32 ? 128u : 256u);
    // steps: [R1 (only when outbar is given: K = n_out padded to 32)] NCH2 x R2, nblk x NCH1 x R3
    constexpr int GR3 = NCH1 >= 2 ? 2 : 1;         // K chunks per accumulator group of R3
    const int o1 = A.outbar ? 1 : 0, i3 = o1 + NCH2;
    const int nblk = (A.K1 + 127) / 128, total = i3 + nblk * NCH1, ngroups = i3 + nblk * (NCH1 / GR3);
    int sb = 0, gb = 0, it = 0;                     // running steps / groups / tiles of this CTA (persistent kernel)

    auto rows_of = [&](int i) { return i < o1 ? H2p : i < i3 ? H1p : min(128, A.K1 - ((i - i3) / NCH1) * 128); };
    if (warp_u == CTL_WARP) {
        // MMA warp (see k_dense_tc_fwd): waits for operands / a free accumulator and issues, nothing else
        Ctl c{bar0, smem_u32(smem + SM_A), smem_u32(smem + SM_B), tmem, 0, 0, A.tf32 != 0};
        for (int tile_idx = blockIdx.x; tile_idx < A.n_tiles; tile_idx += gridDim.x, ++it) {
            c.sb = sb; c.gb = gb;
            for (int i = 0; i < total; ++i) {
                if (i < o1) {
                    mbar_wait(c.bar(BAR_AFULL), (uint32_t)(it & 1));
                    TC_TRACE(1, 0, 2 * i);
                    if (A.tf32) c.mma_chunk_1x(i, 0, H2p, 0, true, true);
                    else c.mma_chunk(i, 0, H2p, i);
                } else if (i < i3) {
                    const int kq = chunk_order(i - o1, NCH2);
                    mbar_wait(c.bar(BAR_AH + kq), (uint32_t)(it & 1));
                    TC_TRACE(1, 0, 2 * i);
                    if (A.tf32) c.mma_chunk_1x(i, kq, H1p, o1, i == o1, i == i3 - 1);
                    else c.mma_chunk(i, kq, H1p, i);
                } else if (A.tf32) {
                    // R3, plain TF32: one accumulator per block of <= 128 output columns (K = H1p)
                    if (i == i3) mbar_wait(c.bar(BAR_ARES), (uint32_t)(it & 1));
                    const int nb = (i - i3) / NCH1, kc = (i - i3) % NCH1;
                    c.mma_chunk_1x(i, kc, rows_of(i), o1 + 1 + nb, kc == 0, kc == NCH1 - 1);
                } else {
                    // R3: groups of GR3 chunks (K = 32 GR3 per accumulator); group index continues after R2
                    if (i == i3) mbar_wait(c.bar(BAR_ARES), (uint32_t)(it & 1));
                    const int kc = (i - i3) % NCH1, g = i3 + (i - i3) / GR3;
                    TC_TRACE(1, 0, 2 * i);
                    if (GR3 == 2) {
                        c.mma_pair_mixed(i, kc, kc + 1, COL_A + KC * (uint32_t)kc, COL_A + KC * (uint32_t)(kc + 1), rows_of(i), g);
                        TC_TRACE(1, 0, 2 * i + 1);
                        ++i;
                        continue;
                    } else {
                        c.mma_chunk(i, kc, rows_of(i), g);
                    }
                }
                TC_TRACE(1, 0, 2 * i + 1);
            }
            sb += total; gb += A.tf32 ? o1 + 1 + nblk : ngroups;
        }
    } else if (warp_u == COPY_WARP) {
        // copy warp: the weight chunks of every step, as far ahead as the ring allows (a slot is free when the MMAs of
        // the step three back have completed)
        Ctl c{bar0, smem_u32(smem + SM_A), smem_u32(smem + SM_B), tmem, 0, 0, A.tf32 != 0};
        for (int tile_idx = blockIdx.x; tile_idx < A.n_tiles; tile_idx += gridDim.x, ++it) {
            const DenseTile tile = A.tiles[tile_idx];
            const DenseWT W = A.w[tile.species];
            c.sb = sb; c.gb = gb;
            for (int i = 0; i < total; ++i) {
                if (i < o1) { c.copy_b(i, W.r1, H2p); continue; }
                if (i < i3) { c.copy_b(i, W.r2 + (size_t)chunk_order(i - o1, NCH2) * (2 * H1p * KC), H1p); continue; }
                const int nb = (i - i3) / NCH1, kc = (i - i3) % NCH1, nr = rows_of(i);
                c.copy_b(i, W.r3 + (size_t)nb * NCH1 * (2 * 128 * KC) + (size_t)kc * (2 * nr * KC), nr);
            }
            sb += total; gb += A.tf32 ? o1 + 1 + nblk : ngroups;
        }
    } else {
        const int m = (warp & 3) * 32 + lane, hf = warp >> 2;
        const uint32_t tl = tmem + ((uint32_t)((warp & 3) * 32) << 16);
        unsigned char *a_base = smem + SM_A;
        for (int tile_idx = blockIdx.x; tile_idx < A.n_tiles; tile_idx += gridDim.x, ++it) {
            const DenseTile tile = A.tiles[tile_idx];
            const DenseWT W = A.w[tile.species];
            const bool valid = m < tile.count;
            const float *zt = A.z_stash + (size_t)tile_idx * A.zs * TM + m * 4;
            if (tid == 0) TC_TRACE(1, 1, 100);
            // ---- h2bar = outbar W3^T: tensor core (K = n_out padded to 32) or, for the energy layer, W3's column;
            //      z2bar = h2bar SiLU'(z2) -> A operand of GEMM R2. The z stash is read ahead of the drains.
            //      (every MMA of the previous tile has completed: its last group was drained by this thread) ----
            {
                float4 z2[CW2 / 4];
#pragma unroll
                for (int k4 = 0; k4 < CW2 / 4; ++k4) {
                    z2[k4] = make_float4(0.f, 0.f, 0.f, 0.f);
                    if (valid) z2[k4] = __ldg(reinterpret_cast<const float4 *>(zt + (size_t)((H1p + hf * CW2 + k4 * 4) >> 2) * (TM * 4)));
                }
                float x[CW2];
                if (o1) {
                    // operand: row m of outbar in columns 0..15 (column half 0), zeros in 16..31 (half 1)
                    float ob[16];
#pragma unroll
                    for (int c = 0; c < 16; ++c) ob[c] = 0.f;
                    if (valid && hf == 0) {
                        const float4 *src =
                            reinterpret_cast<const float4 *>(A.outbar + (size_t)A.sp_list[tile.start + m] * A.outbar_stride);
#pragma unroll
                        for (int q = 0; q < 4; ++q)
                            if (q * 4 < A.nout) {
                                const float4 t = __ldg(src + q);
                                ob[q * 4] = t.x; ob[q * 4 + 1] = t.y; ob[q * 4 + 2] = t.z; ob[q * 4 + 3] = t.w;
                            }
#pragma unroll
                        for (int c = 0; c < 16; ++c)
                            if (c >= A.nout) ob[c] = 0.f;
                    }
#pragma unroll
                    for (int k4 = 0; k4 < 4; ++k4) store_split4(a_base, hf * 4 + k4, m, ob + k4 * 4);
                    fence_async_smem();
                    mbar_arrive(bar0 + 8 * BAR_AFULL);
#pragma unroll
                    for (int c = 0; c < CW2; ++c) x[c] = 0.f;
                    drain_group<CW2>(x, bar0, tl, gb, hf * CW2, true);   // the R1 MMAs have completed: slot 0 is free again
                } else {
#pragma unroll
                    for (int k4 = 0; k4 < CW2 / 4; ++k4) {
                        const float4 w4 = __ldg(reinterpret_cast<const float4 *>(W.w3c0 + hf * CW2 + k4 * 4));
                        x[k4 * 4] = w4.x; x[k4 * 4 + 1] = w4.y; x[k4 * 4 + 2] = w4.z; x[k4 * 4 + 3] = w4.w;
                    }
                }
#pragma unroll
                for (int k4 = 0; k4 < CW2 / 4; ++k4) {
                    const float x4[4] = {valid ? x[k4 * 4] * dsilu_f(z2[k4].x) : 0.f, valid ? x[k4 * 4 + 1] * dsilu_f(z2[k4].y) : 0.f,
                                         valid ? x[k4 * 4 + 2] * dsilu_f(z2[k4].z) : 0.f, valid ? x[k4 * 4 + 3] * dsilu_f(z2[k4].w) : 0.f};
                    store4_publish<CW2>(x4, a_base, bar0, hf * CW2, k4, m);
                }
            }
            if (tid == 0) TC_TRACE(1, 1, 101);
            // ---- GEMM R2: h1bar = z2bar W2^T; z1bar = h1bar SiLU'(z1) -> resident A operand of GEMM R3 ----
            {
                float4 z1[CW1 / 4];
#pragma unroll
                for (int k4 = 0; k4 < CW1 / 4; ++k4) {
                    z1[k4] = make_float4(0.f, 0.f, 0.f, 0.f);
                    if (valid) z1[k4] = __ldg(reinterpret_cast<const float4 *>(zt + (size_t)((hf * CW1 + k4 * 4) >> 2) * (TM * 4)));
                }
                float h1b[CW1];
#pragma unroll
                for (int c = 0; c < CW1; ++c) h1b[c] = 0.f;
                if (A.tf32) drain_group<CW1>(h1b, bar0, tl, gb + o1, hf * CW1, true);
                else {
#pragma unroll 1
                    for (int kc = 0; kc < NCH2; ++kc) drain_group<CW1>(h1b, bar0, tl, gb + o1 + kc, hf * CW1, true);
                }
                // all MMAs of R2 have completed: the A slots may be overwritten
#pragma unroll
                for (int k4 = 0; k4 < CW1 / 4; ++k4) {
                    const int col = hf * CW1 + k4 * 4;
                    const float4 z = z1[k4];
                    const float xv[4] = {valid ? h1b[k4 * 4] * dsilu_f(z.x) : 0.f, valid ? h1b[k4 * 4 + 1] * dsilu_f(z.y) : 0.f,
                                         valid ? h1b[k4 * 4 + 2] * dsilu_f(z.z) : 0.f, valid ? h1b[k4 * 4 + 3] * dsilu_f(z.w) : 0.f};
                    store_split4(a_base + (col >> 5) * A_SLOT, (col & 31) >> 2, m, xv);
                    // R3 reads the hi image from tensor memory (column = K index), the lo image from the slot
                    uint32_t hb[4];
#pragma unroll
                    for (int u = 0; u < 4; ++u) { float h, l; split_tf32(xv[u], h, l); hb[u] = __float_as_uint(h); }
                    tmem_st4(tl + COL_A + (uint32_t)col, hb);
                }
                tmem_wait_st();
                tc_fence_before();
                fence_async_smem();
                mbar_arrive(bar0 + 8 * BAR_ARES);
            }
            if (tid == 0) TC_TRACE(1, 1, 102);
            // ---- GEMM R3: Qbar = z1bar U^T in blocks of <= 128 columns; this thread takes 64 of them ----
            float *qt = A.Qbar + (size_t)tile_idx * A.K1 * TM + m * 4;
#pragma unroll 1
            for (int nb = 0; nb < nblk; ++nb) {
                const int ncols = min(128, A.K1 - nb * 128);
                const bool mine = hf * 64 < ncols;
                float q[64];
#pragma unroll
                for (int c = 0; c < 64; ++c) q[c] = 0.f;
                const int ngr = A.tf32 ? 1 : NCH1 / GR3;
#pragma unroll 1
                for (int gi = 0; gi < ngr; ++gi) {
                    const int g = A.tf32 ? gb + o1 + 1 + nb : gb + i3 + nb * (NCH1 / GR3) + gi;
                    if (ncols - hf * 64 >= 64) drain_group<64>(q, bar0, tl, g, hf * 64, true);
                    else if (ncols - hf * 64 >= 32) drain_group<32>(q, bar0, tl, g, hf * 64, true);
                    else drain_group<32>(q, bar0, tl, g, hf * 64, false);
                    if (tid == 0) TC_TRACE(1, 1, g - gb);
                }
                if (valid && mine) {
#pragma unroll
                    for (int c4 = 0; c4 < 16; ++c4) {
                        const int col = nb * 128 + hf * 64 + c4 * 4;
                        if (col < A.K1)
                            *reinterpret_cast<float4 *>(qt + (size_t)(col >> 2) * (TM * 4)) =
                                make_float4(q[c4 * 4], q[c4 * 4 + 1], q[c4 * 4 + 2], q[c4 * 4 + 3]);
                    }
                }
            }
            if (tid == 0) TC_TRACE(1, 1, 103);
            sb += total; gb += A.tf32 ? o1 + 1 + nblk : ngroups;
        }
    }
    tc_epilogue(tmem);
}

// ============================================================================ host
// persistent grid: one CTA per SM (224 KB of shared memory, all 512 TMEM columns), each walking over its tiles
static int tc_grid(int n_tiles) {
    static int n_sm[64] = {};
    int dev = 0;
    cudaGetDevice(&dev);
    if (dev < 0 || dev >= 64) dev = 0;
    if (!n_sm[dev] && (cudaDeviceGetAttribute(&n_sm[dev], cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n_sm[dev] <= 0))
        n_sm[dev] = 148;
    return n_tiles < n_sm[dev] ? n_tiles : n_sm[dev];
}
template <int N1, int N2>
int run_tc_fwd(const LaunchCtx &ctx, const TcFwdArgs &A, int n_tiles) {
    static bool attr[64] = {};
    int dev = 0;
    cudaGetDevice(&dev);
    if (dev < 0 || dev >= 64) return REANN_ERR_UNSUPPORTED;
    if (!attr[dev]) {   // the attribute is per device
        if (cudaFuncSetAttribute(k_dense_tc_fwd<N1, N2>, cudaFuncAttributeMaxDynamicSharedMemorySize, SM_TOTAL) != cudaSuccess) {
            cudaGetLastError();
            return REANN_ERR_UNSUPPORTED;
        }
        attr[dev] = true;
    }
    LAUNCH(ctx, (k_dense_tc_fwd<N1, N2>), tc_grid(n_tiles), NTHREADS, SM_TOTAL, A);
    return REANN_OK;
}
template <int N1, int N2>
int run_tc_bwd(const LaunchCtx &ctx, const TcBwdArgs &A, int n_tiles) {
    static bool attr[64] = {};
    int dev = 0;
    cudaGetDevice(&dev);
    if (dev < 0 || dev >= 64) return REANN_ERR_UNSUPPORTED;
    if (!attr[dev]) {   // the attribute is per device
        if (cudaFuncSetAttribute(k_dense_tc_bwd<N1, N2>, cudaFuncAttributeMaxDynamicSharedMemorySize, SM_TOTAL) != cudaSuccess) {
            cudaGetLastError();
            return REANN_ERR_UNSUPPORTED;
        }
        attr[dev] = true;
    }
    LAUNCH(ctx, (k_dense_tc_bwd<N1, N2>), tc_grid(n_tiles), NTHREADS, SM_TOTAL, A);
    return REANN_OK;
}
#define TC_DISPATCH(FN, ...)                                                                    \
    switch ((ld.H1p / 32) * 10 + ld.H2p / 32) {                                                 \
        case 11: return FN<1, 1>(__VA_ARGS__); case 12: return FN<1, 2>(__VA_ARGS__);           \
        case 14: return FN<1, 4>(__VA_ARGS__); case 21: return FN<2, 1>(__VA_ARGS__);           \
        case 22: return FN<2, 2>(__VA_ARGS__); case 24: return FN<2, 4>(__VA_ARGS__);           \
        case 41: return FN<4, 1>(__VA_ARGS__); case 42: return FN<4, 2>(__VA_ARGS__);           \
        case 44: return FN<4, 4>(__VA_ARGS__);                                                  \
        default: return REANN_ERR_UNSUPPORTED;                                                  \
    }

} // namespace

#ifdef REANN_TC_TRACE
extern "C" int reann_debug_tc_trace(long long *out) {
    return (int)cudaMemcpyFromSymbol(out, g_tc_trace, sizeof(g_tc_trace));
}
#endif

int launch_dense_tc_fwd(const LaunchCtx &ctx, const ModelDims &md, const LayerDims &ld, const DenseWT *d_w,
                        const DenseTile *tiles, int n_tiles, const int32_t *sp_list, const float *Q, float *z_stash,
                        int zs, float *out, int out_stride, bool tf32) {
    if (n_tiles <= 0) return REANN_OK;
    if (ld.nout > 16) return REANN_ERR_UNSUPPORTED;
    TcFwdArgs A;
    A.w = d_w; A.tiles = tiles; A.sp_list = sp_list; A.Q = Q; A.z_stash = z_stash; A.out = out; A.out_stride = out_stride;
    A.K1 = md.K1; A.nout = ld.nout; A.zs = zs; A.n_tiles = n_tiles; A.tf32 = tf32; A.skip = ctx.skip;
    TC_DISPATCH(run_tc_fwd, ctx, A, n_tiles)
}

int launch_dense_tc_bwd(const LaunchCtx &ctx, const ModelDims &md, const LayerDims &ld, const DenseWT *d_w,
                        const DenseTile *tiles, int n_tiles, const int32_t *sp_list, const float *z_stash, int zs,
                        const float *outbar, int outbar_stride, float *Qbar, bool tf32) {
    if (n_tiles <= 0) return REANN_OK;
    if (ld.nout > 16) return REANN_ERR_UNSUPPORTED;
    TcBwdArgs A;
    A.w = d_w; A.tiles = tiles; A.sp_list = sp_list; A.z_stash = z_stash; A.outbar = outbar; A.Qbar = Qbar;
    A.outbar_stride = outbar_stride; A.K1 = md.K1; A.nout = ld.nout; A.zs = zs; A.n_tiles = n_tiles; A.tf32 = tf32; A.skip = ctx.skip;
    TC_DISPATCH(run_tc_bwd, ctx, A, n_tiles)
}
