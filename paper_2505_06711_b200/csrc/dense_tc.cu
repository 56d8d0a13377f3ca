// dense_tc.cu -- rows A6+A7 / A9 of SURVEY.md section 8(a) on the 5th-generation tensor cores:
// the per-species GEMM chain of the folded contraction + atomic NN (Eq. 1 outer sums + Eq. 2,
// PAPER.md:35-43) and of its reverse pass (Eq. 5 / Appendix B steps 1-2), as tcgen05.mma
// kind::tf32 with FP32 accumulators in tensor memory (TMEM).
//
// FP32-class accuracy from TF32 operands ("3xTF32"): every operand x is split into
//   x_hi = x rounded to 10 mantissa bits,   x_lo = x - x_hi   (exact in FP32)
// and each product is issued as  A_hi B_hi  (main accumulator)  +  A_lo B_hi + A_hi B_lo  (a
// separate correction accumulator); the dropped A_lo B_lo term is 2^-22 relative.
// The tensor core adds into its FP32 accumulator with truncation (measured on B200: a single
// accumulator over K = 576 carries a -6e-6 relative bias, 10x the error of an FP32 FMA loop), so
// K is cut into groups of <= 96 (GEMM over Q) or 64 floats: every group accumulates into a fresh
// pair of TMEM buffers (double-buffered), which the row threads then add into FP32 registers with
// round-to-nearest. Measured error of this scheme: at or below that of a sequential FP32 FMA loop.
//
// One CTA = one tile of 128 atoms of one species (UMMA M = 128, cta_group::1):
//   forward   z1 = Q U + b1;  h1 = SiLU(z1);  z2 = h1 W2 + b2;  h2 = SiLU(z2);  out = h2 W3 + b3
//   reverse   h2bar = outbar W3^T; z2bar = h2bar SiLU'(z2); h1bar = z2bar W2^T; z1bar = h1bar SiLU'(z1);
//             Qbar = z1bar U^T
// (Q = radial-pair products of the neighbour sums b, U = folded contraction x first layer; see
// dense.cu for the algebra.)
//
// Warp roles: warps 0-3 ("row" threads: thread m = tile row m = TMEM lane m) drain the group
// accumulators into registers and turn them into the next GEMM's A operand (bias / activation /
// stash -> hi/lo split -> shared memory) or into the outputs; in the forward kernel warps 4-7
// stream Q from global memory into A chunks; the last warp (one lane) streams the pre-split weight
// chunks into shared memory with cp.async.bulk, issues the MMAs and commits them to mbarriers.
// K is processed in chunks of 32 floats through a 3-stage ring (A slot + B slot per stage).
//
// Shared-memory operand layout (no swizzle, K-major "core matrices" of 8 rows x 16 bytes):
//   element (row r, k) of a [R][32] chunk lives at byte  (k/4)*(R*16) + r*16 + (k%4)*4,
//   i.e. LBO (K direction) = R*16 bytes, SBO (row-group direction) = 128 bytes; the lo image
//   follows the hi image. Weight chunks are stored in global memory in exactly this image
//   (built once in reann_create), so one bulk copy per chunk brings hi and lo.
#include "common.cuh"

namespace {

constexpr int TM = DENSE_TC_TM;        // 128 rows (atoms) per tile
constexpr int KC = 32;                 // floats per K chunk
constexpr int NSTAGE = 3;              // ring depth (A slot + B slot + 3 barriers per stage)
constexpr int NASLOT = 4;              // A slots (the reverse pass keeps z1bar resident in 4)
constexpr int A_HALF = TM * KC * 4;    // bytes of one A image (hi or lo)
constexpr int A_SLOT = 2 * A_HALF;     // 32 KB
constexpr int B_SLOT = 2 * 128 * KC * 4; // 32 KB (N <= 128)
constexpr int SM_A = 0, SM_B = NASLOT * A_SLOT, SM_BAR = SM_B + NSTAGE * B_SLOT;
constexpr int SM_TOTAL = SM_BAR + 256;
constexpr uint32_t A_LBO = TM * 16;
constexpr int GK_Q = 1, GK_H = 1;      // chunks per accumulation group: GEMM over Q / all others

// TMEM (512 columns): group buffer d in {0,1}: main accumulator at 256 d, correction at 256 d + 128
constexpr uint32_t COL_CORR = 128, COL_BUF = 256;

// barrier slots (8 bytes each) in the barrier area
enum { BAR_BFULL = 0, BAR_AFULL = 3, BAR_MMA = 6, BAR_ARES = 9, BAR_DFULL = 10, BAR_DEMPTY = 12, BAR_COUNT = 14 };

// Optional timeline trace of one CTA (development aid, compiled only with -DREANN_TC_TRACE):
// role 0 = control thread, 1 = row thread 0, 2 = first producer thread; slot k = clock64().
#ifdef REANN_TC_TRACE
__device__ long long g_tc_trace[3 * 128];
#define TC_TRACE(role, k)                                                                             \
    do {                                                                                              \
        if (blockIdx.x == 200 && (k) < 128 && (threadIdx.x & 31) == 0) g_tc_trace[(role) * 128 + (k)] = clock64(); \
    } while (0)
#else
#define TC_TRACE(role, k) ((void)0)
#endif

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
    return ok != 0;
}
// Bounded wait: a protocol error traps (the launch fails with an error) instead of hanging the GPU.
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    if (mbar_try(bar, parity)) return;
    const long long t0 = clock64();
    while (!mbar_try(bar, parity))
        if (clock64() - t0 > 4000000000ll) __trap();
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
// D[tmem] (+)= A[smem] . B[smem]^T   (A: M x 8, B: N x 8, both K-major, TF32)
__device__ __forceinline__ void umma_tf32(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc,
                                          uint32_t accumulate) {
    asm volatile(
        "{\n .reg .pred p;\n setp.ne.b32 p, %4, 0;\n tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n}" ::"r"(d_tmem),
        "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
        : "memory");
}
// shared-memory matrix descriptor: no swizzle, version 1 (sm_100), offsets in 16-byte units
__device__ __forceinline__ uint64_t make_desc(uint32_t saddr, uint32_t lbo_bytes) {
    return (uint64_t)((saddr & 0x3FFFFu) >> 4) | ((uint64_t)(lbo_bytes >> 4) << 16) | ((uint64_t)(128u >> 4) << 32) |
           (1ull << 46);
}
// instruction descriptor: D = F32, A = B = TF32, both K-major, M = 128
__device__ __forceinline__ uint32_t make_idesc(int n) {
    return (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(TM >> 4) << 24);
}

__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t *v) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];\n"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
          "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]),
          "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]),
          "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
        : "r"(taddr));
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t *v) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];\n"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
          "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
        : "r"(taddr));
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}

__device__ __forceinline__ void split_tf32(float x, float &hi, float &lo) {
    hi = __uint_as_float((__float_as_uint(x) + 0x1000u) & 0xFFFFE000u);
    lo = __uint_as_float((__float_as_uint(x - hi) + 0x1000u) & 0xFFFFE000u); // x - hi is exact; round it to TF32 here
}
__device__ __forceinline__ void store_split4(unsigned char *a_slot, int k4, int row, const float *x) {
    float4 h, l;
    split_tf32(x[0], h.x, l.x); split_tf32(x[1], h.y, l.y); split_tf32(x[2], h.z, l.z); split_tf32(x[3], h.w, l.w);
    float4 *p = reinterpret_cast<float4 *>(a_slot + k4 * (int)A_LBO + row * 16);
    p[0] = h;
    p[A_HALF / 16] = l;
}

__device__ __forceinline__ float silu_f(float z) { return z / (1.0f + __expf(-z)); }
__device__ __forceinline__ float dsilu_f(float z) {
    const float s = 1.0f / (1.0f + __expf(-z));
    return s * (1.0f + z * (1.0f - s));
}

// ---- common prologue / epilogue of both kernels ----
__device__ __forceinline__ uint32_t tc_prologue(unsigned char *smem, uint32_t *tmem_base_s, int ctl_warp) {
    const int tid = threadIdx.x, warp = tid >> 5;
    const uint32_t bar0 = smem_u32(smem + SM_BAR);
    if (tid == 0) {
        for (int s = 0; s < NSTAGE; ++s) {
            mbar_init(bar0 + 8 * (BAR_BFULL + s), 1);
            mbar_init(bar0 + 8 * (BAR_AFULL + s), 128);
            mbar_init(bar0 + 8 * (BAR_MMA + s), 1);
        }
        mbar_init(bar0 + 8 * BAR_ARES, 128);
        for (int d = 0; d < 2; ++d) {
            mbar_init(bar0 + 8 * (BAR_DFULL + d), 1);
            mbar_init(bar0 + 8 * (BAR_DEMPTY + d), 128);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == ctl_warp) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_base_s)), "r"(512u)
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    return *tmem_base_s;
}
__device__ __forceinline__ void tc_epilogue(uint32_t tmem, int ctl_warp) {
    tc_fence_before();
    __syncthreads();
    if ((int)(threadIdx.x >> 5) == ctl_warp)
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(512u) : "memory");
}

// ---- control-warp helpers (one thread) ----
struct Ctl {
    uint32_t bar0, a0, b0, tmem;
    __device__ __forceinline__ uint32_t bar(int k) const { return bar0 + 8u * (uint32_t)k; }
    // stream the weight chunk of step i into its B slot (after the MMAs of step i-3 released it)
    __device__ __forceinline__ void copy_b(int i, const float *src, int n_rows) const {
        const int s = i % NSTAGE;
        if (i >= NSTAGE) mbar_wait(bar(BAR_MMA + s), (uint32_t)(((i / NSTAGE) - 1) & 1));
        const uint32_t bytes = (uint32_t)n_rows * KC * 4 * 2;
        mbar_expect_tx(bar(BAR_BFULL + s), bytes);
        bulk_g2s(b0 + (uint32_t)s * B_SLOT, src, bytes, bar(BAR_BFULL + s));
    }
    // One K chunk of step i into group buffer d (global group counter gg = ... d = gg & 1):
    //   main[:, 0:n) (+)= A_hi B_hi^T ;  corr[:, 0:n) (+)= A_lo B_hi^T + A_hi B_lo^T
    // first: first chunk of the group (overwrite); last: commit the group's "full" barrier.
    __device__ __forceinline__ void mma_chunk(int i, int a_slot, int n_rows, int gg, bool first, bool last) const {
        const int s = i % NSTAGE, d = gg & 1;
        if (first && gg >= 2) mbar_wait(bar(BAR_DEMPTY + d), (uint32_t)(((gg >> 1) - 1) & 1));
        mbar_wait(bar(BAR_BFULL + s), (uint32_t)((i / NSTAGE) & 1));
        tc_fence_after();
        const uint32_t idesc = make_idesc(n_rows);
        const uint32_t a_hi = a0 + (uint32_t)a_slot * A_SLOT, a_lo = a_hi + A_HALF;
        const uint32_t b_lbo = (uint32_t)n_rows * 16;
        const uint32_t b_hi = b0 + (uint32_t)s * B_SLOT, b_lo = b_hi + (uint32_t)n_rows * KC * 4;
        const uint32_t dm = tmem + COL_BUF * (uint32_t)d, dc = dm + COL_CORR;
#pragma unroll
        for (int kk = 0; kk < KC / 8; ++kk) {
            const uint64_t ah = make_desc(a_hi + kk * 2 * A_LBO, A_LBO), al = make_desc(a_lo + kk * 2 * A_LBO, A_LBO);
            const uint64_t bh = make_desc(b_hi + kk * 2 * b_lbo, b_lbo), bl = make_desc(b_lo + kk * 2 * b_lbo, b_lbo);
            const uint32_t acc = (first && kk == 0) ? 0u : 1u;
            umma_tf32(dm, ah, bh, idesc, acc);
            umma_tf32(dc, al, bl, idesc, acc);
            umma_tf32(dc, al, bh, idesc, 1u);
            umma_tf32(dc, ah, bl, idesc, 1u);
        }
        tc_commit(bar(BAR_MMA + s));
        if (last) tc_commit(bar(BAR_DFULL + d));
    }
};

// ---- row-thread helpers ----
// add group buffer gg (main + correction, NCH*32 columns) into the FP32 register accumulators
template <int NCH>
__device__ __forceinline__ void drain_group(float *acc, uint32_t bar0, uint32_t tl, int gg) {
    const int d = gg & 1;
    mbar_wait(bar0 + 8 * (BAR_DFULL + d), (uint32_t)((gg >> 1) & 1));
    tc_fence_after();
    if (threadIdx.x == 0) TC_TRACE(1, 2 * gg);
#pragma unroll
    for (int c = 0; c < NCH; ++c) {
        uint32_t vm[32], vc[32];
        tmem_ld32(tl + COL_BUF * (uint32_t)d + c * 32, vm);
        tmem_ld32(tl + COL_BUF * (uint32_t)d + COL_CORR + c * 32, vc);
#pragma unroll
        for (int k = 0; k < 32; ++k) acc[c * 32 + k] += __uint_as_float(vm[k]) + __uint_as_float(vc[k]);
    }
    tc_fence_before();
    mbar_arrive(bar0 + 8 * (BAR_DEMPTY + d));
    if (threadIdx.x == 0) TC_TRACE(1, 2 * gg + 1);
}
__device__ __forceinline__ void drain_group16(float *acc, uint32_t bar0, uint32_t tl, int gg) {
    const int d = gg & 1;
    mbar_wait(bar0 + 8 * (BAR_DFULL + d), (uint32_t)((gg >> 1) & 1));
    tc_fence_after();
    uint32_t vm[16], vc[16];
    tmem_ld16(tl + COL_BUF * (uint32_t)d, vm);
    tmem_ld16(tl + COL_BUF * (uint32_t)d + COL_CORR, vc);
#pragma unroll
    for (int k = 0; k < 16; ++k) acc[k] += __uint_as_float(vm[k]) + __uint_as_float(vc[k]);
    tc_fence_before();
    mbar_arrive(bar0 + 8 * (BAR_DEMPTY + d));
}
// wait until the MMAs that last read stage (i % NSTAGE) are complete
__device__ __forceinline__ void wait_stage_free(uint32_t bar0, int i) {
    if (i >= NSTAGE) mbar_wait(bar0 + 8 * (BAR_MMA + i % NSTAGE), (uint32_t)(((i / NSTAGE) - 1) & 1));
}
__host__ __device__ constexpr int cdiv(int a, int b) { return (a + b - 1) / b; }

// ============================================================================ forward
struct TcFwdArgs {
    const DenseWT *w;       // [S]
    const DenseTile *tiles; // 128-atom tiles
    const int32_t *sp_list;
    const float *Q;         // [N][nqp], tile order
    float *z_stash;         // [N][zs], tile order
    float *out;             // rows of stride out_stride, atom order
    int out_stride, nqp, K1, nout, zs;
};
constexpr int FWD_THREADS = 288, FWD_CTL = 8;

// row thread: registers -> (+bias, stash, SiLU, split) -> A chunks of the next GEMM (steps ibase ..)
template <int NCH>
__device__ __forceinline__ void fwd_activate(const float *acc, const float *__restrict__ bias, float *zdst, bool valid,
                                             unsigned char *a_base, uint32_t bar0, int ibase, int m) {
#pragma unroll
    for (int kc = 0; kc < NCH; ++kc) {
        const int i = ibase + kc, s = i % NSTAGE;
        wait_stage_free(bar0, i);
#pragma unroll
        for (int k4 = 0; k4 < 8; ++k4) {
            const float4 b4 = __ldg(reinterpret_cast<const float4 *>(bias + kc * KC) + k4);
            const float z[4] = {acc[kc * 32 + k4 * 4] + b4.x, acc[kc * 32 + k4 * 4 + 1] + b4.y,
                                acc[kc * 32 + k4 * 4 + 2] + b4.z, acc[kc * 32 + k4 * 4 + 3] + b4.w};
            if (valid) reinterpret_cast<float4 *>(zdst + kc * KC)[k4] = make_float4(z[0], z[1], z[2], z[3]);
            const float hv[4] = {silu_f(z[0]), silu_f(z[1]), silu_f(z[2]), silu_f(z[3])};
            store_split4(a_base + s * A_SLOT, k4, m, hv);
        }
        fence_async_smem();
        mbar_arrive(bar0 + 8 * (BAR_AFULL + s));
    }
}

template <int NCH1, int NCH2>
__global__ void __launch_bounds__(FWD_THREADS, 1) k_dense_tc_fwd(TcFwdArgs A) {
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ uint32_t tmem_base_s;
    constexpr int H1p = NCH1 * 32, H2p = NCH2 * 32;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const DenseTile tile = A.tiles[blockIdx.x];
    const DenseWT W = A.w[tile.species];
    const uint32_t bar0 = smem_u32(smem + SM_BAR);
    const uint32_t tmem = tc_prologue(smem, &tmem_base_s, FWD_CTL);
    if (tid == 0) TC_TRACE(1, 103);
    const int n1 = A.K1 / KC, total = n1 + NCH1 + NCH2;
    const int ng1 = cdiv(n1, GK_Q);
    constexpr int ng2 = cdiv(NCH1, GK_H), ng3 = cdiv(NCH2, GK_H);

    if (warp == FWD_CTL) {
        if (lane == 0) {
            Ctl c{bar0, smem_u32(smem + SM_A), smem_u32(smem + SM_B), tmem};
            auto src_of = [&](int i, int &n_rows) -> const float * {
                if (i < n1) { n_rows = H1p; return W.g1 + (size_t)i * (2 * H1p * KC); }
                if (i < n1 + NCH1) { n_rows = H2p; return W.g2 + (size_t)(i - n1) * (2 * H2p * KC); }
                n_rows = 16; return W.g3 + (size_t)(i - n1 - NCH1) * (2 * 16 * KC);
            };
            int nr;
            const float *src = src_of(0, nr);
            c.copy_b(0, src, nr);
            for (int i = 0; i < total; ++i) {
                if (i + 1 < total) { src = src_of(i + 1, nr); c.copy_b(i + 1, src, nr); }
                const int s = i % NSTAGE;
                mbar_wait(c.bar(BAR_AFULL + s), (uint32_t)((i / NSTAGE) & 1));
                TC_TRACE(0, 2 * i);
                if (i < n1) {
                    c.mma_chunk(i, s, H1p, i / GK_Q, i % GK_Q == 0, i % GK_Q == GK_Q - 1 || i == n1 - 1);
                } else if (i < n1 + NCH1) {
                    const int kc = i - n1;
                    c.mma_chunk(i, s, H2p, ng1 + kc / GK_H, kc % GK_H == 0, kc % GK_H == GK_H - 1 || kc == NCH1 - 1);
                } else {
                    const int kc = i - n1 - NCH1;
                    c.mma_chunk(i, s, 16, ng1 + ng2 + kc / GK_H, kc % GK_H == 0, kc % GK_H == GK_H - 1 || kc == NCH2 - 1);
                }
                TC_TRACE(0, 2 * i + 1);
            }
        }
    } else if (warp >= 4) {
        // ---- producers: Q chunks (global -> hi/lo split -> shared) for GEMM 1 ----
        const int pw = warp - 4, r8 = lane & 7, kq = lane >> 3;
        const float *Qt = A.Q + (size_t)tile.start * A.nqp;
        unsigned char *a_base = smem + SM_A;
        for (int i = 0; i < n1; ++i) {
            const int s = i % NSTAGE;
            float4 v[8];
#pragma unroll
            for (int rb = 0; rb < 4; ++rb)
#pragma unroll
                for (int j = 0; j < 2; ++j) {
                    const int row = pw * 32 + rb * 8 + r8, kg = i * KC + (kq + 4 * j) * 4;
                    v[rb * 2 + j] = (row < tile.count && kg < A.nqp)
                                        ? __ldg(reinterpret_cast<const float4 *>(Qt + (size_t)row * A.nqp + kg))
                                        : make_float4(0.f, 0.f, 0.f, 0.f);
                }
            if (tid == 128) TC_TRACE(2, 3 * i);
            wait_stage_free(bar0, i);
            if (tid == 128) TC_TRACE(2, 3 * i + 1);
#pragma unroll
            for (int rb = 0; rb < 4; ++rb)
#pragma unroll
                for (int j = 0; j < 2; ++j) {
                    const float x[4] = {v[rb * 2 + j].x, v[rb * 2 + j].y, v[rb * 2 + j].z, v[rb * 2 + j].w};
                    store_split4(a_base + s * A_SLOT, kq + 4 * j, pw * 32 + rb * 8 + r8, x);
                }
            fence_async_smem();
            mbar_arrive(bar0 + 8 * (BAR_AFULL + s));
            if (tid == 128) TC_TRACE(2, 3 * i + 2);
        }
    } else {
        // ---- row threads ----
        const int m = tid;
        const bool valid = m < tile.count;
        const uint32_t tl = tmem + ((uint32_t)(warp * 32) << 16);
        unsigned char *a_base = smem + SM_A;
        float *zrow = A.z_stash + (size_t)(tile.start + m) * A.zs;
        {
            float z1[H1p];
#pragma unroll
            for (int c = 0; c < H1p; ++c) z1[c] = 0.f;
#pragma unroll 1
            for (int g = 0; g < ng1; ++g) drain_group<NCH1>(z1, bar0, tl, g);
            fwd_activate<NCH1>(z1, W.b1, zrow, valid, a_base, bar0, n1, m);
            if (tid == 0) TC_TRACE(1, 100);
        }
        {
            float z2[H2p];
#pragma unroll
            for (int c = 0; c < H2p; ++c) z2[c] = 0.f;
#pragma unroll 1
            for (int g = 0; g < ng2; ++g) drain_group<NCH2>(z2, bar0, tl, ng1 + g);
            fwd_activate<NCH2>(z2, W.b2, zrow + H1p, valid, a_base, bar0, n1 + NCH1, m);
            if (tid == 0) TC_TRACE(1, 101);
        }
        float o[16];
#pragma unroll
        for (int c = 0; c < 16; ++c) o[c] = 0.f;
#pragma unroll 1
        for (int g = 0; g < ng3; ++g) drain_group16(o, bar0, tl, ng1 + ng2 + g);
        if (valid) {
            float *dst = A.out + (size_t)A.sp_list[tile.start + m] * A.out_stride;
#pragma unroll
            for (int c = 0; c < 16; ++c)
                if (c < A.nout) dst[c] = o[c] + __ldg(W.b3 + c);
        }
    }
    if (tid == 0) TC_TRACE(1, 102);
    tc_epilogue(tmem, FWD_CTL);
}

// ============================================================================ reverse
struct TcBwdArgs {
    const DenseWT *w;
    const DenseTile *tiles;
    const int32_t *sp_list;
    const float *z_stash, *outbar; // outbar == nullptr: energy layer (outbar = 1)
    float *Qbar;                   // [N][nqp], tile order
    int outbar_stride, nqp, K1, nout, zs;
};
constexpr int BWD_THREADS = 160, BWD_CTL = 4;

// row thread: xbar = acc * SiLU'(z) -> split -> A chunk kc into slot slot_of(kc)
template <int NCH, bool RING>
__device__ __forceinline__ void bwd_activate(const float *acc, const float *zsrc, bool valid, unsigned char *a_base,
                                             uint32_t bar0, int ibase, int m) {
#pragma unroll
    for (int kc = 0; kc < NCH; ++kc) {
        const int i = ibase + kc, slot = RING ? i % NSTAGE : kc;
        if (RING) wait_stage_free(bar0, i);
#pragma unroll
        for (int k4 = 0; k4 < 8; ++k4) {
            float4 z = make_float4(0.f, 0.f, 0.f, 0.f);
            if (valid) z = __ldg(reinterpret_cast<const float4 *>(zsrc + kc * KC) + k4);
            const float x[4] = {acc[kc * 32 + k4 * 4] * dsilu_f(z.x), acc[kc * 32 + k4 * 4 + 1] * dsilu_f(z.y),
                                acc[kc * 32 + k4 * 4 + 2] * dsilu_f(z.z), acc[kc * 32 + k4 * 4 + 3] * dsilu_f(z.w)};
            store_split4(a_base + slot * A_SLOT, k4, m, x);
        }
        if (RING) {
            fence_async_smem();
            mbar_arrive(bar0 + 8 * (BAR_AFULL + slot));
        }
    }
}

template <int NCH1, int NCH2>
__global__ void __launch_bounds__(BWD_THREADS, 1) k_dense_tc_bwd(TcBwdArgs A) {
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ uint32_t tmem_base_s;
    constexpr int H1p = NCH1 * 32, H2p = NCH2 * 32;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const DenseTile tile = A.tiles[blockIdx.x];
    const DenseWT W = A.w[tile.species];
    const uint32_t bar0 = smem_u32(smem + SM_BAR);
    const uint32_t tmem = tc_prologue(smem, &tmem_base_s, BWD_CTL);
    constexpr int ng2 = cdiv(NCH2, GK_H), gpb = cdiv(NCH1, GK_H), i3 = 1 + NCH2;
    const int nblk = (A.K1 + 127) / 128, total = i3 + nblk * NCH1;

    if (warp == BWD_CTL) {
        if (lane == 0) {
            Ctl c{bar0, smem_u32(smem + SM_A), smem_u32(smem + SM_B), tmem};
            auto src_of = [&](int i, int &n_rows) -> const float * {
                if (i == 0) { n_rows = H2p; return W.r1; }
                if (i < i3) { n_rows = H1p; return W.r2 + (size_t)(i - 1) * (2 * H1p * KC); }
                const int nb = (i - i3) / NCH1, kc = (i - i3) % NCH1;
                n_rows = min(128, A.K1 - nb * 128);
                return W.r3 + (size_t)nb * NCH1 * (2 * 128 * KC) + (size_t)kc * (2 * n_rows * KC);
            };
            int nr;
            const float *src = src_of(0, nr);
            c.copy_b(0, src, nr);
            for (int i = 0; i < total; ++i) {
                if (i + 1 < total) { src = src_of(i + 1, nr); c.copy_b(i + 1, src, nr); }
                const int s = i % NSTAGE;
                if (i == 0) {
                    mbar_wait(c.bar(BAR_AFULL + s), 0);
                    c.mma_chunk(i, s, H2p, 0, true, true);
                } else if (i < i3) {
                    const int kc = i - 1;
                    mbar_wait(c.bar(BAR_AFULL + s), (uint32_t)((i / NSTAGE) & 1));
                    c.mma_chunk(i, s, H1p, 1 + kc / GK_H, kc % GK_H == 0, kc % GK_H == GK_H - 1 || kc == NCH2 - 1);
                } else {
                    const int nb = (i - i3) / NCH1, kc = (i - i3) % NCH1;
                    if (i == i3) mbar_wait(c.bar(BAR_ARES), 0);
                    c.mma_chunk(i, kc, min(128, A.K1 - nb * 128), 1 + ng2 + nb * gpb + kc / GK_H, kc % GK_H == 0,
                                kc % GK_H == GK_H - 1 || kc == NCH1 - 1);
                }
            }
        }
    } else {
        const int m = tid;
        const bool valid = m < tile.count;
        const uint32_t tl = tmem + ((uint32_t)(warp * 32) << 16);
        unsigned char *a_base = smem + SM_A;
        const float *zrow = A.z_stash + (size_t)(tile.start + m) * A.zs;
        // ---- GEMM R1 operand: outbar (cbar rows of the next layer, or 1 for the energy layer) ----
        {
            float ob[KC];
#pragma unroll
            for (int c = 0; c < KC; ++c) ob[c] = 0.f;
            if (valid) {
                if (A.outbar) {
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
                } else ob[0] = 1.0f;
            }
#pragma unroll
            for (int k4 = 0; k4 < 8; ++k4) store_split4(a_base, k4, m, ob + k4 * 4);
            fence_async_smem();
            mbar_arrive(bar0 + 8 * (BAR_AFULL + 0));
        }
        // ---- z2bar = h2bar * SiLU'(z2) -> GEMM R2 operand (ring) ----
        {
            float h2b[H2p];
#pragma unroll
            for (int c = 0; c < H2p; ++c) h2b[c] = 0.f;
            drain_group<NCH2>(h2b, bar0, tl, 0);
            bwd_activate<NCH2, true>(h2b, zrow + H1p, valid, a_base, bar0, 1, m);
        }
        // ---- z1bar = h1bar * SiLU'(z1) -> resident operand of GEMM R3 (A slots 0..NCH1-1) ----
        {
            float h1b[H1p];
#pragma unroll
            for (int c = 0; c < H1p; ++c) h1b[c] = 0.f;
#pragma unroll 1
            for (int g = 0; g < ng2; ++g) drain_group<NCH1>(h1b, bar0, tl, 1 + g);
            bwd_activate<NCH1, false>(h1b, zrow, valid, a_base, bar0, 0, m);
            fence_async_smem();
            mbar_arrive(bar0 + 8 * BAR_ARES);
        }
        // ---- Qbar blocks of <= 128 columns ----
        float *qrow = A.Qbar + (size_t)(tile.start + m) * A.nqp;
#pragma unroll 1
        for (int nb = 0; nb < nblk; ++nb) {
            float q[128];
#pragma unroll
            for (int c = 0; c < 128; ++c) q[c] = 0.f;
#pragma unroll 1
            for (int g = 0; g < gpb; ++g) drain_group<4>(q, bar0, tl, 1 + ng2 + nb * gpb + g);
            if (valid) {
#pragma unroll
                for (int c4 = 0; c4 < 32; ++c4) {
                    const int col = nb * 128 + c4 * 4;
                    if (col < A.nqp)
                        *reinterpret_cast<float4 *>(qrow + col) = make_float4(q[c4 * 4], q[c4 * 4 + 1], q[c4 * 4 + 2], q[c4 * 4 + 3]);
                }
            }
        }
    }
    tc_epilogue(tmem, BWD_CTL);
}

// ============================================================================ host
template <int N1, int N2>
int run_tc_fwd(const LaunchCtx &ctx, const TcFwdArgs &A, int n_tiles) {
    static bool attr = false;
    if (!attr) {
        if (cudaFuncSetAttribute(k_dense_tc_fwd<N1, N2>, cudaFuncAttributeMaxDynamicSharedMemorySize, SM_TOTAL) != cudaSuccess) {
            cudaGetLastError();
            return REANN_ERR_UNSUPPORTED;
        }
        attr = true;
    }
    LAUNCH(ctx, (k_dense_tc_fwd<N1, N2>), n_tiles, FWD_THREADS, SM_TOTAL, A);
    return REANN_OK;
}
template <int N1, int N2>
int run_tc_bwd(const LaunchCtx &ctx, const TcBwdArgs &A, int n_tiles) {
    static bool attr = false;
    if (!attr) {
        if (cudaFuncSetAttribute(k_dense_tc_bwd<N1, N2>, cudaFuncAttributeMaxDynamicSharedMemorySize, SM_TOTAL) != cudaSuccess) {
            cudaGetLastError();
            return REANN_ERR_UNSUPPORTED;
        }
        attr = true;
    }
    LAUNCH(ctx, (k_dense_tc_bwd<N1, N2>), n_tiles, BWD_THREADS, SM_TOTAL, A);
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
                        int zs, float *out, int out_stride) {
    if (n_tiles <= 0) return REANN_OK;
    if (ld.nout > 16) return REANN_ERR_UNSUPPORTED;
    TcFwdArgs A;
    A.w = d_w; A.tiles = tiles; A.sp_list = sp_list; A.Q = Q; A.z_stash = z_stash; A.out = out; A.out_stride = out_stride;
    A.nqp = md.nqp; A.K1 = md.K1; A.nout = ld.nout; A.zs = zs;
    TC_DISPATCH(run_tc_fwd, ctx, A, n_tiles)
}

int launch_dense_tc_bwd(const LaunchCtx &ctx, const ModelDims &md, const LayerDims &ld, const DenseWT *d_w,
                        const DenseTile *tiles, int n_tiles, const int32_t *sp_list, const float *z_stash, int zs,
                        const float *outbar, int outbar_stride, float *Qbar) {
    if (n_tiles <= 0) return REANN_OK;
    if (ld.nout > 16) return REANN_ERR_UNSUPPORTED;
    TcBwdArgs A;
    A.w = d_w; A.tiles = tiles; A.sp_list = sp_list; A.z_stash = z_stash; A.outbar = outbar; A.Qbar = Qbar;
    A.outbar_stride = outbar_stride; A.nqp = md.nqp; A.K1 = md.K1; A.nout = ld.nout; A.zs = zs;
    TC_DISPATCH(run_tc_bwd, ctx, A, n_tiles)
}
