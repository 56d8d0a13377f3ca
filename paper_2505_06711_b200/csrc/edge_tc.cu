// edge_tc.cu -- row A10 of SURVEY.md section 8(a), the edge backward step, with its two per-atom
// products on the 5th-generation tensor cores (tcgen05.mma kind::tf32, FP32 accumulators in TMEM).
//
// For one atom i with T = bbar_i (N_phi x N_a, the adjoint of the neighbour sums of Eq. 1,
// PAPER.md:35) and its edges e = (i, j) within rc (Eq. 4):
//     S[e,n] = sum_a A_a(r_e) T[n,a]          ( M = edges, K = monomials,  N = N_phi )
//     P[e,a] = sum_n x_e[n]   T[n,a]          ( M = edges, K = N_phi,      N = monomials )
//     g_e = (sum_n c_j[n] R'_n S[e,n]) r_hat + sum_a P[e,a] grad A_a;   kappa_e[n] = R_n S[e,n]  (t >= 1)
// The FP32 ALU kernel (edge.cu) re-reads all of T from shared memory for every edge and is bound by
// that operand delivery; here T is the B operand of an M = 128 MMA tile whose rows are the edges of
// the atom, so it is read once per tile by the tensor core.
//
// FP32-class accuracy from TF32 operands as in dense_tc.cu ("3xTF32"): x = hi + lo, products issued
// as lo.hi + hi.lo first and hi.hi last; K <= 24, so one accumulator sees <= 9 truncating additions.
//
// One CTA = four independent warpgroups (WG) of 128 threads; a WG walks over atoms (persistent grid),
// thread r of the WG = row r of the tile = TMEM lane r:
//   phase 1  (one edge per thread) edge record, c_j gather, radial functions R_n, x_n, y_n = c_j R'_n,
//            monomials; the row (A | x) is split and written to the shared-memory A operand (hi and
//            lo images, K-major core matrices); the WG also writes the B operands (T and T^T images);
//   phase 2  one thread issues the 3 (K/8 + K'/8) tcgen05.mma and commits them to the WG's mbarrier;
//   phase 3  every thread reads its S row and P row from TMEM and finishes g_e, kappa_e (stash
//            written centre-side, read back through rev_rc by k_rev_gather: no atomics).
// While a WG waits for its MMAs the other WGs of the SM run their phases 1 / 3; all global loads of a tile
// are requested one tile ahead (registers / cp.async), so no phase waits on DRAM or L2.
#include <stdlib.h>
#include <string.h>

#include <algorithm>

#include "common.cuh"
#include "edge_common.cuh"
#include "tc_common.cuh"

namespace {
using namespace edge;
using namespace tc;

constexpr int WG_THREADS = 128, N_WG = 4, TC_THREADS = WG_THREADS * N_WG;   // one CTA per SM
constexpr uint32_t TC_TMEM_COLS = 256;   // 64 columns per WG: S at +0 (16), P at +16 (<= 32)

template <int NPHIP, int NA>
struct BwdTc {
    static constexpr int NAK = (NA + 7) & ~7;        // K of the S product (monomials, zero padded)
    static constexpr int NPK = (NPHIP + 7) & ~7;     // K of the P product (radial index, zero padded)
    static constexpr int NS = 16;                    // N of the S product (N_phi <= 16 padded to the M = 128 step of 16)
    static constexpr int NP = (NA + 15) & ~15;       // N of the P product
    static constexpr int KQ = (NAK + NPK) / 4;       // 16-byte k quads per A operand row
    static constexpr int A_LBO = 128 * 16;           // bytes between k quads of the A operand
    static constexpr int A_IMG = KQ * A_LBO;         // one image (hi or lo)
    static constexpr int BS_IMG = (NAK / 4) * NS * 16, BP_IMG = (NPK / 4) * NP * 16;
    static constexpr int OFF_BS = 2 * A_IMG, OFF_BP = OFF_BS + 2 * BS_IMG, OFF_C = OFF_BP + 2 * BP_IMG;
    static constexpr int WG_BYTES = OFF_C + WG_THREADS * NPHIP * 4;   // + staging of the gathered c_j rows
    static constexpr int NTV = (NPHIP * NA + WG_THREADS - 1) / WG_THREADS;
    static constexpr int SMEM = N_WG * WG_BYTES;
    static_assert(NPHIP % 4 == 0 && NPHIP <= 16 && NPHIP >= 8 && NA >= 4 && NA <= 20, "unsupported edge_tc shape");
};

__device__ __forceinline__ void cp_async16(uint32_t dst, const void *src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// The tiles of a WG form one sequence (atom after atom, 128 edges per tile); everything a tile reads from global
// memory is requested one tile ahead: the edge record (registers), the gathered c_j row (cp.async into this
// thread's own staging row), bbar of the next atom (registers) and the row pointers of the atom after next.
template <int NPHIP, int NA, bool VIR>
__global__ void __launch_bounds__(TC_THREADS, 1) k_edge_bwd_tc(int64_t N, const int64_t *__restrict__ rc_ptr,
                                                               const uint32_t *__restrict__ col_rc,
                                                               const float4 *__restrict__ geom,
                                                               const float *__restrict__ c_ext, RadialTab rt, int S,
                                                               const float *__restrict__ bbar, int want_kappa,
                                                               float *__restrict__ kappa, float4 *__restrict__ gst,
                                                               double *__restrict__ vir_part, AtomChunk ch) {
    using C = BwdTc<NPHIP, NA>;
    constexpr int NB = NPHIP * NA;
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ __align__(16) float tab_s[2][REANN_MAX_S * NPHIP];
    __shared__ __align__(8) unsigned long long mbar_s[N_WG];
    __shared__ uint32_t tmem_base_s;
    const int tid = threadIdx.x, wg = tid >> 7, r = tid & 127, warp = tid >> 5, lane = tid & 31;
    unsigned char *wgs = smem + wg * C::WG_BYTES;
    const uint32_t a_hi = smem_u32(wgs), a_lo = a_hi + C::A_IMG;
    const uint32_t bs_hi = a_hi + C::OFF_BS, bs_lo = bs_hi + C::BS_IMG, bp_hi = a_hi + C::OFF_BP, bp_lo = bp_hi + C::BP_IMG;
    const uint32_t mbar = smem_u32(&mbar_s[wg]);
    float4 *crow = reinterpret_cast<float4 *>(wgs + C::OFF_C + r * (NPHIP * 4));      // this thread's staged c_j row
    const uint32_t crow_s = a_hi + C::OFF_C + r * (NPHIP * 4);

    // ---- prologue: tables, zeroed operand padding, barriers, TMEM ----
    for (int k = tid; k < S * NPHIP; k += TC_THREADS) { tab_s[0][k] = rt.rcen[k]; tab_s[1][k] = rt.alpha2[k]; }
    for (int k = tid; k < C::SMEM / 16; k += TC_THREADS) reinterpret_cast<float4 *>(smem)[k] = make_float4(0.f, 0.f, 0.f, 0.f);
    if (r == 0) mbar_init(mbar, 1);
    if (tid == 0) asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    if (warp == 0) tmem_alloc(&tmem_base_s, TC_TMEM_COLS);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = tmem_base_s + (uint32_t)wg * 64u;                          // this WG's accumulator columns
    const uint32_t tlane = tmem + ((uint32_t)((warp & 3) * 32) << 16);               // this warp's TMEM lanes
    const uint32_t idesc_s = make_idesc(C::NS), idesc_p = make_idesc(C::NP);

    float aV[VIR ? 9 : 1];
#pragma unroll
    for (int k = 0; k < (VIR ? 9 : 1); ++k) aV[k] = 0.f;
    const float pi_rc = 3.14159265358979f * rt.inv_rc;
    uint32_t phase = 0;
    const int64_t stride = (int64_t)gridDim.x * N_WG;

    // ---- pipeline state: current tile (i, e0, end), next atom (i_nx, beg_nx, end_nx) ----
    int64_t i = ch.a0 + (int64_t)blockIdx.x * N_WG + wg;
    int64_t e0 = 0, end = 0, i_nx = i + stride, beg_nx = 0, end_nx = 0;
    float4 g = make_float4(0.f, 0.f, 0.f, 1.f);
    uint32_t cj = 0;
    float tv[C::NTV];
    bool new_atom = true;
    if (i < ch.a1) {
        e0 = rc_ptr[i]; end = rc_ptr[i + 1];
        if (i_nx < ch.a1) { beg_nx = rc_ptr[i_nx]; end_nx = rc_ptr[i_nx + 1]; }
        if (e0 + r < end) {
            g = geom[e0 + r]; cj = col_rc[e0 + r];
            const float4 *src = reinterpret_cast<const float4 *>(c_ext + (int64_t)(cj & COL_IDX_MASK) * NPHIP);
#pragma unroll
            for (int n4 = 0; n4 < NPHIP / 4; ++n4) cp_async16(crow_s + n4 * 16, src + n4);
        }
        cp_async_commit();
#pragma unroll
        for (int q = 0; q < C::NTV; ++q) { const int idx = r + q * WG_THREADS; tv[q] = idx < NB ? __ldg(bbar + i * (int64_t)NB + idx) : 0.f; }
    }
    while (i < ch.a1) {
        const int64_t e = e0 + r;
        const bool have = e < end;
        // ---- the tile after this one: same atom or the next atom; request its edge record now ----
        const bool same = e0 + WG_THREADS < end;
        const int64_t e0_n = same ? e0 + WG_THREADS : beg_nx, end_n = same ? end : end_nx, i_n = same ? i : i_nx;
        const bool have_n = i_n < ch.a1 && e0_n + r < end_n;
        float4 g_n = make_float4(0.f, 0.f, 0.f, 1.f);
        uint32_t cj_n = 0;
        if (have_n) { g_n = geom[e0_n + r]; cj_n = col_rc[e0_n + r]; }
        int64_t beg_nn = 0, end_nn = 0;
        const int64_t i_nn = i_nx + stride;
        if (!same && i_nn < ch.a1) { beg_nn = rc_ptr[i_nn]; end_nn = rc_ptr[i_nn + 1]; }
        // ---- B operands of a new atom: T[n][a] as (N = n, K = a) for S and as (N = a, K = n) for P ----
        if (new_atom) {
            float *bsh = reinterpret_cast<float *>(wgs + C::OFF_BS), *bsl = bsh + C::BS_IMG / 4;
            float *bph = reinterpret_cast<float *>(wgs + C::OFF_BP), *bpl = bph + C::BP_IMG / 4;
#pragma unroll
            for (int q = 0; q < C::NTV; ++q) {
                const int idx = r + q * WG_THREADS;
                if (idx < NB) {
                    float hi, lo;
                    split_tf32(tv[q], hi, lo);
                    const int n = idx / NA, a = idx - n * NA;
                    const int os = (a >> 2) * (C::NS * 4) + n * 4 + (a & 3), op = (n >> 2) * (C::NP * 4) + a * 4 + (n & 3);
                    bsh[os] = hi; bsl[os] = lo; bph[op] = hi; bpl[op] = lo;
                }
            }
        }
        float Rn[NPHIP], yn[NPHIP];
        // ---- phase 1: one edge per thread ----
        cp_async_wait_all();
        if (have) {
            const int sj = cj >> COL_SPECIES_SHIFT;
            float sn, cs;
            sincospif(g.w * rt.inv_rc, &sn, &cs);
            const float fc = 0.5f + 0.5f * cs, dfc = -0.5f * pi_rc * sn;
            // monomials -> S part of the row (k = a, zero padded inside the last partial quad)
            {
                float A[(NA + 3) & ~3];
#pragma unroll
                for (int a = NA; a < ((NA + 3) & ~3); ++a) A[a] = 0.f;
                monomials<NA>(g.x, g.y, g.z, A);
#pragma unroll
                for (int q = 0; q < (NA + 3) / 4; ++q) {
                    float4 h, l;
                    split_tf32(A[4 * q], h.x, l.x); split_tf32(A[4 * q + 1], h.y, l.y);
                    split_tf32(A[4 * q + 2], h.z, l.z); split_tf32(A[4 * q + 3], h.w, l.w);
                    *reinterpret_cast<float4 *>(wgs + q * C::A_LBO + r * 16) = h;
                    *reinterpret_cast<float4 *>(wgs + C::A_IMG + q * C::A_LBO + r * 16) = l;
                }
            }
            // radial functions (alpha2 = alpha log2 e: d/dr exp(-alpha d^2) = -2 ln2 alpha2 d ex); two n per packed op
#pragma unroll
            for (int n4 = 0; n4 < NPHIP / 4; ++n4) {
                const float4 cv = crow[n4];
                const float4 rc4 = reinterpret_cast<const float4 *>(tab_s[0] + sj * NPHIP)[n4];
                const float4 al4 = reinterpret_cast<const float4 *>(tab_s[1] + sj * NPHIP)[n4];
                const float cva[4] = {cv.x, cv.y, cv.z, cv.w}, rca[4] = {rc4.x, rc4.y, rc4.z, rc4.w},
                            ala[4] = {al4.x, al4.y, al4.z, al4.w};
                float xn[4];
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const f32x2 al2 = pack2(ala[2 * h], ala[2 * h + 1]), c2 = pack2(cva[2 * h], cva[2 * h + 1]);
                    const f32x2 d2 = fmadd2(pack2(rca[2 * h], rca[2 * h + 1]), pack2(-1.f, -1.f), pack2(g.w, g.w));
                    const f32x2 ad2 = fmul2(al2, d2);
                    float a0, a1;
                    unpack2(fmul2(ad2, d2), a0, a1);
                    const f32x2 ex2 = pack2(exp2f(-a0), exp2f(-a1));
                    const f32x2 R2 = fmul2(ex2, pack2(fc, fc));
                    const f32x2 y2 = fmul2(c2, fmul2(fmadd2(ad2, pack2(-1.3862943611198906f * fc, -1.3862943611198906f * fc),
                                                            pack2(dfc, dfc)), ex2));
                    unpack2(R2, Rn[n4 * 4 + 2 * h], Rn[n4 * 4 + 2 * h + 1]);
                    unpack2(fmul2(c2, R2), xn[2 * h], xn[2 * h + 1]);
                    unpack2(y2, yn[n4 * 4 + 2 * h], yn[n4 * 4 + 2 * h + 1]);
                }
                float4 h4, l4;
                split_tf32(xn[0], h4.x, l4.x); split_tf32(xn[1], h4.y, l4.y);
                split_tf32(xn[2], h4.z, l4.z); split_tf32(xn[3], h4.w, l4.w);
                *reinterpret_cast<float4 *>(wgs + (C::NAK / 4 + n4) * C::A_LBO + r * 16) = h4;
                *reinterpret_cast<float4 *>(wgs + C::A_IMG + (C::NAK / 4 + n4) * C::A_LBO + r * 16) = l4;
            }
        }
        fence_async_smem();
        tc_fence_before();
        if (wg == 0) asm volatile("bar.sync 1, 128;" ::: "memory");                  // the WG's own named barrier
        else if (wg == 1) asm volatile("bar.sync 2, 128;" ::: "memory");
        else if (wg == 2) asm volatile("bar.sync 3, 128;" ::: "memory");
        else asm volatile("bar.sync 4, 128;" ::: "memory");
        // ---- phase 2: the WG's first thread issues the MMAs ----
        if (r == 0) {
            tc_fence_after();
            const uint32_t dS = tmem, dP = tmem + 16u;
#pragma unroll
            for (int ks = 0; ks < C::NAK / 8; ++ks) {
                const uint64_t al = make_desc(a_lo + ks * 2 * C::A_LBO, C::A_LBO), ah = make_desc(a_hi + ks * 2 * C::A_LBO, C::A_LBO);
                const uint64_t bh = make_desc(bs_hi + ks * 2 * (C::NS * 16), C::NS * 16), bl = make_desc(bs_lo + ks * 2 * (C::NS * 16), C::NS * 16);
                umma_tf32(dS, al, bh, idesc_s, ks > 0 ? 1u : 0u);
                umma_tf32(dS, ah, bl, idesc_s, 1u);
            }
#pragma unroll
            for (int ks = 0; ks < C::NPK / 8; ++ks) {
                const uint32_t ao = (C::NAK / 4 + ks * 2) * C::A_LBO;
                const uint64_t al = make_desc(a_lo + ao, C::A_LBO), ah = make_desc(a_hi + ao, C::A_LBO);
                const uint64_t bh = make_desc(bp_hi + ks * 2 * (C::NP * 16), C::NP * 16), bl = make_desc(bp_lo + ks * 2 * (C::NP * 16), C::NP * 16);
                umma_tf32(dP, al, bh, idesc_p, ks > 0 ? 1u : 0u);
                umma_tf32(dP, ah, bl, idesc_p, 1u);
            }
#pragma unroll
            for (int ks = 0; ks < C::NAK / 8; ++ks)
                umma_tf32(dS, make_desc(a_hi + ks * 2 * C::A_LBO, C::A_LBO), make_desc(bs_hi + ks * 2 * (C::NS * 16), C::NS * 16), idesc_s, 1u);
#pragma unroll
            for (int ks = 0; ks < C::NPK / 8; ++ks)
                umma_tf32(dP, make_desc(a_hi + (C::NAK / 4 + ks * 2) * C::A_LBO, C::A_LBO),
                          make_desc(bp_hi + ks * 2 * (C::NP * 16), C::NP * 16), idesc_p, 1u);
            tc_commit(mbar);
        }
        __syncwarp();
        // ---- while the MMAs run: gather the next tile's c_j row, request the next atom's bbar ----
        if (have_n) {
            const float4 *src = reinterpret_cast<const float4 *>(c_ext + (int64_t)(cj_n & COL_IDX_MASK) * NPHIP);
#pragma unroll
            for (int n4 = 0; n4 < NPHIP / 4; ++n4) cp_async16(crow_s + n4 * 16, src + n4);
        }
        cp_async_commit();
        if (!same && i_n < ch.a1) {
#pragma unroll
            for (int q = 0; q < C::NTV; ++q) { const int idx = r + q * WG_THREADS; tv[q] = idx < NB ? __ldg(bbar + i_n * (int64_t)NB + idx) : 0.f; }
        }
        mbar_wait(mbar, phase);
        phase ^= 1u;
        tc_fence_after();
        // ---- phase 3: S row, then P row of this thread's edge ----
        float radial = 0.f;
        {
            uint32_t sv[16];
            tmem_ld16(tlane, sv);
            tmem_wait_ld();
            if (have) {
#pragma unroll
                for (int n = 0; n < NPHIP; ++n) radial = fmaf(yn[n], __uint_as_float(sv[n]), radial);
                if (want_kappa) {
                    float4 *kp = reinterpret_cast<float4 *>(kappa + (e - ch.e_lo) * (int64_t)NPHIP);
#pragma unroll
                    for (int n4 = 0; n4 < NPHIP / 4; ++n4)
                        kp[n4] = make_float4(Rn[4 * n4] * __uint_as_float(sv[4 * n4]), Rn[4 * n4 + 1] * __uint_as_float(sv[4 * n4 + 1]),
                                             Rn[4 * n4 + 2] * __uint_as_float(sv[4 * n4 + 2]), Rn[4 * n4 + 3] * __uint_as_float(sv[4 * n4 + 3]));
                }
            }
        }
        {
            uint32_t pv[(NA + 3) & ~3];
            if constexpr (NA == 20) { tmem_ld16(tlane + 16u, pv); tmem_ld4(tlane + 32u, pv + 16); }
            else if constexpr (NA == 10) { tmem_ld8(tlane + 16u, pv); tmem_ld4(tlane + 24u, pv + 8); }
            else { tmem_ld4(tlane + 16u, pv); }
            tmem_wait_ld();
            tc_fence_before();
            if (have) {
                float A[NA], P[NA];
                monomials<NA>(g.x, g.y, g.z, A);
#pragma unroll
                for (int a = 0; a < NA; ++a) P[a] = __uint_as_float(pv[a]);
                float gx, gy, gz;
                monomial_vjp<NA>(A, P, gx, gy, gz);
                const float rr = __fdividef(radial, g.w);
                gx = fmaf(rr, g.x, gx); gy = fmaf(rr, g.y, gy); gz = fmaf(rr, g.z, gz);
                gst[e] = make_float4(gx, gy, gz, 0.f);
                if constexpr (VIR) {
                    aV[0] -= g.x * gx; aV[1] -= g.x * gy; aV[2] -= g.x * gz;
                    aV[3] -= g.y * gx; aV[4] -= g.y * gy; aV[5] -= g.y * gz;
                    aV[6] -= g.z * gx; aV[7] -= g.z * gy; aV[8] -= g.z * gz;
                }
            }
        }
        // ---- rotate the pipeline ----
        new_atom = !same;
        if (!same) { i = i_nx; i_nx = i_nn; beg_nx = beg_nn; end_nx = end_nn; }
        e0 = e0_n; end = end_n; g = g_n; cj = cj_n;
    }
    // ---- epilogue: virial partial of this block (fixed order; the operand area is free now), TMEM release ----
    tc_fence_before();
    __syncthreads();
    if constexpr (VIR) {
        float(*vir_s)[9] = reinterpret_cast<float(*)[9]>(smem);
#pragma unroll
        for (int d = 16; d >= 1; d >>= 1)
#pragma unroll
            for (int k = 0; k < 9; ++k) aV[k] += __shfl_xor_sync(0xffffffffu, aV[k], d);
        if (lane == 0) {
#pragma unroll
            for (int k = 0; k < 9; ++k) vir_s[warp][k] = aV[k];
        }
        __syncthreads();
        if (tid < 9) {
            double s = 0.0;
#pragma unroll
            for (int w = 0; w < TC_THREADS / 32; ++w) s += (double)vir_s[w][tid];
            vir_part[(int64_t)blockIdx.x * 9 + tid] += s;
        }
    }
    if (warp == 0) tmem_dealloc(tmem_base_s, TC_TMEM_COLS);
}

template <int NPHIP, int NA>
int run_edge_bwd_tc(const LaunchCtx &ctx, int64_t N, const int64_t *rc_ptr, const uint32_t *col_rc, const float4 *geom,
                    const float *c_ext, RadialTab rt, int S, const float *bbar, int want_kappa, float *kappa, float4 *gst,
                    double *vir_part, AtomChunk ch, int n_blocks) {
    using C = BwdTc<NPHIP, NA>;
    static bool attr_set[64] = {};
    int dev = 0;
    cudaGetDevice(&dev);
    if (dev < 0 || dev >= 64) return REANN_ERR_UNSUPPORTED;
    if (!attr_set[dev]) {
        if (cudaFuncSetAttribute(k_edge_bwd_tc<NPHIP, NA, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM) != cudaSuccess ||
            cudaFuncSetAttribute(k_edge_bwd_tc<NPHIP, NA, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM) != cudaSuccess) {
            cudaGetLastError();
            return REANN_ERR_CUDA;
        }
        attr_set[dev] = true;
    }
    if (vir_part)
        LAUNCH(ctx, (k_edge_bwd_tc<NPHIP, NA, true>), n_blocks, TC_THREADS, C::SMEM, N, rc_ptr, col_rc, geom, c_ext, rt, S, bbar,
               want_kappa, kappa, gst, vir_part, ch);
    else
        LAUNCH(ctx, (k_edge_bwd_tc<NPHIP, NA, false>), n_blocks, TC_THREADS, C::SMEM, N, rc_ptr, col_rc, geom, c_ext, rt, S, bbar,
               want_kappa, kappa, gst, vir_part, ch);
    return REANN_OK;
}

} // namespace

bool edge_bwd_tc_supported(const ModelDims &md) {
    return (md.nphip == 8 || md.nphip == 12 || md.nphip == 16) && (md.Na == 4 || md.Na == 10 || md.Na == 20);
}

// persistent grid: one CTA of four warpgroups per SM (shared memory), fewer for small systems
int edge_bwd_tc_blocks(int64_t n_atoms) {
    static int n_sm = 0;
    if (!n_sm) {
        int dev = 0;
        cudaGetDevice(&dev);
        if (cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n_sm <= 0) n_sm = 148;
    }
    const int64_t want = (n_atoms + N_WG - 1) / N_WG;
    return (int)std::max<int64_t>(1, std::min<int64_t>(n_sm, want));
}

int launch_edge_bwd_tc(const LaunchCtx &ctx, const ModelDims &md, int t, int64_t N, const int64_t *rc_ptr,
                       const uint32_t *col_rc, const float4 *geom, const float *c_ext, const float *rcen,
                       const float *alpha, const float *bbar, float *kappa, float4 *gst, double *vir_part, int64_t a0,
                       int64_t a1, int64_t e_lo) {
    if (N <= 0 || a1 <= a0) return REANN_OK;
    const AtomChunk ch{a0, a1, e_lo};
    RadialTab rt{rcen + (size_t)t * md.S * md.nphip, alpha + (size_t)t * md.S * md.nphip, (float)(1.0 / md.rc)};
    const int want_kappa = t >= 1, nb = edge_bwd_tc_blocks(a1 - a0);
#define M(NP, NA_) return run_edge_bwd_tc<NP, NA_>(ctx, N, rc_ptr, col_rc, geom, c_ext, rt, md.S, bbar, want_kappa, kappa, gst, vir_part, ch, nb);
    switch (md.nphip * 100 + md.Na) {
        case 804: M(8, 4) case 810: M(8, 10) case 820: M(8, 20)
        case 1204: M(12, 4) case 1210: M(12, 10) case 1220: M(12, 20)
        case 1604: M(16, 4) case 1610: M(16, 10) case 1620: M(16, 20)
        default: return REANN_ERR_UNSUPPORTED;
    }
#undef M
}
