// edge.cu -- per-evaluation edge work: rows A4 (skin check), A5 (edge forward), A8 (ghost gather),
// A10 (edge backward), A11 (reverse gather) and A12 (outputs) of SURVEY.md section 8(a), plus the
// per-step rc-filter that compacts the skin list into the r < rc edges all layers reuse
// (one list, reused by every MP layer).
//
// Orbitals (Eq. 1; readings A-2..A-5 of SURVEY.md 8(c)):
//   x_e[n] = c_j[n] * exp(-alpha_n (r_e - r_n)^2) * f_c(r_e),   f_c(r) = (1 + cos(pi r / rc)) / 2
//   A_a(r_e) = x^lx y^ly z^lz,  a = (lx,ly,lz), lx+ly+lz <= L (graded order, see monomials<>())
//   b_i[n,a] = sum_{e in row(i), r_e < rc} x_e[n] A_a(r_e)
// Backward (Eqs. 3-5, vector-Jacobian products):
//   S_n = sum_a bbar_i[n,a] A_a;  P_a = sum_n bbar_i[n,a] x_e[n]
//   g_e = (sum_n c_j[n] R'_n S_n) r_hat + sum_a P_a grad A_a;   kappa_e[n] = R_n S_n  (t >= 1)
//   cbar_k[n] = sum_{e in row(k)} kappa_{rev(e)}[n];   F_k = sum_{e in row(k)} (g_e - g_{rev(e)})
// No floating-point atomics anywhere: the neighbour-side sums are gathers through rev[].
#include <stdlib.h>
#include <string.h>

#include <algorithm>

#include "common.cuh"
#include "edge_common.cuh"

namespace {
using namespace edge;

constexpr int EW = 4; // warps per block in the edge kernels
constexpr int RW = 2; // warps per block of the row-streaming kernels (rc-filter, reverse gather): a warp takes one row

// ------------------------------------------------------------------------------------------ A4
__global__ void k_skin_check(const double *__restrict__ pos, const double *__restrict__ pos_build, int64_t n3,
                             double thr2, int32_t *__restrict__ flag) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    bool moved = false;
    if (i * 3 < n3) {
        double dx = pos[3 * i] - pos_build[3 * i], dy = pos[3 * i + 1] - pos_build[3 * i + 1],
               dz = pos[3 * i + 2] - pos_build[3 * i + 2];
        moved = (dx * dx + dy * dy + dz * dz) > thr2;
    }
    if (__syncthreads_or(moved) && threadIdx.x == 0) atomicOr(flag, 1);
}

// positions of all ext atoms in the build-time wrapped frame; layer-0 coefficients c^0 = c0[species]
__global__ void k_refresh(XRec *__restrict__ xrec, int64_t n_ext, const int32_t *__restrict__ perm,
                          const int32_t *__restrict__ wshift, const double *__restrict__ pos, BoxP B,
                          float *__restrict__ c_ext0, const float *__restrict__ c0, int nphip) {
    int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n_ext) return;
    XRec r = xrec[k];
    const int64_t i = perm[r.owner];
    double hx, hy, hz;
    box_shift(B, (double)wshift[3 * i], (double)wshift[3 * i + 1], (double)wshift[3 * i + 2], hx, hy, hz);
    r.x = __dsub_rn(pos[3 * i], hx);
    r.y = __dsub_rn(pos[3 * i + 1], hy);
    r.z = __dsub_rn(pos[3 * i + 2], hz);
    xrec[k] = r;
    for (int n = 0; n < nphip; ++n) c_ext0[k * nphip + n] = c0[r.species * nphip + n];
}

__device__ __forceinline__ double edge_d2(const XRec &me, const XRec &o, const BoxP &B, double *dx, double *dy, double *dz) {
    double hx, hy, hz;
    box_shift(B, (double)o.sx, (double)o.sy, (double)o.sz, hx, hy, hz);
    *dx = __dadd_rn(__dsub_rn(o.x, me.x), hx);
    *dy = __dadd_rn(__dsub_rn(o.y, me.y), hy);
    *dz = __dadd_rn(__dsub_rn(o.z, me.z), hz);
    return __dadd_rn(__dadd_rn(__dmul_rn(*dx, *dx), __dmul_rn(*dy, *dy)), __dmul_rn(*dz, *dz));
}

// rc-filter, pass 1: rank of every accepted list entry inside its row (0xFFFF = rejected)
__global__ void __launch_bounds__(RW * 32) k_filter_count(const XRec *__restrict__ xrec,
                                                          const int64_t *__restrict__ row_ptr,
                                                          const int32_t *__restrict__ col, int64_t N, BoxP B, double rc2,
                                                          uint16_t *__restrict__ rank16, int32_t *__restrict__ rc_cnt) {
    const int lane = threadIdx.x & 31;
    const int64_t i = (int64_t)blockIdx.x * RW + (threadIdx.x >> 5);
    if (i >= N) return;
    const XRec me = xrec[i];
    const int64_t r0 = row_ptr[i], r1 = row_ptr[i + 1];
    int cnt = 0;
    // two batches of 32 list entries per iteration: both gathers are in flight together
    for (int64_t eb = r0; eb < r1; eb += 64) {
        const int64_t e0 = eb + lane, e1 = e0 + 32;
        int32_t j0 = 0, j1 = 0;
        if (e0 < r1) j0 = col[e0];
        if (e1 < r1) j1 = col[e1];
        XRec o0 = me, o1 = me;
        if (e0 < r1) o0 = xrec[j0];
        if (e1 < r1) o1 = xrec[j1];
        double dx, dy, dz;
        const bool in0 = e0 < r1 && edge_d2(me, o0, B, &dx, &dy, &dz) < rc2;
        const bool in1 = e1 < r1 && edge_d2(me, o1, B, &dx, &dy, &dz) < rc2;
        const unsigned m0 = __ballot_sync(0xffffffffu, in0), m1 = __ballot_sync(0xffffffffu, in1);
        if (e0 < r1) rank16[e0] = in0 ? (uint16_t)(cnt + __popc(m0 & ((1u << lane) - 1))) : (uint16_t)0xFFFF;
        cnt += __popc(m0);
        if (e1 < r1) rank16[e1] = in1 ? (uint16_t)(cnt + __popc(m1 & ((1u << lane) - 1))) : (uint16_t)0xFFFF;
        cnt += __popc(m1);
    }
    if (lane == 0) rc_cnt[i] = cnt;
}

// offset of the compact row of the owner of every ext atom (ghosts: their owner's row), so that the fill pass below
// finds the row of a reverse edge with one 4-byte gather that does not wait for the neighbour's record
__global__ void k_rc_ext(const XRec *__restrict__ xrec, const int64_t *__restrict__ rc_ptr, int64_t N, int64_t n_ext,
                         uint32_t *__restrict__ rcx, const int32_t *__restrict__ skip) {
    SKIP_GUARD(skip);
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n_ext) return;
    rcx[k] = (uint32_t)rc_ptr[k < N ? k : (int64_t)xrec[k].owner];
}

// rc-filter, pass 2: compact rows (neighbour ext index | species<<28, edge vector + length in FP32
// rounded once from the FP64 difference, index of the reverse compact edge). Two levels of dependent loads per
// iteration: (rank, col, rev) of the entry, then (record, rank of the reverse entry, row offset of the owner).
// Bound by the latency of its gathers: 64 registers (16 two-warp blocks per SM) with two entries per lane in flight
// measured best on config 3 (prep 0.55 -> 0.50 ms per step against four entries at 94 registers = 10 blocks per SM;
// one entry or 20+ blocks spill and are slower).
__global__ void __launch_bounds__(RW * 32, 16) k_filter_fill(const XRec *__restrict__ xrec,
                                                         const int64_t *__restrict__ row_ptr,
                                                         const int32_t *__restrict__ col,
                                                         const uint32_t *__restrict__ rev, int64_t N, BoxP B,
                                                         const uint16_t *__restrict__ rank16,
                                                         const int64_t *__restrict__ rc_ptr,
                                                         const uint32_t *__restrict__ rcx,
                                                         uint32_t *__restrict__ col_rc, float4 *__restrict__ geom,
                                                         uint32_t *__restrict__ rev_rc, const int32_t *__restrict__ skip) {
    SKIP_GUARD(skip);
    const int lane = threadIdx.x & 31;
    const int64_t i = (int64_t)blockIdx.x * RW + (threadIdx.x >> 5);
    if (i >= N) return;
    const XRec me = xrec[i];
    const int64_t r0 = row_ptr[i], r1 = row_ptr[i + 1], c0 = rc_ptr[i];
    // two list entries per lane and iteration: their gathers are all in flight together
    constexpr int U = 2;
    for (int64_t eb = r0 + lane; eb < r1; eb += 32 * U) {
        uint16_t rk[U];
        int32_t j[U];
        uint32_t rv[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int64_t e = eb + 32 * u;
            rk[u] = 0xFFFF; j[u] = 0; rv[u] = 0;
            if (e < r1) { rk[u] = rank16[e]; j[u] = col[e]; rv[u] = rev[e]; }
        }
        XRec o[U];
        uint16_t rrk[U];
        uint32_t base[U];
#pragma unroll
        for (int u = 0; u < U; ++u)
            if (rk[u] != 0xFFFF) { o[u] = xrec[j[u]]; rrk[u] = rank16[rv[u]]; base[u] = rcx[j[u]]; }
#pragma unroll
        for (int u = 0; u < U; ++u)
            if (rk[u] != 0xFFFF) {
                double dx, dy, dz;
                const double d2 = edge_d2(me, o[u], B, &dx, &dy, &dz);
                const int64_t ce = c0 + rk[u];
                col_rc[ce] = (uint32_t)j[u] | ((uint32_t)o[u].species << COL_SPECIES_SHIFT);
                geom[ce] = make_float4((float)dx, (float)dy, (float)dz, (float)sqrt(d2));
                rev_rc[ce] = base[u] + rrk[u];
            }
    }
}

// ------------------------------------------------------------------------------------------ A8
// c_ext[N+g][:] = c[owner[g]][:]  -- the paper's forward LA -> GA message.
__global__ void k_ghost_gather(float *__restrict__ c_ext, const XRec *__restrict__ xrec, int64_t N, int64_t n_ext,
                               int nphip, const int32_t *__restrict__ skip) {
    SKIP_GUARD(skip);
    const int q4 = nphip >> 2;
    int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int64_t g = N + idx / q4;
    if (g >= n_ext) return;
    int part = (int)(idx % q4);
    const float4 *src = reinterpret_cast<const float4 *>(c_ext + (int64_t)xrec[g].owner * nphip);
    reinterpret_cast<float4 *>(c_ext + g * nphip)[part] = src[part];
}

// ------------------------------------------------------------------------------------------ A5
// Warp-autonomous: a warp owns APW = 32/LPA atoms; lane group `sub` (LPA lanes) owns atom `sub` and
// every lane of it a PN x PA block of b_i[n,a] in registers. Per round the warp stages 32 edges,
// EPA = 32/APW of each of its atoms (staged row = lane):
//   1a  one edge per lane: edge record, cutoff function, monomials A_a -> shared memory;
//   1b  NPHIP/4 lanes per edge: each gathers one float4 of c_j (a load instruction then touches
//       whole 64-byte rows) and stores its four x_e[n];
//   2   every lane accumulates its block over the staged edges of its atom (operands read as
//       vectors from shared memory, no atomics).
// Shared memory delivers 128 B per clock to the lanes whether or not they read the same word, so
// what counts is operand floats per FMA: (PN + PA) / (PN PA) -- hence the large register blocks.
template <int NPHIP, int NA, int PN, int PA>
struct FwdCfg {
    static constexpr int NG = NPHIP / PN, AG = (NA + PA - 1) / PA, LPA = NG * AG, APW = 32 / LPA, EPA = 32 / APW;
    static constexpr int AST = (PA + 3) & ~3;            // floats reserved per a-group (16-B aligned)
    static constexpr int ROW = NPHIP + AG * AST + 4;     // +4: de-phase rows across banks
    static constexpr int SMEM = EW * 32 * ROW * 4;
    static_assert(NPHIP % PN == 0 && 32 % LPA == 0 && NPHIP % 4 == 0, "bad edge-forward tiling");
};

template <int NPHIP, int NA, int PN, int PA>
__global__ void __launch_bounds__(EW * 32) k_edge_fwd(int64_t N, const int64_t *__restrict__ rc_ptr,
                                                      const uint32_t *__restrict__ col_rc,
                                                      const float4 *__restrict__ geom,
                                                      const float *__restrict__ c_ext, RadialTab rt,
                                                      float *__restrict__ b, const int32_t *__restrict__ skip) {
    SKIP_GUARD(skip);
    using C = FwdCfg<NPHIP, NA, PN, PA>;
    extern __shared__ __align__(16) float smem_f[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    float *stage = smem_f + (size_t)warp * 32 * C::ROW;
    const int sub = lane / C::LPA, sl = lane % C::LPA, p = sl % C::NG, q = sl / C::NG;
    const int64_t atom0 = ((int64_t)blockIdx.x * EW + warp) * C::APW;
    if (atom0 >= N) return;
    const int64_t my_atom = atom0 + sub;
    int64_t my_beg = 0, my_end = 0;
    if (my_atom < N) { my_beg = rc_ptr[my_atom]; my_end = rc_ptr[my_atom + 1]; }
    int64_t maxlen = my_end - my_beg;
#pragma unroll
    for (int d = 16; d >= 1; d >>= 1) maxlen = max(maxlen, __shfl_xor_sync(0xffffffffu, maxlen, d));
    // phase 1a: lane -> (atom slot, edge within the round); EPA == LPA, so slot == sub
    const int le = lane % C::EPA;
    float acc[PN][PA];
#pragma unroll
    for (int a = 0; a < PN; ++a)
#pragma unroll
        for (int c = 0; c < PA; ++c) acc[a][c] = 0.0f;

    for (int64_t c0 = 0; c0 < maxlen; c0 += C::EPA) {
        // ---- phase 1a ----
        const int64_t e = my_beg + c0 + le;
        float4 g = make_float4(0.f, 0.f, 0.f, 0.f);
        uint32_t cj = 0;
        float fc = 0.f;
        const bool have = e < my_end;
        if (have) {
            g = geom[e];
            cj = col_rc[e];
            fc = 0.5f + 0.5f * cospif(g.w * rt.inv_rc);
            float *row = stage + (size_t)lane * C::ROW;
            float A[C::AG * C::AST];
#pragma unroll
            for (int a = 0; a < C::AG * C::AST; ++a) A[a] = 0.0f;
            float Am[NA];
            monomials<NA>(g.x, g.y, g.z, Am);
#pragma unroll
            for (int a = 0; a < NA; ++a) A[(a / PA) * C::AST + a % PA] = Am[a];
#pragma unroll
            for (int v4 = 0; v4 < C::AG * C::AST / 4; ++v4)
                reinterpret_cast<float4 *>(row + NPHIP)[v4] = make_float4(A[4 * v4], A[4 * v4 + 1], A[4 * v4 + 2], A[4 * v4 + 3]);
        }
        // ---- phase 1b ----
        {
            constexpr int PARTS = NPHIP / 4, EPI = 32 / PARTS, ROUNDS = (32 + EPI - 1) / EPI;
            const int part = lane % PARTS;
#pragma unroll
            for (int r = 0; r < ROUNDS; ++r) {
                const int rr = r * EPI + lane / PARTS;            // staged row = lane that holds its record
                const bool mine = lane < EPI * PARTS && rr < 32;
                const int src = mine ? rr : 0;
                const uint32_t cje = __shfl_sync(0xffffffffu, cj, src);
                const float we = __shfl_sync(0xffffffffu, g.w, src);
                const float fce = __shfl_sync(0xffffffffu, fc, src);
                const int ok = __shfl_sync(0xffffffffu, (int)have, src);
                if (mine && ok) {
                    const int sj = cje >> COL_SPECIES_SHIFT;
                    const float4 cv = reinterpret_cast<const float4 *>(c_ext + (int64_t)(cje & COL_IDX_MASK) * NPHIP)[part];
                    const float4 rc4 = reinterpret_cast<const float4 *>(rt.rcen + sj * NPHIP)[part];
                    const float4 al4 = reinterpret_cast<const float4 *>(rt.alpha2 + sj * NPHIP)[part];
                    float4 xv;
                    float d;
                    d = we - rc4.x; xv.x = cv.x * (ex2_ftz(-al4.x * d * d) * fce);
                    d = we - rc4.y; xv.y = cv.y * (ex2_ftz(-al4.y * d * d) * fce);
                    d = we - rc4.z; xv.z = cv.z * (ex2_ftz(-al4.z * d * d) * fce);
                    d = we - rc4.w; xv.w = cv.w * (ex2_ftz(-al4.w * d * d) * fce);
                    reinterpret_cast<float4 *>(stage + (size_t)rr * C::ROW)[part] = xv;
                }
            }
        }
        __syncwarp();
        // ---- phase 2: register-tiled accumulation over the staged edges of my atom ----
        int64_t cnt64 = my_end - (my_beg + c0);
        const int cnt = cnt64 > C::EPA ? C::EPA : (cnt64 < 0 ? 0 : (int)cnt64);
        const float *rowb = stage + (size_t)(sub * C::EPA) * C::ROW;
#pragma unroll 4
        for (int k = 0; k < cnt; ++k) {
            const float *row = rowb + (size_t)k * C::ROW;
            float xv[PN], av[PA];
            if constexpr (PN % 4 == 0) {
#pragma unroll
                for (int a4 = 0; a4 < PN / 4; ++a4) {
                    const float4 v = *reinterpret_cast<const float4 *>(row + p * PN + a4 * 4);
                    xv[a4 * 4] = v.x; xv[a4 * 4 + 1] = v.y; xv[a4 * 4 + 2] = v.z; xv[a4 * 4 + 3] = v.w;
                }
            } else if constexpr (PN == 2) {
                const float2 v = *reinterpret_cast<const float2 *>(row + p * 2);
                xv[0] = v.x; xv[1] = v.y;
            } else {
#pragma unroll
                for (int a = 0; a < PN; ++a) xv[a] = row[p * PN + a];
            }
            const float *ar = row + NPHIP + q * C::AST;
#pragma unroll
            for (int c4 = 0; c4 < PA / 4; ++c4) {
                const float4 v = *reinterpret_cast<const float4 *>(ar + c4 * 4);
                av[c4 * 4] = v.x; av[c4 * 4 + 1] = v.y; av[c4 * 4 + 2] = v.z; av[c4 * 4 + 3] = v.w;
            }
            if constexpr (PA % 4 >= 2) {
                const float2 v = *reinterpret_cast<const float2 *>(ar + (PA / 4) * 4);
                av[(PA / 4) * 4] = v.x; av[(PA / 4) * 4 + 1] = v.y;
            }
            if constexpr (PA % 2 == 1) av[PA - 1] = ar[PA - 1];
#pragma unroll
            for (int a = 0; a < PN; ++a)
#pragma unroll
                for (int c = 0; c < PA; ++c) acc[a][c] = fmaf(xv[a], av[c], acc[a][c]);
        }
        __syncwarp();
    }
    if (my_atom < N) {
        float *bi = b + my_atom * (int64_t)(NPHIP * NA);
#pragma unroll
        for (int a = 0; a < PN; ++a)
#pragma unroll
            for (int c = 0; c < PA; ++c)
                if (q * PA + c < NA) bi[(p * PN + a) * NA + q * PA + c] = acc[a][c];
    }
}

// ------------------------------------------------------------------------------------------ A5 (MMA)
// Edge forward with the neighbour sum on the tensor cores: b_i[n,a] = sum_e X[e,n] A[e,a] is a
// (N_phi x edges) x (edges x N_a) product with K = the edges of atom i. Warp per atom, rounds of 32 edges:
// phase 1 as in k_edge_fwd (edge record / monomials one edge per lane, x_e[n] by N_phi/4 lanes per edge)
// but staged transposed, XT[n][e] | AT[a][e] with a row stride of 36 floats, so that both the scalar
// stores and the mma.sync fragment loads are conflict-free; phase 2: four K = 8 steps of
// mma.sync.m16n8k8 TF32 (3xTF32: lo.hi + hi.lo + hi.hi into a fresh accumulator per step, summed in FP32
// registers: accumulating the ~36 steps of an atom inside the MMA truncates like tcgen05 does and was measured
// to cost 1.4e-6 eV/atom on config 2, above the 1e-6 gate). N_phi (padded to 4) in {8, 12, 16}: the M = 16 rows
// beyond N_phi are zero.
constexpr int FW = 1; // warps per block of the mma.sync edge forward kernel: a warp takes one atom and leaves
template <int NA>
struct FwdMma {
    static constexpr int NAP = (NA + 7) & ~7, AT = NAP / 8, TS = 36;
    static constexpr int ROWS = 16 + NAP, SMEM = FW * ROWS * TS * 4;
};

template <int NPHIP, int NA>
__global__ void __launch_bounds__(FW * 32) k_edge_fwd_mma(int64_t N, const int64_t *__restrict__ rc_ptr,
                                                          const uint32_t *__restrict__ col_rc,
                                                          const float4 *__restrict__ geom,
                                                          const float *__restrict__ c_ext, RadialTab rt,
                                                          float *__restrict__ b, const int32_t *__restrict__ skip) {
    SKIP_GUARD(skip);
    using C = FwdMma<NA>;
    constexpr int NAP = C::NAP, AT = C::AT, TS = C::TS;
    static_assert(NPHIP == 8 || NPHIP == 12 || NPHIP == 16, "mma.sync edge forward: N_phi padded to 8, 12 or 16");
    extern __shared__ __align__(16) float smem_f[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, g8 = lane >> 2, t4 = lane & 3;
    float *XT = smem_f + (size_t)warp * C::ROWS * TS, *AT_s = XT + 16 * TS;
    const int64_t i = (int64_t)blockIdx.x * FW + warp;
    if (i >= N) return;
    const int64_t beg = rc_ptr[i], end = rc_ptr[i + 1];
    float acc[AT][4];
#pragma unroll
    for (int at = 0; at < AT; ++at) acc[at][0] = acc[at][1] = acc[at][2] = acc[at][3] = 0.f;
    float4 g_nx = make_float4(0.f, 0.f, 0.f, 0.f);
    uint32_t cj_nx = 0;
    if (beg + lane < end) { g_nx = geom[beg + lane]; cj_nx = col_rc[beg + lane]; }
    for (int64_t e0 = beg; e0 < end; e0 += 32) {
        // ---- phase 1a: one edge per lane (the next round's record is fetched one round ahead) ----
        const int64_t e = e0 + lane;
        const bool have = e < end;
        const float4 g = g_nx;
        const uint32_t cj = cj_nx;
        if (e + 32 < end) { g_nx = geom[e + 32]; cj_nx = col_rc[e + 32]; }
        float fc = 0.f;
        {
            float A[NAP];
#pragma unroll
            for (int a = 0; a < NAP; ++a) A[a] = 0.f;
            if (have) {
                fc = 0.5f + 0.5f * cospif(g.w * rt.inv_rc);
                monomials<NA>(g.x, g.y, g.z, A);
            }
#pragma unroll
            for (int a = 0; a < NAP; ++a) AT_s[a * TS + lane] = A[a];       // zeros for the lanes past the row's end
        }
        // ---- phase 1b: four lanes per edge, one float4 of c_j each ----
        {
            const int part = lane & 3;
#pragma unroll
            for (int r = 0; r < 4; ++r) {
                const int rr = r * 8 + (lane >> 2);
                const uint32_t cje = __shfl_sync(0xffffffffu, cj, rr);
                const float we = __shfl_sync(0xffffffffu, g.w, rr);
                const float fce = __shfl_sync(0xffffffffu, fc, rr);
                float4 xv = make_float4(0.f, 0.f, 0.f, 0.f);
                if (e0 + rr < end && part * 4 < NPHIP) {
                    const int sj = cje >> COL_SPECIES_SHIFT;
                    const float4 cv = reinterpret_cast<const float4 *>(c_ext + (int64_t)(cje & COL_IDX_MASK) * NPHIP)[part];
                    const float4 rc4 = reinterpret_cast<const float4 *>(rt.rcen + sj * NPHIP)[part];
                    const float4 al4 = reinterpret_cast<const float4 *>(rt.alpha2 + sj * NPHIP)[part];
                    // x_n = c_j[n] exp2(-alpha2 (r - r_n)^2) f_c(r), two n per packed operation
                    const f32x2 w2 = pack2(we, we), m1 = pack2(-1.f, -1.f), f2 = pack2(fce, fce);
                    const f32x2 da = fmadd2(pack2(rc4.x, rc4.y), m1, w2), db = fmadd2(pack2(rc4.z, rc4.w), m1, w2);
                    float a0, a1, a2, a3;
                    unpack2(fmul2(fmul2(pack2(al4.x, al4.y), da), da), a0, a1);
                    unpack2(fmul2(fmul2(pack2(al4.z, al4.w), db), db), a2, a3);
                    unpack2(fmul2(pack2(cv.x, cv.y), fmul2(pack2(ex2_ftz(-a0), ex2_ftz(-a1)), f2)), xv.x, xv.y);
                    unpack2(fmul2(pack2(cv.z, cv.w), fmul2(pack2(ex2_ftz(-a2), ex2_ftz(-a3)), f2)), xv.z, xv.w);
                }
                float *dst = XT + (part * 4) * TS + rr;
                dst[0] = xv.x; dst[TS] = xv.y; dst[2 * TS] = xv.z; dst[3 * TS] = xv.w;
            }
        }
        __syncwarp();
        // ---- phase 2: K = 8 edges per step ----
        const int nks = (int)((end - e0 + 7) >> 3) < 4 ? (int)((end - e0 + 7) >> 3) : 4;
#pragma unroll 1
        for (int ks = 0; ks < nks; ++ks) {
            const float *xa = XT + g8 * TS + ks * 8 + t4;
            uint32_t ah[4], al[4];
            split_bits(xa[0], ah[0], al[0]); split_bits(xa[8 * TS], ah[1], al[1]);
            split_bits(xa[4], ah[2], al[2]); split_bits(xa[8 * TS + 4], ah[3], al[3]);
#pragma unroll
            for (int at = 0; at < AT; ++at) {
                const float *ba = AT_s + (at * 8 + g8) * TS + ks * 8 + t4;
                uint32_t bh0, bl0, bh1, bl1;
                split_bits(ba[0], bh0, bl0); split_bits(ba[4], bh1, bl1);
                float d[4] = {0.f, 0.f, 0.f, 0.f};
                mma_tf32(d, al, bh0, bh1);
                mma_tf32(d, ah, bl0, bl1);
                mma_tf32(d, ah, bh0, bh1);
                acc[at][0] += d[0]; acc[at][1] += d[1]; acc[at][2] += d[2]; acc[at][3] += d[3];
            }
        }
        __syncwarp();
    }
    // C fragment: rows n = g, g + 8; columns a = at*8 + 2t, +1
    float *bi = b + i * (int64_t)(NPHIP * NA);
#pragma unroll
    for (int at = 0; at < AT; ++at) {
        const int a = at * 8 + 2 * t4;
        if (a < NA) {
            *reinterpret_cast<float2 *>(bi + g8 * NA + a) = make_float2(acc[at][0], acc[at][1]);
            if (g8 + 8 < NPHIP) *reinterpret_cast<float2 *>(bi + (g8 + 8) * NA + a) = make_float2(acc[at][2], acc[at][3]);
        }
    }
}

// ------------------------------------------------------------------------------------------ A10
// Warp per atom; bbar_i is broadcast from shared memory, S_n and P_a stay in the lane's registers, so there is no
// cross-lane reduction per edge. Orbitals are recomputed (nothing per-edge is kept from the forward pass). Writes
// the per-edge stash g_e (float4) and kappa_e; the forces are gathered from the g_e stash by k_rev_gather.
// Shared memory delivers 128 B per clock to the lanes whether or not they read the same word, and every float of
// bbar_i feeds only two FMAs per edge (S and P), so a lane takes NE = 2 edges per pass while more than 32 remain:
// one 16-byte read then feeds 16 FMAs instead of 8 (the last <= 32 edges of a row go one per lane).
// VIR: accumulate the virial (only when the caller asked for it).
template <int NPHIP, int NA, bool VIR, int NE>
__device__ __forceinline__ void edge_bwd_pass(int64_t e0, int64_t end, const uint32_t *__restrict__ col_rc,
                                              const float4 *__restrict__ geom, const float *__restrict__ c_ext,
                                              const float *__restrict__ tab_rc, const float *__restrict__ tab_al,
                                              float inv_rc, const float *__restrict__ bb, int want_kappa,
                                              float *__restrict__ kappa, float4 *__restrict__ gst, int64_t e_lo, float *aV,
                                              const float4 *g_s, const uint32_t *cj_s /* prefetched records of the row's first 64 edges, or nullptr */) {
    constexpr bool PAIRS = NA % 2 == 0;                   // (a, a+1) pairs never straddle a row of bbar_i
    constexpr int NP2 = PAIRS ? NA / 2 : 1;
    static_assert(PAIRS || NE == 1, "two edges per lane need an even number of monomials");
    const float pi_rc = 3.14159265358979f * inv_rc;
    int64_t e[NE];
    bool have[NE];
    float4 g[NE];
    int sj[NE];
    const float4 *cptr[NE];
    float fc[NE], dfc[NE], radial[NE];
    float A[NE][NA], P[NE][NA];
    f32x2 A2[NE][NP2], P2[NE][NP2];
#pragma unroll
    for (int k = 0; k < NE; ++k) {
        e[k] = e0 + 32 * k;
        have[k] = e[k] < end;
        g[k] = make_float4(0.f, 0.f, 0.f, 1.f);
        uint32_t cj = 0;
        if (have[k]) {
            if (g_s) { g[k] = g_s[32 * k]; cj = cj_s[32 * k]; }
            else { g[k] = geom[e[k]]; cj = col_rc[e[k]]; }
        }
        sj[k] = cj >> COL_SPECIES_SHIFT;
        cptr[k] = reinterpret_cast<const float4 *>(c_ext + (int64_t)(cj & COL_IDX_MASK) * NPHIP);
    }
#pragma unroll
    for (int k = 0; k < NE; ++k) {
        float sn, cs;
        sincospif(g[k].w * inv_rc, &sn, &cs);
        fc[k] = 0.5f + 0.5f * cs; dfc[k] = -0.5f * pi_rc * sn;
        monomials<NA>(g[k].x, g[k].y, g[k].z, A[k]);
        radial[k] = 0.f;
#pragma unroll
        for (int a = 0; a < NA; ++a) P[k][a] = 0.f;
        if constexpr (PAIRS) {
#pragma unroll
            for (int a2 = 0; a2 < NP2; ++a2) { A2[k][a2] = pack2(A[k][2 * a2], A[k][2 * a2 + 1]); P2[k][a2] = pack2(0.f, 0.f); }
        }
    }
    // four rows n of bbar_i per outer iteration (one float4 of c_j / r_n / alpha_n / kappa);
    // the outer loop is kept rolled so that the shared-memory loads are not all hoisted. The gathered c_j quad of
    // the next iteration is requested one iteration ahead (an L2 round trip).
    float4 cvc[NE];
#pragma unroll
    for (int k = 0; k < NE; ++k) cvc[k] = cptr[k][0];
#pragma unroll 1
    for (int n4 = 0; n4 < NPHIP / 4; ++n4) {
        float Rn[NE][4], xn[NE][4], yn[NE][4], Sn[NE][4];
        float4 cvn[NE];
#pragma unroll
        for (int k = 0; k < NE; ++k) cvn[k] = cptr[k][n4 + 1 < NPHIP / 4 ? n4 + 1 : n4];
#pragma unroll
        for (int k = 0; k < NE; ++k) {
            const float4 cv = cvc[k];
            const float4 rc4 = reinterpret_cast<const float4 *>(tab_rc + sj[k] * NPHIP)[n4];
            const float4 al4 = reinterpret_cast<const float4 *>(tab_al + sj[k] * NPHIP)[n4];
            const float cva[4] = {cv.x, cv.y, cv.z, cv.w}, rca[4] = {rc4.x, rc4.y, rc4.z, rc4.w},
                        ala[4] = {al4.x, al4.y, al4.z, al4.w};
            // alpha2 = alpha*log2(e): d/dr exp(-alpha d^2) = -2 ln2 alpha2 d ex; two n per packed operation
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const f32x2 al2 = pack2(ala[2 * h], ala[2 * h + 1]), c2 = pack2(cva[2 * h], cva[2 * h + 1]);
                const f32x2 d2 = fmadd2(pack2(rca[2 * h], rca[2 * h + 1]), pack2(-1.f, -1.f), pack2(g[k].w, g[k].w));
                const f32x2 ad2 = fmul2(al2, d2);
                float a0, a1;
                unpack2(fmul2(ad2, d2), a0, a1);
                const f32x2 ex2 = pack2(ex2_ftz(-a0), ex2_ftz(-a1));
                const f32x2 R2 = fmul2(ex2, pack2(fc[k], fc[k]));
                const f32x2 y2 = fmul2(c2, fmul2(fmadd2(ad2, pack2(-1.3862943611198906f * fc[k], -1.3862943611198906f * fc[k]),
                                                        pack2(dfc[k], dfc[k])), ex2));
                unpack2(R2, Rn[k][2 * h], Rn[k][2 * h + 1]);
                unpack2(fmul2(c2, R2), xn[k][2 * h], xn[k][2 * h + 1]);
                unpack2(y2, yn[k][2 * h], yn[k][2 * h + 1]);
                Sn[k][2 * h] = Sn[k][2 * h + 1] = 0.f;
            }
        }
        const float4 *bb4 = reinterpret_cast<const float4 *>(bb + n4 * 4 * NA);
        if constexpr (PAIRS) {
            f32x2 S2[NE][4], x2[NE][4];
#pragma unroll
            for (int k = 0; k < NE; ++k)
#pragma unroll
                for (int u = 0; u < 4; ++u) { S2[k][u] = pack2(0.f, 0.f); x2[k][u] = pack2(xn[k][u], xn[k][u]); }
#pragma unroll
            for (int f4 = 0; f4 < NA; ++f4) { // 4 rows x NA values = NA float4 = 2 NA pairs
                const float4 v = bb4[f4];
                const f32x2 v2[2] = {pack2(v.x, v.y), pack2(v.z, v.w)};
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const int f = f4 * 4 + 2 * h, nl = f / NA, a2 = (f % NA) / 2;
#pragma unroll
                    for (int k = 0; k < NE; ++k) {
                        ffma2(S2[k][nl], v2[h], A2[k][a2]);
                        ffma2(P2[k][a2], v2[h], x2[k][nl]);
                    }
                }
            }
#pragma unroll
            for (int k = 0; k < NE; ++k)
#pragma unroll
                for (int u = 0; u < 4; ++u) { float lo, hi; unpack2(S2[k][u], lo, hi); Sn[k][u] = lo + hi; }
        } else {
#pragma unroll
            for (int f4 = 0; f4 < NA; ++f4) {
                const float4 v = bb4[f4];
                const float va[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int f = f4 * 4 + u, nl = f / NA, a = f % NA;
                    Sn[0][nl] = fmaf(va[u], A[0][a], Sn[0][nl]);
                    P[0][a] = fmaf(va[u], xn[0][nl], P[0][a]);
                }
            }
        }
#pragma unroll
        for (int k = 0; k < NE; ++k) {
#pragma unroll
            for (int u = 0; u < 4; ++u) radial[k] = fmaf(yn[k][u], Sn[k][u], radial[k]);
            if ((want_kappa & BWD_KAPPA) && have[k])
                reinterpret_cast<float4 *>(kappa + (e[k] - e_lo) * (int64_t)NPHIP)[n4] =
                    make_float4(Rn[k][0] * Sn[k][0], Rn[k][1] * Sn[k][1], Rn[k][2] * Sn[k][2], Rn[k][3] * Sn[k][3]);
            cvc[k] = cvn[k];
        }
    }
#pragma unroll
    for (int k = 0; k < NE; ++k) {
        if constexpr (PAIRS) {
#pragma unroll
            for (int a2 = 0; a2 < NP2; ++a2) unpack2(P2[k][a2], P[k][2 * a2], P[k][2 * a2 + 1]);
        }
        float gx, gy, gz;
        monomial_vjp<NA>(A[k], P[k], gx, gy, gz);
        const float rr = __fdividef(radial[k], g[k].w);
        gx = fmaf(rr, g[k].x, gx); gy = fmaf(rr, g[k].y, gy); gz = fmaf(rr, g[k].z, gz);
        if (have[k]) {
            if (want_kappa & BWD_G_ADD) red_add_f32x4(gst + e[k], gx, gy, gz, 0.f);
            else gst[e[k]] = make_float4(gx, gy, gz, 0.f);
            if constexpr (VIR) {
                aV[0] -= g[k].x * gx; aV[1] -= g[k].x * gy; aV[2] -= g[k].x * gz;
                aV[3] -= g[k].y * gx; aV[4] -= g[k].y * gy; aV[5] -= g[k].y * gz;
                aV[6] -= g[k].z * gx; aV[7] -= g[k].z * gy; aV[8] -= g[k].z * gz;
            }
        }
    }
}

// Persistent warps: a warp walks over atoms (stride = warps of the grid); bbar_i and the records of the row's first
// 64 edges of the NEXT atom arrive by cp.async while the current atom is processed (double-buffered in shared
// memory, no registers held), so an atom starts without waiting on DRAM. One-warp blocks (N_a > 10) stage the records of
// the row's first 96 edges with bbar_i, so the later passes of a row do not wait for theirs either.
// two edges per lane where the registers allow three blocks per SM with it (N_a <= 10); at N_a = 20 the pair of edges
// costs a quarter of the resident warps and measured slower (1.09 vs 1.03 ms on config 3)
#ifndef REANN_BWD_MINB
#define REANN_BWD_MINB 16
#endif
#ifndef REANN_BWD_NREC
#define REANN_BWD_NREC 96
#endif
template <int NA>
struct BwdShape {
    static constexpr int NE = (NA % 2 == 0 && NA <= 10) ? 2 : 1;
    static constexpr int WPB = NE == 2 ? EW : 1;        // warps per block: one where a warp takes one atom and leaves (no waiting for block mates)
    static constexpr int MINB = NE == 2 ? 3 : REANN_BWD_MINB;
    static constexpr int NREC = NE == 2 ? 64 : REANN_BWD_NREC;   // staged edge records per row
};

template <int NPHIP, int NA, bool VIR>
__global__ void __launch_bounds__(BwdShape<NA>::WPB * 32, BwdShape<NA>::MINB) k_edge_bwd(int64_t N, const int64_t *__restrict__ rc_ptr,
                                                      const uint32_t *__restrict__ col_rc,
                                                      const float4 *__restrict__ geom,
                                                      const float *__restrict__ c_ext, RadialTab rt, int S,
                                                      const float *__restrict__ bbar, int want_kappa,
                                                      float *__restrict__ kappa, float4 *__restrict__ gst,
                                                      double *__restrict__ vir_part, AtomChunk ch, const int32_t *__restrict__ skip) {
    SKIP_GUARD(skip);
    constexpr int NB = NPHIP * NA, WPB = BwdShape<NA>::WPB;
    __shared__ __align__(16) float bb_s[WPB][2][NB];
    constexpr int NREC = BwdShape<NA>::NREC;            // records of the row's first NREC edges are staged with bbar_i
    __shared__ __align__(16) float4 g_s[WPB][2][NREC];
    __shared__ uint32_t cj_s[WPB][2][NREC];
    __shared__ __align__(16) float tab_s[2][REANN_MAX_S * NPHIP];
    __shared__ float vir_s[VIR ? WPB : 1][9];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int k = threadIdx.x; k < S * NPHIP; k += WPB * 32) { tab_s[0][k] = rt.rcen[k]; tab_s[1][k] = rt.alpha2[k]; }
    __syncthreads();
    float aV[VIR ? 9 : 1];
#pragma unroll
    for (int k = 0; k < (VIR ? 9 : 1); ++k) aV[k] = 0.f;
    const int64_t stride = (int64_t)gridDim.x * WPB;
    int64_t i = ch.a0 + (int64_t)blockIdx.x * WPB + warp;
    // request bbar and the first-pass records of atom `a` (row [b0, b1)) into buffer `buf`
    auto request = [&](int64_t a, int64_t b0, int64_t b1, int buf) {
        const float4 *src = reinterpret_cast<const float4 *>(bbar + a * (int64_t)NB);
        for (int k = lane; k < NB / 4; k += 32) cp_async16(reinterpret_cast<float4 *>(bb_s[warp][buf]) + k, src + k);
#pragma unroll
        for (int k = 0; k < NREC / 32; ++k) {
            const int64_t e = b0 + lane + 32 * k;
            if (e < b1) { cp_async16(&g_s[warp][buf][lane + 32 * k], geom + e); cp_async4(&cj_s[warp][buf][lane + 32 * k], col_rc + e); }
        }
    };
    int64_t beg = 0, end = 0, beg_n = 0, end_n = 0;
    int buf = 0;
    if (i < ch.a1) {
        beg = rc_ptr[i]; end = rc_ptr[i + 1];
        request(i, beg, end, 0);
        if (i + stride < ch.a1) { beg_n = rc_ptr[i + stride]; end_n = rc_ptr[i + stride + 1]; }
    }
    cp_async_commit();
    for (; i < ch.a1; i += stride) {
        const int64_t i_n = i + stride;
        if (i_n < ch.a1) request(i_n, beg_n, end_n, buf ^ 1);
        cp_async_commit();
        int64_t beg_nn = 0, end_nn = 0;
        if (i_n + stride < ch.a1) { beg_nn = rc_ptr[i_n + stride]; end_nn = rc_ptr[i_n + stride + 1]; }
        cp_async_wait<1>();                                  // this atom's group (the one committed an iteration ago)
        __syncwarp();
        int64_t p0 = beg;                                    // first edge of the pass (warp-uniform)
        while (p0 < end) {
            if constexpr (BwdShape<NA>::NE == 2) {       // two-edge shape: the first pass of a row reads the staged records
                const bool first = p0 == beg;
                const float4 *gp = first ? &g_s[warp][buf][lane] : nullptr;
                const uint32_t *cp = first ? &cj_s[warp][buf][lane] : nullptr;
                if (end - p0 > 32) {
                    edge_bwd_pass<NPHIP, NA, VIR, 2>(p0 + lane, end, col_rc, geom, c_ext, tab_s[0], tab_s[1], rt.inv_rc,
                                                     bb_s[warp][buf], want_kappa, kappa, gst, ch.e_lo, aV, gp, cp);
                    p0 += 64;
                    continue;
                }
                edge_bwd_pass<NPHIP, NA, VIR, 1>(p0 + lane, end, col_rc, geom, c_ext, tab_s[0], tab_s[1], rt.inv_rc,
                                                 bb_s[warp][buf], want_kappa, kappa, gst, ch.e_lo, aV, gp, cp);
            } else {                                     // every pass whose edges are all among the staged records reads them there
                const int off = (int)(p0 - beg);
                const bool st = off + 32 <= NREC;
                const float4 *gp = st ? &g_s[warp][buf][off + lane] : nullptr;
                const uint32_t *cp = st ? &cj_s[warp][buf][off + lane] : nullptr;
                edge_bwd_pass<NPHIP, NA, VIR, 1>(p0 + lane, end, col_rc, geom, c_ext, tab_s[0], tab_s[1], rt.inv_rc,
                                                 bb_s[warp][buf], want_kappa, kappa, gst, ch.e_lo, aV, gp, cp);
            }
            p0 += 32;
        }
        __syncwarp();                                        // every lane is done with bb_s[buf] before it is refilled
        buf ^= 1;
        beg = beg_n; end = end_n; beg_n = beg_nn; end_n = end_nn;
    }
    cp_async_wait<0>();
    // fixed-order reductions: lanes (butterfly, FP32), then FP64 accumulation across layers / warps
    if constexpr (VIR) {
#pragma unroll
        for (int d = 16; d >= 1; d >>= 1)
#pragma unroll
            for (int k = 0; k < 9; ++k) aV[k] += __shfl_xor_sync(0xffffffffu, aV[k], d);
        if (lane == 0) {
#pragma unroll
            for (int k = 0; k < 9; ++k) vir_s[warp][k] = aV[k];
        }
        __syncthreads();
        if (threadIdx.x < 9) {
            double s = 0.0;
#pragma unroll
            for (int w = 0; w < WPB; ++w) s += (double)vir_s[w][threadIdx.x];
            atomicAdd(&vir_part[(int64_t)blockIdx.x * 9 + threadIdx.x], s);   // result unused = RED: one add per address and launch, no wait for the old value
        }
    }
}

// ------------------------------------------------------------------------------------------ A11
// Reverse gather (the paper's backward GA -> LA gradient message as a vJp of N_phi numbers per
// edge): cbar_k[n] = sum_{e in row(k)} kappa[rev(e)][n];  F_k += sum_{e in row(k)} (g_e - g_rev(e))
// (Eq. 3).
template <int NPHIP>
__global__ void __launch_bounds__(RW * 32) k_rev_gather(int64_t N, const int64_t *__restrict__ rc_ptr,
                                                        const uint32_t *__restrict__ rev_rc,
                                                        const float *__restrict__ kappa,
                                                        const float4 *__restrict__ gst, int want_cbar,
                                                        float *__restrict__ cbar, double *__restrict__ Fc,
                                                        StashChunk ch, const int32_t *__restrict__ skip) {
    SKIP_GUARD(skip);
    constexpr int PARTS = NPHIP / 4, EPS = 32 / PARTS; // float4 parts per edge, edges per warp step
    __shared__ float4 red_s[RW][32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t k = (int64_t)blockIdx.x * RW + warp;
    if (k >= N) return;
    const int64_t beg = rc_ptr[k], end = rc_ptr[k + 1];
    if (ch.do_forces) {
        double f0 = 0.0, f1 = 0.0, f2 = 0.0;
        // four edges per lane and iteration: the index loads, then the eight stash loads, are in flight together
        constexpr int U = 4;
        for (int64_t eb = beg + lane; eb < end; eb += 32 * U) {
            uint32_t r[U];
            float4 g[U], o[U];
#pragma unroll
            for (int u = 0; u < U; ++u) r[u] = eb + 32 * u < end ? rev_rc[eb + 32 * u] : 0u;
#pragma unroll
            for (int u = 0; u < U; ++u) {
                g[u] = o[u] = make_float4(0.f, 0.f, 0.f, 0.f);
                if (eb + 32 * u < end) { g[u] = gst[r[u]]; o[u] = gst[eb + 32 * u]; }
            }
#pragma unroll
            for (int u = 0; u < U; ++u) {       // same order of additions as one edge per iteration
                f0 += (double)(o[u].x - g[u].x); f1 += (double)(o[u].y - g[u].y); f2 += (double)(o[u].z - g[u].z);
            }
        }
#pragma unroll
        for (int d = 16; d >= 1; d >>= 1) {
            f0 += __shfl_xor_sync(0xffffffffu, f0, d);
            f1 += __shfl_xor_sync(0xffffffffu, f1, d);
            f2 += __shfl_xor_sync(0xffffffffu, f2, d);
        }
        if (lane == 0) { Fc[3 * k] += f0; Fc[3 * k + 1] += f1; Fc[3 * k + 2] += f2; }
    }
    if (!want_cbar) return;
    const int eo = lane / PARTS, part = lane % PARTS;
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    if (eo < EPS)
        for (int64_t e = beg + eo; e < end; e += EPS) {
            const int64_t r = rev_rc[e];
            if (r < ch.e_lo || r >= ch.e_hi) continue;       // stash chunk: only the edges kappa currently holds
            const float4 v = reinterpret_cast<const float4 *>(kappa + (r - ch.e_lo) * NPHIP)[part];
            acc.x += v.x; acc.y += v.y; acc.z += v.z; acc.w += v.w;
        }
    red_s[warp][lane] = (eo < EPS) ? acc : make_float4(0.f, 0.f, 0.f, 0.f);
    __syncwarp();
    if (lane < PARTS) {
        float4 s = make_float4(0.f, 0.f, 0.f, 0.f);
        for (int q = 0; q < EPS; ++q) {
            const float4 v = red_s[warp][q * PARTS + lane];
            s.x += v.x; s.y += v.y; s.z += v.z; s.w += v.w;
        }
        float4 *dst = reinterpret_cast<float4 *>(cbar + k * (int64_t)NPHIP) + lane;
        if (ch.accumulate) { const float4 o = *dst; s.x += o.x; s.y += o.y; s.z += o.z; s.w += o.w; }
        *dst = s;
    }
}

// ------------------------------------------------------------------------------------------ A12
constexpr int OUT_TPB = 256;
// Two-level, fixed-order FP64 reductions. Block b of k_output_a: caller atoms [256 b, 256 (b+1)) (un-permute F, E_i)
// and its share of the virial partials of the edge backward blocks; partial[b][0] = sum E_i, [1..9] = virial.
__global__ void __launch_bounds__(OUT_TPB) k_output_a(int64_t N, const int32_t *__restrict__ inv_perm,
                                                      const double *__restrict__ Fc, const float *__restrict__ Ei,
                                                      double *__restrict__ F_out, double *__restrict__ Ei_caller,
                                                      const double *__restrict__ vir_part, int n_vir, int want_vir,
                                                      double *__restrict__ partial, const uint8_t *__restrict__ halo,
                                                      const int32_t *__restrict__ skip) {
    SKIP_GUARD(skip);
    __shared__ double red[OUT_TPB];
    const int64_t i = (int64_t)blockIdx.x * OUT_TPB + threadIdx.x; // caller index
    double e = 0.0;
    if (i < N) {
        const int64_t k = inv_perm[i];
        e = (halo && halo[i]) ? 0.0 : (double)Ei[k];    // ghost atoms of a decomposed run: E_i belongs to the owning rank
        if (Ei_caller) Ei_caller[i] = e;
        if (F_out) { F_out[3 * i] = Fc[3 * k]; F_out[3 * i + 1] = Fc[3 * k + 1]; F_out[3 * i + 2] = Fc[3 * k + 2]; }
    }
    red[threadIdx.x] = e;
    __syncthreads();
    for (int s = OUT_TPB / 2; s > 0; s >>= 1) {
        if (threadIdx.x < s) red[threadIdx.x] += red[threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x == 0) partial[(int64_t)blockIdx.x * 10] = red[0];
    if (!want_vir) return;
    // virial partials [v0, v1) of this block, nine sums: thread t takes component t % 9 of every (t / 9)-th entry
    const int per = (n_vir + gridDim.x - 1) / gridDim.x;
    const int v0 = min(n_vir, (int)blockIdx.x * per), v1 = min(n_vir, v0 + per);
    const int q = threadIdx.x % 9, lane9 = threadIdx.x / 9;                       // 28 groups of 9 threads (252 used)
    double s = 0.0;
    if (lane9 < 28)
        for (int k = v0 + lane9; k < v1; k += 28) s += vir_part[(int64_t)k * 9 + q];
    __syncthreads();
    red[threadIdx.x] = s;
    __syncthreads();
    if (threadIdx.x < 9) {
        double t = 0.0;
        for (int g = 0; g < 28; ++g) t += red[g * 9 + threadIdx.x];
        partial[(int64_t)blockIdx.x * 10 + 1 + threadIdx.x] = t;
    }
}
__global__ void __launch_bounds__(OUT_TPB) k_output_b(int n_part, const double *__restrict__ partial,
                                                      double *__restrict__ E_out, double *__restrict__ vir_out, const int32_t *__restrict__ skip) {
    SKIP_GUARD(skip);
    __shared__ double red[OUT_TPB];
    for (int q = 0; q < 10; ++q) {
        if (q > 0 && !vir_out) break;
        double s = 0.0;
        for (int k = threadIdx.x; k < n_part; k += OUT_TPB) s += partial[(int64_t)k * 10 + q];
        red[threadIdx.x] = s;
        __syncthreads();
        for (int st = OUT_TPB / 2; st > 0; st >>= 1) {
            if (threadIdx.x < st) red[threadIdx.x] += red[threadIdx.x + st];
            __syncthreads();
        }
        if (threadIdx.x == 0) {
            if (q == 0) { if (E_out) *E_out = red[0]; }
            else vir_out[q - 1] = red[0];
        }
        __syncthreads();
    }
}

__global__ void k_verlet(int64_t N, double *__restrict__ pos, double *__restrict__ vel, const double *__restrict__ F,
                         const double *__restrict__ inv_mass, double dt, double acc_unit, int drift) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const double s = 0.5 * dt * acc_unit * inv_mass[i];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        double v = vel[3 * i + d] + s * F[3 * i + d];
        vel[3 * i + d] = v;
        if (drift) pos[3 * i + d] += dt * v;
    }
}

} // namespace

// ============================================================================================ host
void launch_skin_check(const LaunchCtx &ctx, const double *pos, const double *pos_build, int64_t N, double thr2,
                       int32_t *flag) {
    if (N > 0) LAUNCH(ctx, k_skin_check, div_up(N, 256), 256, 0, pos, pos_build, 3 * N, thr2, flag);
}
void launch_refresh(const LaunchCtx &ctx, XRec *xrec, int64_t n_ext, const int32_t *perm, const int32_t *wshift,
                    const double *pos, const BoxP &box, float *c_ext0, const float *c0, int nphip) {
    if (n_ext > 0) LAUNCH(ctx, k_refresh, div_up(n_ext, 256), 256, 0, xrec, n_ext, perm, wshift, pos, box, c_ext0, c0, nphip);
}
void launch_filter_count(const LaunchCtx &ctx, const XRec *xrec, const int64_t *row_ptr, const int32_t *col,
                         int64_t N, const BoxP &box, double rc2, uint16_t *rank16, int32_t *rc_cnt) {
    if (N > 0) LAUNCH(ctx, k_filter_count, div_up(N, RW), RW * 32, 0, xrec, row_ptr, col, N, box, rc2, rank16, rc_cnt);
}
void launch_filter_fill(const LaunchCtx &ctx, const XRec *xrec, const int64_t *row_ptr, const int32_t *col,
                        const uint32_t *rev, int64_t N, int64_t n_ext, const BoxP &box, const uint16_t *rank16,
                        const int64_t *rc_ptr, uint32_t *rcx, uint32_t *col_rc, float4 *geom, uint32_t *rev_rc) {
    if (N <= 0) return;
    LAUNCH(ctx, k_rc_ext, div_up(n_ext, 256), 256, 0, xrec, rc_ptr, N, n_ext, rcx, ctx.skip);
    LAUNCH(ctx, k_filter_fill, div_up(N, RW), RW * 32, 0, xrec, row_ptr, col, rev, N, box, rank16, rc_ptr, rcx, col_rc, geom, rev_rc, ctx.skip);
}
void launch_ghost_gather(const LaunchCtx &ctx, float *c_ext, const XRec *xrec, int64_t N, int64_t n_ext, int nphip) {
    const int64_t work = (n_ext - N) * (nphip / 4);
    if (work > 0) LAUNCH(ctx, k_ghost_gather, div_up(work, 256), 256, 0, c_ext, xrec, N, n_ext, nphip, ctx.skip);
}

template <int NPHIP, int NA>
static int run_edge_fwd_mma(const LaunchCtx &ctx, int64_t N, const int64_t *rc_ptr, const uint32_t *col_rc,
                            const float4 *geom, const float *c_ext, RadialTab rt, float *b) {
    using C = FwdMma<NA>;
    LAUNCH(ctx, (k_edge_fwd_mma<NPHIP, NA>), div_up(N, FW), FW * 32, C::SMEM, N, rc_ptr, col_rc, geom, c_ext, rt, b, ctx.skip);
    return REANN_OK;
}

template <int NPHIP, int NA, int PN, int PA>
static int run_edge_fwd(const LaunchCtx &ctx, int64_t N, const int64_t *rc_ptr, const uint32_t *col_rc,
                        const float4 *geom, const float *c_ext, RadialTab rt, float *b) {
    using C = FwdCfg<NPHIP, NA, PN, PA>;
    static bool attr_set[64] = {};
    int dev = 0;
    cudaGetDevice(&dev);
    if (dev < 0 || dev >= 64) return REANN_ERR_UNSUPPORTED;
    if (!attr_set[dev]) {   // the attribute is per device
        if (cudaFuncSetAttribute(k_edge_fwd<NPHIP, NA, PN, PA>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM) != cudaSuccess)
            return REANN_ERR_CUDA;
        attr_set[dev] = true;
    }
    LAUNCH(ctx, (k_edge_fwd<NPHIP, NA, PN, PA>), div_up(N, (int64_t)EW * C::APW), EW * 32, C::SMEM, N, rc_ptr, col_rc, geom, c_ext, rt, b, ctx.skip);
    return REANN_OK;
}

#define EDGE_DISPATCH(M)                                                                                 \
    switch (md.nphip * 100 + md.Na) {                                                                    \
        case 401: M(4, 1, 1, 1) case 404: M(4, 4, 1, 4) case 410: M(4, 10, 1, 5) case 420: M(4, 20, 1, 5)      \
        case 801: M(8, 1, 2, 1) case 804: M(8, 4, 2, 4) case 810: M(8, 10, 2, 5) case 820: M(8, 20, 2, 5)      \
        case 1201: M(12, 1, 3, 1) case 1204: M(12, 4, 3, 4) case 1210: M(12, 10, 3, 5) case 1220: M(12, 20, 3, 5) \
        case 1601: M(16, 1, 2, 1) case 1604: M(16, 4, 2, 4) case 1610: M(16, 10, 2, 5) case 1620: M(16, 20, 4, 5) \
        default: return REANN_ERR_UNSUPPORTED;                                                           \
    }

int launch_edge_fwd(const LaunchCtx &ctx, const ModelDims &md, int t, int64_t N, const int64_t *rc_ptr,
                    const uint32_t *col_rc, const float4 *geom, const float *c_ext, const float *rcen,
                    const float *alpha, float *b, bool allow_mma) {
    if (N <= 0) return REANN_OK;
    RadialTab rt{rcen + (size_t)t * md.S * md.nphip, alpha + (size_t)t * md.S * md.nphip, (float)(1.0 / md.rc)};
    if (md.nphip >= 8 && md.Na >= 10 && allow_mma) {
        switch (md.nphip * 100 + md.Na) {
            case 1620: return run_edge_fwd_mma<16, 20>(ctx, N, rc_ptr, col_rc, geom, c_ext, rt, b);
            case 1610: return run_edge_fwd_mma<16, 10>(ctx, N, rc_ptr, col_rc, geom, c_ext, rt, b);
            case 1220: return run_edge_fwd_mma<12, 20>(ctx, N, rc_ptr, col_rc, geom, c_ext, rt, b);
            case 1210: return run_edge_fwd_mma<12, 10>(ctx, N, rc_ptr, col_rc, geom, c_ext, rt, b);
            case 820: return run_edge_fwd_mma<8, 20>(ctx, N, rc_ptr, col_rc, geom, c_ext, rt, b);
            case 810: return run_edge_fwd_mma<8, 10>(ctx, N, rc_ptr, col_rc, geom, c_ext, rt, b);
            default: break;
        }
    }
#define M(NP, NA_, PN_, PA_) return run_edge_fwd<NP, NA_, PN_, PA_>(ctx, N, rc_ptr, col_rc, geom, c_ext, rt, b);
    EDGE_DISPATCH(M)
#undef M
}

// upper bound of the grid of the edge backward kernel (= entries of the virial partial array)
static int sm_count() {
    static int n_sm[64] = {};
    int dev = 0;
    cudaGetDevice(&dev);
    if (dev < 0 || dev >= 64) dev = 0;
    if (!n_sm[dev] && (cudaDeviceGetAttribute(&n_sm[dev], cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n_sm[dev] <= 0))
        n_sm[dev] = 148;
    return n_sm[dev];
}
// upper bound of the grid of the edge backward kernel (= entries of the virial partial array): one-warp blocks, one per
// atom, in the one-edge-per-lane shape; a persistent grid of MINB blocks per SM in the two-edges-per-lane shape
int edge_bwd_blocks(int64_t N, int Na) {
    const int64_t n = std::max<int64_t>(N, 1);
    const bool two = Na % 2 == 0 && Na <= 10;               // BwdShape<NA>::NE == 2
    return (int)(two ? std::min<int64_t>((n + EW - 1) / EW, (int64_t)3 * sm_count()) : n);
}

int launch_edge_bwd(const LaunchCtx &ctx, const ModelDims &md, int t, int64_t N, const int64_t *rc_ptr,
                    const uint32_t *col_rc, const float4 *geom, const float *c_ext, const float *rcen,
                    const float *alpha, const float *bbar, float *kappa, float4 *gst, double *vir_part,
                    int64_t a0, int64_t a1, int64_t e_lo, bool g_add) {
    if (N <= 0 || a1 <= a0) return REANN_OK;
    const AtomChunk ch{a0, a1, e_lo};
    RadialTab rt{rcen + (size_t)t * md.S * md.nphip, alpha + (size_t)t * md.S * md.nphip, (float)(1.0 / md.rc)};
    const int want_kappa = (t >= 1 ? BWD_KAPPA : 0) | (g_add ? BWD_G_ADD : 0);
#define M(NP, NA_, PN_, PA_) {                                                                                    \
    /* two edges per lane: persistent warps, one wave of resident blocks; else one atom per warp (measured faster) */ \
    const unsigned nblk_all = div_up(a1 - a0, BwdShape<NA_>::WPB);                                                \
    const unsigned nblk = BwdShape<NA_>::NE == 2 ? std::min(nblk_all, (unsigned)(BwdShape<NA_>::MINB * sm_count())) : nblk_all; \
    if (vir_part)                                                                                                 \
        LAUNCH(ctx, (k_edge_bwd<NP, NA_, true>), nblk, BwdShape<NA_>::WPB * 32, 0, N, rc_ptr, col_rc, geom, c_ext, rt,            \
               md.S, bbar, want_kappa, kappa, gst, vir_part, ch, ctx.skip);                                       \
    else                                                                                                          \
        LAUNCH(ctx, (k_edge_bwd<NP, NA_, false>), nblk, BwdShape<NA_>::WPB * 32, 0, N, rc_ptr, col_rc, geom, c_ext, rt,           \
               md.S, bbar, want_kappa, kappa, gst, vir_part, ch, ctx.skip);                                       \
    return REANN_OK; }
    EDGE_DISPATCH(M)
#undef M
}

void launch_rev_gather(const LaunchCtx &ctx, int64_t N, const int64_t *rc_ptr, const uint32_t *rev_rc,
                       const float *kappa, const float4 *gst, int nphip, int want_cbar, float *cbar, double *Fc,
                       int64_t e_lo, int64_t e_hi, int do_forces, int accumulate) {
    if (N <= 0) return;
    const StashChunk ch{e_lo, e_hi, do_forces, accumulate};
    switch (nphip) {
        case 4: LAUNCH(ctx, k_rev_gather<4>, div_up(N, RW), RW * 32, 0, N, rc_ptr, rev_rc, kappa, gst, want_cbar, cbar, Fc, ch, ctx.skip); break;
        case 8: LAUNCH(ctx, k_rev_gather<8>, div_up(N, RW), RW * 32, 0, N, rc_ptr, rev_rc, kappa, gst, want_cbar, cbar, Fc, ch, ctx.skip); break;
        case 12: LAUNCH(ctx, k_rev_gather<12>, div_up(N, RW), RW * 32, 0, N, rc_ptr, rev_rc, kappa, gst, want_cbar, cbar, Fc, ch, ctx.skip); break;
        default: LAUNCH(ctx, k_rev_gather<16>, div_up(N, RW), RW * 32, 0, N, rc_ptr, rev_rc, kappa, gst, want_cbar, cbar, Fc, ch, ctx.skip); break;
    }
}

void launch_output(const LaunchCtx &ctx, int64_t N, const int32_t *inv_perm, const double *Fc, const float *Ei,
                   const double *vir_part, int n_vir_blocks, double *E_out, double *F_out, double *vir_out,
                   double *Ei_caller, double *scratch, const uint8_t *halo) {
    const int nb = (int)div_up(N > 0 ? N : 1, OUT_TPB);
    LAUNCH(ctx, k_output_a, nb, OUT_TPB, 0, N, inv_perm, Fc, Ei, F_out, Ei_caller, vir_part, n_vir_blocks, vir_out != nullptr, scratch, halo, ctx.skip);
    LAUNCH(ctx, k_output_b, 1, OUT_TPB, 0, nb, (const double *)scratch, E_out, vir_out, ctx.skip);
}

void launch_verlet(const LaunchCtx &ctx, int64_t N, double *pos, double *vel, const double *F, const double *inv_mass,
                   double dt, double acc_unit, int drift) {
    if (N > 0) LAUNCH(ctx, k_verlet, div_up(N, 256), 256, 0, N, pos, vel, F, inv_mass, dt, acc_unit, drift);
}
