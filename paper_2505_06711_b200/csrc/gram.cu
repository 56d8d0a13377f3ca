// gram.cu -- the two per-atom "gram" steps of rows A6 / A9 of SURVEY.md section 8(a): the density
// of Eq. 1 in its radial-pair form (see dense.cu for the algebra)
//     forward   Q[l, n<=n'] = sum_{|a|=l} mu_a b[n,a] b[n',a]
//     reverse   bbar[n,a]   = mu_a sum_n' G_l(a)[n,n'] b[n',a],   G_l[n,n'] = Qbar[l,min,max] (1 + delta_nn')
// Both are HBM-bound streaming kernels: a block owns 8 consecutive rows of Q / Qbar, one warp per
// row (= atom); b rows are staged with coalesced float4 loads and Q rows go through shared memory so
// that the block reads / writes them in full 128-byte lines in either of the two layouts:
//   tile-quad (tensor-core path, see dense_tc.cu): [tile][q/4][128 rows][4], KQ = K1 columns;
//   row-major (SIMT path, dense.cu):               [p][KQ = nqp], row p belongs to atom sp_list[p].
// Column q = l * NPp + pair(n, n'), pair(n, n') = n nphi - n (n - 1) / 2 + (n' - n); columns that
// are padding are written as zeros.
#include <algorithm>

#include "common.cuh"
#include "edge_common.cuh"

namespace {

constexpr int GW = 8;           // warps (= rows) per block

__host__ __device__ constexpr float mu_of(int a) { // l! / (lx! ly! lz!) in the graded monomial order of edge.cu
    return (a == 5 || a == 6 || a == 8) ? 2.f
           : (a == 11 || a == 12 || a == 13 || a == 15 || a == 17 || a == 18) ? 3.f
           : a == 14 ? 6.f : 1.f;
}
__host__ __device__ constexpr int l_of(int a) { return a >= 10 ? 3 : a >= 4 ? 2 : a >= 1 ? 1 : 0; }
__constant__ float c_mu[20] = {1, 1, 1, 1, 1, 2, 2, 1, 2, 1, 1, 3, 3, 3, 6, 3, 1, 3, 3, 1};

// hi = x rounded to TF32, lo = (x - hi) rounded to TF32 (nearest; split_bits() leaves lo's low bits to the MMA's truncation)
__device__ __forceinline__ void split_rn(float x, uint32_t &hi, uint32_t &lo) {
    hi = (__float_as_uint(x) + 0x1000u) & 0xFFFFE000u;
    lo = (__float_as_uint(x - __uint_as_float(hi)) + 0x1000u) & 0xFFFFE000u;
}

template <int NA>
__device__ __forceinline__ void load_row(const float *__restrict__ src, float *x) {
    if constexpr (NA % 4 == 0) {
#pragma unroll
        for (int k = 0; k < NA / 4; ++k) {
            const float4 v = reinterpret_cast<const float4 *>(src)[k];
            x[4 * k] = v.x; x[4 * k + 1] = v.y; x[4 * k + 2] = v.z; x[4 * k + 3] = v.w;
        }
    } else if constexpr (NA % 2 == 0) {
#pragma unroll
        for (int k = 0; k < NA / 2; ++k) {
            const float2 v = reinterpret_cast<const float2 *>(src)[k];
            x[2 * k] = v.x; x[2 * k + 1] = v.y;
        }
    } else {
#pragma unroll
        for (int k = 0; k < NA; ++k) x[k] = src[k];
    }
}

// row of this warp: tile-quad mode (tiles != nullptr): block = (tile, group of 8 rows); else p = 8 block + warp
struct RowId {
    int64_t p;      // position in sp_list, -1 if the row is padding
    int tile, r0;   // tile-quad mode: tile index, first row of the block's group
};
__device__ __forceinline__ RowId row_of_block(const DenseTile *__restrict__ tiles, int64_t N, int warp) {
    RowId r;
    if (tiles) {
        r.tile = blockIdx.x >> 4; r.r0 = (blockIdx.x & 15) * 8;
        const DenseTile t = tiles[r.tile];
        r.p = (r.r0 + warp < t.count) ? (int64_t)t.start + r.r0 + warp : -1;
    } else {
        r.tile = 0; r.r0 = 0;
        r.p = (int64_t)blockIdx.x * GW + warp;
        if (r.p >= N) r.p = -1;
    }
    return r;
}
// the same for group g of 8 rows (persistent kernels walk over groups): tile-quad mode g = (tile, group of 8 rows)
__device__ __forceinline__ RowId row_of_group(const DenseTile *__restrict__ tiles, int64_t N, int64_t g, int warp) {
    RowId r;
    if (tiles) {
        r.tile = (int)(g >> 4); r.r0 = (int)(g & 15) * 8;
        const DenseTile t = tiles[r.tile];
        r.p = (r.r0 + warp < t.count) ? (int64_t)t.start + r.r0 + warp : -1;
    } else {
        r.tile = 0; r.r0 = 0;
        r.p = g * GW + warp;
        if (r.p >= N) r.p = -1;
    }
    return r;
}
__device__ __forceinline__ int64_t quad_index_g(const DenseTile *tiles, const RowId &r, int64_t g, int r8, int q4, int KQ) {
    if (tiles) return ((int64_t)r.tile * (KQ >> 2) + q4) * DENSE_TC_TM + r.r0 + r8;
    return (g * GW + r8) * (KQ >> 2) + q4;
}
// float4 index in global memory of (row r8 of this block, column quad q4)
__device__ __forceinline__ int64_t quad_index(const DenseTile *tiles, const RowId &r, int r8, int q4, int KQ) {
    if (tiles) return ((int64_t)r.tile * (KQ >> 2) + q4) * DENSE_TC_TM + r.r0 + r8;
    return ((int64_t)blockIdx.x * GW + r8) * (KQ >> 2) + q4;
}

// ---------------------------------------------------------------------------------------- forward
template <int NPHIP, int NA>
__global__ void __launch_bounds__(GW * 32) k_gram_fwd(int64_t N, const int32_t *__restrict__ sp_list,
                                                      const DenseTile *__restrict__ tiles,
                                                      const float *__restrict__ b, float *__restrict__ Q, int nphi,
                                                      int npairs, int NPp, int KQ, const int32_t *__restrict__ skip) {
    SKIP_GUARD(skip);
    constexpr int NB = NPHIP * NA, LMAX = l_of(NA - 1);
    extern __shared__ __align__(16) float sm[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, QS = KQ + 4;
    float *bs = sm + warp * NB, *qs = sm + GW * NB + warp * QS;
    const RowId row = row_of_block(tiles, N, warp);
    for (int f = lane; f < KQ / 4; f += 32) reinterpret_cast<float4 *>(qs)[f] = make_float4(0.f, 0.f, 0.f, 0.f);
    if (row.p >= 0) {
        const float4 *bi = reinterpret_cast<const float4 *>(b + (int64_t)sp_list[row.p] * NB);
#pragma unroll
        for (int f = lane; f < NB / 4; f += 32) reinterpret_cast<float4 *>(bs)[f] = __ldg(bi + f);
        __syncwarp();
        if constexpr (NA == 20) {
            // Q_l = B_l diag(mu) B_l^T per l on the tensor cores: M = N = rows n (16), K = the monomials of degree l in steps
            // of 8 (l = 0: 1 of 8 used, l = 1: 3, l = 2: 6, l = 3: 8 + 2). mma.sync m16n8k8 TF32, operands split hi + lo; the
            // chains are at most two steps long. The B fragments (K = a, N = n') are the A fragment's own registers times
            // mu_a: column tile j = 0 is rows n' = g (a0, a2), j = 1 rows n' = g + 8 (a1, a3). Shared-memory traffic: four
            // LDS.32 per K step instead of 80 LDS.128 per atom in the FP32 ALU form this replaces.
            const int g8 = lane >> 2, t4 = lane & 3;
            constexpr int NKS = NA == 20 ? 5 : NA == 10 ? 3 : NA == 4 ? 2 : 1;
            constexpr int KS_A0[5] = {0, 1, 4, 10, 18}, KS_CNT[5] = {1, 3, 6, 8, 2}, KS_L[5] = {0, 1, 2, 3, 3};
            float acc[LMAX + 1][2][4];
#pragma unroll
            for (int l = 0; l <= LMAX; ++l)
#pragma unroll
                for (int j = 0; j < 2; ++j) acc[l][j][0] = acc[l][j][1] = acc[l][j][2] = acc[l][j][3] = 0.f;
#pragma unroll
            for (int ks = 0; ks < NKS; ++ks) {
                const int a0 = KS_A0[ks] + t4, a1 = a0 + 4;
                const bool v0 = t4 < KS_CNT[ks], v1 = t4 + 4 < KS_CNT[ks];
                const bool r0 = g8 < NPHIP, r1 = g8 + 8 < NPHIP;
                const float x00 = (v0 && r0) ? bs[g8 * NA + a0] : 0.f, x10 = (v0 && r1) ? bs[(g8 + 8) * NA + a0] : 0.f;
                const float x01 = (v1 && r0) ? bs[g8 * NA + a1] : 0.f, x11 = (v1 && r1) ? bs[(g8 + 8) * NA + a1] : 0.f;
                const float m0 = v0 ? c_mu[a0] : 0.f, m1 = v1 ? c_mu[a1] : 0.f;
                uint32_t ah[4], al[4], bh[2][2], bl[2][2];
                split_rn(x00, ah[0], al[0]); split_rn(x10, ah[1], al[1]);
                split_rn(x01, ah[2], al[2]); split_rn(x11, ah[3], al[3]);
                split_rn(m0 * x00, bh[0][0], bl[0][0]); split_rn(m1 * x01, bh[0][1], bl[0][1]);
                split_rn(m0 * x10, bh[1][0], bl[1][0]); split_rn(m1 * x11, bh[1][1], bl[1][1]);
#pragma unroll
                for (int j = 0; j < 2; ++j) {
                    if (j == 1 && NPHIP <= 8) continue;
                    edge::mma_tf32(acc[KS_L[ks]][j], al, bl[j][0], bl[j][1]);      // Q is quadratic in b and feeds E_i: all four
                    edge::mma_tf32(acc[KS_L[ks]][j], al, bh[j][0], bh[j][1]);      // partial products, smallest first
                    edge::mma_tf32(acc[KS_L[ks]][j], ah, bl[j][0], bl[j][1]);
                    edge::mma_tf32(acc[KS_L[ks]][j], ah, bh[j][0], bh[j][1]);
                }
            }
            // C fragment: rows n = g, g + 8; columns n' = 8 j + 2 t, + 1; kept where n <= n' < nphi
#pragma unroll
            for (int j = 0; j < 2; ++j)
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    const int n = g8 + 8 * (c >> 1), m = 8 * j + 2 * t4 + (c & 1);
                    if (n <= m && m < nphi) {
                        const int pi = n * nphi - (n * (n - 1)) / 2 + (m - n);
#pragma unroll
                        for (int l = 0; l <= LMAX; ++l) qs[l * NPp + pi] = acc[l][j][c];
                    }
                }
        } else {
            // 2 x 2 blocks of row pairs: block (I <= J) = rows {2I, 2I+1} x {2J, 2J+1}; four rows loaded for (up to)
            // four products -- half the shared-memory operand traffic of one pair per lane
            constexpr int NBK = NPHIP / 2, NBLOCKS = NBK * (NBK + 1) / 2;
#pragma unroll
            for (int j = 0; j < (NBLOCKS + 31) / 32; ++j) {
                const int bi = lane + 32 * j;
                if (bi < NBLOCKS) {
                    int I = 0, rem = bi;
                    while (rem >= NBK - I) { rem -= NBK - I; ++I; }
                    const int J = I + rem, n0 = 2 * I, m0 = 2 * J;
                    float s[4][LMAX + 1];                       // (n0,m0) (n0,m1) (n1,m0) (n1,m1)
#pragma unroll
                    for (int k = 0; k < 4; ++k)
#pragma unroll
                        for (int l = 0; l <= LMAX; ++l) s[k][l] = 0.f;
                    float x0[NA], x1[NA], y0[NA], y1[NA];
                    load_row<NA>(bs + n0 * NA, x0); load_row<NA>(bs + (n0 + 1) * NA, x1);
                    load_row<NA>(bs + m0 * NA, y0); load_row<NA>(bs + (m0 + 1) * NA, y1);
#pragma unroll
                    for (int a = 0; a < NA; ++a) {
                        const float u0 = mu_of(a) * x0[a], u1 = mu_of(a) * x1[a];
                        s[0][l_of(a)] = fmaf(u0, y0[a], s[0][l_of(a)]); s[1][l_of(a)] = fmaf(u0, y1[a], s[1][l_of(a)]);
                        s[2][l_of(a)] = fmaf(u1, y0[a], s[2][l_of(a)]); s[3][l_of(a)] = fmaf(u1, y1[a], s[3][l_of(a)]);
                    }
#pragma unroll
                    for (int k = 0; k < 4; ++k) {
                        const int n = n0 + (k >> 1), m = m0 + (k & 1);
                        if (n <= m && m < nphi) {                // diagonal block: (n1, m0) is the mirror of (n0, m1)
                            const int pi = n * nphi - (n * (n - 1)) / 2 + (m - n);
#pragma unroll
                            for (int l = 0; l <= LMAX; ++l) qs[l * NPp + pi] = s[k][l];
                        }
                    }
                }
            }
        }
    }
    __syncthreads();
    if (!tiles && (int64_t)blockIdx.x * GW >= N) return;
    const float *q0 = sm + GW * NB;
    float4 *Q4 = reinterpret_cast<float4 *>(Q);
    const int nq4 = KQ >> 2;
    if (tiles) {
        for (int idx = threadIdx.x; idx < GW * nq4; idx += GW * 32) {
            const int q4 = idx >> 3, r8 = idx & 7;
            Q4[quad_index(tiles, row, r8, q4, KQ)] = *reinterpret_cast<const float4 *>(q0 + r8 * QS + q4 * 4);
        }
    } else {
        for (int idx = threadIdx.x; idx < GW * nq4; idx += GW * 32) {
            const int r8 = idx / nq4, q4 = idx - r8 * nq4;
            if ((int64_t)blockIdx.x * GW + r8 < N)
                Q4[quad_index(tiles, row, r8, q4, KQ)] = *reinterpret_cast<const float4 *>(q0 + r8 * QS + q4 * 4);
        }
    }
}

// ---------------------------------------------------------------------------------------- reverse
template <int NPHIP, int NA>
struct BwdCfg {
    static constexpr int PARTS = NPHIP == 4 ? 8 : NPHIP == 8 ? 4 : 2; // lanes per row n
    static constexpr int CNT = (NA + PARTS - 1) / PARTS;              // monomials per lane
    static constexpr int TS = NPHIP + 4;                              // row stride of the transposed b
    static constexpr int PER_WARP = NA * TS + NPHIP * NA;             // floats: bT | outs
};

// Persistent: a block walks over groups of 8 rows (one warp = one row); the Qbar rows and the b rows of the NEXT group
// arrive by cp.async while the current group is computed (double-buffered in shared memory), so the kernel streams at
// the pace of HBM instead of waiting out a DRAM round trip per group.
template <int NPHIP, int NA>
__global__ void __launch_bounds__(GW * 32, 3) k_gram_bwd(int64_t N, const int32_t *__restrict__ sp_list,
                                                      const DenseTile *__restrict__ tiles,
                                                      const float *__restrict__ b, const float *__restrict__ Qbar,
                                                      float *__restrict__ bbar, int nphi, int NPp, int KQ, int64_t n_groups,
                                                      const int32_t *__restrict__ skip) {
    SKIP_GUARD(skip);
    using C = BwdCfg<NPHIP, NA>;
    constexpr int NB = NPHIP * NA, WORK = NA == 20 ? NB : C::PER_WARP;
    extern __shared__ __align__(16) float sm[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, QS = KQ + 4, RS = QS + NB;   // row of a buffer: Qbar row | b row
    float *work = sm + (size_t)2 * GW * RS + warp * WORK;
    const float4 *Q4 = reinterpret_cast<const float4 *>(Qbar);
    const int nq4 = KQ >> 2;
    auto issue = [&](int64_t g, int buf) {
        float *in = sm + (size_t)buf * GW * RS;
        const RowId row = row_of_group(tiles, N, g, warp);
        if (tiles) {
            for (int idx = threadIdx.x; idx < GW * nq4; idx += GW * 32) {
                const int q4 = idx >> 3, r8 = idx & 7;
                edge::cp_async16(in + r8 * RS + q4 * 4, Q4 + quad_index_g(tiles, row, g, r8, q4, KQ));
            }
        } else {
            for (int idx = threadIdx.x; idx < GW * nq4; idx += GW * 32) {
                const int r8 = idx / nq4, q4 = idx - r8 * nq4;
                if (g * GW + r8 < N) edge::cp_async16(in + r8 * RS + q4 * 4, Q4 + quad_index_g(tiles, row, g, r8, q4, KQ));
            }
        }
        if (row.p >= 0) {
            const float4 *bi = reinterpret_cast<const float4 *>(b + (int64_t)sp_list[row.p] * NB);
            for (int f = lane; f < NB / 4; f += 32) edge::cp_async16(in + warp * RS + QS + f * 4, bi + f);
        }
    };
    // lane constants of the tensor-core path: triangular offsets and (1 + delta) factors of this lane's A-fragment elements
    const int g8 = lane >> 2, t4 = lane & 3;
    int gi[2][4];
    float gf[2][4];
#pragma unroll
    for (int k = 0; k < 2; ++k)
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            const int n = g8 + 8 * (c & 1), m = 8 * k + t4 + 4 * (c >> 1);       // a0 (g, t), a1 (g+8, t), a2 (g, t+4), a3 (g+8, t+4)
            const int lo = min(n, m), hi = max(n, m);
            const bool ok = n < nphi && m < nphi;
            gi[k][c] = ok ? lo * nphi - (lo * (lo - 1)) / 2 + (hi - lo) : 0;
            gf[k][c] = ok ? (n == m ? 2.0f : 1.0f) : 0.0f;
        }
    int64_t g = blockIdx.x;
    int buf = 0;
    if (g < n_groups) issue(g, 0);
    edge::cp_async_commit();
    for (; g < n_groups; g += gridDim.x, buf ^= 1) {
        if (g + gridDim.x < n_groups) issue(g + gridDim.x, buf ^ 1);
        edge::cp_async_commit();
        edge::cp_async_wait<1>();
        __syncthreads();                       // the Qbar rows were brought in by all threads of the block
        const RowId row = row_of_group(tiles, N, g, warp);
        if (row.p >= 0) {
            const int64_t atom = sp_list[row.p];
            const float *qs = sm + (size_t)buf * GW * RS + warp * RS, *bs = qs + QS;
            if constexpr (NA == 20) {
                // bbar_l = mu . (G_l B_l) per l on the tensor cores: M = n (16), K = n' (two steps of 8), N = the monomials of
                // degree l in tiles of 8 (l = 0: 1 of 8 columns used, l = 1: 3, l = 2: 6, l = 3: 8 + 2). A fragments = G_l
                // gathered from the triangular Qbar row, B fragments = b (row-major, as it arrived), 3xTF32.
                float *outs = work;
                constexpr int NTL = 5;
                constexpr int NT_A0[NTL] = {0, 1, 4, 10, 18}, NT_CNT[NTL] = {1, 3, 6, 8, 2}, NT_L[NTL] = {0, 1, 2, 3, 3};
                uint32_t ah[2][4], al[2][4];
#pragma unroll
                for (int nt = 0; nt < NTL; ++nt) {
                    if (nt == 0 || NT_L[nt] != NT_L[nt - 1]) {
                        const float *ql = qs + NT_L[nt] * NPp;
#pragma unroll
                        for (int k = 0; k < 2; ++k)
#pragma unroll
                            for (int c = 0; c < 4; ++c) edge::split_bits(ql[gi[k][c]] * gf[k][c], ah[k][c], al[k][c]);
                    }
                    float acc[4] = {0.f, 0.f, 0.f, 0.f};
                    const int a = NT_A0[nt] + g8;
                    const bool va = g8 < NT_CNT[nt];
                    uint32_t bh[2][2], bl[2][2];
#pragma unroll
                    for (int k = 0; k < 2; ++k) {
                        const int r0 = 8 * k + t4, r1 = r0 + 4;
                        edge::split_bits((va && r0 < NPHIP) ? bs[r0 * NA + a] : 0.f, bh[k][0], bl[k][0]);
                        edge::split_bits((va && r1 < NPHIP) ? bs[r1 * NA + a] : 0.f, bh[k][1], bl[k][1]);
                    }
#pragma unroll
                    for (int k = 0; k < 2; ++k) {
                        if (k == 1 && NPHIP <= 8) continue;
                        edge::mma_tf32(acc, al[k], bh[k][0], bh[k][1]);
                        edge::mma_tf32(acc, ah[k], bl[k][0], bl[k][1]);
                    }
#pragma unroll
                    for (int k = 0; k < 2; ++k) {
                        if (k == 1 && NPHIP <= 8) continue;
                        edge::mma_tf32(acc, ah[k], bh[k][0], bh[k][1]);
                    }
                    // C fragment: rows n = g, g + 8; columns a = a0 + 2t, + 1
#pragma unroll
                    for (int c = 0; c < 4; ++c) {
                        const int n = g8 + 8 * (c >> 1), col = 2 * t4 + (c & 1);
                        if (col < NT_CNT[nt] && n < NPHIP) outs[n * NA + NT_A0[nt] + col] = c_mu[NT_A0[nt] + col] * acc[c];
                    }
                }
            } else {
                float *bT = work, *outs = work + NA * C::TS;
                for (int e = lane; e < NB; e += 32) bT[(e % NA) * C::TS + e / NA] = bs[e];
                __syncwarp();
                const int n = lane / C::PARTS, a0 = (lane % C::PARTS) * C::CNT;
                if (n < NPHIP) {
                    // triangular offsets of G[n, k] and the (1 + delta) factor; 0 for padded rows / columns
                    int idx[NPHIP];
                    float fac[NPHIP];
#pragma unroll
                    for (int k = 0; k < NPHIP; ++k) {
                        const int lo = min(n, k), hi = max(n, k);
                        const bool ok = n < nphi && k < nphi;
                        idx[k] = ok ? lo * nphi - (lo * (lo - 1)) / 2 + (hi - lo) : 0;
                        fac[k] = ok ? (k == n ? 2.0f : 1.0f) : 0.0f;
                    }
                    float G[NPHIP];
                    int lcur = -1;
#pragma unroll
                    for (int ai = 0; ai < C::CNT; ++ai) {
                        const int a = a0 + ai;
                        if (a < NA) {
                            const int l = l_of(a);
                            if (l != lcur) {
                                const float *ql = qs + l * NPp;
#pragma unroll
                                for (int k = 0; k < NPHIP; ++k) G[k] = ql[idx[k]] * fac[k];
                                lcur = l;
                            }
                            float s = 0.f;
#pragma unroll
                            for (int k4 = 0; k4 < NPHIP / 4; ++k4) {
                                const float4 v = *reinterpret_cast<const float4 *>(bT + a * C::TS + 4 * k4);
                                s = fmaf(G[4 * k4], v.x, s); s = fmaf(G[4 * k4 + 1], v.y, s);
                                s = fmaf(G[4 * k4 + 2], v.z, s); s = fmaf(G[4 * k4 + 3], v.w, s);
                            }
                            outs[n * NA + a] = c_mu[a] * s;
                        }
                    }
                }
            }
            __syncwarp();
            float4 *bo = reinterpret_cast<float4 *>(bbar + atom * NB);
            const float *outs = NA == 20 ? work : work + NA * C::TS;
#pragma unroll
            for (int f = lane; f < NB / 4; f += 32) bo[f] = reinterpret_cast<const float4 *>(outs)[f];
        }
        __syncthreads();                       // every warp is done with this buffer before the next prefetch refills it
    }
    edge::cp_async_wait<0>();
}

template <class K>
int set_smem(K kernel, size_t smem, size_t &attr) {
    if (smem > attr) {
        if (cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) {
            cudaGetLastError();
            return REANN_ERR_UNSUPPORTED;
        }
        attr = smem;
    }
    return REANN_OK;
}

static int gram_grid(int64_t n_groups, size_t smem) {
    int dev = 0, n_sm = 148;
    cudaGetDevice(&dev);
    if (cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n_sm <= 0) n_sm = 148;
    const int per_sm = (int)std::max<size_t>(1, std::min<size_t>(3, (size_t)(220 * 1024) / smem));
    return (int)std::min<int64_t>(n_groups, (int64_t)per_sm * n_sm);
}

template <int NPHIP, int NA>
int run_gram_fwd(const LaunchCtx &ctx, const ModelDims &md, int64_t N, const int32_t *sp_list, const DenseTile *tiles,
                 int n_tiles, const float *b, float *Q) {
    const int KQ = tiles ? md.K1 : md.nqp;
    const size_t smem = sizeof(float) * GW * (size_t)(NPHIP * NA + KQ + 4);
    static size_t attr = 48 * 1024;
    if (int rc = set_smem(k_gram_fwd<NPHIP, NA>, smem, attr)) return rc;
    const unsigned grid = tiles ? (unsigned)n_tiles * 16u : div_up(N, GW);
    LAUNCH(ctx, (k_gram_fwd<NPHIP, NA>), grid, GW * 32, smem, N, sp_list, tiles, b, Q, md.nphi, md.npairs, md.NPp, KQ, ctx.skip);
    return REANN_OK;
}
template <int NPHIP, int NA>
int run_gram_bwd(const LaunchCtx &ctx, const ModelDims &md, int64_t N, const int32_t *sp_list, const DenseTile *tiles,
                 int n_tiles, const float *b, const float *Qbar, float *bbar) {
    using C = BwdCfg<NPHIP, NA>;
    const int KQ = tiles ? md.K1 : md.nqp;
    constexpr int NB = NPHIP * NA, WORK = NA == 20 ? NB : C::PER_WARP;
    const size_t smem = sizeof(float) * GW * (size_t)(2 * (KQ + 4 + NB) + WORK);
    static size_t attr = 48 * 1024;
    if (int rc = set_smem(k_gram_bwd<NPHIP, NA>, smem, attr)) return rc;
    const int64_t n_groups = tiles ? (int64_t)n_tiles * 16 : (N + GW - 1) / GW;
    LAUNCH(ctx, (k_gram_bwd<NPHIP, NA>), (unsigned)gram_grid(n_groups, smem), GW * 32, smem, N, sp_list, tiles, b, Qbar, bbar, md.nphi, md.NPp,
           KQ, n_groups, ctx.skip);
    return REANN_OK;
}

#define GRAM_DISPATCH(FN, ...)                                                                                     \
    switch (md.nphip * 100 + md.Na) {                                                                              \
        case 401: return FN<4, 1>(__VA_ARGS__); case 404: return FN<4, 4>(__VA_ARGS__);                            \
        case 410: return FN<4, 10>(__VA_ARGS__); case 420: return FN<4, 20>(__VA_ARGS__);                          \
        case 801: return FN<8, 1>(__VA_ARGS__); case 804: return FN<8, 4>(__VA_ARGS__);                            \
        case 810: return FN<8, 10>(__VA_ARGS__); case 820: return FN<8, 20>(__VA_ARGS__);                          \
        case 1201: return FN<12, 1>(__VA_ARGS__); case 1204: return FN<12, 4>(__VA_ARGS__);                        \
        case 1210: return FN<12, 10>(__VA_ARGS__); case 1220: return FN<12, 20>(__VA_ARGS__);                      \
        case 1601: return FN<16, 1>(__VA_ARGS__); case 1604: return FN<16, 4>(__VA_ARGS__);                        \
        case 1610: return FN<16, 10>(__VA_ARGS__); case 1620: return FN<16, 20>(__VA_ARGS__);                      \
        default: return REANN_ERR_UNSUPPORTED;                                                                     \
    }

} // namespace

int launch_gram_fwd(const LaunchCtx &ctx, const ModelDims &md, int64_t N, const int32_t *sp_list, const DenseTile *tiles,
                    int n_tiles, const float *b, float *Q) {
    if (N <= 0) return REANN_OK;
    GRAM_DISPATCH(run_gram_fwd, ctx, md, N, sp_list, tiles, n_tiles, b, Q)
}

int launch_gram_bwd(const LaunchCtx &ctx, const ModelDims &md, int64_t N, const int32_t *sp_list, const DenseTile *tiles,
                    int n_tiles, const float *b, const float *Qbar, float *bbar) {
    if (N <= 0) return REANN_OK;
    GRAM_DISPATCH(run_gram_bwd, ctx, md, N, sp_list, tiles, n_tiles, b, Qbar, bbar)
}
