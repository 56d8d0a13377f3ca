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
#include "common.cuh"

namespace {

constexpr int GW = 8;           // warps (= rows) per block

__host__ __device__ constexpr float mu_of(int a) { // l! / (lx! ly! lz!) in the graded monomial order of edge.cu
    return (a == 5 || a == 6 || a == 8) ? 2.f
           : (a == 11 || a == 12 || a == 13 || a == 15 || a == 17 || a == 18) ? 3.f
           : a == 14 ? 6.f : 1.f;
}
__host__ __device__ constexpr int l_of(int a) { return a >= 10 ? 3 : a >= 4 ? 2 : a >= 1 ? 1 : 0; }
__constant__ float c_mu[20] = {1, 1, 1, 1, 1, 2, 2, 1, 2, 1, 1, 3, 3, 3, 6, 3, 1, 3, 3, 1};

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

template <int NPHIP, int NA>
__global__ void __launch_bounds__(GW * 32, 4) k_gram_bwd(int64_t N, const int32_t *__restrict__ sp_list,
                                                      const DenseTile *__restrict__ tiles,
                                                      const float *__restrict__ b, const float *__restrict__ Qbar,
                                                      float *__restrict__ bbar, int nphi, int NPp, int KQ, const int32_t *__restrict__ skip) {
    SKIP_GUARD(skip);
    using C = BwdCfg<NPHIP, NA>;
    constexpr int NB = NPHIP * NA;
    extern __shared__ __align__(16) float sm[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, QS = KQ + 4;
    float *bT = sm + warp * C::PER_WARP, *outs = bT + NA * C::TS, *q0 = sm + GW * C::PER_WARP, *qs = q0 + warp * QS;
    const RowId row = row_of_block(tiles, N, warp);
    if (!tiles && (int64_t)blockIdx.x * GW >= N) return;
    // ---- block: the 8 Qbar rows, full lines ----
    {
        const float4 *Q4 = reinterpret_cast<const float4 *>(Qbar);
        const int nq4 = KQ >> 2;
        if (tiles) {
            for (int idx = threadIdx.x; idx < GW * nq4; idx += GW * 32) {
                const int q4 = idx >> 3, r8 = idx & 7;
                *reinterpret_cast<float4 *>(q0 + r8 * QS + q4 * 4) = __ldg(Q4 + quad_index(tiles, row, r8, q4, KQ));
            }
        } else {
            for (int idx = threadIdx.x; idx < GW * nq4; idx += GW * 32) {
                const int r8 = idx / nq4, q4 = idx - r8 * nq4;
                if ((int64_t)blockIdx.x * GW + r8 < N)
                    *reinterpret_cast<float4 *>(q0 + r8 * QS + q4 * 4) = __ldg(Q4 + quad_index(tiles, row, r8, q4, KQ));
            }
        }
    }
    int64_t atom = 0;
    if (row.p >= 0) {
        atom = sp_list[row.p];
        const float4 *bi = reinterpret_cast<const float4 *>(b + atom * NB);
#pragma unroll
        for (int f = lane; f < NB / 4; f += 32) {
            const float4 v = __ldg(bi + f);
            const float va[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int e = f * 4 + u;
                bT[(e % NA) * C::TS + e / NA] = va[u];
            }
        }
    }
    __syncthreads();
    if (row.p < 0) return;
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
    __syncwarp();
    float4 *bo = reinterpret_cast<float4 *>(bbar + atom * NB);
#pragma unroll
    for (int f = lane; f < NB / 4; f += 32) bo[f] = reinterpret_cast<const float4 *>(outs)[f];
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
    const size_t smem = sizeof(float) * GW * (size_t)(C::PER_WARP + KQ + 4);
    static size_t attr = 48 * 1024;
    if (int rc = set_smem(k_gram_bwd<NPHIP, NA>, smem, attr)) return rc;
    const unsigned grid = tiles ? (unsigned)n_tiles * 16u : div_up(N, GW);
    LAUNCH(ctx, (k_gram_bwd<NPHIP, NA>), grid, GW * 32, smem, N, sp_list, tiles, b, Qbar, bbar, md.nphi, md.NPp, KQ, ctx.skip);
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
