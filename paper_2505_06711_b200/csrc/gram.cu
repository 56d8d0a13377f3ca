// gram.cu -- the two per-atom "gram" steps of rows A6 / A9 of SURVEY.md section 8(a): the density
// of Eq. 1 in its radial-pair form (see dense.cu for the algebra)
//     forward   Q[l, n<=n'] = sum_{|a|=l} mu_a b[n,a] b[n',a]
//     reverse   bbar[n,a]   = mu_a sum_n' G_l(a)[n,n'] b[n',a],   G_l[n,n'] = Qbar[l,min,max] (1 + delta_nn')
// Both are HBM-bound streaming kernels: a warp owns one atom at a time (grid-stride), stages its
// b row (and Qbar row) in shared memory with coalesced float4 loads and writes coalesced rows.
// Q / Qbar rows are in tile order (row p belongs to atom sp_list[p]), row stride nqp,
// column l * NPp + pair(n, n'), pair(n, n') = n nphi - n (n - 1) / 2 + (n' - n).
#include "common.cuh"

namespace {

constexpr int GW = 8;           // warps per block
constexpr int GRID_PER_SM = 6;  // resident blocks per SM the grid is sized for

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

// ---------------------------------------------------------------------------------------- forward
template <int NPHIP, int NA>
__global__ void __launch_bounds__(GW * 32) k_gram_fwd(int64_t N, const int32_t *__restrict__ sp_list,
                                                      const float *__restrict__ b, float *__restrict__ Q, int nphi,
                                                      int npairs, int NPp, int nqp) {
    constexpr int NB = NPHIP * NA, JMAX = (NPHIP * (NPHIP + 1) / 2 + 31) / 32, LMAX = l_of(NA - 1);
    __shared__ __align__(16) float bs_all[GW][NB];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    float *bs = bs_all[warp];
    // this lane's pairs: pair index lane + 32 j -> (n, n') with n <= n'
    int pn[JMAX], pn2[JMAX];
#pragma unroll
    for (int j = 0; j < JMAX; ++j) {
        int pi = lane + 32 * j, lo = 0;
        while (lo < nphi && pi >= nphi - lo) { pi -= nphi - lo; ++lo; }
        pn[j] = lo; pn2[j] = lo + pi;           // lo == nphi: beyond the last pair (padding column)
    }
    for (int64_t p = (int64_t)blockIdx.x * GW + warp; p < N; p += (int64_t)gridDim.x * GW) {
        const float4 *bi = reinterpret_cast<const float4 *>(b + (int64_t)sp_list[p] * NB);
#pragma unroll
        for (int f = lane; f < NB / 4; f += 32) reinterpret_cast<float4 *>(bs)[f] = __ldg(bi + f);
        __syncwarp();
        float *qo = Q + p * nqp;
#pragma unroll
        for (int j = 0; j < JMAX; ++j) {
            const int pi = lane + 32 * j;
            if (pi < NPp) {
                float s[LMAX + 1];
#pragma unroll
                for (int l = 0; l <= LMAX; ++l) s[l] = 0.f;
                if (pi < npairs) {
                    float x[NA], y[NA];
                    load_row<NA>(bs + pn[j] * NA, x);
                    load_row<NA>(bs + pn2[j] * NA, y);
#pragma unroll
                    for (int a = 0; a < NA; ++a) s[l_of(a)] = fmaf(mu_of(a) * x[a], y[a], s[l_of(a)]);
                }
#pragma unroll
                for (int l = 0; l <= LMAX; ++l) qo[l * NPp + pi] = s[l];
            }
        }
        __syncwarp();
    }
}

// ---------------------------------------------------------------------------------------- reverse
template <int NPHIP, int NA>
struct BwdCfg {
    static constexpr int PARTS = NPHIP == 4 ? 8 : NPHIP == 8 ? 4 : 2; // lanes per row n
    static constexpr int CNT = (NA + PARTS - 1) / PARTS;              // monomials per lane
    static constexpr int TS = NPHIP + 4;                              // row stride of the transposed b
};

template <int NPHIP, int NA>
__global__ void __launch_bounds__(GW * 32) k_gram_bwd(int64_t N, const int32_t *__restrict__ sp_list,
                                                      const float *__restrict__ b, const float *__restrict__ Qbar,
                                                      float *__restrict__ bbar, int nphi, int NPp, int nqp) {
    using C = BwdCfg<NPHIP, NA>;
    constexpr int NB = NPHIP * NA;
    extern __shared__ __align__(16) float sm[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int per_warp = NA * C::TS + NB + nqp;
    float *bT = sm + (size_t)warp * per_warp, *outs = bT + NA * C::TS, *qs = outs + NB;
    const int n = lane / C::PARTS, a0 = (lane % C::PARTS) * C::CNT;
    const bool row_ok = n < nphi;
    // triangular offsets of G[n, k] and the (1 + delta) factor; 0 for padded rows / columns
    int idx[NPHIP];
    float fac[NPHIP];
#pragma unroll
    for (int k = 0; k < NPHIP; ++k) {
        const int lo = min(n, k), hi = max(n, k);
        const bool ok = row_ok && k < nphi;
        idx[k] = ok ? lo * nphi - (lo * (lo - 1)) / 2 + (hi - lo) : 0;
        fac[k] = ok ? (k == n ? 2.0f : 1.0f) : 0.0f;
    }
    for (int64_t p = (int64_t)blockIdx.x * GW + warp; p < N; p += (int64_t)gridDim.x * GW) {
        const int64_t atom = sp_list[p];
        const float4 *bi = reinterpret_cast<const float4 *>(b + atom * NB);
        const float4 *qi = reinterpret_cast<const float4 *>(Qbar + p * nqp);
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
        for (int f = lane; f < nqp / 4; f += 32) reinterpret_cast<float4 *>(qs)[f] = __ldg(qi + f);
        __syncwarp();
        if (n < NPHIP) {
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
        __syncwarp();
    }
}

int gram_grid(int64_t N) {
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int64_t want = (N + GW - 1) / GW, cap = (int64_t)sms * GRID_PER_SM;
    return (int)(want < cap ? want : cap);
}

template <int NPHIP, int NA>
int run_gram_fwd(const LaunchCtx &ctx, const ModelDims &md, int64_t N, const int32_t *sp_list, const float *b, float *Q) {
    LAUNCH(ctx, (k_gram_fwd<NPHIP, NA>), gram_grid(N), GW * 32, 0, N, sp_list, b, Q, md.nphi, md.npairs, md.NPp, md.nqp);
    return REANN_OK;
}
template <int NPHIP, int NA>
int run_gram_bwd(const LaunchCtx &ctx, const ModelDims &md, int64_t N, const int32_t *sp_list, const float *b,
                 const float *Qbar, float *bbar) {
    using C = BwdCfg<NPHIP, NA>;
    const size_t smem = sizeof(float) * GW * (size_t)(NA * C::TS + NPHIP * NA + md.nqp);
    static size_t attr = 48 * 1024;
    if (smem > attr) {
        if (cudaFuncSetAttribute(k_gram_bwd<NPHIP, NA>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) {
            cudaGetLastError();
            return REANN_ERR_UNSUPPORTED;
        }
        attr = smem;
    }
    LAUNCH(ctx, (k_gram_bwd<NPHIP, NA>), gram_grid(N), GW * 32, smem, N, sp_list, b, Qbar, bbar, md.nphi, md.NPp, md.nqp);
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

int launch_gram_fwd(const LaunchCtx &ctx, const ModelDims &md, int64_t N, const int32_t *sp_list, const float *b,
                    float *Q) {
    if (N <= 0) return REANN_OK;
    GRAM_DISPATCH(run_gram_fwd, ctx, md, N, sp_list, b, Q)
}

int launch_gram_bwd(const LaunchCtx &ctx, const ModelDims &md, int64_t N, const int32_t *sp_list, const float *b,
                    const float *Qbar, float *bbar) {
    if (N <= 0) return REANN_OK;
    GRAM_DISPATCH(run_gram_bwd, ctx, md, N, sp_list, b, Qbar, bbar)
}
