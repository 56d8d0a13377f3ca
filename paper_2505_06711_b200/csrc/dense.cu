// dense.cu -- rows A6+A7 (contraction, density, per-species MLP) and A9 (their reverse pass) of
// FP32 SIMT GEMM-chain tile kernels (64 atoms of one species per CTA). The
// gram kernels (b <-> radial-pair products Q) live in gram.cu, the tcgen05 chain in dense_tc.cu.
//
// Eq. 1 with the learned contraction (reading A-1):
//     d[a,m] = sum_n Wc[l(a)][n][m] b[n,a],   rho[m] = sum_a mu_a d[a,m]^2
// is evaluated in the algebraically identical "radial-pair" form
//     rho[m] = sum_q V[q][m] Q[q],   q = (l, n <= n'),
//     Q[q]   = sum_{|a|=l} mu_a b[n,a] b[n',a],       V[q][m] = (2 - delta_nn') Wc[l][n][m] Wc[l][n'][m]
// and, because the first MLP layer (Eq. 2) is linear in rho, V is folded into it once
// at reann_create (FP64 on the host):   z1 = U^T Q + b1,   U = V W1   ([n_q][H1]).
// n_q = (L+1) N_phi (N_phi+1)/2 is exactly the paper's feature count, so the GEMM
// has the same shape as W1 while the N_a x N_phi x n_orb contraction and the 2x as expensive
// reverse contraction disappear. Reverse pass (Eq. 5 / Appendix B steps 1-2):
//     Qbar = U z1bar;   bbar[n,a] = mu_a sum_n' G_l(a)[n,n'] b[n',a],  G_l[n,n'] = Qbar[l,min,max] (1 + delta_nn')
// The oracle evaluates the literal form; parity between the two is the test of this refactoring.
#include "common.cuh"

namespace {

constexpr int TM = 64;       // atoms per tile
constexpr int DT = 256;      // threads per CTA: 16 (row groups of 4 atoms) x 16 (column groups)
constexpr int KC = 32;       // K-chunk of the B operand staged in shared memory
static_assert(TM == DENSE_TM, "tile size");


__device__ __forceinline__ float silu_f(float z) { return z / (1.0f + __expf(-z)); }
__device__ __forceinline__ float dsilu_f(float z) {
    const float s = 1.0f / (1.0f + __expf(-z));
    return s * (1.0f + z * (1.0f - s));
}

template <int NC>
__device__ __forceinline__ int col_of(int tn, int c) {
    if constexpr (NC == 8) return (c >> 2) * 64 + tn * 4 + (c & 3);
    else return tn * NC + c;
}

// acc[4][NC] += As[k0..k0+kc)[tm*4..] (x) Bs[kk][cols]      As: [K][TM], Bs: [KC][16*NC]
template <int NC>
__device__ __forceinline__ void mm_chunk(float (&acc)[4][NC], const float *__restrict__ As, const float *__restrict__ Bs,
                                         int kc, int tm, int tn) {
    constexpr int LDB = 16 * NC;
#pragma unroll 4
    for (int kk = 0; kk < kc; ++kk) {
        const float4 a4 = *reinterpret_cast<const float4 *>(As + kk * TM + tm * 4);
        const float a[4] = {a4.x, a4.y, a4.z, a4.w};
        float bv[NC];
        if constexpr (NC == 8) {
            const float4 b0 = *reinterpret_cast<const float4 *>(Bs + kk * LDB + tn * 4);
            const float4 b1 = *reinterpret_cast<const float4 *>(Bs + kk * LDB + 64 + tn * 4);
            bv[0] = b0.x; bv[1] = b0.y; bv[2] = b0.z; bv[3] = b0.w; bv[4] = b1.x; bv[5] = b1.y; bv[6] = b1.z; bv[7] = b1.w;
        } else if constexpr (NC == 4) {
            const float4 b0 = *reinterpret_cast<const float4 *>(Bs + kk * LDB + tn * 4);
            bv[0] = b0.x; bv[1] = b0.y; bv[2] = b0.z; bv[3] = b0.w;
        } else if constexpr (NC == 2) {
            const float2 b0 = *reinterpret_cast<const float2 *>(Bs + kk * LDB + tn * 2);
            bv[0] = b0.x; bv[1] = b0.y;
        } else {
            bv[0] = Bs[kk * LDB + tn];
        }
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
            for (int c = 0; c < NC; ++c) acc[r][c] = fmaf(a[r], bv[c], acc[r][c]);
    }
}

// stage rows [k0, k0+kc) x columns [col0, col0+16*NC) of a row-major global matrix into Bs
template <int NC>
__device__ __forceinline__ void load_b_chunk(float *__restrict__ Bs, const float *__restrict__ Bg, int ldg, int k0,
                                             int kc, int col0) {
    constexpr int LDB = 16 * NC;
    for (int idx = threadIdx.x; idx < kc * LDB; idx += DT) {
        const int kk = idx / LDB, c = idx % LDB;
        Bs[idx] = __ldg(Bg + (size_t)(k0 + kk) * ldg + col0 + c);
    }
}

// full GEMM over K with the A operand resident in shared memory ([K][TM])
template <int NC>
__device__ __forceinline__ void gemm_smemA(float (&acc)[4][NC], const float *__restrict__ As, int K,
                                           const float *__restrict__ Bg, int ldg, int col0, float *__restrict__ Bs,
                                           int tm, int tn) {
#pragma unroll
    for (int r = 0; r < 4; ++r)
#pragma unroll
        for (int c = 0; c < NC; ++c) acc[r][c] = 0.f;
    for (int k0 = 0; k0 < K; k0 += KC) {
        const int kc = min(KC, K - k0);
        __syncthreads();
        load_b_chunk<NC>(Bs, Bg, ldg, k0, kc, col0);
        __syncthreads();
        mm_chunk<NC>(acc, As + (size_t)k0 * TM, Bs, kc, tm, tn);
    }
}


// ============================================================================ GEMM-chain tile kernels (SIMT)
struct FwdArgs {
    const DenseW *w;        // [S]
    const DenseTile *tiles;
    const int32_t *sp_list;
    const float *Q;         // [N][nqp], tile order
    float *z_stash;         // [N][zs], tile order
    float *out;             // rows of stride out_stride, atom order
    int out_stride, nqp, H1p, H2p, nout, zs;
    const int32_t *skip;    // see LaunchCtx
};

// A chunk from row-major global rows -> K-major shared [KC][TM]
__device__ __forceinline__ void load_a_chunk(float *__restrict__ As, const float *__restrict__ Ag, int ldg, int k0,
                                             int kc, int rows_valid) {
    // thread -> (row m = tid % TM, k-quad = tid / TM + 4 j): lanes run over m => conflict-free stores
    const int m = threadIdx.x & (TM - 1);
    for (int kq = threadIdx.x / TM; kq * 4 < kc; kq += DT / TM) {
        float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
        if (m < rows_valid) v = __ldg(reinterpret_cast<const float4 *>(Ag + (size_t)m * ldg + k0) + kq);
        As[(kq * 4 + 0) * TM + m] = v.x; As[(kq * 4 + 1) * TM + m] = v.y;
        As[(kq * 4 + 2) * TM + m] = v.z; As[(kq * 4 + 3) * TM + m] = v.w;
    }
}

template <int NC1, int NC2>
__global__ void __launch_bounds__(DT) k_dense_fwd(FwdArgs A) {
    SKIP_GUARD(A.skip);
    extern __shared__ __align__(16) float sm[];
    const DenseTile tile = A.tiles[blockIdx.x];
    const DenseW W = A.w[tile.species];
    const int tid = threadIdx.x, tm = tid >> 4, tn = tid & 15;
    // carve-up (floats): Ac [KC][TM] | Bs [KC][128] | Hs [H1p][TM] | H2s [H2p][TM]
    float *Ac = sm, *Bs = Ac + KC * TM, *Hs = Bs + KC * 128, *H2s = Hs + A.H1p * TM;
    __shared__ int32_t atom_s[TM];
    if (tid < TM) atom_s[tid] = (tid < tile.count) ? A.sp_list[tile.start + tid] : -1;
    const float *Qt = A.Q + (size_t)tile.start * A.nqp;
    // 1. z1 = U^T Q + b1
    float acc1[4][NC1];
#pragma unroll
    for (int r = 0; r < 4; ++r)
#pragma unroll
        for (int c = 0; c < NC1; ++c) acc1[r][c] = 0.f;
    for (int q0 = 0; q0 < A.nqp; q0 += KC) {
        const int kc = min(KC, A.nqp - q0);
        __syncthreads();
        load_a_chunk(Ac, Qt, A.nqp, q0, kc, tile.count);
        load_b_chunk<NC1>(Bs, W.U, A.H1p, q0, kc, 0);
        __syncthreads();
        mm_chunk<NC1>(acc1, Ac, Bs, kc, tm, tn);
    }
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const int m = tm * 4 + r;
#pragma unroll
        for (int c = 0; c < NC1; ++c) {
            const int n = col_of<NC1>(tn, c);
            const float z = acc1[r][c] + __ldg(W.b1 + n);
            if (m < tile.count) A.z_stash[(size_t)(tile.start + m) * A.zs + n] = z;
            Hs[n * TM + m] = silu_f(z);
        }
    }
    // 2. z2 = W2^T h1 + b2
    float acc2[4][NC2];
    gemm_smemA<NC2>(acc2, Hs, A.H1p, W.W2, A.H2p, 0, Bs, tm, tn);
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const int m = tm * 4 + r;
#pragma unroll
        for (int c = 0; c < NC2; ++c) {
            const int n = col_of<NC2>(tn, c);
            const float z = acc2[r][c] + __ldg(W.b2 + n);
            if (m < tile.count) A.z_stash[(size_t)(tile.start + m) * A.zs + A.H1p + n] = z;
            H2s[n * TM + m] = silu_f(z);
        }
    }
    __syncthreads();
    // 3. out = W3^T h2 + b3   (nout = N_phi or 1)
    for (int idx = tid; idx < TM * A.nout; idx += DT) {
        const int m = idx & (TM - 1), o = idx / TM;
        float s = __ldg(W.b3 + o);
        const float *w3 = W.W3T + (size_t)o * A.H2p;
        for (int k = 0; k < A.H2p; ++k) s = fmaf(H2s[k * TM + m], __ldg(w3 + k), s);
        if (atom_s[m] >= 0) A.out[(size_t)atom_s[m] * A.out_stride + o] = s;
    }
}

struct BwdArgs {
    const DenseW *w;
    const DenseTile *tiles;
    const int32_t *sp_list;
    const float *z_stash, *outbar; // outbar == nullptr: energy layer, outbar = 1
    float *Qbar;                   // [N][nqp], tile order
    int outbar_stride, nqp, H1p, H2p, nout, zs;
    const int32_t *skip;
};

template <int NC1, int NC2>
__global__ void __launch_bounds__(DT) k_dense_bwd(BwdArgs A) {
    SKIP_GUARD(A.skip);
    extern __shared__ __align__(16) float sm[];
    const DenseTile tile = A.tiles[blockIdx.x];
    const DenseW W = A.w[tile.species];
    const int tid = threadIdx.x, tm = tid >> 4, tn = tid & 15;
    // carve-up: Z1s [H1p][TM] | Z2s [H2p][TM] | Bs [KC][128] | ob [TM][nout+1]
    float *Z1s = sm, *Z2s = Z1s + A.H1p * TM, *Bs = Z2s + A.H2p * TM, *ob = Bs + KC * 128;
    __shared__ int32_t atom_s[TM];
    if (tid < TM) atom_s[tid] = (tid < tile.count) ? A.sp_list[tile.start + tid] : -1;
    __syncthreads();
    const int OLD = A.nout + 1;
    for (int idx = tid; idx < TM * A.nout; idx += DT) {
        const int m = idx / A.nout, o = idx % A.nout;
        float v = 0.f;
        if (atom_s[m] >= 0) v = A.outbar ? __ldg(A.outbar + (size_t)atom_s[m] * A.outbar_stride + o) : 1.0f;
        ob[m * OLD + o] = v;
    }
    __syncthreads();
    // 1. z2bar[m][g] = (sum_o W3[g][o] outbar[m][o]) * SiLU'(z2[m][g])  -> Z2s [g][m]
    for (int idx = tid; idx < TM * A.H2p; idx += DT) {
        const int m = idx & (TM - 1), g = idx / TM;
        float s = 0.f;
        const float *w3 = W.W3 + (size_t)g * A.nout;
        for (int o = 0; o < A.nout; ++o) s = fmaf(__ldg(w3 + o), ob[m * OLD + o], s);
        const float z2 = (m < tile.count) ? __ldg(A.z_stash + (size_t)(tile.start + m) * A.zs + A.H1p + g) : 0.f;
        Z2s[g * TM + m] = s * dsilu_f(z2);
    }
    // 2. z1bar = (W2 z2bar) * SiLU'(z1)  -> Z1s [h][m]      (B operand: W2T [H2p][H1p])
    float acc1[4][NC1];
    gemm_smemA<NC1>(acc1, Z2s, A.H2p, W.W2T, A.H1p, 0, Bs, tm, tn);
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const int m = tm * 4 + r;
#pragma unroll
        for (int c = 0; c < NC1; ++c) {
            const int n = col_of<NC1>(tn, c);
            const float z1 = (m < tile.count) ? __ldg(A.z_stash + (size_t)(tile.start + m) * A.zs + n) : 0.f;
            Z1s[n * TM + m] = acc1[r][c] * dsilu_f(z1);
        }
    }
    // 3. Qbar = z1bar . UT  ([TM][nqp]),  UT: [H1p][nqp] row-major; column blocks of 128 / 64 / 32 / 16
    float *Qt = A.Qbar + (size_t)tile.start * A.nqp;
    for (int col0 = 0; col0 < A.nqp;) {
        const int rem = A.nqp - col0;
        if (rem >= 128) {
            float acc[4][8];
            gemm_smemA<8>(acc, Z1s, A.H1p, W.UT, A.nqp, col0, Bs, tm, tn);
#pragma unroll
            for (int r = 0; r < 4; ++r)
                if (tm * 4 + r < tile.count) {
                    float *d = Qt + (size_t)(tm * 4 + r) * A.nqp + col0;
                    *reinterpret_cast<float4 *>(d + tn * 4) = make_float4(acc[r][0], acc[r][1], acc[r][2], acc[r][3]);
                    *reinterpret_cast<float4 *>(d + 64 + tn * 4) = make_float4(acc[r][4], acc[r][5], acc[r][6], acc[r][7]);
                }
            col0 += 128;
        } else if (rem >= 64) {
            float acc[4][4];
            gemm_smemA<4>(acc, Z1s, A.H1p, W.UT, A.nqp, col0, Bs, tm, tn);
#pragma unroll
            for (int r = 0; r < 4; ++r)
                if (tm * 4 + r < tile.count)
                    *reinterpret_cast<float4 *>(Qt + (size_t)(tm * 4 + r) * A.nqp + col0 + tn * 4) =
                        make_float4(acc[r][0], acc[r][1], acc[r][2], acc[r][3]);
            col0 += 64;
        } else if (rem >= 32) {
            float acc[4][2];
            gemm_smemA<2>(acc, Z1s, A.H1p, W.UT, A.nqp, col0, Bs, tm, tn);
#pragma unroll
            for (int r = 0; r < 4; ++r)
                if (tm * 4 + r < tile.count)
                    *reinterpret_cast<float2 *>(Qt + (size_t)(tm * 4 + r) * A.nqp + col0 + tn * 2) = make_float2(acc[r][0], acc[r][1]);
            col0 += 32;
        } else {
            float acc[4][1];
            gemm_smemA<1>(acc, Z1s, A.H1p, W.UT, A.nqp, col0, Bs, tm, tn);
#pragma unroll
            for (int r = 0; r < 4; ++r)
                if (tm * 4 + r < tile.count) Qt[(size_t)(tm * 4 + r) * A.nqp + col0 + tn] = acc[r][0];
            col0 += 16;
        }
    }
}

template <int NC1, int NC2>
int run_fwd(const LaunchCtx &ctx, const FwdArgs &A, int n_tiles, size_t smem) {
    static size_t attr = 0;
    if (smem > attr) {
        if (cudaFuncSetAttribute(k_dense_fwd<NC1, NC2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
            return REANN_ERR_UNSUPPORTED;
        attr = smem;
    }
    LAUNCH(ctx, (k_dense_fwd<NC1, NC2>), n_tiles, DT, smem, A);
    return REANN_OK;
}
template <int NC1, int NC2>
int run_bwd(const LaunchCtx &ctx, const BwdArgs &A, int n_tiles, size_t smem) {
    static size_t attr = 0;
    if (smem > attr) {
        if (cudaFuncSetAttribute(k_dense_bwd<NC1, NC2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
            return REANN_ERR_UNSUPPORTED;
        attr = smem;
    }
    LAUNCH(ctx, (k_dense_bwd<NC1, NC2>), n_tiles, DT, smem, A);
    return REANN_OK;
}

#define NC_DISPATCH(FN, ...)                                                                \
    switch ((ld.H1p / 16) * 10 + ld.H2p / 16) {                                             \
        case 11: return FN<1, 1>(__VA_ARGS__); case 12: return FN<1, 2>(__VA_ARGS__);       \
        case 14: return FN<1, 4>(__VA_ARGS__); case 18: return FN<1, 8>(__VA_ARGS__);       \
        case 21: return FN<2, 1>(__VA_ARGS__); case 22: return FN<2, 2>(__VA_ARGS__);       \
        case 24: return FN<2, 4>(__VA_ARGS__); case 28: return FN<2, 8>(__VA_ARGS__);       \
        case 41: return FN<4, 1>(__VA_ARGS__); case 42: return FN<4, 2>(__VA_ARGS__);       \
        case 44: return FN<4, 4>(__VA_ARGS__); case 48: return FN<4, 8>(__VA_ARGS__);       \
        case 81: return FN<8, 1>(__VA_ARGS__); case 82: return FN<8, 2>(__VA_ARGS__);       \
        case 84: return FN<8, 4>(__VA_ARGS__); case 88: return FN<8, 8>(__VA_ARGS__);       \
        default: return REANN_ERR_UNSUPPORTED;                                              \
    }

} // namespace

int launch_dense_fwd(const LaunchCtx &ctx, const ModelDims &md, const LayerDims &ld, const DenseW *d_w,
                     const DenseTile *tiles, int n_tiles, const int32_t *sp_list, const float *Q, float *z_stash, int zs,
                     float *out, int out_stride) {
    if (n_tiles <= 0) return REANN_OK;
    FwdArgs A;
    A.w = d_w; A.tiles = tiles; A.sp_list = sp_list; A.Q = Q; A.z_stash = z_stash; A.out = out;
    A.out_stride = out_stride; A.nqp = md.nqp; A.H1p = ld.H1p; A.H2p = ld.H2p; A.nout = ld.nout; A.zs = zs; A.skip = ctx.skip;
    const size_t smem = sizeof(float) * ((size_t)KC * TM + KC * 128 + (size_t)TM * (A.H1p + A.H2p));
    NC_DISPATCH(run_fwd, ctx, A, n_tiles, smem)
}

int launch_dense_bwd(const LaunchCtx &ctx, const ModelDims &md, const LayerDims &ld, const DenseW *d_w,
                     const DenseTile *tiles, int n_tiles, const int32_t *sp_list, const float *z_stash, int zs,
                     const float *outbar, int outbar_stride, float *Qbar) {
    if (n_tiles <= 0) return REANN_OK;
    BwdArgs A;
    A.w = d_w; A.tiles = tiles; A.sp_list = sp_list; A.z_stash = z_stash; A.outbar = outbar; A.Qbar = Qbar;
    A.outbar_stride = outbar_stride; A.nqp = md.nqp; A.H1p = ld.H1p; A.H2p = ld.H2p; A.nout = ld.nout; A.zs = zs; A.skip = ctx.skip;
    const size_t smem = sizeof(float) * ((size_t)TM * (A.H1p + A.H2p) + KC * 128 + TM * (A.nout + 1));
    NC_DISPATCH(run_bwd, ctx, A, n_tiles, smem)
}
