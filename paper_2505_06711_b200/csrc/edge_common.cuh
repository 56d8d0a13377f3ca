// edge_common.cuh -- device helpers of the edge kernels (edge.cu): Cartesian monomials and their vector-Jacobian
// product, packed FP32 pairs, launch structs.
#pragma once
#include "common.cuh"

namespace edge {

// ------------------------------------------------------------------------------------------ orbitals
// Cartesian monomials in graded order: 1 | x y z | xx xy xz yy yz zz | xxx xxy xxz xyy xyz xzz yyy yyz yzz zzz
template <int NA>
__device__ __forceinline__ void monomials(float x, float y, float z, float *A) {
    A[0] = 1.0f;
    if constexpr (NA > 1) { A[1] = x; A[2] = y; A[3] = z; }
    if constexpr (NA > 4) { A[4] = x * x; A[5] = x * y; A[6] = x * z; A[7] = y * y; A[8] = y * z; A[9] = z * z; }
    if constexpr (NA > 10) {
        A[10] = A[4] * x; A[11] = A[4] * y; A[12] = A[4] * z; A[13] = A[7] * x; A[14] = A[5] * z;
        A[15] = A[9] * x; A[16] = A[7] * y; A[17] = A[7] * z; A[18] = A[9] * y; A[19] = A[9] * z;
    }
}
// sum_a P_a grad A_a
template <int NA>
__device__ __forceinline__ void monomial_vjp(const float *A, const float *P, float &gx, float &gy, float &gz) {
    gx = gy = gz = 0.0f;
    if constexpr (NA > 1) { gx = P[1]; gy = P[2]; gz = P[3]; }
    if constexpr (NA > 4) {
        const float x = A[1], y = A[2], z = A[3];
        gx += 2.0f * x * P[4] + y * P[5] + z * P[6];
        gy += x * P[5] + 2.0f * y * P[7] + z * P[8];
        gz += x * P[6] + y * P[8] + 2.0f * z * P[9];
    }
    if constexpr (NA > 10) {
        gx += 3.0f * A[4] * P[10] + 2.0f * A[5] * P[11] + 2.0f * A[6] * P[12] + A[7] * P[13] + A[8] * P[14] + A[9] * P[15];
        gy += A[4] * P[11] + 2.0f * A[5] * P[13] + A[6] * P[14] + 3.0f * A[7] * P[16] + 2.0f * A[8] * P[17] + A[9] * P[18];
        gz += A[4] * P[12] + A[5] * P[14] + 2.0f * A[6] * P[15] + A[7] * P[17] + 2.0f * A[8] * P[18] + 3.0f * A[9] * P[19];
    }
}

// 2^x as one MUFU.EX2 (exp2f() wraps it in a range check for denormal results, six more instructions per call)
__device__ __forceinline__ float ex2_ftz(float x) { float r; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }

// Packed FP32 pairs: Blackwell's fma.rn.f32x2 (SASS FFMA2) does two FP32 FMAs per issue slot at the same FLOP
// rate (measured 74 TFLOP/s either way), which halves the instruction count of the FMA loops below.
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pack2(float lo, float hi) {
    f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void unpack2(f32x2 v, float &lo, float &hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ void ffma2(f32x2 &c, f32x2 a, f32x2 b) { asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(c) : "l"(a), "l"(b)); }
__device__ __forceinline__ f32x2 fmadd2(f32x2 a, f32x2 b, f32x2 c) { f32x2 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
__device__ __forceinline__ f32x2 fmul2(f32x2 a, f32x2 b) { f32x2 r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }

__device__ __forceinline__ f32x2 fadd2(f32x2 a, f32x2 b) { f32x2 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }

// ---- warp-level tensor-core helpers (mma.sync TF32, 3xTF32 splitting) ----
__device__ __forceinline__ void mma_tf32(float (&d)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
    asm("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ void split_bits(float x, uint32_t &hi, uint32_t &lo) {
    // hi rounded to nearest TF32, lo = x - hi exact (<= 13 significant bits, of which the MMA reads the top 11):
    // |x - hi - lo_read| <= 2^-22 |x|
    hi = (__float_as_uint(x) + 0x1000u) & 0xFFFFE000u;
    lo = __float_as_uint(x - __uint_as_float(hi));
}

// ---- cp.async (LDGSTS): global -> shared without registers ----
__device__ __forceinline__ void cp_async16(void *dst_smem, const void *src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(dst_smem)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async4(void *dst_smem, const void *src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"((uint32_t)__cvta_generic_to_shared(dst_smem)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N_>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N_) : "memory"); }

// g_e stash accumulated over the layers: one 16-byte reduction per edge, resolved in L2, nothing returned (no register is
// held for the old value and no latency is exposed). Every address receives exactly one add per launch and launches
// are ordered on the stream, so the sum is deterministic.
__device__ __forceinline__ void red_add_f32x4(float4 *dst, float x, float y, float z, float w) {
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(dst), "f"(x), "f"(y), "f"(z), "f"(w) : "memory");
}
constexpr int BWD_KAPPA = 1, BWD_G_ADD = 2;   // flag word of k_edge_bwd: write the kappa stash / add g_e to the stash instead of storing it

struct StashChunk { // reverse gather: kappa holds the edges [e_lo, e_hi); forces once; cbar = or +=
    int64_t e_lo, e_hi;
    int do_forces, accumulate;
};
struct AtomChunk { // edge backward: atoms [a0, a1) (a0 % EW == 0); kappa holds the edges from e_lo on
    int64_t a0, a1, e_lo;
};
struct RadialTab { // per layer: [S][NPHIP]; alpha pre-multiplied by log2(e)
    const float *rcen, *alpha2;
    float inv_rc;
};


} // namespace edge
