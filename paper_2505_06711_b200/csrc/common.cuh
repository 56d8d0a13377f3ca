// common.cuh -- shared declarations of the CUDA implementation (sm_100a only).
// Notation follows the paper / SURVEY.md section 8: N atoms, G ghosts (periodic images),
// N_ext = N + G, nphi = N_phi primitives, Na Cartesian monomials, NB = nphip * Na,
// n_q = (L+1) nphi (nphi+1) / 2 radial-pair products (see dense.cu), H1/H2 MLP widths.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <math.h>

#include <string>
#include <vector>

#include "../../include/reann.h"

#define REANN_MAX_S 32
#define REANN_MAX_T 8
#define REANN_MAX_NA 20
#define REANN_MAX_NPHI 16

// ---------------------------------------------------------------------------------------------
// Ext-atom record, 32 B (one DRAM sector): the WRAPPED position of the owner in FP64, the owner's
// internal index and the image shift. Edge vectors are formed as (x_owner(j) - x_i) + S*L in
// FP64, which is exactly antisymmetric under (i <-> j, S <-> -S): both directions of an edge
// take the same r < rc decision and the same |r|.
struct __align__(32) XRec {
    double x, y, z;
    int32_t owner;     // internal index of the owning local atom (== own index for locals)
    int8_t sx, sy, sz; // image shift in {-1,0,1}
    uint8_t species;
};
static_assert(sizeof(XRec) == 32, "XRec must be 32 bytes");

// shift code 0..26 = (sx+1)*9 + (sy+1)*3 + (sz+1); 13 = no shift; reverse code = 26 - code
__host__ __device__ inline int shift_code(int sx, int sy, int sz) { return (sx + 1) * 9 + (sy + 1) * 3 + (sz + 1); }

// Periodic cell in the lower-triangular form of include/reann.h: a = (ax, 0, 0), b = (bx, by, 0), c = (cx, cy, cz);
// orthorhombic: bx = cx = cy = 0. wa / wb / wc = distance between the two faces spanned by the other two vectors.
// The arithmetic below is the reading B-9 of DESIGN.md (A-15 extended): FP64, round to nearest, no contraction, in
// exactly this order -- the r < R decisions of the neighbour list depend on it bit for bit. For an orthorhombic cell
// every expression reduces to the x - floor(x / L) L and (x_j - x_i) + S L of A-15 with the same bits.
struct BoxP {
    double ax, bx, by, cx, cy, cz;
    double wa, wb, wc;
};
inline BoxP make_boxp(const double *box9) {
    BoxP B{box9[0], box9[3], box9[4], box9[6], box9[7], box9[8], 0, 0, 0};
    const double n0 = B.by * B.cz, n1 = -B.bx * B.cz, n2 = B.bx * B.cy - B.by * B.cx;      // b x c
    B.wa = B.ax * B.by * B.cz / sqrt(n0 * n0 + n1 * n1 + n2 * n2);
    B.wb = B.by * B.cz / sqrt(B.cy * B.cy + B.cz * B.cz);
    B.wc = B.cz;
    return B;
}
#ifdef __CUDACC__
// fractional coordinates by back substitution: x = sa a + sb b + sc c
__device__ __forceinline__ void box_frac(const BoxP &B, double x, double y, double z, double &sa, double &sb, double &sc) {
    sc = __ddiv_rn(z, B.cz);
    sb = __ddiv_rn(__dsub_rn(y, __dmul_rn(sc, B.cy)), B.by);
    sa = __ddiv_rn(__dsub_rn(__dsub_rn(x, __dmul_rn(sb, B.bx)), __dmul_rn(sc, B.cx)), B.ax);
}
// S . box for whole periods (sa, sb, sc): ((sa ax + sb bx) + sc cx, sb by + sc cy, sc cz)
__device__ __forceinline__ void box_shift(const BoxP &B, double sa, double sb, double sc, double &hx, double &hy, double &hz) {
    hx = __dadd_rn(__dadd_rn(__dmul_rn(sa, B.ax), __dmul_rn(sb, B.bx)), __dmul_rn(sc, B.cx));
    hy = __dadd_rn(__dmul_rn(sb, B.by), __dmul_rn(sc, B.cy));
    hz = __dmul_rn(sc, B.cz);
}
#endif

// col_rc entries carry the neighbour's species in the top 5 bits (S <= 32, N_ext < 2^27)
#define COL_IDX_MASK 0x07FFFFFFu
#define COL_SPECIES_SHIFT 27

struct DevBuf {
    void *p = nullptr;
    size_t bytes = 0;
};

// Per-(layer, species) dense weights, FP32, padded (see dense.cu / api.cu fold_weights()).
struct DenseW {
    const float *U;   // [n_qp][H1p]      folded  U = V . W1   (K-major for the forward GEMM)
    const float *UT;  // [H1p][n_qp]      transposed (K-major for the backward GEMM)
    const float *b1;  // [H1p]
    const float *W2;  // [H1p][H2p]
    const float *W2T; // [H2p][H1p]
    const float *b2;  // [H2p]
    const float *W3;  // [H2p][noutp]
    const float *W3T; // [noutp][H2p]
    const float *b3;  // [noutp]
};

// Tensor-core path (dense_tc.cu): pre-split (hi | lo) TF32 weight chunk images, see dense_tc.cu.
struct DenseWT {
    const float *g1, *g2;      // forward:  U^T chunks [K1/32], W2^T chunks [H1p/32]
    const float *r1, *r2, *r3; // reverse:  W3 chunk (K = n_out padded to 32), W2 chunks [H2p/32], U blocks of <= 128 rows x [H1p/32]
    const float *b1, *b2, *b3; // biases (FP32)
    const float *w3p;          // FP32 [H2p][16]: W3 rows zero-padded to 16 outputs (ALU GEMM with n_out <= 16)
    const float *w3c0;         // FP32 [H2p]: first column of W3 (energy layer, n_out = 1)
};

struct LayerDims {
    int H1p, H2p, nout, noutp;
};

struct ModelDims {
    int S, T, L, nphi, nphip, Na, NB, norb;
    int npairs, NPp, nqp; // pairs n<=n' per l; stride of an l block in Q (= npairs); (L+1)*NPp rounded up to 16
    int K1;               // nqp rounded up to 32 (K extent of the tensor-core GEMM over Q)
    double rc, skin;
};

// launch counter (kernels launched by the handle) -- every launch goes through LAUNCH()
struct LaunchCtx {
    cudaStream_t stream;
    int64_t *n_launches;
    // device flag word: non-zero = this evaluation is void (the skin criterion asks for a rebuild, or the compact
    // edge list outgrew its buffers); every kernel after the rc-filter count returns at once when it is set, the
    // host reads it after the evaluation and redoes the step (api.cu). nullptr: no guard.
    const int32_t *skip;
};
#define SKIP_GUARD(skip) do { if ((skip) != nullptr && *(skip) != 0) return; } while (0)
#define LAUNCH(ctx, kernel, grid, block, smem, ...)                          \
    do {                                                                     \
        kernel<<<(grid), (block), (smem), (ctx).stream>>>(__VA_ARGS__);      \
        ++*(ctx).n_launches;                                                 \
    } while (0)

static inline unsigned div_up(int64_t a, int64_t b) { return (unsigned)((a + b - 1) / b); }

// ---- scan.cu ----
// exclusive scan of int32 counts into int64 offsets: out[0] = 0, out[i+1] = sum_{k<=i} in[k]
size_t scan_workspace_bytes(int64_t n);
void exclusive_scan_i32_to_i64(const LaunchCtx &ctx, const int32_t *in, int64_t *out, int64_t n, void *workspace);

// ---- neighbor.cu ----
struct reann; // handle (api.cu)
int neighbor_build(reann *h, const double *d_pos);   // returns REANN_* code
int neighbor_export(reann *h, int64_t *n_edges, int64_t *row_ptr, int32_t *j, int8_t *shift);
int neighbor_export_rows(reann *h, int64_t n_sel, const int64_t *atoms, int64_t *row_ptr, int32_t *j, int8_t *shift);

// ---- edge.cu ----
void launch_skin_check(const LaunchCtx &ctx, const double *pos, const double *pos_build, int64_t N, double thr2,
                       int32_t *flag);
void launch_refresh(const LaunchCtx &ctx, XRec *xrec, int64_t n_ext, const int32_t *perm, const int32_t *wshift,
                    const double *pos, const BoxP &box, float *c_ext0, const float *c0, int nphip);
void launch_filter_count(const LaunchCtx &ctx, const XRec *xrec, const int64_t *row_ptr, const int32_t *col,
                         int64_t N, const BoxP &box, double rc2, uint16_t *rank16, int32_t *rc_cnt);
void launch_filter_fill(const LaunchCtx &ctx, const XRec *xrec, const int64_t *row_ptr, const int32_t *col,
                        const uint32_t *rev, int64_t N, int64_t n_ext, const BoxP &box, const uint16_t *rank16,
                        const int64_t *rc_ptr, uint32_t *rcx, uint32_t *col_rc, float4 *geom, uint32_t *rev_rc);
void launch_ghost_gather(const LaunchCtx &ctx, float *c_ext, const XRec *xrec, int64_t N, int64_t n_ext, int nphip);
int launch_edge_fwd(const LaunchCtx &ctx, const ModelDims &md, int t, int64_t N, const int64_t *rc_ptr,
                    const uint32_t *col_rc, const float4 *geom, const float *c_ext, const float *rcen,
                    const float *alpha, float *b, bool allow_mma);
int launch_edge_bwd(const LaunchCtx &ctx, const ModelDims &md, int t, int64_t N, const int64_t *rc_ptr,
                    const uint32_t *col_rc, const float4 *geom, const float *c_ext, const float *rcen,
                    const float *alpha, const float *bbar, float *kappa, float4 *gst, double *vir_part,
                    int64_t a0, int64_t a1, int64_t e_lo /* atoms [a0, a1), a0 % 4 == 0; kappa holds edges from e_lo on */,
                    bool g_add /* gst += g_e (layers below the top one: the stash then holds the sum over the layers) */);
int edge_bwd_blocks(int64_t N, int Na);
void launch_rev_gather(const LaunchCtx &ctx, int64_t N, const int64_t *rc_ptr, const uint32_t *rev_rc,
                       const float *kappa, const float4 *gst, int nphip, int want_cbar, float *cbar, double *Fc,
                       int64_t e_lo, int64_t e_hi, int do_forces, int accumulate /* kappa holds edges [e_lo, e_hi) */);
void launch_output(const LaunchCtx &ctx, int64_t N, const int32_t *inv_perm, const double *Fc, const float *Ei,
                   const double *vir_part, int n_vir_blocks, double *E_out, double *F_out, double *vir_out,
                   double *Ei_sorted, double *scratch, const uint8_t *halo_caller /* or nullptr */);
void launch_verlet(const LaunchCtx &ctx, int64_t N, double *pos, double *vel, const double *F, const double *inv_mass,
                   double dt, double acc_unit, int drift);

// ---- md.cu ----
int md_blocks(int64_t N);
void launch_md_kick(const LaunchCtx &ctx, int64_t N, double *pos, double *vel, const double *F, const double *inv_mass,
                    double dt, double acc_unit, int drift, const double *state /* or nullptr */, double *ke_partial /* or nullptr */);
void launch_nh_update(const LaunchCtx &ctx, int64_t N, const double *ke_partial, double *state, double h, double g_kT,
                      double Q, double acc_unit, int mode, int nvt);
void launch_md_scale(const LaunchCtx &ctx, int64_t N, double *vel, const double *state);

// ---- gram.cu / dense.cu ----
struct DenseTile {
    int32_t species, start, count; // atoms sp_list[start .. start+count) all of `species`
};
// tiles != nullptr: Q / Qbar in the tile-quad layout of dense_tc.cu (K1 columns, 128-row tiles);
// tiles == nullptr: row-major [N][nqp] rows in sp_list order (SIMT path)
int launch_gram_fwd(const LaunchCtx &ctx, const ModelDims &md, int64_t N, const int32_t *sp_list, const DenseTile *tiles,
                    int n_tiles, const float *b, float *Q);
int launch_gram_bwd(const LaunchCtx &ctx, const ModelDims &md, int64_t N, const int32_t *sp_list, const DenseTile *tiles,
                    int n_tiles, const float *b, const float *Qbar, float *bbar);
int launch_dense_fwd(const LaunchCtx &ctx, const ModelDims &md, const LayerDims &ld, const DenseW *d_w /*[S]*/,
                     const DenseTile *tiles, int n_tiles, const int32_t *sp_list, const float *Q, float *z_stash,
                     int zs, float *out /* c_ext[t+1] rows (stride nphip) or Ei (stride 1) */, int out_stride);
int launch_dense_bwd(const LaunchCtx &ctx, const ModelDims &md, const LayerDims &ld, const DenseW *d_w,
                     const DenseTile *tiles, int n_tiles, const int32_t *sp_list, const float *z_stash, int zs,
                     const float *outbar /* cbar rows or NULL for the energy layer */, int outbar_stride,
                     float *Qbar /* [N][nqp], tile order */);
#define DENSE_TM 64 // atoms per dense tile (SIMT path)

// ---- dense_tc.cu (tcgen05 path; same contracts as the SIMT launchers, 128-atom tiles) ----
#define DENSE_TC_TM 128
int launch_dense_tc_fwd(const LaunchCtx &ctx, const ModelDims &md, const LayerDims &ld, const DenseWT *d_w,
                        const DenseTile *tiles, int n_tiles, const int32_t *sp_list, const float *Q, float *z_stash,
                        int zs, float *out, int out_stride, bool tf32 /* REANN_MLP_MODE=tf32 */);
int launch_dense_tc_bwd(const LaunchCtx &ctx, const ModelDims &md, const LayerDims &ld, const DenseWT *d_w,
                        const DenseTile *tiles, int n_tiles, const int32_t *sp_list, const float *z_stash, int zs,
                        const float *outbar, int outbar_stride, float *Qbar, bool tf32);
