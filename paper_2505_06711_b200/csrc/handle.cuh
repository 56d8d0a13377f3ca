// handle.cuh -- the opaque reann handle (host-side state + device buffers).
#pragma once
#include "common.cuh"

struct reann {
    ModelDims md{};
    LayerDims ld[REANN_MAX_T]{};
    int64_t N = 0;
    cudaStream_t stream = nullptr;      // the stream every kernel of the handle runs on (never the legacy default stream)
    cudaStream_t own_stream = nullptr;  // used while the caller has set no stream of their own
    // CUDA graph of the steady-state evaluation (api.cu): replayed while this key stays the same
    struct GraphKey { const void *pos, *E, *F, *V; int64_t n_rebuilds, cap_rc; cudaStream_t stream; };
    cudaGraphExec_t gexec = nullptr;
    GraphKey gkey{};
    int64_t g_kernels = 0;
    bool use_graph = true;              // REANN_GRAPH=0 switches the graph off
    int64_t n_launches = 0;
    std::string err;

    // ---- model (device, FP32) ----
    DevBuf w_all;                 // every dense weight, one allocation
    DevBuf w_tab;                 // DenseW[T][S]
    DevBuf wt_all, wt_tab;        // tensor-core weight images, DenseWT[T][S]
    // kernel selection, read from the environment once at reann_create
    bool dense_tc = true;         // REANN_DENSE=simt selects the FP32 SIMT GEMM chain instead
    bool edge_fwd_mma = true;     // REANN_EDGE_FWD=simt: FP32 ALU edge forward where the mma.sync kernel applies
    int stash_chunks_forced = 0;  // REANN_STASH_CHUNKS=n
    bool mlp_tf32 = false;        // REANN_MLP_MODE=tf32: plain TF32 GEMMs (one accumulator per GEMM), tolerance restated
    DevBuf rcen, alpha, c0;       // [T][S][nphip] (alpha pre-multiplied by log2(e)), [S][nphip]
    std::vector<DenseW> h_wtab;   // host copy of the table (device pointers inside)

    // ---- atoms (device) ----
    DevBuf species_caller;        // int32 [N]
    DevBuf tiles;                 // DenseTile[n_tiles]  (tiles of DENSE_TM or DENSE_TC_TM atoms)
    int n_tiles = 0, tile_rows = 0;
    std::vector<int64_t> species_count;

    // ---- neighbour list, rebuilt on demand ----
    bool have_list = false;
    bool eval_bufs_ready = false;  // every per-evaluation buffer of do_build() is allocated
    double box_build[9]{};
    int64_t G = 0, n_ext = 0, E_list = 0, E_rc_build = 0;
    DevBuf pos_build;             // double [N][3], caller order
    DevBuf wshift;                // int32 [N][3], caller order: floor(x/L) at build
    DevBuf perm, inv_perm;        // int32 [N]: internal -> caller, caller -> internal
    DevBuf xrec;                  // XRec [n_ext]
    DevBuf img_index;             // int32 [N][27]: ext index of image (owner, code) or -1
    DevBuf cell_start;            // int32 [ncell+1] (internal indices are cell-contiguous)
    DevBuf cell_rank;             // int32 [ncell]: linear cell id -> position in Morton order
    int nc_cached[3]{0, 0, 0};
    DevBuf row_ptr;               // int64 [N+1]
    DevBuf col;                   // int32 [E_list] ext index, rows sorted ascending
    DevBuf rev;                   // uint32 [E_list] index of the reverse entry
    DevBuf sp_list;               // int32 [N] internal indices grouped by species
    DevBuf scratch_a, scratch_b, scratch_c, scan_ws;
    DevBuf nbr_mask;              // uint32 [N][27 MB]: ballot words of the count pass of the list build

    // ---- per-evaluation buffers ----
    DevBuf pos_stage;             // double [N][3] when the caller passes host positions
    DevBuf rank16;                // uint16 [E_list]
    DevBuf rc_cnt;                // int32 [N]
    DevBuf rc_ptr;                // int64 [N+1]
    DevBuf rcx;                   // uint32 [n_ext]: rc_ptr of the owner of every ext atom
    DevBuf col_rc, geom, rev_rc;  // uint32 / float4 / uint32 [cap_rc]
    int64_t cap_rc = 0, E_rc = 0;
    int stash_chunks = 1;         // kappa stash held for 1/stash_chunks of the atoms at a time (memory-limited systems)
    DevBuf c_ext;                 // float [T][n_ext][nphip]
    DevBuf b;                     // float [T][N][NB]
    DevBuf z_stash;               // float [T][N][zs]  (z1 | z2 pre-activations)
    int zs = 0;
    DevBuf bbar;                  // float [N][NB]
    DevBuf Qbuf;                  // float [N][nqp] radial-pair products Q (forward) / Qbar (reverse), tile order
    DevBuf cbar;                  // float [N][nphip]
    DevBuf kappa;                 // float [cap_rc][nphip]
    DevBuf gst;                   // float4 [cap_rc]
    DevBuf Ei;                    // float [N] internal order
    DevBuf Fc;                    // double [N][3] internal order
    DevBuf vir_part;              // double [n_vir_blocks][9]
    int n_vir_blocks = 0;
    DevBuf out_stage;             // double [1 + 9 + 3N] device staging for host outputs; + Ei sorted
    DevBuf Ei_caller;             // double [N]
    DevBuf red_scratch;           // double [N/256 + 2] partial sums of the energy reduction
    DevBuf flags;                 // int32 [4] device flags
    int32_t *h_flags = nullptr;   // pinned mirror [8] (+ int64 n_rc)

    // ---- decomposed runs (NEXT-1 groundwork): ghost atoms of other ranks, layer-by-layer state ----
    bool have_halo = false;
    DevBuf halo_caller;           // uint8 [N], caller order: 1 = ghost atom (copy of another rank's atom)
    DevBuf xch_idx, xch_val;      // staging of reann_coeff_* / reann_cbar_* (int64 indices, float rows)
    int step_state = 0;           // 0 = idle, 1 = after reann_step_begin (forward), 2 = reverse pass started
    bool step_vir = false;

    // ---- device-resident MD (reann_md_run, md.cu) ----
    DevBuf md_state;              // double [8]: xi, vxi, pending scale, 2 KE, final scale
    DevBuf md_partial;            // double [N/256 + 1] block partials of sum m v^2
    DevBuf md_E;                  // double [1] potential energy of the last step

    // ---- stats / profiling ----
    int64_t n_rebuilds = 0, n_calls = 0, n_prof_calls = 0;
    bool profiling = false;
    double ms[10]{};              // build, prep, edge_fwd, dense_fwd, gather, dense_bwd, edge_bwd, rev_gather (t >= 1), output, rev_gather (t = 0)
    std::vector<cudaEvent_t> ev;  // event pool
    size_t bytes_device = 0;

    LaunchCtx ctx() { return LaunchCtx{stream, &n_launches, nullptr}; }
};

// api.cu helpers used by neighbor.cu
int dev_ensure(reann *h, DevBuf &b, size_t bytes);       // grow-only; REANN_OK / REANN_ERR_OOM
int set_err(reann *h, int code, const char *fmt, ...);
#define CU(h, call)                                                                                    \
    do {                                                                                               \
        cudaError_t e_ = (call);                                                                       \
        if (e_ != cudaSuccess)                                                                         \
            return set_err((h), REANN_ERR_CUDA, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), \
                           __FILE__, __LINE__);                                                        \
    } while (0)
#define RC(call)                   \
    do {                           \
        int rc_ = (call);          \
        if (rc_ != REANN_OK) return rc_; \
    } while (0)
