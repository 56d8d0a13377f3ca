/*
 * reann.h -- C ABI of libreann_b200.so: the REANN energy + force (+ virial) hot path on one B200.
 *
 * The model is the recursively embedded atom neural network of arXiv 2505.06711
 * (Eqs. 1-2; forces by the chain rule of PAPER.md:59-80, Eqs. 3-5), with the
 * readings of SURVEY.md section 8(c) / DESIGN.md where the paper is silent. Everything behind
 * these calls runs in hand-written CUDA kernels for sm_100a; there is no CPU fallback.
 *
 * Conventions
 *  - Units: Angstrom, eV, eV/Angstrom.
 *  - `pos`, `E`, `F`, `virial`, `species`, `weights` may each be HOST or DEVICE pointers
 *    (detected with cudaPointerGetAttributes). `box` is always a HOST pointer to 9 doubles:
 *    row-major lattice vectors a = box[0..2], b = box[3..5], c = box[6..8] in lower-triangular form,
 *    a = (ax, 0, 0), b = (bx, by, 0), c = (cx, cy, cz) with ax, by, cz > 0 (orthorhombic: bx = cx = cy = 0;
 *    any triclinic cell can be rotated into this form). The distance between opposite faces of the cell
 *    must be >= rc + skin in all three directions (so only images -1,0,+1 of the wrapped atoms occur);
 *    entries box[1], box[2], box[5] other than 0 give REANN_ERR_UNSUPPORTED. Positions need not be
 *    wrapped into the cell. The pair test is FP64 with the operation order of DESIGN.md A-15 / B-9.
 *  - Ownership: the caller owns every array it passes; the library copies what it keeps
 *    (weights, species) and never retains caller pointers past the call.
 *  - Synchronisation: reann_energy_forces enqueues the whole evaluation on the handle's stream
 *    without a host round trip in the middle (the skin criterion and the capacity of the
 *    compact-edge buffers are checked on the device; the kernels after the check return at once
 *    when either fails) and synchronises the stream ONCE, at the end, to read that flag word: a
 *    rebuild or a buffer growth is followed by a second pass inside the same call. When the
 *    call returns, the outputs are complete (device or host pointers alike). The steady-state
 *    launch sequence is a CUDA graph, re-captured after every rebuild and whenever the device
 *    addresses it works on change (the caller's device pointers, or the handle's staging buffers
 *    when host pointers are passed; REANN_GRAPH=0 switches it off). The handle never works on the legacy default stream (a
 *    graph cannot be captured there): until reann_set_stream gives it a stream, or when that
 *    stream is 0, it uses a blocking stream of its own, which is ordered after earlier work of
 *    the default stream. Systems whose per-edge stash is held in chunks synchronise once more.
 *  - Every function returns a REANN_* code, never throws or aborts; reann_last_error() gives
 *    text for the last failure on that handle.
 *  - Determinism: same inputs give bitwise-identical outputs (no floating-point atomics;
 *    fixed reduction order) for a given build, kernel selection and stash chunk count.
 *  - Memory: device buffers grow on demand and are kept; list-sized buffers carry head-room so
 *    that skin-triggered rebuilds do not allocate. When the per-edge stash of the reverse pass
 *    (4 n_gauss bytes per edge within rc) does not fit into the free device memory it is held
 *    for a fraction of the atoms at a time (transparent to the caller).
 *  - Environment switches, read once per handle at reann_create:
 *    REANN_DENSE=simt, REANN_EDGE_FWD=simt (kernel selection, for testing), REANN_STASH_CHUNKS=n,
 *    REANN_GRAPH=0, REANN_MLP_MODE=tf32 (plain TF32 MLP GEMMs; accuracy restated in DESIGN.md).
 */
#ifndef REANN_H
#define REANN_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct reann reann_t; /* opaque; owns all device memory */

enum {
    REANN_OK = 0,
    REANN_ERR_ARG = 1,          /* NULL / out-of-range argument                         */
    REANN_ERR_WEIGHTS = 2,      /* bad blob, or blob header disagrees with arguments    */
    REANN_ERR_BOX = 3,          /* box length < rc + skin, or non-positive              */
    REANN_ERR_NO_NEIGHBORS = 4, /* reann_energy_forces before any reann_build_neighbors */
    REANN_ERR_CUDA = 5,         /* a CUDA runtime call failed (text in last_error)      */
    REANN_ERR_OOM = 6,          /* device allocation failed                             */
    REANN_ERR_UNSUPPORTED = 7   /* lattice not lower-triangular, n_gauss > 16, L > 3, row too long ... */
};

/*
 * reann_create -- build a model instance for a fixed set of atoms (per-element
 * orbital coefficients, per-element atomic NNs, T message-passing layers).
 *   weights, weights_bytes : the blob described in gen/weights.py (header + float64 arrays:
 *                            r_center, alpha [T][S][n_gauss]; c0 [S][n_gauss];
 *                            Wc [T][L+1][n_gauss][n_orb]; per (t, s) W1,b1,W2,b2,W3,b3).
 *                            Copied; folded/converted to FP32 device copies.
 *   species[n_atoms]       : 0..S-1 in caller order; copied.
 *   rc, skin               : cutoff of Eq. 1 and the neighbour-list skin.
 *   T, L, n_gauss          : must equal the blob header (else REANN_ERR_WEIGHTS);
 *                            T >= 1, 0 <= L <= 3, 1 <= n_gauss <= 16 in this version.
 */
int reann_create(reann_t **out, const void *weights, size_t weights_bytes, const int32_t *species,
                 int64_t n_atoms, double rc, double skin, int T, int L, int n_gauss);

/*
 * reann_build_neighbors -- force a rebuild of the skin neighbour list (one list
 * with cutoff rc(+skin), reused by every layer; local atoms, ghost atoms).
 * Sorts atoms by cell (Morton order), generates the periodic-image ("ghost") map, and emits
 * CSR rows of all (i, j_image) with |r_j + S o box - r_i|^2 < (rc+skin)^2, strict, FP64,
 * plus the index of every reverse edge.   pos: [n_atoms][3] doubles.
 */
int reann_build_neighbors(reann_t *h, const double *pos, const double *box9);

/*
 * reann_energy_forces -- one evaluation of E = sum_i E_i, F_k = -dE/dr_k
 * (Eq. 3) and optionally the virial  -sum_e r_e (x) dE/dr_e  (3x3 row-major, eV; = -dE/d(strain)).
 * Runs the skin check itself (rebuild when any atom moved > skin/2 since the last build, or
 * the box changed), then T forward layers (Eq. 1, Eq. 2) and the analytic reverse pass
 * (Eqs. 3-5).   E: 1 double; F: [n_atoms][3] doubles, caller order; virial: 9 doubles or NULL.
 */
int reann_energy_forces(reann_t *h, const double *pos, const double *box9, double *E, double *F,
                        double *virial);

void reann_destroy(reann_t *h);
const char *reann_last_error(const reann_t *h); /* h may be NULL: error of the last failed create */

/* ---- introspection for the parity tests and bench.py (not needed by an MD code) ---- */

typedef struct {
    int64_t n_atoms, n_ext;          /* local atoms, local + image ("ghost") atoms            */
    int64_t n_edges_list, n_edges_rc;/* list entries (r < rc+skin); entries with r < rc now   */
    int64_t n_rebuilds, n_calls;     /* builds so far; reann_energy_forces calls so far       */
    int64_t n_launches;              /* kernels launched by this handle so far                */
    double ms_build;                 /* accumulated, only while profiling is on (ms):         */
    double ms_prep, ms_edge_fwd, ms_dense_fwd, ms_gather, ms_dense_bwd, ms_edge_bwd,
           ms_rev_gather, ms_output;
    int64_t n_profiled_calls;        /* calls the ms_* fields (except ms_build) accumulate    */
    size_t bytes_device;             /* device memory currently held by the handle            */
    double ms_rev_gather_t0;         /* the layer-0 reverse gather (forces only, no cbar); ms_rev_gather = layers t >= 1 */
    int64_t stash_chunks;            /* atom chunks the per-edge stash is currently held in (1 = whole) */
} reann_stats_t;

/* Neighbour list in the CALLER's order and frame (for exact pair-set parity):
 *   call with row_ptr = j = shift = NULL to get *n_edges; then with arrays of sizes
 *   row_ptr[n_atoms+1], j[n_edges] (caller index of the neighbour), shift[n_edges][3] such
 *   that the edge vector is pos[j] + shift o box - pos[i] for the positions given at build.
 *   All three are HOST pointers. */
int reann_get_neighbors(reann_t *h, int64_t *n_edges, int64_t *row_ptr, int32_t *j, int8_t *shift);

/* The same for n_sel selected atoms only (caller indices, HOST array): row_ptr[n_sel+1] is always written; j and
 * shift (both or neither; HOST arrays of row_ptr[n_sel] entries) when given. For sampled exact pair-set parity
 * on systems whose whole list (up to 2^32 entries) is too large to export. */
int reann_get_neighbor_rows(reann_t *h, int64_t n_sel, const int64_t *atoms, int64_t *row_ptr, int32_t *j,
                            int8_t *shift);

int reann_get_stats(reann_t *h, reann_stats_t *out);
int reann_set_profiling(reann_t *h, int on);            /* CUDA-event timing of kernel groups  */
int reann_set_stream(reann_t *h, void *cuda_stream);    /* e.g. torch.cuda.current_stream().cuda_stream */

/* Per-atom energies E_i of the last evaluation, caller order (host or device pointer). */
int reann_get_atomic_energies(reann_t *h, double *Ei);

/*
 * ---- One rank of a spatially decomposed run (the paper's scheme, Fig. 3-4; groundwork for NEXT-1) ----
 * The handle is created over the rank's local atoms (LAs) AND copies of the other ranks' atoms that lie within
 * rc + skin of its domain (ghost atoms, GAs); reann_set_halo flags the GAs (HOST array [n_atoms], 1 = GA; NULL
 * clears). GAs serve as neighbours only: their E_i is not counted, they are not centres of edges on this rank
 * ("local parts computed in place"). One evaluation, driven by the caller, all ranks in lock step:
 *   reann_step_begin(pos, box, want_virial)      skin check / rebuild, compact edge list, c^0
 *   for t = 0 .. T-1:                             forward (Fig. 4a)
 *     [t >= 1] reann_coeff_set(t, GAs, rows)      c^t of the GAs, received from their owners (reann_coeff_get there)
 *     reann_step_forward(t)                       rho^t and c^{t+1} (or E_i) of the LAs
 *   for t = T-1 .. 0:                             reverse (Fig. 4b; vector-Jacobian products)
 *     [t < T-1] reann_cbar_add(LAs, rows)         dE/dc^{t+1} contributions received from the ranks that hold the
 *                                                 atom as a GA (reann_cbar_get there, after their step_backward(t+1))
 *     reann_step_backward(t)                      this rank's edges: dE/dc^t rows (t >= 1), forces accumulate
 *   reann_step_end(E, F, virial)                  E = sum over LAs; F[n_atoms][3]: the rows of GAs are this rank's
 *                                                 contributions to forces on other ranks' atoms (to be sent and added
 *                                                 there, Eq. 3); virial = this rank's edges
 * Row arrays are HOST float arrays [n][n_gauss]; idx are caller indices (HOST int64, unique within a call).
 * Every call synchronises the stream. Not available while the per-edge stash is held in chunks.
 */
int reann_set_halo(reann_t *h, const uint8_t *is_halo);
int reann_step_begin(reann_t *h, const double *pos, const double *box9, int want_virial);
int reann_step_forward(reann_t *h, int t);
int reann_coeff_get(reann_t *h, int t, int64_t n, const int64_t *idx, float *out);
int reann_coeff_set(reann_t *h, int t, int64_t n, const int64_t *idx, const float *in);
int reann_step_backward(reann_t *h, int t);
int reann_cbar_get(reann_t *h, int64_t n, const int64_t *idx, float *out);
int reann_cbar_add(reann_t *h, int64_t n, const int64_t *idx, const float *in);
int reann_step_end(reann_t *h, double *E, double *F, double *virial);

/*
 * Harness support, outside the energy/force path: one velocity-Verlet step on device arrays
 * (all DEVICE pointers, caller order): v += dt/2 * F * acc_unit / m ; x += dt * v  (kick_drift),
 * or only the half kick. inv_mass[n_atoms] in 1/amu, acc_unit converts eV/(A amu) to A/fs^2.
 */
int reann_verlet(reann_t *h, double *pos, double *vel, const double *F, const double *inv_mass,
                 double dt, double acc_unit, int drift);

/*
 * ---- Device-resident molecular dynamics ----
 * The paper drives its potentials in NVT molecular dynamics at 300 K (MD driver of
 * section 4.2). reann_md_run advances n_steps of velocity Verlet, optionally with a Nose-Hoover
 * thermostat (one thermostat variable; half step before and after every velocity-Verlet step; g = 3 n_atoms degrees of
 * freedom; Q = g kT tau^2 -- the integrator is written out in DESIGN.md section 2, B-8, and in oracle/md.py):
 *   pos, vel [n_atoms][3], inv_mass [n_atoms] (1/amu), F [n_atoms][3], virial [9] or NULL: DEVICE pointers, caller
 *     order; pos and vel are advanced in place, F and virial hold the values at the final positions on return
 *     (F need not be initialised: the forces at the initial positions are evaluated first, unless st->forces_valid
 *     says that F already holds them, e.g. from the previous reann_md_run of the same trajectory);
 *   dt in fs, acc_unit converts eV/(A amu) to A/fs^2, kT = kB T in eV (kT <= 0: no thermostat, NVE), tau in fs;
 *   st: in  xi, vxi (0, 0 to start; pass the values a previous call returned to continue a run), forces_valid,
 *       out xi, vxi, kinetic and potential energy (eV) after the last step, the conserved quantity
 *           KE + PE + Q vxi^2 / 2 + g kT xi, steps done, rebuilds of the neighbour list during the run.
 * Nothing but the thermostat scalars and E crosses to the host; every step is one reann_energy_forces (skin check on
 * the device, CUDA graph of the evaluation) plus three small kernels. Builds the list first if there is none.
 * Errors: as reann_energy_forces; REANN_ERR_ARG for host pointers or non-positive dt / acc_unit / tau.
 */
typedef struct {
    double xi, vxi;
    int64_t forces_valid;            /* in: non-zero = F holds the forces at pos (skip the initial evaluation; then
                                        `potential` / `conserved` are only defined when n_steps > 0) */
    double kinetic, potential, conserved;
    int64_t n_steps_done, n_rebuilds;
} reann_md_state_t;
int reann_md_run(reann_t *h, double *pos, double *vel, const double *inv_mass, const double *box9, int64_t n_steps,
                 double dt, double acc_unit, double kT, double tau, double *F, double *virial, reann_md_state_t *st);

/*
 * ---- An entry point that allocates nothing ----
 * For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid it): the step of the neighbour build that turns per-atom neighbour counts into the CSR row pointers of the
 * list ("neighbor list" of PAPER.md:57-59, section 2.2), with no handle and no allocation.
 *   row_ptr[0] = 0, row_ptr[i + 1] = counts[0] + ... + counts[i]      (exact, 64-bit sums)
 *   counts  [n_rows]      int32, DEVICE pointer, read only (may be NULL when n_rows == 0);
 *   row_ptr [n_rows + 1]  int64, DEVICE pointer, written; both stay the caller's;
 *   cuda_stream           cudaStream_t to enqueue on (NULL = the default stream); the call does not synchronise.
 * Same kernels as the handle's build; their workspace (block totals and offsets) is a file-scope device array of
 * fixed size instead of a cudaMalloc'ed buffer: 133 120 bytes that every GPU loading the library holds until the
 * process exits. Limit: n_rows <= REANN_NOALLOC_MAX_ROWS; larger -> REANN_ERR_UNSUPPORTED, nothing launched.
 * Calls no cudaMalloc / cudaFree or allocating library routine. All calls on one device share the array: calls that
 * overlap on the GPU (different streams without ordering between them, or different host threads) RACE -- order
 * them. The array keeps the previous call's contents; no word of it is read before this call has written it.
 * Errors: REANN_ERR_ARG (NULL pointer, n_rows < 0), REANN_ERR_UNSUPPORTED (over the limit), REANN_ERR_CUDA;
 * the text is returned by reann_last_error(NULL) on the calling thread.
 */
#define REANN_NOALLOC_MAX_ROWS (1 << 24)
int reann_row_ptr_noalloc(const int32_t *counts, int64_t n_rows, int64_t *row_ptr, void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* REANN_H */
