// neighbor.cu -- rows A1-A3 of SURVEY.md section 8(a): cell assignment + Morton-ordered counting
// sort, periodic-image ("ghost") map, CSR neighbour list with skin, reverse-edge index.
//
// PAPER.md:49  "only the original neighbor list is required for each atom, and once computed, it
//              can be repeatedly used in different MP layers"
// PAPER.md:51  local atoms (LAs) with complete neighbour lists; ghost atoms (GAs) within the
//              cutoff sphere of LAs -- here: periodic images of the atoms of the one GPU domain.
// PAPER.md:23  skin distance to reduce the frequency of neighbour-list updates.
//
// Pair test: FP64, round-to-nearest, no FMA contraction:
//   x_w = x - floor(x/L) L;  d = (x_w[j] - x_w[i]) + S L;  d2 = (dx dx + dy dy) + dz dz;  d2 < (rc+skin)^2
// and for a triclinic cell (lower-triangular lattice, reading B-9) the same with fractional coordinates by
// back substitution and S . box = ((S0 ax + S1 bx) + S2 cx, S1 by + S2 cy, S2 cz): box_frac / box_shift of common.cuh.
// Integer atomics (cell histogram, scatter slots, counters) are used; their effect on ordering is
// removed by sorting each cell by caller index and each CSR row by ext index, so the list is
// bitwise deterministic.
#include <algorithm>
#include <numeric>

#include "handle.cuh"

namespace {

constexpr int ROWCAP = 1024; // max list entries per atom (smem row buffer per warp)
constexpr int NB_WARPS = 4;  // warps per block in the row kernels

// whole periods w = floor(fractional coordinates) and the wrapped position x - w . box (reading B-9)
__device__ __forceinline__ void wrap_pos(const BoxP &B, double x, double y, double z, int32_t *w, double *xw, double *yw,
                                         double *zw) {
    double sa, sb, sc;
    box_frac(B, x, y, z, sa, sb, sc);
    const double fa = floor(sa), fb = floor(sb), fc = floor(sc);
    w[0] = (int32_t)fa; w[1] = (int32_t)fb; w[2] = (int32_t)fc;
    double hx, hy, hz;
    box_shift(B, fa, fb, fc, hx, hy, hz);
    *xw = __dsub_rn(x, hx); *yw = __dsub_rn(y, hy); *zw = __dsub_rn(z, hz);
}
// cell of a wrapped position: cells are equal slices of the fractional coordinates
__device__ __forceinline__ void cell_of(const BoxP &B, double xw, double yw, double zw, int ncx, int ncy, int ncz, int *cx,
                                        int *cy, int *cz) {
    double sa, sb, sc;
    box_frac(B, xw, yw, zw, sa, sb, sc);
    *cx = min(ncx - 1, max(0, (int)floor(sa * ncx)));
    *cy = min(ncy - 1, max(0, (int)floor(sb * ncy)));
    *cz = min(ncz - 1, max(0, (int)floor(sc * ncz)));
}

__global__ void k_wrap_cell(const double *__restrict__ pos, int64_t N, BoxP B, int ncx,
                            int ncy, int ncz, const int32_t *__restrict__ cell_rank, int32_t *__restrict__ wshift,
                            int32_t *__restrict__ cellkey, int32_t *__restrict__ cell_count) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    int32_t w[3];
    double x, y, z;
    wrap_pos(B, pos[3 * i], pos[3 * i + 1], pos[3 * i + 2], w, &x, &y, &z);
    wshift[3 * i] = w[0]; wshift[3 * i + 1] = w[1]; wshift[3 * i + 2] = w[2];
    int cx, cy, cz;
    cell_of(B, x, y, z, ncx, ncy, ncz, &cx, &cy, &cz);
    int key = cell_rank[(cx * ncy + cy) * ncz + cz];
    cellkey[i] = key;
    atomicAdd(&cell_count[key], 1);
}

__global__ void k_max_i32(const int32_t *__restrict__ v, int64_t n, int32_t *__restrict__ out) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int m = i < n ? v[i] : 0;
#pragma unroll
    for (int d = 16; d >= 1; d >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, d));
    if ((threadIdx.x & 31) == 0 && m > 0) atomicMax(out, m);
}

__global__ void k_scatter(const int32_t *__restrict__ cellkey, int64_t N, const int64_t *__restrict__ cell_start,
                          int32_t *__restrict__ cell_fill, int32_t *__restrict__ perm) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    int key = cellkey[i];
    int slot = atomicAdd(&cell_fill[key], 1);
    perm[cell_start[key] + slot] = (int32_t)i;
}

// one warp per cell: rank sort by caller index (a cell holds a few dozen atoms) -> deterministic internal order
__global__ void k_sort_cells(int32_t *__restrict__ perm, const int64_t *__restrict__ cell_start, int64_t ncell) {
    const int lane = threadIdx.x & 31;
    const int64_t c = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (c >= ncell) return;
    const int64_t a = cell_start[c], b = cell_start[c + 1];
    const int n = (int)(b - a);
    if (n <= 1) return;
    if (n <= 64) {
        const int v0 = lane < n ? perm[a + lane] : 0x7fffffff, v1 = lane + 32 < n ? perm[a + 32 + lane] : 0x7fffffff;
        int r0 = 0, r1 = 0;
        for (int q = 0; q < n; ++q) {
            const int w = __shfl_sync(0xffffffffu, q < 32 ? v0 : v1, q & 31);
            r0 += w < v0; r1 += w < v1;
        }
        __syncwarp();
        if (lane < n) perm[a + r0] = v0;
        if (lane + 32 < n) perm[a + r1] = v1;
    } else if (lane == 0) {                      // very dense cell: insertion sort by one lane
        for (int64_t p = a + 1; p < b; ++p) {
            int32_t v = perm[p];
            int64_t q = p - 1;
            while (q >= a && perm[q] > v) { perm[q + 1] = perm[q]; --q; }
            perm[q + 1] = v;
        }
    }
}

__global__ void k_local_records(const int32_t *__restrict__ perm, const double *__restrict__ pos,
                                const int32_t *__restrict__ wshift, const int32_t *__restrict__ species_caller,
                                int64_t N, BoxP B, XRec *__restrict__ xrec,
                                int32_t *__restrict__ inv_perm, double *__restrict__ pos_build) {
    int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= N) return;
    int64_t i = perm[k];
    XRec r;
    double hx, hy, hz;
    box_shift(B, (double)wshift[3 * i], (double)wshift[3 * i + 1], (double)wshift[3 * i + 2], hx, hy, hz);
    r.x = __dsub_rn(pos[3 * i], hx);
    r.y = __dsub_rn(pos[3 * i + 1], hy);
    r.z = __dsub_rn(pos[3 * i + 2], hz);
    r.owner = (int32_t)k; r.sx = r.sy = r.sz = 0; r.species = (uint8_t)species_caller[i];
    xrec[k] = r;
    inv_perm[i] = (int32_t)k;
    pos_build[3 * i] = pos[3 * i]; pos_build[3 * i + 1] = pos[3 * i + 1]; pos_build[3 * i + 2] = pos[3 * i + 2];
}

// A2: images of atom k that can lie within R of some wrapped local atom. In the direction of lattice vector d the atom
// is s_d w_d away from the low face and (1 - s_d) w_d from the high one (s = fractional coordinate, w = distance between
// the faces): shift +1 needs s_d w_d < R (+margin), shift -1 needs (1 - s_d) w_d <= R (+margin). Superset of the images
// referenced.
__device__ __forceinline__ int allowed_mask(double s, double w, double Rm) {
    int m = 2; // bit1: s=0
    if (s * w < Rm) m |= 4;             // s=+1
    if ((1.0 - s) * w <= Rm) m |= 1;    // s=-1
    return m;
}
__device__ __forceinline__ void image_masks(const BoxP &B, const XRec &r, double Rm, int *mx, int *my, int *mz) {
    double sa, sb, sc;
    box_frac(B, r.x, r.y, r.z, sa, sb, sc);
    *mx = allowed_mask(sa, B.wa, Rm); *my = allowed_mask(sb, B.wb, Rm); *mz = allowed_mask(sc, B.wc, Rm);
}

__global__ void k_ghost_count(const XRec *__restrict__ xrec, int64_t N, BoxP B, double Rm,
                              int32_t *__restrict__ gcnt) {
    int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= N) return;
    XRec r = xrec[k];
    int mx, my, mz;
    image_masks(B, r, Rm, &mx, &my, &mz);
    gcnt[k] = __popc(mx) * __popc(my) * __popc(mz) - 1;
}

__global__ void k_ghost_fill(XRec *__restrict__ xrec, int64_t N, BoxP B, double Rm,
                             const int64_t *__restrict__ goff, int32_t *__restrict__ img_index) {
    int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= N) return;
    XRec r = xrec[k];
    int mx, my, mz;
    image_masks(B, r, Rm, &mx, &my, &mz);
    int64_t g = N + goff[k];
    for (int sx = -1; sx <= 1; ++sx)
        for (int sy = -1; sy <= 1; ++sy)
            for (int sz = -1; sz <= 1; ++sz) {
                int code = shift_code(sx, sy, sz);
                bool ok = ((mx >> (sx + 1)) & 1) && ((my >> (sy + 1)) & 1) && ((mz >> (sz + 1)) & 1);
                if (code == 13) { img_index[k * 27 + code] = (int32_t)k; continue; }
                if (!ok) { img_index[k * 27 + code] = -1; continue; }
                XRec q = r; q.sx = (int8_t)sx; q.sy = (int8_t)sy; q.sz = (int8_t)sz;
                xrec[g] = q;
                img_index[k * 27 + code] = (int32_t)g;
                ++g;
            }
}

struct Grid {
    BoxP B;
    int ncx, ncy, ncz;
    double R2, rc2;
};

__device__ __forceinline__ bool pair_in(const XRec &a, const XRec &b, double shx, double shy, double shz, double R2,
                                        double *d2out) {
    double dx = __dadd_rn(__dsub_rn(b.x, a.x), shx);
    double dy = __dadd_rn(__dsub_rn(b.y, a.y), shy);
    double dz = __dadd_rn(__dsub_rn(b.z, a.z), shz);
    double d2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
    *d2out = d2;
    return d2 < R2;
}

// Warp per atom over the 27-cell stencil. FILL = false: count; FILL = true: collect ext indices in
// shared memory (in ascending order where the stencil cells are distinct, else rank-sorted), write the CSR row.
template <bool FILL>
__global__ void __launch_bounds__(NB_WARPS * 32) k_nbr(const XRec *__restrict__ xrec, int64_t N, Grid g,
                                                       const int32_t *__restrict__ cell_rank,
                                                       const int64_t *__restrict__ cell_start,
                                                       const int32_t *__restrict__ img_index,
                                                       int32_t *__restrict__ row_cnt,
                                                       unsigned long long *__restrict__ n_rc_total,
                                                       const int64_t *__restrict__ row_ptr, int32_t *__restrict__ col,
                                                       int32_t *__restrict__ err_flag, uint32_t *__restrict__ mask, int MB) {
    // mask != nullptr: the count pass leaves the ballot word of every batch of 32 candidates (27 cells x MB batches per
    // atom), and the fill pass reads them back instead of gathering the records and testing the distances again
    __shared__ int32_t rowbuf[FILL ? NB_WARPS * ROWCAP : 1];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t i = (int64_t)blockIdx.x * NB_WARPS + warp;
    if (i >= N) return;
    const XRec me = xrec[i];
    int cx, cy, cz;
    cell_of(g.B, me.x, me.y, me.z, g.ncx, g.ncy, g.ncz, &cx, &cy, &cz);
    int cnt = 0, cnt_rc = 0;
    int32_t *buf = rowbuf + (FILL ? warp * ROWCAP : 0);
    // Fill pass with at least three cells per direction: the 27 stencil cells are distinct, so visiting first the
    // unshifted ones and then the shifted ones, each kind by ascending Morton rank, yields the row already sorted by
    // ext index (internal indices are cell-rank-major, image indices owner-major and all above N) -- no sort needed.
    const bool presorted = FILL && g.ncx >= 3 && g.ncy >= 3 && g.ncz >= 3;
    __shared__ int8_t order_s[FILL ? NB_WARPS : 1][32];
    // lane o < 27 looks up stencil cell o once (rank, first atom, atom count, shift code): one chain of two dependent
    // loads for the whole stencil, and the loop below gets them by shuffle, so its only loads are the candidates' records
    // (or the count pass's ballot words), fetched one batch ahead
    int l_c0 = 0, l_n = 0, l_code = 13, l_key = 0x7fffffff;
    if (lane < 27) {
        const int ox = lane / 9 - 1, oy = (lane / 3) % 3 - 1, oz = lane % 3 - 1;
        int ax = cx + ox, ay = cy + oy, az = cz + oz, sx = 0, sy = 0, sz = 0;
        if (ax < 0) { ax += g.ncx; sx = -1; } else if (ax >= g.ncx) { ax -= g.ncx; sx = 1; }
        if (ay < 0) { ay += g.ncy; sy = -1; } else if (ay >= g.ncy) { ay -= g.ncy; sy = 1; }
        if (az < 0) { az += g.ncz; sz = -1; } else if (az >= g.ncz) { az -= g.ncz; sz = 1; }
        const int key = cell_rank[(ax * g.ncy + ay) * g.ncz + az];
        const int64_t c0 = cell_start[key];
        l_c0 = (int)c0;
        l_n = (int)(cell_start[key + 1] - c0);
        l_code = shift_code(sx, sy, sz);
        l_key = key | (l_code != 13 ? 0x40000000 : 0);      // ncell <= 2^30
    }
    int l_o = lane;                                          // stencil cell visited at position `lane`
    if (FILL && presorted) {
        int r = 0;
        for (int q = 0; q < 27; ++q) r += __shfl_sync(0xffffffffu, l_key, q) < l_key;
        if (lane < 27) order_s[warp][r] = (int8_t)lane;
        __syncwarp();
        l_o = lane < 27 ? order_s[warp][lane] : lane;
    }
    // parameters in visiting order: lane p holds those of the p-th visited cell
    const int v_c0 = __shfl_sync(0xffffffffu, l_c0, l_o), v_n = __shfl_sync(0xffffffffu, l_n, l_o),
              v_code = __shfl_sync(0xffffffffu, l_code, l_o);
    const bool use_mask = FILL && mask != nullptr;
    const uint32_t *mrow = mask ? mask + (size_t)i * (27 * MB) : nullptr;
    XRec nxt = me;
    unsigned nxt_m = 0;
    // state of the cell being visited (warp-uniform)
    int oi = 0, bi = 0;
    int c0 = __shfl_sync(0xffffffffu, v_c0, 0), n = __shfl_sync(0xffffffffu, v_n, 0);
    int code = __shfl_sync(0xffffffffu, v_code, 0), o = __shfl_sync(0xffffffffu, l_o, 0);
    double shx, shy, shz;
    box_shift(g.B, (double)(code / 9 - 1), (double)((code / 3) % 3 - 1), (double)(code % 3 - 1), shx, shy, shz);
    if (use_mask) { if (n > 0) nxt_m = mrow[o * MB]; }
    else if (lane < n) nxt = xrec[c0 + lane];
    while (oi < 27) {
        const int k = 32 * bi + lane;                        // candidate k of the cell
        const int64_t j = (int64_t)c0 + k;
        const XRec cur = nxt;
        unsigned m = nxt_m;
        // next batch (of this cell, else the first one of the next cell) in flight while this one is tested
        const bool more = 32 * (bi + 1) < n;
        int c0n = c0, nn = n, coden = code, on = o;
        if (more) {
            if (use_mask) nxt_m = mrow[o * MB + bi + 1];
            else if (k + 32 < n) nxt = xrec[j + 32];
        } else if (oi + 1 < 27) {
            c0n = __shfl_sync(0xffffffffu, v_c0, oi + 1); nn = __shfl_sync(0xffffffffu, v_n, oi + 1);
            coden = __shfl_sync(0xffffffffu, v_code, oi + 1); on = __shfl_sync(0xffffffffu, l_o, oi + 1);
            if (use_mask) { if (nn > 0) nxt_m = mrow[on * MB]; }
            else if (lane < nn) nxt = xrec[c0n + lane];
        }
        if (n > 0) {                                         // warp-uniform: the batch holds candidates
            bool in = false, in_rc = false;
            if (use_mask) {
                in = (m >> lane) & 1u;
            } else {
                if (k < n && !(j == i && code == 13)) {
                    double d2;
                    in = pair_in(me, cur, shx, shy, shz, g.R2, &d2);
                    in_rc = d2 < g.rc2;
                }
                m = __ballot_sync(0xffffffffu, in);
                if (!FILL && mask && lane == 0) mask[(size_t)i * (27 * MB) + o * MB + bi] = m;
            }
            if (FILL) {
                if (in) {
                    const int slot = cnt + __popc(m & ((1u << lane) - 1));
                    const int32_t e = (code == 13) ? (int32_t)j : img_index[j * 27 + code];
                    if (e < 0) atomicOr(err_flag, 2);
                    if (slot < ROWCAP) buf[slot] = e;
                }
            } else {
                cnt_rc += __popc(__ballot_sync(0xffffffffu, in_rc));
            }
            cnt += __popc(m);
        }
        if (more) ++bi;
        else {
            ++oi; bi = 0;
            if (coden != code) box_shift(g.B, (double)(coden / 9 - 1), (double)((coden / 3) % 3 - 1), (double)(coden % 3 - 1), shx, shy, shz);
            c0 = c0n; n = nn; code = coden; o = on;
        }
    }
    if (!FILL) {
        if (lane == 0) {
            row_cnt[i] = cnt;
            if (cnt > ROWCAP) atomicOr(err_flag, 1);
            atomicAdd(n_rc_total, (unsigned long long)cnt_rc);
        }
        return;
    }
    __syncwarp();
    if (cnt > ROWCAP) return; // flagged in the count pass
    const int64_t base = row_ptr[i];
    if (presorted) {
        for (int e = lane; e < cnt; e += 32) col[base + e] = buf[e];
        return;
    }
    for (int e = lane; e < cnt; e += 32) {       // small boxes (a cell met with several shifts): rank sort
        const int32_t v = buf[e];
        int rank = 0;
        for (int q = 0; q < cnt; ++q) rank += (buf[q] < v);
        col[base + rank] = v;
    }
}

// rev[e]: for entry e = (i -> image of owner oj with shift S), the position of the entry
// (oj -> image of i with shift -S) in row oj (rows are sorted: binary search).
__global__ void __launch_bounds__(128) k_rev(const XRec *__restrict__ xrec, int64_t N,
                                             const int64_t *__restrict__ row_ptr, const int32_t *__restrict__ col,
                                             const int32_t *__restrict__ img_index, uint32_t *__restrict__ rev,
                                             int32_t *__restrict__ err_flag) {
    const int lane = threadIdx.x & 31;
    const int64_t i = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (i >= N) return;
    const int64_t r0 = row_ptr[i], r1 = row_ptr[i + 1];
    for (int64_t e = r0 + lane; e < r1; e += 32) {
        const int32_t j = col[e];
        const XRec rj = xrec[j];
        const int code = shift_code(rj.sx, rj.sy, rj.sz);
        const int32_t target = (code == 13) ? (int32_t)i : img_index[i * 27 + (26 - code)];
        int64_t lo = row_ptr[rj.owner], hi = row_ptr[rj.owner + 1];
        int64_t found = -1;
        while (lo < hi) {
            int64_t mid = (lo + hi) >> 1;
            int32_t v = col[mid];
            if (v == target) { found = mid; break; }
            if (v < target) lo = mid + 1; else hi = mid;
        }
        if (found < 0 || target < 0) { atomicOr(err_flag, 4); found = 0; }
        rev[e] = (uint32_t)found;
    }
}

__global__ void k_species_flags(const XRec *__restrict__ xrec, int64_t N, int s, int32_t *__restrict__ flag) {
    int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k < N) flag[k] = (xrec[k].species == s);
}
__global__ void k_species_scatter(const XRec *__restrict__ xrec, int64_t N, int s, const int64_t *__restrict__ off,
                                  int64_t base, int32_t *__restrict__ sp_list) {
    int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k < N && xrec[k].species == s) sp_list[base + off[k]] = (int32_t)k;
}

// Introspection: rows of selected atoms (caller indices) in the caller's order and frame, one warp per row.
// pass 0 (j_out == nullptr): cnt[k] = length of the row; pass 1: entries written from off[k] on.
__global__ void __launch_bounds__(128) k_export_rows(const XRec *__restrict__ xrec, const int64_t *__restrict__ row_ptr,
                                                     const int32_t *__restrict__ col, const int32_t *__restrict__ perm,
                                                     const int32_t *__restrict__ inv_perm,
                                                     const int32_t *__restrict__ wshift, int64_t n_sel,
                                                     const int64_t *__restrict__ atoms, int64_t *__restrict__ cnt,
                                                     const int64_t *__restrict__ off, int32_t *__restrict__ j_out,
                                                     int8_t *__restrict__ shift_out) {
    const int lane = threadIdx.x & 31;
    const int64_t k = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (k >= n_sel) return;
    const int64_t i = atoms[k], ki = inv_perm[i];
    const int64_t r0 = row_ptr[ki], r1 = row_ptr[ki + 1];
    if (!j_out) { if (lane == 0) cnt[k] = r1 - r0; return; }
    for (int64_t e = r0 + lane; e < r1; e += 32) {
        const XRec r = xrec[col[e]];
        const int32_t jc = perm[r.owner];
        const int64_t o = off[k] + (e - r0);
        j_out[o] = jc;
        shift_out[3 * o + 0] = (int8_t)(r.sx + wshift[3 * i + 0] - wshift[3 * (int64_t)jc + 0]);
        shift_out[3 * o + 1] = (int8_t)(r.sy + wshift[3 * i + 1] - wshift[3 * (int64_t)jc + 1]);
        shift_out[3 * o + 2] = (int8_t)(r.sz + wshift[3 * i + 2] - wshift[3 * (int64_t)jc + 2]);
    }
}

uint32_t morton3(uint32_t x, uint32_t y, uint32_t z) {
    auto spread = [](uint64_t v) {
        v &= 0x1fffff;
        v = (v | v << 32) & 0x1f00000000ffffULL;
        v = (v | v << 16) & 0x1f0000ff0000ffULL;
        v = (v | v << 8) & 0x100f00f00f00f00fULL;
        v = (v | v << 4) & 0x10c30c30c30c30c3ULL;
        v = (v | v << 2) & 0x1249249249249249ULL;
        return v;
    };
    return (uint32_t)(spread(x) | (spread(y) << 1) | (spread(z) << 2));
}

} // namespace

int neighbor_build(reann *h, const double *d_pos) {
    const int64_t N = h->N;
    const ModelDims &md = h->md;
    LaunchCtx ctx = h->ctx();
    const double R = md.rc + md.skin;
    const BoxP B = make_boxp(h->box_build);
    // cells: equal slices of the fractional coordinates, at least R between their faces
    Grid g{B, std::max(1, (int)floor(B.wa / R)), std::max(1, (int)floor(B.wb / R)),
           std::max(1, (int)floor(B.wc / R)), R * R, md.rc * md.rc};
    const int64_t ncell = (int64_t)g.ncx * g.ncy * g.ncz;
    if (ncell > (int64_t)1 << 30) return set_err(h, REANN_ERR_UNSUPPORTED, "too many cells");

    // cell -> Morton rank table (host; only when the grid changes)
    if (g.ncx != h->nc_cached[0] || g.ncy != h->nc_cached[1] || g.ncz != h->nc_cached[2]) {
        std::vector<uint64_t> keyed((size_t)ncell);
        for (int x = 0; x < g.ncx; ++x)
            for (int y = 0; y < g.ncy; ++y)
                for (int z = 0; z < g.ncz; ++z) {
                    uint64_t lin = ((uint64_t)x * g.ncy + y) * g.ncz + z;
                    keyed[lin] = ((uint64_t)morton3(x, y, z) << 32) | lin;
                }
        std::sort(keyed.begin(), keyed.end());
        std::vector<int32_t> rank((size_t)ncell);
        for (int64_t r = 0; r < ncell; ++r) rank[(size_t)(keyed[(size_t)r] & 0xffffffffu)] = (int32_t)r;
        RC(dev_ensure(h, h->cell_rank, sizeof(int32_t) * (size_t)ncell));
        CU(h, cudaMemcpyAsync(h->cell_rank.p, rank.data(), sizeof(int32_t) * (size_t)ncell, cudaMemcpyHostToDevice,
                              h->stream));
        CU(h, cudaStreamSynchronize(h->stream));
        h->nc_cached[0] = g.ncx; h->nc_cached[1] = g.ncy; h->nc_cached[2] = g.ncz;
    }
    const int TPB = 256;
    const size_t scan_n = (size_t)std::max<int64_t>(N, ncell) + 1;
    RC(dev_ensure(h, h->scan_ws, scan_workspace_bytes((int64_t)scan_n)));
    RC(dev_ensure(h, h->cell_start, sizeof(int64_t) * ((size_t)ncell + 1)));
    RC(dev_ensure(h, h->scratch_a, sizeof(int32_t) * scan_n));              // cellkey / gcnt / row_cnt / flags
    RC(dev_ensure(h, h->scratch_b, sizeof(int32_t) * 2 * ((size_t)ncell + 1))); // cell_count | cell_fill
    RC(dev_ensure(h, h->scratch_c, sizeof(int64_t) * (scan_n + 1)));        // goff / species offsets
    RC(dev_ensure(h, h->wshift, sizeof(int32_t) * 3 * (size_t)N));
    RC(dev_ensure(h, h->perm, sizeof(int32_t) * (size_t)N));
    RC(dev_ensure(h, h->inv_perm, sizeof(int32_t) * (size_t)N));
    RC(dev_ensure(h, h->pos_build, sizeof(double) * 3 * (size_t)N));
    RC(dev_ensure(h, h->img_index, sizeof(int32_t) * 27 * (size_t)N));
    RC(dev_ensure(h, h->row_ptr, sizeof(int64_t) * ((size_t)N + 1)));
    RC(dev_ensure(h, h->sp_list, sizeof(int32_t) * (size_t)N));
    RC(dev_ensure(h, h->xrec, sizeof(XRec) * (size_t)N)); // grown below once G is known

    int32_t *cellkey = (int32_t *)h->scratch_a.p;
    int32_t *cell_count = (int32_t *)h->scratch_b.p, *cell_fill = cell_count + ncell + 1;
    int32_t *flags = (int32_t *)h->flags.p;
    CU(h, cudaMemsetAsync(h->scratch_b.p, 0, sizeof(int32_t) * 2 * ((size_t)ncell + 1), h->stream));
    CU(h, cudaMemsetAsync(flags, 0, sizeof(int32_t) * 8, h->stream));

    // A1: wrap, cell key, counting sort in Morton cell order, deterministic inside each cell
    LAUNCH(ctx, k_wrap_cell, div_up(N, TPB), TPB, 0, d_pos, N, B, g.ncx, g.ncy, g.ncz,
           (const int32_t *)h->cell_rank.p, (int32_t *)h->wshift.p, cellkey, cell_count);
    LAUNCH(ctx, k_max_i32, div_up(ncell, TPB), TPB, 0, (const int32_t *)cell_count, ncell, flags + 6);
    exclusive_scan_i32_to_i64(ctx, cell_count, (int64_t *)h->cell_start.p, ncell, h->scan_ws.p);
    LAUNCH(ctx, k_scatter, div_up(N, TPB), TPB, 0, cellkey, N, (const int64_t *)h->cell_start.p, cell_fill,
           (int32_t *)h->perm.p);
    LAUNCH(ctx, k_sort_cells, div_up(ncell, 4), 128, 0, (int32_t *)h->perm.p, (const int64_t *)h->cell_start.p, ncell);
    LAUNCH(ctx, k_local_records, div_up(N, TPB), TPB, 0, (const int32_t *)h->perm.p, d_pos,
           (const int32_t *)h->wshift.p, (const int32_t *)h->species_caller.p, N, B, (XRec *)h->xrec.p,
           (int32_t *)h->inv_perm.p, (double *)h->pos_build.p);

    // A2: ghost / image map
    const double Rm = R + 1e-6 * std::max(B.ax, std::max(B.by, B.cz)) + 1e-9;
    int32_t *gcnt = (int32_t *)h->scratch_a.p;
    int64_t *goff = (int64_t *)h->scratch_c.p;
    LAUNCH(ctx, k_ghost_count, div_up(N, TPB), TPB, 0, (const XRec *)h->xrec.p, N, B, Rm, gcnt);
    exclusive_scan_i32_to_i64(ctx, gcnt, goff, N, h->scan_ws.p);
    int64_t G = 0;
    CU(h, cudaMemcpyAsync(&G, goff + N, sizeof(int64_t), cudaMemcpyDeviceToHost, h->stream));
    CU(h, cudaStreamSynchronize(h->stream));
    if (N + G >= ((int64_t)1 << COL_SPECIES_SHIFT))
        return set_err(h, REANN_ERR_UNSUPPORTED, "N_ext = %lld exceeds 2^27", (long long)(N + G));
    {   // grow xrec preserving the local records
        size_t need = sizeof(XRec) * (size_t)(N + G);
        if (h->xrec.bytes < need) {
            DevBuf nb;
            RC(dev_ensure(h, nb, need + need / 8));
            CU(h, cudaMemcpyAsync(nb.p, h->xrec.p, sizeof(XRec) * (size_t)N, cudaMemcpyDeviceToDevice, h->stream));
            CU(h, cudaStreamSynchronize(h->stream));
            cudaFree(h->xrec.p);
            h->bytes_device -= h->xrec.bytes;
            h->xrec = nb;
        }
    }
    h->G = G; h->n_ext = N + G;
    LAUNCH(ctx, k_ghost_fill, div_up(N, TPB), TPB, 0, (XRec *)h->xrec.p, N, B, Rm, (const int64_t *)goff,
           (int32_t *)h->img_index.p);

    // A3: count -> scan -> fill (+ row sort) -> reverse index
    // ballot words of the count pass for the fill pass: 27 x MB words per atom (MB = batches of 32 that cover the fullest
    // cell); skipped (the fill pass then repeats the pair tests) when they would take more than 4 GB
    int max_cell = 0;
    CU(h, cudaMemcpyAsync(&max_cell, flags + 6, sizeof(int32_t), cudaMemcpyDeviceToHost, h->stream));
    CU(h, cudaStreamSynchronize(h->stream));
    const int MB = std::max(1, (max_cell + 31) / 32);
    uint32_t *mask = nullptr;
    if ((size_t)N * 27 * MB * sizeof(uint32_t) <= ((size_t)4 << 30)) {
        RC(dev_ensure(h, h->nbr_mask, (size_t)N * 27 * MB * sizeof(uint32_t)));
        mask = (uint32_t *)h->nbr_mask.p;
    }
    int32_t *row_cnt = (int32_t *)h->scratch_a.p;
    unsigned long long *n_rc_total = (unsigned long long *)(flags + 4);
    LAUNCH(ctx, k_nbr<false>, div_up(N, NB_WARPS), NB_WARPS * 32, 0, (const XRec *)h->xrec.p, N, g,
           (const int32_t *)h->cell_rank.p, (const int64_t *)h->cell_start.p, (const int32_t *)h->img_index.p, row_cnt,
           n_rc_total, (const int64_t *)nullptr, (int32_t *)nullptr, flags, mask, MB);
    exclusive_scan_i32_to_i64(ctx, row_cnt, (int64_t *)h->row_ptr.p, N, h->scan_ws.p);
    int64_t E = 0;
    CU(h, cudaMemcpyAsync(&E, (int64_t *)h->row_ptr.p + N, sizeof(int64_t), cudaMemcpyDeviceToHost, h->stream));
    CU(h, cudaMemcpyAsync(h->h_flags, flags, sizeof(int32_t) * 8, cudaMemcpyDeviceToHost, h->stream));
    CU(h, cudaStreamSynchronize(h->stream));
    if (h->h_flags[0] & 1) return set_err(h, REANN_ERR_UNSUPPORTED, "a neighbour row exceeds %d entries", ROWCAP);
    if (E >= ((int64_t)1 << 32)) return set_err(h, REANN_ERR_UNSUPPORTED, "more than 2^32 list entries");
    h->E_list = E;
    h->E_rc_build = (int64_t)(*(unsigned long long *)(h->h_flags + 4));
    // list-sized buffers get 3 % head-room: the list length fluctuates from rebuild to rebuild, and a
    // cudaFree + cudaMalloc of a few hundred MB in the middle of an MD run costs tens of milliseconds
    const size_t e_cap = (size_t)std::max<int64_t>(E, 1) + (size_t)E / 32 + 1024;
    if (h->col.bytes < sizeof(int32_t) * (size_t)std::max<int64_t>(E, 1)) RC(dev_ensure(h, h->col, sizeof(int32_t) * e_cap));
    if (h->rev.bytes < sizeof(uint32_t) * (size_t)std::max<int64_t>(E, 1)) RC(dev_ensure(h, h->rev, sizeof(uint32_t) * e_cap));
    LAUNCH(ctx, k_nbr<true>, div_up(N, NB_WARPS), NB_WARPS * 32, 0, (const XRec *)h->xrec.p, N, g,
           (const int32_t *)h->cell_rank.p, (const int64_t *)h->cell_start.p, (const int32_t *)h->img_index.p,
           (int32_t *)nullptr, (unsigned long long *)nullptr, (const int64_t *)h->row_ptr.p, (int32_t *)h->col.p,
           flags, mask, MB);
    LAUNCH(ctx, k_rev, div_up(N, 4), 128, 0, (const XRec *)h->xrec.p, N, (const int64_t *)h->row_ptr.p,
           (const int32_t *)h->col.p, (const int32_t *)h->img_index.p, (uint32_t *)h->rev.p, flags);

    // species-grouped atom lists for the dense tiles (counts per species are fixed at create)
    int64_t base = 0;
    for (int s = 0; s < md.S; ++s) {
        int32_t *fl = (int32_t *)h->scratch_a.p;
        int64_t *off = (int64_t *)h->scratch_c.p;
        LAUNCH(ctx, k_species_flags, div_up(N, TPB), TPB, 0, (const XRec *)h->xrec.p, N, s, fl);
        exclusive_scan_i32_to_i64(ctx, fl, off, N, h->scan_ws.p);
        LAUNCH(ctx, k_species_scatter, div_up(N, TPB), TPB, 0, (const XRec *)h->xrec.p, N, s, (const int64_t *)off,
               base, (int32_t *)h->sp_list.p);
        base += h->species_count[(size_t)s];
    }
    CU(h, cudaMemcpyAsync(h->h_flags, flags, sizeof(int32_t) * 4, cudaMemcpyDeviceToHost, h->stream));
    CU(h, cudaStreamSynchronize(h->stream));
    if (h->h_flags[0] & 2) return set_err(h, REANN_ERR_CUDA, "internal: image index missing for a list entry");
    if (h->h_flags[0] & 4) return set_err(h, REANN_ERR_CUDA, "internal: reverse edge not found");
    CU(h, cudaGetLastError());
    return REANN_OK;
}

// Introspection (host assembly; not on the hot path): rows in caller order and caller frame,
// S_caller = S_wrapped + w_i - w_j with w = floor(x/L) at build.
int neighbor_export(reann *h, int64_t *n_edges, int64_t *row_ptr_out, int32_t *j_out, int8_t *shift_out) {
    if (!h->have_list) return set_err(h, REANN_ERR_NO_NEIGHBORS, "no neighbour list built yet");
    const int64_t N = h->N, E = h->E_list;
    if (n_edges) *n_edges = E;
    if (!row_ptr_out && !j_out && !shift_out) return REANN_OK;
    if (!row_ptr_out || !j_out || !shift_out) return set_err(h, REANN_ERR_ARG, "pass all three arrays or none");
    std::vector<int64_t> rp((size_t)N + 1);
    std::vector<int32_t> col((size_t)std::max<int64_t>(E, 1)), perm((size_t)N), wsh((size_t)3 * N);
    std::vector<XRec> xr((size_t)h->n_ext);
    CU(h, cudaStreamSynchronize(h->stream));
    CU(h, cudaMemcpy(rp.data(), h->row_ptr.p, sizeof(int64_t) * ((size_t)N + 1), cudaMemcpyDeviceToHost));
    CU(h, cudaMemcpy(col.data(), h->col.p, sizeof(int32_t) * (size_t)E, cudaMemcpyDeviceToHost));
    CU(h, cudaMemcpy(perm.data(), h->perm.p, sizeof(int32_t) * (size_t)N, cudaMemcpyDeviceToHost));
    CU(h, cudaMemcpy(wsh.data(), h->wshift.p, sizeof(int32_t) * 3 * (size_t)N, cudaMemcpyDeviceToHost));
    CU(h, cudaMemcpy(xr.data(), h->xrec.p, sizeof(XRec) * (size_t)h->n_ext, cudaMemcpyDeviceToHost));
    std::vector<int32_t> inv((size_t)N);
    for (int64_t k = 0; k < N; ++k) inv[(size_t)perm[(size_t)k]] = (int32_t)k;
    row_ptr_out[0] = 0;
    for (int64_t i = 0; i < N; ++i) {
        int64_t k = inv[(size_t)i];
        row_ptr_out[i + 1] = row_ptr_out[i] + (rp[(size_t)k + 1] - rp[(size_t)k]);
    }
    for (int64_t i = 0; i < N; ++i) {
        int64_t k = inv[(size_t)i], o = row_ptr_out[i];
        for (int64_t e = rp[(size_t)k]; e < rp[(size_t)k + 1]; ++e, ++o) {
            const XRec &r = xr[(size_t)col[(size_t)e]];
            int32_t jc = perm[(size_t)r.owner];
            j_out[o] = jc;
            shift_out[3 * o + 0] = (int8_t)(r.sx + wsh[3 * (size_t)i + 0] - wsh[3 * (size_t)jc + 0]);
            shift_out[3 * o + 1] = (int8_t)(r.sy + wsh[3 * (size_t)i + 1] - wsh[3 * (size_t)jc + 1]);
            shift_out[3 * o + 2] = (int8_t)(r.sz + wsh[3 * (size_t)i + 2] - wsh[3 * (size_t)jc + 2]);
        }
    }
    return REANN_OK;
}


// Rows of selected atoms only (for sampled pair-set parity on systems whose full list is too large to export).
int neighbor_export_rows(reann *h, int64_t n_sel, const int64_t *atoms, int64_t *row_ptr_out, int32_t *j_out,
                         int8_t *shift_out) {
    if (!h->have_list) return set_err(h, REANN_ERR_NO_NEIGHBORS, "no neighbour list built yet");
    if (n_sel < 0 || !atoms || !row_ptr_out || (!!j_out != !!shift_out)) return set_err(h, REANN_ERR_ARG, "bad argument");
    for (int64_t k = 0; k < n_sel; ++k)
        if (atoms[k] < 0 || atoms[k] >= h->N) return set_err(h, REANN_ERR_ARG, "atom index out of range");
    row_ptr_out[0] = 0;
    if (n_sel == 0) return REANN_OK;
    LaunchCtx ctx = h->ctx();
    DevBuf d_atoms, d_cnt, d_off, d_j, d_sh;
    auto cleanup = [&]() { for (DevBuf *b : {&d_atoms, &d_cnt, &d_off, &d_j, &d_sh}) if (b->p) { cudaFree(b->p); h->bytes_device -= b->bytes; b->p = nullptr; } };
#define XRC(call) do { int r_ = (call); if (r_ != REANN_OK) { cleanup(); return r_; } } while (0)
#define XCU(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { cleanup(); return set_err(h, REANN_ERR_CUDA, "%s: %s", #call, cudaGetErrorString(e_)); } } while (0)
    XRC(dev_ensure(h, d_atoms, sizeof(int64_t) * (size_t)n_sel));
    XRC(dev_ensure(h, d_cnt, sizeof(int64_t) * (size_t)n_sel));
    XRC(dev_ensure(h, d_off, sizeof(int64_t) * (size_t)n_sel));
    XCU(cudaMemcpyAsync(d_atoms.p, atoms, sizeof(int64_t) * (size_t)n_sel, cudaMemcpyHostToDevice, h->stream));
    LAUNCH(ctx, k_export_rows, div_up(n_sel, 4), 128, 0, (const XRec *)h->xrec.p, (const int64_t *)h->row_ptr.p,
           (const int32_t *)h->col.p, (const int32_t *)h->perm.p, (const int32_t *)h->inv_perm.p,
           (const int32_t *)h->wshift.p, n_sel, (const int64_t *)d_atoms.p, (int64_t *)d_cnt.p, (const int64_t *)nullptr,
           (int32_t *)nullptr, (int8_t *)nullptr);
    std::vector<int64_t> cnt((size_t)n_sel);
    XCU(cudaMemcpyAsync(cnt.data(), d_cnt.p, sizeof(int64_t) * (size_t)n_sel, cudaMemcpyDeviceToHost, h->stream));
    XCU(cudaStreamSynchronize(h->stream));
    for (int64_t k = 0; k < n_sel; ++k) row_ptr_out[k + 1] = row_ptr_out[k] + cnt[(size_t)k];
    const int64_t tot = row_ptr_out[n_sel];
    if (j_out && tot > 0) {
        XRC(dev_ensure(h, d_j, sizeof(int32_t) * (size_t)tot));
        XRC(dev_ensure(h, d_sh, 3 * (size_t)tot));
        XCU(cudaMemcpyAsync(d_off.p, row_ptr_out, sizeof(int64_t) * (size_t)n_sel, cudaMemcpyHostToDevice, h->stream));
        LAUNCH(ctx, k_export_rows, div_up(n_sel, 4), 128, 0, (const XRec *)h->xrec.p, (const int64_t *)h->row_ptr.p,
               (const int32_t *)h->col.p, (const int32_t *)h->perm.p, (const int32_t *)h->inv_perm.p,
               (const int32_t *)h->wshift.p, n_sel, (const int64_t *)d_atoms.p, (int64_t *)d_cnt.p,
               (const int64_t *)d_off.p, (int32_t *)d_j.p, (int8_t *)d_sh.p);
        XCU(cudaMemcpyAsync(j_out, d_j.p, sizeof(int32_t) * (size_t)tot, cudaMemcpyDeviceToHost, h->stream));
        XCU(cudaMemcpyAsync(shift_out, d_sh.p, 3 * (size_t)tot, cudaMemcpyDeviceToHost, h->stream));
        XCU(cudaStreamSynchronize(h->stream));
    }
    cleanup();
#undef XRC
#undef XCU
    return REANN_OK;
}
