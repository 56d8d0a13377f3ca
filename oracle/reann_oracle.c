/*
 * reann_oracle.c -- float64 CPU ORACLE for the REANN energy+force path.
 *
 * TEST INFRASTRUCTURE ONLY. Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call this file. It shares
 * no code with paper_2505_06711_b200/ (the CUDA path); neither includes the other.
 *
 * It is the paper's recursion written out step by step, in the paper's order, with no
 * blocking, fusion or reordering (SURVEY.md 8(c) holds the readings A-1..A-18 of the
 * points where PAPER.md is silent or garbled; DESIGN.md lists them again):
 *
 *   Eq. 1   rho_i = sum_l sum_{lx+ly+lz=l} l!/(lx!ly!lz!) [ sum_{j!=i} c_j G_j(r_ij) ]^2
 *   Eq. 2   c_i^t = M_i^{t-1}[ rho_i^{t-1} ],  1 <= t <= T-1;  last atomic NN -> E_i (:43)
 *   Eqs. 3-5   F_k = -dE/dr_k by the chain rule through all T layers
 *                               (dc^0/dr = 0), written as vector-Jacobian
 *                               products, SURVEY.md Appendix B.
 *
 * Pins (tests/test_oracle_*.py, all "-m 'not gpu'"): brute-force O(N^2*27) neighbour sets;
 * an independent NumPy pair-form of Eq. 1 via the multinomial theorem; NumPy matmul MLP;
 * central finite differences for F and the virial; translation / rotation / permutation
 * invariance; 2x2x2 supercell; cluster additivity; receptive field T*rc; fcc symmetry.
 * Absolute E/F values on the synthetic configs have no external reference:
 * "parity unpinned" for those beyond the pins above (the paper prints no worked example).
 *
 * Build: gcc -O2 -std=c11 -ffp-contract=off -fopenmp -shared -fPIC reann_oracle.c -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_OK 0
#define ORC_ERR_ARG 1
#define ORC_ERR_WEIGHTS 2
#define ORC_ERR_BOX 3
#define ORC_ERR_MEM 6
#define ORC_ERR_UNSUPPORTED 7

#define MAXL 5
#define ORC_PI 3.14159265358979323846
#define MAXA 56 /* (L+1)(L+2)(L+3)/6 at L=5 */

typedef struct {
    int S, T, L, nphi, norb, H1c, H2c, H1e, H2e, act;
    double rc;
    const double *rcen, *alpha, *c0, *Wc;
    const double **W1, **b1, **W2, **b2, **W3, **b3; /* [T*S] */
    int Na;
    int lx[MAXA], ly[MAXA], lz[MAXA], la[MAXA];
    double mu[MAXA]; /* l!/(lx! ly! lz!), Eq. 1 */
} model_t;

static double factorial(int n) { double f = 1; for (int i = 2; i <= n; ++i) f *= i; return f; }

static void model_free(model_t *m) {
    free((void *)m->W1); free((void *)m->b1); free((void *)m->W2);
    free((void *)m->b2); free((void *)m->W3); free((void *)m->b3);
}

/* Parse the weights blob (layout: gen/weights.py docstring). */
static int model_parse(model_t *m, const void *blob, size_t nbytes) {
    memset(m, 0, sizeof(*m));
    if (!blob || nbytes < 64) return ORC_ERR_WEIGHTS;
    const unsigned char *p = (const unsigned char *)blob;
    if (memcmp(p, "REANNB2\0", 8) != 0) return ORC_ERR_WEIGHTS;
    uint32_t h[12];
    memcpy(h, p + 8, sizeof(h));
    if (h[0] != 1) return ORC_ERR_WEIGHTS;
    m->S = (int)h[1]; m->T = (int)h[2]; m->L = (int)h[3]; m->nphi = (int)h[4]; m->norb = (int)h[5];
    m->H1c = (int)h[6]; m->H2c = (int)h[7]; m->H1e = (int)h[8]; m->H2e = (int)h[9]; m->act = (int)h[10];
    memcpy(&m->rc, p + 56, 8);
    if (m->S < 1 || m->T < 1 || m->L < 0 || m->L > MAXL || m->nphi < 1 || m->nphi > 256 || m->norb < 1 ||
        m->act != 0 ||
        !(m->rc > 0))
        return ORC_ERR_WEIGHTS;
    const double *q = (const double *)(p + 64);
    size_t avail = (nbytes - 64) / 8, used = 0;
#define TAKE(dst, n) do { size_t n_ = (size_t)(n); if (used + n_ > avail) { model_free(m); return ORC_ERR_WEIGHTS; } \
                          (dst) = q + used; used += n_; } while (0)
    int TS = m->T * m->S;
    m->W1 = calloc(TS, sizeof(double *)); m->b1 = calloc(TS, sizeof(double *));
    m->W2 = calloc(TS, sizeof(double *)); m->b2 = calloc(TS, sizeof(double *));
    m->W3 = calloc(TS, sizeof(double *)); m->b3 = calloc(TS, sizeof(double *));
    TAKE(m->rcen, (size_t)m->T * m->S * m->nphi);
    TAKE(m->alpha, (size_t)m->T * m->S * m->nphi);
    TAKE(m->c0, (size_t)m->S * m->nphi);
    TAKE(m->Wc, (size_t)m->T * (m->L + 1) * m->nphi * m->norb);
    for (int t = 0; t < m->T; ++t) {
        int last = (t == m->T - 1);
        int H1 = last ? m->H1e : m->H1c, H2 = last ? m->H2e : m->H2c, out = last ? 1 : m->nphi;
        for (int s = 0; s < m->S; ++s) {
            int k = t * m->S + s;
            TAKE(m->W1[k], (size_t)m->norb * H1); TAKE(m->b1[k], H1);
            TAKE(m->W2[k], (size_t)H1 * H2);      TAKE(m->b2[k], H2);
            TAKE(m->W3[k], (size_t)H2 * out);     TAKE(m->b3[k], out);
        }
    }
#undef TAKE
    if (used != avail || (nbytes - 64) % 8 != 0) { model_free(m); return ORC_ERR_WEIGHTS; }
    /* Cartesian monomials a = (lx,ly,lz), lx+ly+lz = l <= L, with multinomial weight (Eq. 1) */
    int a = 0;
    for (int l = 0; l <= m->L; ++l)
        for (int lx = l; lx >= 0; --lx)
            for (int ly = l - lx; ly >= 0; --ly) {
                int lz = l - lx - ly;
                m->lx[a] = lx; m->ly[a] = ly; m->lz[a] = lz; m->la[a] = l;
                m->mu[a] = factorial(l) / (factorial(lx) * factorial(ly) * factorial(lz));
                ++a;
            }
    m->Na = a;
    return ORC_OK;
}

/* ------------------------------------------------------------------------------------------
 * Edges (readings A-12, A-13, A-15)
 *   E = {(i, j, S): S in Z^3, (j,S) != (i,0), |r_j + S o box - r_i| < R}, strict "<" on d^2,
 *   arithmetic: wrap x <- x - floor(x/L) L; d = (x_j - x_i) + S L; d2 = (dx dx + dy dy) + dz dz (orthorhombic box;
 *   the triclinic form is written out at wrap_all() and pair_test()).
 * ---------------------------------------------------------------------------------------- */
typedef struct { int32_t j; int32_t S[3]; double d[3]; } edge_t;
typedef struct { int64_t n; int64_t *off; edge_t *e; double *xw; int32_t *w; } edges_t;

static void edges_free(edges_t *E) { free(E->off); free(E->e); free(E->xw); free(E->w); memset(E, 0, sizeof(*E)); }

/* Box: row-major lattice vectors a = box9[0..2], b = box9[3..5], c = box9[6..8] in the lower-triangular form
 * a = (ax, 0, 0), b = (bx, by, 0), c = (cx, cy, cz) with ax, by, cz > 0 (orthorhombic: bx = cx = cy = 0; any cell can be
 * brought to this form by a rotation). H = {ax, bx, by, cx, cy, cz}; wd[d] = distance between the two faces of the cell
 * that are spanned by the other two lattice vectors: images with S in {-1,0,1}^3 of WRAPPED atoms are enough when
 * every wd[d] >= R (a point within R of the cell is less than one period away in every fractional coordinate). */
static int box_params(const double *box9, double H[6], double wd[3]) {
    if (box9[1] != 0.0 || box9[2] != 0.0 || box9[5] != 0.0) return ORC_ERR_UNSUPPORTED; /* not lower-triangular */
    H[0] = box9[0]; H[1] = box9[3]; H[2] = box9[4]; H[3] = box9[6]; H[4] = box9[7]; H[5] = box9[8];
    if (!(H[0] > 0) || !(H[2] > 0) || !(H[5] > 0)) return ORC_ERR_BOX;
    const double ax = H[0], bx = H[1], by = H[2], cx = H[3], cy = H[4], cz = H[5];
    const double n0 = by * cz, n1 = -bx * cz, n2 = bx * cy - by * cx;       /* b x c */
    wd[0] = ax * by * cz / sqrt(n0 * n0 + n1 * n1 + n2 * n2);
    wd[1] = by * cz / sqrt(cy * cy + cz * cz);                                /* a x c = (0, -ax cz, ax cy) */
    wd[2] = cz;
    return ORC_OK;
}

/* Wrapping (reading A-15, extended to a triclinic cell in DESIGN.md B-9): fractional coordinates by back substitution,
 *   sc = z / cz;  sb = (y - sc cy) / by;  sa = ((x - sb bx) - sc cx) / ax;   w = floor(s)  (whole periods, per lattice vector)
 * and the wrapped position is x - ((wa ax + wb bx) + wc cx), y - (wb by + wc cy), z - wc cz. For an orthorhombic box
 * this is x - floor(x / L) L, bit for bit. */
static void wrap_all(const double *pos, int64_t N, const double H[6], double *xw, int32_t *w) {
    const double ax = H[0], bx = H[1], by = H[2], cx = H[3], cy = H[4], cz = H[5];
    for (int64_t i = 0; i < N; ++i) {
        const double x = pos[3 * i], y = pos[3 * i + 1], z = pos[3 * i + 2];
        const double sc = z / cz;
        const double sb = (y - sc * cy) / by;
        const double sa = ((x - sb * bx) - sc * cx) / ax;
        const double fa = floor(sa), fb = floor(sb), fc = floor(sc);
        w[3 * i] = (int32_t)fa; w[3 * i + 1] = (int32_t)fb; w[3 * i + 2] = (int32_t)fc;
        xw[3 * i] = x - ((fa * ax + fb * bx) + fc * cx);
        xw[3 * i + 1] = y - (fb * by + fc * cy);
        xw[3 * i + 2] = z - fc * cz;
    }
}

/* d = (x_j - x_i) + S . box with S . box = ((S0 ax + S1 bx) + S2 cx, S1 by + S2 cy, S2 cz) */
static inline int pair_test(const double *xi, const double *xj, const int S[3], const double H[6],
                            double R2, double d[3]) {
    d[0] = (xj[0] - xi[0]) + ((S[0] * H[0] + S[1] * H[1]) + S[2] * H[3]);
    d[1] = (xj[1] - xi[1]) + (S[1] * H[2] + S[2] * H[4]);
    d[2] = (xj[2] - xi[2]) + S[2] * H[5];
    double d2 = (d[0] * d[0] + d[1] * d[1]) + d[2] * d[2];
    return d2 < R2;
}

/* mode 0: O(N^2 * 27) brute force over S in {-1,0,1}^3; mode 1: cell list (cells in fractional coordinates, at least R
 * wide between their faces). Both need wd[d] >= R.
 * sel == NULL: rows of all N atoms (row k = atom k); else rows of the n_sel atoms sel[k] only (row k = atom
 * sel[k]; the same pair test over the same candidates -- used for sampled pair-set parity on systems whose
 * full list would not fit the host). */
static int build_edges_sel(const double *pos, int64_t N, const double *box9, double R, int mode, edges_t *E,
                           const int64_t *sel, int64_t n_sel) {
    memset(E, 0, sizeof(*E));
    double H[6], wd[3];
    int rc_ = box_params(box9, H, wd);
    if (rc_) return rc_;
    for (int d = 0; d < 3; ++d) if (wd[d] < R) return ORC_ERR_BOX;
    const double R2 = R * R;
    E->xw = malloc(sizeof(double) * 3 * (size_t)(N > 0 ? N : 1));
    E->w = malloc(sizeof(int32_t) * 3 * (size_t)(N > 0 ? N : 1));
    const int64_t n_rows = sel ? n_sel : N;
    E->off = calloc((size_t)n_rows + 1, sizeof(int64_t));
    if (!E->xw || !E->w || !E->off) return ORC_ERR_MEM;
    wrap_all(pos, N, H, E->xw, E->w);
    int nc[3]; int64_t ncell = 1;
    int32_t *cell_of = NULL; int64_t *cstart = NULL; int32_t *catoms = NULL;
    if (mode == 1) {
        for (int d = 0; d < 3; ++d) { nc[d] = (int)floor(wd[d] / R); if (nc[d] < 1) nc[d] = 1; ncell *= nc[d]; }
        cell_of = malloc(sizeof(int32_t) * 3 * (size_t)(N > 0 ? N : 1));
        cstart = calloc((size_t)ncell + 1, sizeof(int64_t));
        catoms = malloc(sizeof(int32_t) * (size_t)(N > 0 ? N : 1));
        if (!cell_of || !cstart || !catoms) return ORC_ERR_MEM;
        for (int64_t i = 0; i < N; ++i) {
            int64_t lin = 0;
            /* fractional coordinates of the wrapped position: x = sa a + sb b + sc c */
            double sf[3];
            sf[2] = E->xw[3 * i + 2] / H[5];
            sf[1] = (E->xw[3 * i + 1] - sf[2] * H[4]) / H[2];
            sf[0] = ((E->xw[3 * i] - sf[1] * H[1]) - sf[2] * H[3]) / H[0];
            for (int d = 0; d < 3; ++d) {
                int c = (int)floor(sf[d] * nc[d]);
                if (c >= nc[d]) c = nc[d] - 1;
                if (c < 0) c = 0;
                cell_of[3 * i + d] = c;
                lin = lin * nc[d] + c;
            }
            cstart[lin + 1]++;
        }
        for (int64_t c = 0; c < ncell; ++c) cstart[c + 1] += cstart[c];
        int64_t *fill = malloc(sizeof(int64_t) * (size_t)ncell);
        memcpy(fill, cstart, sizeof(int64_t) * (size_t)ncell);
        for (int64_t i = 0; i < N; ++i) {
            int64_t lin = ((int64_t)cell_of[3 * i] * nc[1] + cell_of[3 * i + 1]) * nc[2] + cell_of[3 * i + 2];
            catoms[fill[lin]++] = (int32_t)i;
        }
        free(fill);
    }
    /* two passes: count, then fill */
    for (int pass = 0; pass < 2; ++pass) {
        if (pass == 1) {
            int64_t tot = 0;
            for (int64_t i = 0; i < n_rows; ++i) { int64_t c = E->off[i + 1]; E->off[i + 1] = tot + c; tot += c; }
            /* off[i+1] now holds end of row i; off[0] = 0 */
            E->n = tot;
            E->e = malloc(sizeof(edge_t) * (size_t)(tot > 0 ? tot : 1));
            if (!E->e) return ORC_ERR_MEM;
        }
#pragma omp parallel for schedule(dynamic, 64)
        for (int64_t row = 0; row < n_rows; ++row) {
            const int64_t i = sel ? sel[row] : row;
            int64_t cnt = 0;
            int64_t base = (pass == 1) ? (row == 0 ? 0 : E->off[row]) : 0;
            const double *xi = E->xw + 3 * i;
            double d[3];
            if (mode == 0) {
                for (int64_t j = 0; j < N; ++j)
                    for (int sx = -1; sx <= 1; ++sx) for (int sy = -1; sy <= 1; ++sy) for (int sz = -1; sz <= 1; ++sz) {
                        if (j == i && sx == 0 && sy == 0 && sz == 0) continue;
                        int S[3] = {sx, sy, sz};
                        if (pair_test(xi, E->xw + 3 * j, S, H, R2, d)) {
                            if (pass == 1) { edge_t *e = &E->e[base + cnt]; e->j = (int32_t)j;
                                e->S[0] = sx; e->S[1] = sy; e->S[2] = sz; e->d[0] = d[0]; e->d[1] = d[1]; e->d[2] = d[2]; }
                            ++cnt;
                        }
                    }
            } else {
                for (int ox = -1; ox <= 1; ++ox) for (int oy = -1; oy <= 1; ++oy) for (int oz = -1; oz <= 1; ++oz) {
                    int o[3] = {ox, oy, oz}, S[3], cc[3];
                    for (int dd = 0; dd < 3; ++dd) {
                        int c = cell_of[3 * i + dd] + o[dd]; S[dd] = 0;
                        if (c < 0) { c += nc[dd]; S[dd] = -1; } else if (c >= nc[dd]) { c -= nc[dd]; S[dd] = 1; }
                        cc[dd] = c;
                    }
                    int64_t lin = ((int64_t)cc[0] * nc[1] + cc[1]) * nc[2] + cc[2];
                    for (int64_t q = cstart[lin]; q < cstart[lin + 1]; ++q) {
                        int64_t j = catoms[q];
                        if (j == i && S[0] == 0 && S[1] == 0 && S[2] == 0) continue;
                        if (pair_test(xi, E->xw + 3 * j, S, H, R2, d)) {
                            if (pass == 1) { edge_t *e = &E->e[base + cnt]; e->j = (int32_t)j;
                                e->S[0] = S[0]; e->S[1] = S[1]; e->S[2] = S[2]; e->d[0] = d[0]; e->d[1] = d[1]; e->d[2] = d[2]; }
                            ++cnt;
                        }
                    }
                }
            }
            if (pass == 0) E->off[row + 1] = cnt;
        }
    }
    free(cell_of); free(cstart); free(catoms);
    return ORC_OK;
}
static int build_edges(const double *pos, int64_t N, const double *box9, double R, int mode, edges_t *E) {
    return build_edges_sel(pos, N, box9, R, mode, E, NULL, 0);
}

static int cmp_row5(const void *a, const void *b) {
    const int32_t *x = a, *y = b;
    for (int k = 0; k < 5; ++k) if (x[k] != y[k]) return x[k] < y[k] ? -1 : 1;
    return 0;
}

/* Neighbour oracle: rows (i, j, Sx, Sy, Sz) in the CALLER's frame (positions as given, not
 * wrapped): r_j + S o box - r_i is the edge vector. Sorted lexicographically.
 * With w = floor(x/L): S_caller = S_wrapped + w_i - w_j.
 * Returns the number of edges (>= 0) or -(error code). Writes at most `cap` rows. */
int64_t oracle_neighbors(const double *pos, int64_t N, const double *box9, double R, int mode,
                         int32_t *rows, int64_t cap) {
    edges_t E;
    int rc_ = build_edges(pos, N, box9, R, mode, &E);
    if (rc_) { edges_free(&E); return -(int64_t)rc_; }
    int64_t n = E.n;
    if (rows && cap >= n) {
        for (int64_t i = 0; i < N; ++i)
            for (int64_t q = E.off[i]; q < E.off[i + 1]; ++q) {
                edge_t *e = &E.e[q]; int32_t *r = rows + 5 * q;
                r[0] = (int32_t)i; r[1] = e->j;
                for (int d = 0; d < 3; ++d) r[2 + d] = e->S[d] + E.w[3 * i + d] - E.w[3 * e->j + d];
            }
        qsort(rows, (size_t)n, 5 * sizeof(int32_t), cmp_row5);
    }
    edges_free(&E);
    return n;
}

/* The same rows for the selected atoms sel[0..n_sel) only (cell list): rows (i, j, Sx, Sy, Sz), caller frame,
 * sorted; row_ptr[n_sel+1] gives each selected atom's slice after sorting by (i, ...) -- sel must be
 * strictly ascending so that the sorted order is the selection order. Returns the row count or -(error). */
int64_t oracle_neighbor_rows(const double *pos, int64_t N, const double *box9, double R, const int64_t *sel,
                             int64_t n_sel, int64_t *row_ptr, int32_t *rows, int64_t cap) {
    for (int64_t k = 0; k < n_sel; ++k)
        if (sel[k] < 0 || sel[k] >= N || (k > 0 && sel[k] <= sel[k - 1])) return -(int64_t)ORC_ERR_ARG;
    edges_t E;
    int rc_ = build_edges_sel(pos, N, box9, R, 1, &E, sel, n_sel);
    if (rc_) { edges_free(&E); return -(int64_t)rc_; }
    int64_t n = E.n;
    if (row_ptr) memcpy(row_ptr, E.off, sizeof(int64_t) * (size_t)(n_sel + 1));
    if (rows && cap >= n) {
        for (int64_t k = 0; k < n_sel; ++k)
            for (int64_t q = E.off[k]; q < E.off[k + 1]; ++q) {
                edge_t *e = &E.e[q]; int32_t *r = rows + 5 * q;
                const int64_t i = sel[k];
                r[0] = (int32_t)i; r[1] = e->j;
                for (int d = 0; d < 3; ++d) r[2 + d] = e->S[d] + E.w[3 * i + d] - E.w[3 * e->j + d];
            }
        qsort(rows, (size_t)n, 5 * sizeof(int32_t), cmp_row5);
    }
    edges_free(&E);
    return n;
}

/* ------------------------------------------------------------------------------------------
 * Per-edge functions (readings A-4, A-5)
 *   R_n(r) = exp(-alpha_n (r - r_n)^2) f_c(r),  f_c(r) = (1 + cos(pi r / rc)) / 2  (r < rc)
 *   A_a(r_vec) = x^lx y^ly z^lz  (raw Cartesian components)
 * ---------------------------------------------------------------------------------------- */
static inline double fcut(double r, double rc) { return r < rc ? 0.5 * (1.0 + cos(ORC_PI * r / rc)) : 0.0; }
static inline double dfcut(double r, double rc) { return r < rc ? -0.5 * (ORC_PI / rc) * sin(ORC_PI * r / rc) : 0.0; }

static void powers(const double d[3], int L, double px[MAXL + 1], double py[MAXL + 1], double pz[MAXL + 1]) {
    px[0] = py[0] = pz[0] = 1.0;
    for (int k = 1; k <= L; ++k) { px[k] = px[k - 1] * d[0]; py[k] = py[k - 1] * d[1]; pz[k] = pz[k - 1] * d[2]; }
}
static void monomials(const model_t *m, const double d[3], double *A) {
    double px[MAXL + 1], py[MAXL + 1], pz[MAXL + 1];
    powers(d, m->L, px, py, pz);
    for (int a = 0; a < m->Na; ++a) A[a] = px[m->lx[a]] * py[m->ly[a]] * pz[m->lz[a]];
}
static void monomial_grads(const model_t *m, const double d[3], double (*dA)[3]) {
    double px[MAXL + 1], py[MAXL + 1], pz[MAXL + 1];
    powers(d, m->L, px, py, pz);
    for (int a = 0; a < m->Na; ++a) {
        int lx = m->lx[a], ly = m->ly[a], lz = m->lz[a];
        dA[a][0] = lx ? lx * px[lx - 1] * py[ly] * pz[lz] : 0.0;
        dA[a][1] = ly ? ly * px[lx] * py[ly - 1] * pz[lz] : 0.0;
        dA[a][2] = lz ? lz * px[lx] * py[ly] * pz[lz - 1] : 0.0;
    }
}

static inline double silu(double z) { return z / (1.0 + exp(-z)); }
static inline double dsilu(double z) { double s = 1.0 / (1.0 + exp(-z)); return s * (1.0 + z * (1.0 - s)); }

/* Per-atom dense part of layer t:
 *   d[a][m] = sum_n Wc[t][l(a)][n][m] b[n][a];  rho[m] = sum_a mu_a d[a][m]^2      (Eq. 1)
 *   out = W3^T SiLU(W2^T SiLU(W1^T rho + b1) + b2) + b3                             (Eq. 2 / E_i)
 * If outbar != NULL also the reverse pass: rhobar, dbar = 2 mu d rhobar, bbar = Wc dbar. */
static void atom_dense(const model_t *m, int t, int s, const double *b, double *out, double *rho_out,
                       const double *outbar, double *bbar, double *work) {
    const int nphi = m->nphi, Na = m->Na, norb = m->norb;
    const int last = (t == m->T - 1);
    const int H1 = last ? m->H1e : m->H1c, H2 = last ? m->H2e : m->H2c, nout = last ? 1 : nphi;
    const int k = t * m->S + s;
    double *d = work;                       /* [Na][norb] */
    double *rho = d + (size_t)Na * norb;    /* [norb] */
    double *z1 = rho + norb, *h1 = z1 + H1, *z2 = h1 + H1, *h2 = z2 + H2;
    double *z2bar = h2 + H2, *z1bar = z2bar + H2, *rhobar = z1bar + H1;   /* [H2],[H1],[norb] */
    for (int mm = 0; mm < norb; ++mm) rho[mm] = 0.0;
    for (int a = 0; a < Na; ++a) {
        double *da = d + (size_t)a * norb;
        const double *W = m->Wc + ((size_t)t * (m->L + 1) + m->la[a]) * nphi * norb;
        for (int mm = 0; mm < norb; ++mm) da[mm] = 0.0;
        for (int n = 0; n < nphi; ++n) {
            const double bna = b[n * Na + a];
            const double *Wn = W + (size_t)n * norb;
            for (int mm = 0; mm < norb; ++mm) da[mm] += Wn[mm] * bna;
        }
        for (int mm = 0; mm < norb; ++mm) rho[mm] += m->mu[a] * (da[mm] * da[mm]);
    }
    if (rho_out) memcpy(rho_out, rho, sizeof(double) * norb);
    const double *W1 = m->W1[k], *W2 = m->W2[k], *W3 = m->W3[k];
    for (int h = 0; h < H1; ++h) z1[h] = m->b1[k][h];
    for (int mm = 0; mm < norb; ++mm) for (int h = 0; h < H1; ++h) z1[h] += W1[(size_t)mm * H1 + h] * rho[mm];
    for (int h = 0; h < H1; ++h) h1[h] = silu(z1[h]);
    for (int h = 0; h < H2; ++h) z2[h] = m->b2[k][h];
    for (int g = 0; g < H1; ++g) for (int h = 0; h < H2; ++h) z2[h] += W2[(size_t)g * H2 + h] * h1[g];
    for (int h = 0; h < H2; ++h) h2[h] = silu(z2[h]);
    if (out) {
        for (int o = 0; o < nout; ++o) out[o] = m->b3[k][o];
        for (int g = 0; g < H2; ++g) for (int o = 0; o < nout; ++o) out[o] += W3[(size_t)g * nout + o] * h2[g];
    }
    if (!outbar) return;
    for (int g = 0; g < H2; ++g) {
        double acc = 0.0;
        for (int o = 0; o < nout; ++o) acc += W3[(size_t)g * nout + o] * outbar[o];
        z2bar[g] = acc * dsilu(z2[g]);
    }
    for (int g = 0; g < H1; ++g) {
        double acc = 0.0;
        for (int h = 0; h < H2; ++h) acc += W2[(size_t)g * H2 + h] * z2bar[h];
        z1bar[g] = acc * dsilu(z1[g]);
    }
    for (int mm = 0; mm < norb; ++mm) {
        double acc = 0.0;
        for (int h = 0; h < H1; ++h) acc += W1[(size_t)mm * H1 + h] * z1bar[h];
        rhobar[mm] = acc;
    }
    for (int a = 0; a < Na; ++a) {
        const double *da = d + (size_t)a * norb;
        const double *W = m->Wc + ((size_t)t * (m->L + 1) + m->la[a]) * nphi * norb;
        for (int n = 0; n < nphi; ++n) {
            const double *Wn = W + (size_t)n * norb;
            double acc = 0.0;
            for (int mm = 0; mm < norb; ++mm) acc += Wn[mm] * (2.0 * m->mu[a] * da[mm] * rhobar[mm]);
            bbar[n * Na + a] = acc;
        }
    }
}

static size_t dense_work_doubles(const model_t *m) {
    int H1 = m->H1c > m->H1e ? m->H1c : m->H1e, H2 = m->H2c > m->H2e ? m->H2c : m->H2e;
    return (size_t)m->Na * m->norb + 2 * (size_t)m->norb + 3 * (size_t)H1 + 3 * (size_t)H2 + 16;
}

/* E, F, virial for one configuration.
 * Optional dumps (NULL to skip): Ei[N]; c_out[T][N][nphi] (c^t, t=0..T-1); b_out[T][N][nphi*Na];
 * rho_out[T][N][norb]. do_forces = 0 skips the reverse pass (F, virial untouched).
 * Returns 0 or an error code. */
int oracle_energy_forces(const void *blob, size_t nbytes, const int32_t *species, int64_t N,
                         const double *pos, const double *box9, int do_forces,
                         double *E_out, double *F, double *virial, double *Ei,
                         double *c_out, double *b_out, double *rho_out, int nthreads) {
    model_t M;
    int rc_ = model_parse(&M, blob, nbytes);
    if (rc_) return rc_;
    if (N < 0 || !species || !pos || !box9) { model_free(&M); return ORC_ERR_ARG; }
    for (int64_t i = 0; i < N; ++i) if (species[i] < 0 || species[i] >= M.S) { model_free(&M); return ORC_ERR_ARG; }
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#else
    (void)nthreads;
#endif
    edges_t Eg;
    rc_ = build_edges(pos, N, box9, M.rc, N > 400 ? 1 : 0, &Eg);
    if (rc_) { edges_free(&Eg); model_free(&M); return rc_; }
    const int nphi = M.nphi, Na = M.Na, NB = nphi * Na, T = M.T;
    double *c = malloc(sizeof(double) * (size_t)T * N * nphi + 8);       /* c^t_i[n] */
    double *b = malloc(sizeof(double) * (size_t)T * N * NB + 8);         /* b^t_i[n][a] */
    double *Eat = malloc(sizeof(double) * (size_t)N + 8);
    if (!c || !b || !Eat) return ORC_ERR_MEM;
    const size_t wd = dense_work_doubles(&M);

    /* ---- forward, t = 0 .. T-1 ---- */
    for (int64_t i = 0; i < N; ++i) memcpy(c + (size_t)i * nphi, M.c0 + (size_t)species[i] * nphi, sizeof(double) * nphi);
    for (int t = 0; t < T; ++t) {
        const double *ct = c + (size_t)t * N * nphi;
        double *bt = b + (size_t)t * N * NB;
#pragma omp parallel
        {
            double *work = malloc(sizeof(double) * wd);
            double A[MAXA], x[256], outv[256];
#pragma omp for schedule(dynamic, 16)
            for (int64_t i = 0; i < N; ++i) {
                double *bi = bt + (size_t)i * NB;
                for (int q = 0; q < NB; ++q) bi[q] = 0.0;
                for (int64_t q = Eg.off[i]; q < Eg.off[i + 1]; ++q) {
                    const edge_t *e = &Eg.e[q];
                    const int sj = species[e->j];
                    const double r = sqrt((e->d[0] * e->d[0] + e->d[1] * e->d[1]) + e->d[2] * e->d[2]);
                    const double fc = fcut(r, M.rc);
                    const double *rcen = M.rcen + ((size_t)t * M.S + sj) * nphi;
                    const double *alpha = M.alpha + ((size_t)t * M.S + sj) * nphi;
                    const double *cj = ct + (size_t)e->j * nphi;
                    for (int n = 0; n < nphi; ++n) {
                        double dr = r - rcen[n];
                        x[n] = cj[n] * (exp(-alpha[n] * dr * dr) * fc);
                    }
                    monomials(&M, e->d, A);
                    for (int n = 0; n < nphi; ++n) for (int a = 0; a < Na; ++a) bi[n * Na + a] += x[n] * A[a];
                }
                double *rho_o = rho_out ? rho_out + ((size_t)t * N + i) * M.norb : NULL;
                atom_dense(&M, t, species[i], bi, outv, rho_o, NULL, NULL, work);
                if (t < T - 1) memcpy(c + ((size_t)(t + 1) * N + i) * nphi, outv, sizeof(double) * nphi);
                else Eat[i] = outv[0];
            }
            free(work);
        }
    }
    double Etot = 0.0;
    for (int64_t i = 0; i < N; ++i) Etot += Eat[i];
    if (E_out) *E_out = Etot;
    if (Ei) memcpy(Ei, Eat, sizeof(double) * (size_t)N);
    if (c_out) memcpy(c_out, c, sizeof(double) * (size_t)T * N * nphi);
    if (b_out) memcpy(b_out, b, sizeof(double) * (size_t)T * N * NB);

    /* ---- reverse, t = T-1 .. 0 (Eqs. 3-5) ---- */
    if (do_forces) {
        double *cbar_next = calloc((size_t)N * nphi + 8, sizeof(double)); /* dE/dc^{t+1} */
        double *cbar = calloc((size_t)N * nphi + 8, sizeof(double));      /* dE/dc^{t}   */
        double *bbar = malloc(sizeof(double) * (size_t)N * NB + 8);
        double *g = calloc((size_t)Eg.n * 3 + 8, sizeof(double));         /* g_e = dE/dr_e, summed over layers */
        if (!cbar_next || !cbar || !bbar || !g) return ORC_ERR_MEM;
        for (int t = T - 1; t >= 0; --t) {
            const double *ct = c + (size_t)t * N * nphi;
            const double *bt = b + (size_t)t * N * NB;
            memset(cbar, 0, sizeof(double) * (size_t)N * nphi);
#pragma omp parallel
            {
                double *work = malloc(sizeof(double) * wd);
                double one = 1.0;
#pragma omp for schedule(dynamic, 16)
                for (int64_t i = 0; i < N; ++i) {
                    const double *outbar = (t == T - 1) ? &one : cbar_next + (size_t)i * nphi;
                    atom_dense(&M, t, species[i], bt + (size_t)i * NB, NULL, NULL, outbar, bbar + (size_t)i * NB, work);
                }
                free(work);
            }
#pragma omp parallel
            {
                double A[MAXA], dA[MAXA][3], Sn[256], Pa[MAXA];
#pragma omp for schedule(dynamic, 16)
                for (int64_t i = 0; i < N; ++i) {
                    const double *bb = bbar + (size_t)i * NB;
                    for (int64_t q = Eg.off[i]; q < Eg.off[i + 1]; ++q) {
                        const edge_t *e = &Eg.e[q];
                        const int sj = species[e->j];
                        const double r = sqrt((e->d[0] * e->d[0] + e->d[1] * e->d[1]) + e->d[2] * e->d[2]);
                        const double fc = fcut(r, M.rc), dfc = dfcut(r, M.rc);
                        const double *rcen = M.rcen + ((size_t)t * M.S + sj) * nphi;
                        const double *alpha = M.alpha + ((size_t)t * M.S + sj) * nphi;
                        const double *cj = ct + (size_t)e->j * nphi;
                        monomials(&M, e->d, A);
                        monomial_grads(&M, e->d, dA);
                        for (int a = 0; a < Na; ++a) Pa[a] = 0.0;
                        double radial = 0.0; /* sum_n c_j[n] R'_n S_n */
                        for (int n = 0; n < nphi; ++n) {
                            double dr = r - rcen[n];
                            double ex = exp(-alpha[n] * dr * dr);
                            double Rn = ex * fc;
                            double dRn = (-2.0 * alpha[n] * dr * fc + dfc) * ex;
                            double s = 0.0;
                            for (int a = 0; a < Na; ++a) s += bb[n * Na + a] * A[a];
                            Sn[n] = s;
                            for (int a = 0; a < Na; ++a) Pa[a] += bb[n * Na + a] * (cj[n] * Rn);
                            radial += cj[n] * dRn * s;
                            if (t >= 1) {           /* coefficient path of Eq. 4; dc^0/dr = 0 */
                                double add = Rn * s;
#pragma omp atomic
                                cbar[(size_t)e->j * nphi + n] += add;
                            }
                        }
                        double ge[3];
                        for (int dd = 0; dd < 3; ++dd) ge[dd] = radial * (e->d[dd] / r);
                        for (int a = 0; a < Na; ++a) for (int dd = 0; dd < 3; ++dd) ge[dd] += Pa[a] * dA[a][dd];
                        for (int dd = 0; dd < 3; ++dd) g[3 * q + dd] += ge[dd];
                    }
                }
            }
            double *tmp = cbar_next; cbar_next = cbar; cbar = tmp;
        }
        /* F_k = sum_{e: centre = k} g_e - sum_{e: neighbour = k} g_e;  virial = - sum_e r_e (x) g_e */
        if (F) memset(F, 0, sizeof(double) * 3 * (size_t)N);
        double vir[9] = {0};
        for (int64_t i = 0; i < N; ++i)
            for (int64_t q = Eg.off[i]; q < Eg.off[i + 1]; ++q) {
                const edge_t *e = &Eg.e[q];
                for (int dd = 0; dd < 3; ++dd) {
                    if (F) { F[3 * i + dd] += g[3 * q + dd]; F[3 * (size_t)e->j + dd] -= g[3 * q + dd]; }
                    for (int ee = 0; ee < 3; ++ee) vir[3 * dd + ee] -= e->d[dd] * g[3 * q + ee];
                }
            }
        if (virial) memcpy(virial, vir, sizeof(vir));
        free(cbar_next); free(cbar); free(bbar); free(g);
    }
    free(c); free(b); free(Eat);
    edges_free(&Eg); model_free(&M);
    return ORC_OK;
}

/* Header fields of a blob, for tests: out[10] = S,T,L,nphi,norb,H1c,H2c,H1e,H2e,Na; returns code. */
int oracle_blob_info(const void *blob, size_t nbytes, int32_t *out, double *rc) {
    model_t M;
    int rc_ = model_parse(&M, blob, nbytes);
    if (rc_) return rc_;
    out[0] = M.S; out[1] = M.T; out[2] = M.L; out[3] = M.nphi; out[4] = M.norb;
    out[5] = M.H1c; out[6] = M.H2c; out[7] = M.H1e; out[8] = M.H2e; out[9] = M.Na;
    if (rc) *rc = M.rc;
    model_free(&M);
    return ORC_OK;
}

/* Monomial table in the oracle's order a = 0..Na-1: rows (lx, ly, lz); mu[a]. */
int oracle_monomials(int L, int32_t *lxyz, double *mu) {
    if (L < 0 || L > MAXL) return -1;
    int a = 0;
    for (int l = 0; l <= L; ++l)
        for (int lx = l; lx >= 0; --lx)
            for (int ly = l - lx; ly >= 0; --ly) {
                int lz = l - lx - ly;
                lxyz[3 * a] = lx; lxyz[3 * a + 1] = ly; lxyz[3 * a + 2] = lz;
                mu[a] = factorial(l) / (factorial(lx) * factorial(ly) * factorial(lz));
                ++a;
            }
    return a;
}

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
