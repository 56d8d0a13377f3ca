// api.cu -- the C ABI of include/reann.h: handle, weights folding/upload, the evaluation schedule.
// Host logic only; every arithmetic step of the path runs in the kernels of neighbor.cu, edge.cu,
// dense.cu, scan.cu. There is deliberately no CPU fallback: without a CUDA device every call fails.
#include <math.h>
#include <stdarg.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>

#include "handle.cuh"

static thread_local std::string g_create_error;

int set_err(reann *h, int code, const char *fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof(buf), fmt, ap);
    va_end(ap);
    if (h) h->err = buf; else g_create_error = buf;
    return code;
}

int dev_ensure(reann *h, DevBuf &b, size_t bytes) {
    if (bytes == 0) bytes = 16;
    if (b.bytes >= bytes) return REANN_OK;
    if (b.p) { cudaFree(b.p); h->bytes_device -= b.bytes; b.p = nullptr; b.bytes = 0; }
    const size_t want = (bytes + 255) & ~(size_t)255;
    cudaError_t e = cudaMalloc(&b.p, want);
    if (e != cudaSuccess) {
        cudaGetLastError();
        b.p = nullptr;
        return set_err(h, REANN_ERR_OOM, "cudaMalloc(%zu bytes) failed: %s", want, cudaGetErrorString(e));
    }
    b.bytes = want;
    h->bytes_device += want;
    return REANN_OK;
}

static void dev_free(reann *h, DevBuf &b) {
    if (b.p) { cudaFree(b.p); h->bytes_device -= b.bytes; }
    b.p = nullptr; b.bytes = 0;
}

static bool is_device_ptr(const void *p) {
    if (!p) return false;
    cudaPointerAttributes at;
    cudaError_t e = cudaPointerGetAttributes(&at, p);
    if (e != cudaSuccess) { cudaGetLastError(); return false; }
    return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

static int pad_pow2_32(int H) { int p = 32; while (p < H) p <<= 1; return p; }

// x = hi + lo with hi rounded to TF32 (10 mantissa bits), lo = x - hi exact (same split as dense_tc.cu)
static void split_tf32_host(float x, float *hi, float *lo) {
    uint32_t u;
    memcpy(&u, &x, 4);
    u = (u + 0x1000u) & 0xFFFFE000u;
    memcpy(hi, &u, 4);
    *lo = x - *hi;                 // exact; then rounded to TF32 as well
    memcpy(&u, lo, 4);
    u = (u + 0x1000u) & 0xFFFFE000u;
    memcpy(lo, &u, 4);
}

// Append the chunk images of a K-major operand B[n][k] (n < N, k < K, K % 32 == 0) in the shared-memory
// layout of dense_tc.cu: per chunk of 32 k: hi image [k/4][n][k%4], then the lo image.
template <class F>
static size_t push_images(std::vector<float> &img, int N, int K, F Bnk) {
    const size_t off = img.size();
    img.resize(off + (size_t)2 * N * K, 0.f);
    for (int kc = 0; kc < K / 32; ++kc) {
        float *hi = img.data() + off + (size_t)kc * 2 * N * 32, *lo = hi + (size_t)N * 32;
        for (int ki = 0; ki < 8; ++ki)
            for (int n = 0; n < N; ++n)
                for (int j = 0; j < 4; ++j)
                    split_tf32_host(Bnk(n, kc * 32 + ki * 4 + j), &hi[((size_t)ki * N + n) * 4 + j], &lo[((size_t)ki * N + n) * 4 + j]);
    }
    return off;
}

// ---------------------------------------------------------------------------------------------
// Blob parsing (layout: gen/weights.py) -- this side's own parser.
struct BlobView {
    int S, T, L, nphi, norb, H1c, H2c, H1e, H2e;
    double rc;
    const double *rcen, *alpha, *c0, *Wc;
    std::vector<const double *> W1, b1, W2, b2, W3, b3;
};

static int parse_blob(const unsigned char *p, size_t nbytes, BlobView &v, std::string &why) {
    if (nbytes < 64 || memcmp(p, "REANNB2\0", 8) != 0) { why = "bad magic or truncated header"; return REANN_ERR_WEIGHTS; }
    uint32_t hd[12];
    memcpy(hd, p + 8, sizeof(hd));
    if (hd[0] != 1 || hd[10] != 0) { why = "unsupported version or activation"; return REANN_ERR_WEIGHTS; }
    v.S = hd[1]; v.T = hd[2]; v.L = hd[3]; v.nphi = hd[4]; v.norb = hd[5];
    v.H1c = hd[6]; v.H2c = hd[7]; v.H1e = hd[8]; v.H2e = hd[9];
    memcpy(&v.rc, p + 56, 8);
    if (v.S < 1 || v.T < 1 || v.nphi < 1 || v.norb < 1 || v.L < 0 || !(v.rc > 0) || v.H1c < 1 || v.H2c < 1 || v.H1e < 1 ||
        v.H2e < 1 || v.S > 1024 || v.T > 1024 || v.nphi > 4096 || v.L > 64 || v.norb > (1 << 20) || v.H1c > (1 << 16) ||
        v.H2c > (1 << 16) || v.H1e > (1 << 16) || v.H2e > (1 << 16)) {
        why = "header fields out of range"; return REANN_ERR_WEIGHTS;
    }
    size_t need = (size_t)2 * v.T * v.S * v.nphi + (size_t)v.S * v.nphi + (size_t)v.T * (v.L + 1) * v.nphi * v.norb;
    for (int t = 0; t < v.T; ++t) {
        const bool last = t == v.T - 1;
        const size_t H1 = last ? v.H1e : v.H1c, H2 = last ? v.H2e : v.H2c, out = last ? 1 : v.nphi;
        need += (size_t)v.S * ((size_t)v.norb * H1 + H1 + H1 * H2 + H2 + H2 * out + out);
    }
    if (nbytes != 64 + 8 * need) { why = "blob size does not match its header"; return REANN_ERR_WEIGHTS; }
    const double *q = reinterpret_cast<const double *>(p + 64);
    v.rcen = q; q += (size_t)v.T * v.S * v.nphi;
    v.alpha = q; q += (size_t)v.T * v.S * v.nphi;
    v.c0 = q; q += (size_t)v.S * v.nphi;
    v.Wc = q; q += (size_t)v.T * (v.L + 1) * v.nphi * v.norb;
    for (int t = 0; t < v.T; ++t) {
        const bool last = t == v.T - 1;
        const size_t H1 = last ? v.H1e : v.H1c, H2 = last ? v.H2e : v.H2c, out = last ? 1 : v.nphi;
        for (int s = 0; s < v.S; ++s) {
            v.W1.push_back(q); q += (size_t)v.norb * H1;
            v.b1.push_back(q); q += H1;
            v.W2.push_back(q); q += H1 * H2;
            v.b2.push_back(q); q += H2;
            v.W3.push_back(q); q += H2 * out;
            v.b3.push_back(q); q += out;
        }
    }
    return REANN_OK;
}

// ---------------------------------------------------------------------------------------------
extern "C" int reann_create(reann_t **out, const void *weights, size_t weights_bytes, const int32_t *species,
                            int64_t n_atoms, double rc, double skin, int T, int L, int n_gauss) {
    if (!out) return set_err(nullptr, REANN_ERR_ARG, "out is NULL");
    *out = nullptr;
    if (!weights || !species || n_atoms < 0 || !(rc > 0) || !(skin >= 0) || T < 1)
        return set_err(nullptr, REANN_ERR_ARG, "bad argument (NULL pointer, n_atoms < 0, rc <= 0, skin < 0 or T < 1)");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        return set_err(nullptr, REANN_ERR_CUDA, "no CUDA device: this library has no CPU path");
    }
    if (n_atoms >= ((int64_t)1 << COL_SPECIES_SHIFT)) return set_err(nullptr, REANN_ERR_UNSUPPORTED, "n_atoms >= 2^27");
    // bring blob and species to the host
    std::vector<unsigned char> blob(weights_bytes);
    if (is_device_ptr(weights)) {
        if (cudaMemcpy(blob.data(), weights, weights_bytes, cudaMemcpyDeviceToHost) != cudaSuccess)
            return set_err(nullptr, REANN_ERR_CUDA, "copy of weights failed");
    } else memcpy(blob.data(), weights, weights_bytes);
    std::vector<int32_t> sp((size_t)n_atoms);
    if (n_atoms > 0) {
        if (is_device_ptr(species)) {
            if (cudaMemcpy(sp.data(), species, sizeof(int32_t) * (size_t)n_atoms, cudaMemcpyDeviceToHost) != cudaSuccess)
                return set_err(nullptr, REANN_ERR_CUDA, "copy of species failed");
        } else memcpy(sp.data(), species, sizeof(int32_t) * (size_t)n_atoms);
    }
    BlobView v;
    std::string why;
    int rcode = parse_blob(blob.data(), weights_bytes, v, why);
    if (rcode) return set_err(nullptr, rcode, "weights blob: %s", why.c_str());
    if (v.T != T || v.L != L || v.nphi != n_gauss || fabs(v.rc - rc) > 1e-12 * rc)
        return set_err(nullptr, REANN_ERR_WEIGHTS, "blob header (T=%d L=%d n_gauss=%d rc=%g) disagrees with arguments (T=%d L=%d n_gauss=%d rc=%g)",
                       v.T, v.L, v.nphi, v.rc, T, L, n_gauss, rc);
    if (L > 3 || n_gauss > REANN_MAX_NPHI || T > REANN_MAX_T || v.S > REANN_MAX_S)
        return set_err(nullptr, REANN_ERR_UNSUPPORTED, "this version supports L <= 3, n_gauss <= %d, T <= %d, S <= %d",
                       REANN_MAX_NPHI, REANN_MAX_T, REANN_MAX_S);
    if (std::max(std::max(v.H1c, v.H2c), std::max(v.H1e, v.H2e)) > 128)
        return set_err(nullptr, REANN_ERR_UNSUPPORTED, "MLP hidden width > 128 not supported in this version");
    for (int64_t i = 0; i < n_atoms; ++i)
        if (sp[(size_t)i] < 0 || sp[(size_t)i] >= v.S) return set_err(nullptr, REANN_ERR_ARG, "species[%lld] = %d out of range", (long long)i, sp[(size_t)i]);

    reann *h = new reann();
    h->N = n_atoms;
    ModelDims &md = h->md;
    md.S = v.S; md.T = T; md.L = L; md.nphi = n_gauss; md.nphip = (n_gauss + 3) & ~3;
    md.Na = (L + 1) * (L + 2) * (L + 3) / 6; md.NB = md.nphip * md.Na; md.norb = v.norb;
    md.npairs = n_gauss * (n_gauss + 1) / 2; md.NPp = md.npairs; md.nqp = ((L + 1) * md.NPp + 15) & ~15;
    md.K1 = (md.nqp + 31) & ~31;
    {
        auto is = [](const char *name, const char *val) { const char *e = getenv(name); return e && strcmp(e, val) == 0; };
        h->dense_tc = !is("REANN_DENSE", "simt");
        h->edge_fwd_mma = !is("REANN_EDGE_FWD", "simt");
        h->mlp_tf32 = is("REANN_MLP_MODE", "tf32") && h->dense_tc;
        if (const char *e = getenv("REANN_STASH_CHUNKS")) h->stash_chunks_forced = std::max(0, atoi(e));
        h->use_graph = !is("REANN_GRAPH", "0");
    }
    md.rc = rc; md.skin = skin;
    h->zs = 0;
    for (int t = 0; t < T; ++t) {
        const bool last = t == T - 1;
        h->ld[t].H1p = pad_pow2_32(last ? v.H1e : v.H1c);
        h->ld[t].H2p = pad_pow2_32(last ? v.H2e : v.H2c);
        h->ld[t].nout = last ? 1 : n_gauss;
        h->ld[t].noutp = h->ld[t].nout;
        h->zs = std::max(h->zs, h->ld[t].H1p + h->ld[t].H2p);
    }
#define CREATE_FAIL(code, ...) do { int c_ = set_err(nullptr, code, __VA_ARGS__); reann_destroy(h); return c_; } while (0)
#define CCU(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) CREATE_FAIL(REANN_ERR_CUDA, "%s: %s", #call, cudaGetErrorString(e_)); } while (0)
#define CRC(call) do { int r_ = (call); if (r_ != REANN_OK) { g_create_error = h->err; reann_destroy(h); return r_; } } while (0)

    // ---- radial tables and c0 (FP32, padded to nphip) ----
    const double LOG2E = 1.4426950408889634;
    {
        const size_t n = (size_t)T * md.S * md.nphip;
        std::vector<float> rcen(n, 0.f), al(n, 0.f), c0((size_t)md.S * md.nphip, 0.f);
        for (int t = 0; t < T; ++t)
            for (int s = 0; s < md.S; ++s)
                for (int k = 0; k < md.nphi; ++k) {
                    rcen[((size_t)t * md.S + s) * md.nphip + k] = (float)v.rcen[((size_t)t * md.S + s) * md.nphi + k];
                    al[((size_t)t * md.S + s) * md.nphip + k] = (float)(v.alpha[((size_t)t * md.S + s) * md.nphi + k] * LOG2E);
                }
        for (int s = 0; s < md.S; ++s)
            for (int k = 0; k < md.nphi; ++k) c0[(size_t)s * md.nphip + k] = (float)v.c0[(size_t)s * md.nphi + k];
        CRC(dev_ensure(h, h->rcen, n * 4)); CRC(dev_ensure(h, h->alpha, n * 4)); CRC(dev_ensure(h, h->c0, c0.size() * 4));
        CCU(cudaMemcpy(h->rcen.p, rcen.data(), n * 4, cudaMemcpyHostToDevice));
        CCU(cudaMemcpy(h->alpha.p, al.data(), n * 4, cudaMemcpyHostToDevice));
        CCU(cudaMemcpy(h->c0.p, c0.data(), c0.size() * 4, cudaMemcpyHostToDevice));
    }
    // ---- fold the contraction into the first MLP layer (FP64), pad, transpose (see dense.cu) ----
    {
        std::vector<float> all;
        auto reserve = [&](size_t n) { size_t o = all.size(); all.resize(o + ((n + 3) & ~(size_t)3), 0.f); return o; };
        struct Off { size_t U, UT, b1, W2, W2T, b2, W3, W3T, b3, W3p, W3c0; };
        std::vector<Off> offs((size_t)T * md.S);
        std::vector<double> Vq((size_t)v.norb);
        for (int t = 0; t < T; ++t) {
            const bool last = t == T - 1;
            const int H1 = last ? v.H1e : v.H1c, H2 = last ? v.H2e : v.H2c, nout = h->ld[t].nout;
            const int H1p = h->ld[t].H1p, H2p = h->ld[t].H2p;
            for (int s = 0; s < md.S; ++s) {
                const int k = t * md.S + s;
                Off o;
                o.U = reserve((size_t)md.nqp * H1p); o.UT = reserve((size_t)H1p * md.nqp);
                o.b1 = reserve(H1p); o.W2 = reserve((size_t)H1p * H2p); o.W2T = reserve((size_t)H2p * H1p);
                o.b2 = reserve(H2p); o.W3 = reserve((size_t)H2p * nout); o.W3T = reserve((size_t)nout * H2p);
                o.b3 = reserve(nout);
                o.W3p = reserve((size_t)H2p * 16); o.W3c0 = reserve(H2p);   // tensor-core path: ALU GEMM over W3
                offs[(size_t)k] = o;
                const double *W1 = v.W1[(size_t)k];
                for (int l = 0; l <= L; ++l) {
                    const double *Wl = v.Wc + ((size_t)t * (L + 1) + l) * md.nphi * v.norb;
                    int pp = 0;
                    for (int n = 0; n < md.nphi; ++n)
                        for (int n2 = n; n2 < md.nphi; ++n2, ++pp) {
                            const double fac = (n == n2) ? 1.0 : 2.0;
                            for (int m = 0; m < v.norb; ++m) Vq[(size_t)m] = fac * Wl[(size_t)n * v.norb + m] * Wl[(size_t)n2 * v.norb + m];
                            const size_t q = (size_t)l * md.NPp + pp;
                            for (int hh = 0; hh < H1; ++hh) {
                                double acc = 0.0;
                                for (int m = 0; m < v.norb; ++m) acc += Vq[(size_t)m] * W1[(size_t)m * H1 + hh];
                                all[o.U + q * H1p + hh] = (float)acc;
                                all[o.UT + (size_t)hh * md.nqp + q] = (float)acc;
                            }
                        }
                }
                for (int a = 0; a < H1; ++a) all[o.b1 + a] = (float)v.b1[(size_t)k][a];
                for (int a = 0; a < H1; ++a)
                    for (int b = 0; b < H2; ++b) {
                        const float w = (float)v.W2[(size_t)k][(size_t)a * H2 + b];
                        all[o.W2 + (size_t)a * H2p + b] = w;
                        all[o.W2T + (size_t)b * H1p + a] = w;
                    }
                for (int b = 0; b < H2; ++b) all[o.b2 + b] = (float)v.b2[(size_t)k][b];
                for (int b = 0; b < H2; ++b)
                    for (int c = 0; c < nout; ++c) {
                        const float w = (float)v.W3[(size_t)k][(size_t)b * nout + c];
                        all[o.W3 + (size_t)b * nout + c] = w;
                        all[o.W3T + (size_t)c * H2p + b] = w;
                        if (c < 16) all[o.W3p + (size_t)b * 16 + c] = w;
                        if (c == 0) all[o.W3c0 + b] = w;
                    }
                for (int c = 0; c < nout; ++c) all[o.b3 + c] = (float)v.b3[(size_t)k][c];
            }
        }
        CRC(dev_ensure(h, h->w_all, all.size() * 4));
        CCU(cudaMemcpy(h->w_all.p, all.data(), all.size() * 4, cudaMemcpyHostToDevice));
        const float *base = (const float *)h->w_all.p;
        h->h_wtab.resize((size_t)T * md.S);
        for (size_t k = 0; k < offs.size(); ++k) {
            const Off &o = offs[k];
            h->h_wtab[k] = DenseW{base + o.U, base + o.UT, base + o.b1, base + o.W2, base + o.W2T, base + o.b2,
                                  base + o.W3, base + o.W3T, base + o.b3};
        }
        CRC(dev_ensure(h, h->w_tab, sizeof(DenseW) * h->h_wtab.size()));
        CCU(cudaMemcpy(h->w_tab.p, h->h_wtab.data(), sizeof(DenseW) * h->h_wtab.size(), cudaMemcpyHostToDevice));
        // tensor-core chunk images (dense_tc.cu): pre-split hi | lo TF32 operands
        {
            std::vector<float> img;
            struct OffT { size_t g1, g2, r1, r2, r3; };
            std::vector<OffT> ot(offs.size());
            for (int t = 0; t < T; ++t) {
                const int H1p = h->ld[t].H1p, H2p = h->ld[t].H2p, nout = h->ld[t].nout;
                for (int s = 0; s < md.S; ++s) {
                    const Off &o = offs[(size_t)t * md.S + s];
                    OffT &q = ot[(size_t)t * md.S + s];
                    const float *A = all.data();
                    auto Uqh = [&](int qq, int hh) { return qq < md.nqp ? A[o.U + (size_t)qq * H1p + hh] : 0.f; };
                    q.g1 = push_images(img, H1p, md.K1, [&](int n, int k) { return Uqh(k, n); });
                    q.g2 = push_images(img, H2p, H1p, [&](int n, int k) { return A[o.W2 + (size_t)k * H2p + n]; });
                    q.r1 = push_images(img, H2p, 32, [&](int n, int k) { return k < nout ? A[o.W3 + (size_t)n * nout + k] : 0.f; });
                    q.r2 = push_images(img, H1p, H2p, [&](int n, int k) { return A[o.W2 + (size_t)n * H2p + k]; });
                    q.r3 = img.size();
                    for (int nb = 0; nb * 128 < md.K1; ++nb) {
                        const int rows = std::min(128, md.K1 - nb * 128);
                        push_images(img, rows, H1p, [&](int n, int k) { return Uqh(nb * 128 + n, k); });
                    }
                }
            }
            CRC(dev_ensure(h, h->wt_all, img.size() * 4));
            CCU(cudaMemcpy(h->wt_all.p, img.data(), img.size() * 4, cudaMemcpyHostToDevice));
            const float *ib = (const float *)h->wt_all.p;
            std::vector<DenseWT> wt(offs.size());
            for (size_t k = 0; k < offs.size(); ++k)
                wt[k] = DenseWT{ib + ot[k].g1, ib + ot[k].g2, ib + ot[k].r1, ib + ot[k].r2, ib + ot[k].r3,
                                base + offs[k].b1, base + offs[k].b2, base + offs[k].b3, base + offs[k].W3p, base + offs[k].W3c0};
            CRC(dev_ensure(h, h->wt_tab, sizeof(DenseWT) * wt.size()));
            CCU(cudaMemcpy(h->wt_tab.p, wt.data(), sizeof(DenseWT) * wt.size(), cudaMemcpyHostToDevice));
        }
    }
    // ---- atoms: species, dense tiles ----
    CRC(dev_ensure(h, h->species_caller, sizeof(int32_t) * (size_t)std::max<int64_t>(n_atoms, 1)));
    if (n_atoms > 0) CCU(cudaMemcpy(h->species_caller.p, sp.data(), sizeof(int32_t) * (size_t)n_atoms, cudaMemcpyHostToDevice));
    h->species_count.assign((size_t)md.S, 0);
    for (int64_t i = 0; i < n_atoms; ++i) h->species_count[(size_t)sp[(size_t)i]]++;
    {
        std::vector<DenseTile> tiles;
        h->tile_rows = h->dense_tc ? DENSE_TC_TM : DENSE_TM;
        int64_t base = 0;
        for (int s = 0; s < md.S; ++s) {
            for (int64_t o = 0; o < h->species_count[(size_t)s]; o += h->tile_rows)
                tiles.push_back(DenseTile{s, (int32_t)(base + o), (int32_t)std::min<int64_t>(h->tile_rows, h->species_count[(size_t)s] - o)});
            base += h->species_count[(size_t)s];
        }
        h->n_tiles = (int)tiles.size();
        CRC(dev_ensure(h, h->tiles, sizeof(DenseTile) * std::max<size_t>(tiles.size(), 1)));
        if (!tiles.empty()) CCU(cudaMemcpy(h->tiles.p, tiles.data(), sizeof(DenseTile) * tiles.size(), cudaMemcpyHostToDevice));
    }
    CRC(dev_ensure(h, h->flags, 64));
    CCU(cudaMemset(h->flags.p, 0, 64));
    CCU(cudaStreamCreate(&h->own_stream));
    h->stream = h->own_stream;
    CCU(cudaMallocHost((void **)&h->h_flags, 64));
    *out = h;
    return REANN_OK;
}

extern "C" void reann_destroy(reann_t *h) {
    if (!h) return;
    if (h->stream) cudaStreamSynchronize(h->stream); else cudaDeviceSynchronize();
    if (h->gexec) cudaGraphExecDestroy(h->gexec);
    if (h->own_stream) cudaStreamDestroy(h->own_stream);
    DevBuf *bufs[] = {&h->w_all, &h->w_tab, &h->wt_all, &h->wt_tab, &h->rcen, &h->alpha, &h->c0, &h->species_caller, &h->tiles,
                      &h->pos_build, &h->wshift, &h->perm, &h->inv_perm, &h->xrec, &h->img_index, &h->cell_start,
                      &h->cell_rank, &h->row_ptr, &h->col, &h->rev, &h->sp_list, &h->scratch_a, &h->scratch_b,
                      &h->scratch_c, &h->scan_ws, &h->pos_stage, &h->rank16, &h->rc_cnt, &h->rc_ptr, &h->col_rc,
                      &h->geom, &h->rev_rc, &h->c_ext, &h->b, &h->z_stash, &h->bbar, &h->cbar, &h->kappa, &h->gst,
                      &h->Ei, &h->Fc, &h->vir_part, &h->out_stage, &h->Ei_caller, &h->flags, &h->red_scratch, &h->Qbuf,
                      &h->halo_caller, &h->xch_idx, &h->xch_val, &h->md_state, &h->md_partial, &h->md_E, &h->nbr_mask, &h->rcx};
    for (DevBuf *b : bufs) dev_free(h, *b);
    if (h->h_flags) cudaFreeHost(h->h_flags);
    for (cudaEvent_t e : h->ev) cudaEventDestroy(e);
    delete h;
}

extern "C" const char *reann_last_error(const reann_t *h) { return h ? h->err.c_str() : g_create_error.c_str(); }

static void graph_drop(reann *h) {
    if (h->gexec) { cudaGraphExecDestroy(h->gexec); h->gexec = nullptr; }
}

// The legacy default stream (0) cannot be captured into a CUDA graph, so the handle then works on a blocking stream
// of its own: it is ordered after earlier work of the default stream, and every call ends with a synchronisation.
extern "C" int reann_set_stream(reann_t *h, void *cuda_stream) {
    if (!h) return REANN_ERR_ARG;
    cudaStreamSynchronize(h->stream);
    graph_drop(h);
    h->stream = cuda_stream ? (cudaStream_t)cuda_stream : h->own_stream;
    return REANN_OK;
}

extern "C" int reann_set_profiling(reann_t *h, int on) {
    if (!h) return REANN_ERR_ARG;
    h->profiling = on != 0;
    return REANN_OK;
}

static int check_box(reann *h, const double *box9) {
    if (!box9) return set_err(h, REANN_ERR_ARG, "box is NULL");
    if (box9[1] != 0.0 || box9[2] != 0.0 || box9[5] != 0.0)
        return set_err(h, REANN_ERR_UNSUPPORTED, "lattice vectors must be in lower-triangular form: a = (ax,0,0), b = (bx,by,0), c = (cx,cy,cz)");
    if (!(box9[0] > 0.0) || !(box9[4] > 0.0) || !(box9[8] > 0.0)) return set_err(h, REANN_ERR_BOX, "ax, by, cz must be positive");
    if (h->have_halo && (box9[3] != 0.0 || box9[6] != 0.0 || box9[7] != 0.0))
        return set_err(h, REANN_ERR_UNSUPPORTED, "decomposed runs (reann_set_halo) take orthorhombic boxes only");
    const BoxP B = make_boxp(box9);
    const double R = h->md.rc + h->md.skin, wd[3] = {B.wa, B.wb, B.wc};
    for (int d = 0; d < 3; ++d)
        if (!(wd[d] >= R)) return set_err(h, REANN_ERR_BOX, "distance %g between the cell faces along lattice vector %d < rc + skin = %g", wd[d], d, R);
    return REANN_OK;
}

// positions on the device (staged when the caller passed a host pointer)
static int device_positions(reann *h, const double *pos, const double **d_pos) {
    if (h->N == 0) { *d_pos = nullptr; return REANN_OK; }
    if (!pos) return set_err(h, REANN_ERR_ARG, "pos is NULL");
    if (is_device_ptr(pos)) { *d_pos = pos; return REANN_OK; }
    RC(dev_ensure(h, h->pos_stage, sizeof(double) * 3 * (size_t)h->N));
    CU(h, cudaMemcpyAsync(h->pos_stage.p, pos, sizeof(double) * 3 * (size_t)h->N, cudaMemcpyHostToDevice, h->stream));
    *d_pos = (const double *)h->pos_stage.p;
    return REANN_OK;
}

static int do_build(reann *h, const double *d_pos, const double *box9) {
    memcpy(h->box_build, box9, sizeof(double) * 9);
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (h->profiling) { cudaEventCreate(&e0); cudaEventCreate(&e1); cudaEventRecord(e0, h->stream); }
    h->have_list = false;
    if (h->N > 0) RC(neighbor_build(h, d_pos));
    const ModelDims &md = h->md;
    const int64_t N = h->N;
    if (N == 0) { h->G = 0; h->n_ext = 0; h->E_list = 0; h->E_rc_build = 0; }
    // per-evaluation buffers whose size follows the list
    if (h->rank16.bytes < sizeof(uint16_t) * (size_t)std::max<int64_t>(h->E_list, 1))
        RC(dev_ensure(h, h->rank16, sizeof(uint16_t) * ((size_t)std::max<int64_t>(h->E_list, 1) + (size_t)h->E_list / 32 + 1024)));
    RC(dev_ensure(h, h->rc_cnt, sizeof(int32_t) * (size_t)(N + 1)));
    RC(dev_ensure(h, h->rc_ptr, sizeof(int64_t) * (size_t)(N + 1)));
    RC(dev_ensure(h, h->rcx, sizeof(uint32_t) * (size_t)std::max<int64_t>(h->n_ext, 1)));
    RC(dev_ensure(h, h->scan_ws, scan_workspace_bytes(N + 1)));
    {
        const size_t need = sizeof(float) * (size_t)md.T * (size_t)std::max<int64_t>(h->n_ext, 1) * md.nphip;
        if (h->c_ext.bytes < need) { RC(dev_ensure(h, h->c_ext, need + need / 16)); }
        CU(h, cudaMemsetAsync(h->c_ext.p, 0, h->c_ext.bytes, h->stream)); // padded coefficients stay 0
    }
    if (!h->eval_bufs_ready) {
        RC(dev_ensure(h, h->b, sizeof(float) * (size_t)md.T * (size_t)std::max<int64_t>(N, 1) * md.NB));
        // dense rows: tensor-core path = 128-row tiles (tile-quad layout, dense_tc.cu), SIMT path = sp_list rows
        const size_t rows = h->dense_tc ? (size_t)std::max(h->n_tiles, 1) * DENSE_TC_TM : (size_t)std::max<int64_t>(N, 1);
        RC(dev_ensure(h, h->z_stash, sizeof(float) * (size_t)md.T * rows * h->zs));
        RC(dev_ensure(h, h->bbar, sizeof(float) * (size_t)std::max<int64_t>(N, 1) * md.NB));
        CU(h, cudaMemsetAsync(h->bbar.p, 0, h->bbar.bytes, h->stream));       // padded rows stay 0
        RC(dev_ensure(h, h->cbar, sizeof(float) * (size_t)std::max<int64_t>(N, 1) * md.nphip));
        RC(dev_ensure(h, h->Qbuf, sizeof(float) * rows * md.K1));
        CU(h, cudaMemsetAsync(h->Qbuf.p, 0, h->Qbuf.bytes, h->stream));       // padding rows of ragged tiles stay finite
        RC(dev_ensure(h, h->Ei, sizeof(float) * (size_t)std::max<int64_t>(N, 1)));
        RC(dev_ensure(h, h->Ei_caller, sizeof(double) * (size_t)std::max<int64_t>(N, 1)));
        RC(dev_ensure(h, h->Fc, sizeof(double) * 3 * (size_t)std::max<int64_t>(N, 1)));
        h->n_vir_blocks = edge_bwd_blocks(std::max<int64_t>(N, 1), md.Na);
        RC(dev_ensure(h, h->vir_part, sizeof(double) * 9 * (size_t)h->n_vir_blocks));
        RC(dev_ensure(h, h->red_scratch, sizeof(double) * 10 * ((size_t)N / 256 + 2)));
        RC(dev_ensure(h, h->out_stage, sizeof(double) * (16 + 3 * (size_t)N)));
        h->eval_bufs_ready = true;   // only now: a failed allocation above is retried by the next build
    }
    h->have_list = true;
    h->n_rebuilds++;
    if (h->profiling) {
        cudaEventRecord(e1, h->stream); cudaEventSynchronize(e1);
        float ms = 0; cudaEventElapsedTime(&ms, e0, e1); h->ms[0] += ms;
        cudaEventDestroy(e0); cudaEventDestroy(e1);
    }
    return REANN_OK;
}

extern "C" int reann_build_neighbors(reann_t *h, const double *pos, const double *box9) {
    if (!h) return REANN_ERR_ARG;
    RC(check_box(h, box9));
    const double *d_pos = nullptr;
    RC(device_positions(h, pos, &d_pos));
    return do_build(h, d_pos, box9);
}

// profiling marks: event before each kernel group; slot = index into h->ms of the group that follows
struct Marks {
    reann *h; std::vector<std::pair<int, int>> m; // (event index, slot)
    void mark(int slot) {
        if (!h->profiling) return;
        const size_t k = m.size();
        if (h->ev.size() <= k) { cudaEvent_t e; cudaEventCreate(&e); h->ev.push_back(e); }
        cudaEventRecord(h->ev[k], h->stream);
        m.push_back({(int)k, slot});
    }
    void finish() {
        if (!h->profiling || m.size() < 2) return;
        cudaEventSynchronize(h->ev[(size_t)m.back().first]);
        for (size_t k = 0; k + 1 < m.size(); ++k) {
            float ms = 0; cudaEventElapsedTime(&ms, h->ev[(size_t)m[k].first], h->ev[(size_t)m[k + 1].first]);
            h->ms[m[k].second] += ms;
        }
        h->n_prof_calls++;
    }
};

// ---- device flag word (h->flags[0]) of one evaluation; the kernels after the rc-filter count return at once when
// it is non-zero (LaunchCtx::skip), the host reads it after the evaluation ----
enum { FLAG_REBUILD = 1, FLAG_OVERFLOW = 2 };

__global__ void k_cap_check(const int64_t *__restrict__ n_rc, int64_t cap, int32_t *__restrict__ flags,
                            int64_t *__restrict__ n_rc_out) {
    if (*n_rc > cap) atomicOr(flags, FLAG_OVERFLOW);
    *n_rc_out = *n_rc;
}

// A4 + per-step prep on the current list: skin check (sets FLAG_REBUILD), positions of the ext atoms, rc-filter count,
// offsets of the compact rows, capacity check (sets FLAG_OVERFLOW). No host synchronisation.
static int enqueue_prep(reann *h, const double *d_pos) {
    LaunchCtx ctx = h->ctx();
    const int64_t N = h->N;
    const BoxP B = make_boxp(h->box_build);
    int32_t *flags = (int32_t *)h->flags.p;
    CU(h, cudaMemsetAsync(flags, 0, 16, h->stream));
    const double thr = 0.5 * h->md.skin;
    launch_skin_check(ctx, d_pos, (const double *)h->pos_build.p, N, thr * thr, flags);
    launch_refresh(ctx, (XRec *)h->xrec.p, h->n_ext, (const int32_t *)h->perm.p, (const int32_t *)h->wshift.p, d_pos,
                   B, (float *)h->c_ext.p, (const float *)h->c0.p, h->md.nphip);
    launch_filter_count(ctx, (const XRec *)h->xrec.p, (const int64_t *)h->row_ptr.p, (const int32_t *)h->col.p, N, B,
                        h->md.rc * h->md.rc, (uint16_t *)h->rank16.p, (int32_t *)h->rc_cnt.p);
    exclusive_scan_i32_to_i64(ctx, (const int32_t *)h->rc_cnt.p, (int64_t *)h->rc_ptr.p, N, h->scan_ws.p);
    LAUNCH(ctx, k_cap_check, 1, 1, 0, (const int64_t *)h->rc_ptr.p + N, h->cap_rc, flags, (int64_t *)(flags + 2));
    return REANN_OK;
}

// (re)size the buffers that follow the compact edge count; chooses the stash chunk count (config 5)
static int ensure_rc_capacity(reann *h, int64_t n_rc) {
    if (n_rc <= h->cap_rc) return REANN_OK;
    const ModelDims &md = h->md;
    const int64_t cap = n_rc + n_rc / 16 + 1024;
    dev_free(h, h->kappa);
    RC(dev_ensure(h, h->col_rc, sizeof(uint32_t) * (size_t)cap));
    RC(dev_ensure(h, h->rev_rc, sizeof(uint32_t) * (size_t)cap));
    RC(dev_ensure(h, h->geom, sizeof(float4) * (size_t)cap));
    RC(dev_ensure(h, h->gst, sizeof(float4) * (size_t)cap));
    // kappa stash (4 N_phi bytes per edge, one layer live): whole if it fits into what is left of the device
    // memory, else in chunks of atoms -- k_edge_bwd / k_rev_gather then run once per chunk (config 5)
    const size_t whole = sizeof(float) * (size_t)cap * md.nphip;
    size_t free_b = 0, total_b = 0;
    CU(h, cudaMemGetInfo(&free_b, &total_b));
    const size_t budget = free_b > ((size_t)3 << 30) ? free_b - ((size_t)3 << 30) : free_b / 2;
    int C = 1;
    if (h->stash_chunks_forced > 0) C = h->stash_chunks_forced;
    else while (C < 64 && (C == 1 ? whole : whole / C + whole / (8 * C)) > budget) ++C;
    h->stash_chunks = C;
    RC(dev_ensure(h, h->kappa, C == 1 ? whole : whole / C + whole / (8 * C)));
    h->cap_rc = cap;
    return REANN_OK;
}

struct OutPtrs {      // where the kernels write (device), and what has to be copied back to host pointers
    double *dE, *dF, *dV;
    bool E_host, F_host, V_host;
};

// ---- the pieces of one evaluation (used by reann_energy_forces and by the layer-by-layer calls of a decomposed run) ----
struct LayerPtrs {
    size_t cstride, bstride, zstride;
    float *c_ext, *b, *zst;
    const DenseW *wtab;
    const DenseWT *wttab;
    const DenseTile *gram_tiles;
};
static LayerPtrs layer_ptrs(reann *h) {
    const ModelDims &md = h->md;
    LayerPtrs p;
    p.cstride = (size_t)h->n_ext * md.nphip; p.bstride = (size_t)h->N * md.NB;
    p.zstride = (h->dense_tc ? (size_t)h->n_tiles * DENSE_TC_TM : (size_t)h->N) * h->zs;
    p.c_ext = (float *)h->c_ext.p; p.b = (float *)h->b.p; p.zst = (float *)h->z_stash.p;
    p.wtab = (const DenseW *)h->w_tab.p; p.wttab = (const DenseWT *)h->wt_tab.p;
    p.gram_tiles = h->dense_tc ? (const DenseTile *)h->tiles.p : nullptr;
    return p;
}

static void enqueue_filter_fill(reann *h, const LaunchCtx &ctx) {
    const BoxP B = make_boxp(h->box_build);
    launch_filter_fill(ctx, (const XRec *)h->xrec.p, (const int64_t *)h->row_ptr.p, (const int32_t *)h->col.p,
                       (const uint32_t *)h->rev.p, h->N, h->n_ext, B, (const uint16_t *)h->rank16.p,
                       (const int64_t *)h->rc_ptr.p, (uint32_t *)h->rcx.p, (uint32_t *)h->col_rc.p, (float4 *)h->geom.p, (uint32_t *)h->rev_rc.p);
}

// layer t of the forward pass (Eq. 1, Eq. 2): b^t, rho^t (radial-pair form), c^{t+1} of the local atoms or E_i
static int enqueue_forward_layer(reann *h, const LaunchCtx &ctx, Marks &mk, int t) {
    const ModelDims &md = h->md;
    const int64_t N = h->N;
    const LayerPtrs p = layer_ptrs(h);
    mk.mark(2);
    int rcode = launch_edge_fwd(ctx, md, t, N, (const int64_t *)h->rc_ptr.p, (const uint32_t *)h->col_rc.p,
                                (const float4 *)h->geom.p, p.c_ext + t * p.cstride, (const float *)h->rcen.p,
                                (const float *)h->alpha.p, p.b + t * p.bstride, h->edge_fwd_mma);
    if (rcode) return set_err(h, rcode, "edge forward: unsupported (n_gauss, L) combination");
    mk.mark(3);
    const bool last = t == md.T - 1;
    launch_gram_fwd(ctx, md, N, (const int32_t *)h->sp_list.p, p.gram_tiles, h->n_tiles, p.b + t * p.bstride, (float *)h->Qbuf.p);
    rcode = h->dense_tc
                ? launch_dense_tc_fwd(ctx, md, h->ld[t], p.wttab + (size_t)t * md.S, (const DenseTile *)h->tiles.p, h->n_tiles,
                                      (const int32_t *)h->sp_list.p, (const float *)h->Qbuf.p, p.zst + t * p.zstride, h->zs,
                                      last ? (float *)h->Ei.p : p.c_ext + (t + 1) * p.cstride, last ? 1 : md.nphip, h->mlp_tf32)
                : launch_dense_fwd(ctx, md, h->ld[t], p.wtab + (size_t)t * md.S, (const DenseTile *)h->tiles.p, h->n_tiles,
                                   (const int32_t *)h->sp_list.p, (const float *)h->Qbuf.p, p.zst + t * p.zstride, h->zs,
                                   last ? (float *)h->Ei.p : p.c_ext + (t + 1) * p.cstride, last ? 1 : md.nphip);
    if (rcode) return set_err(h, rcode, "dense forward: unsupported MLP shape or shared-memory size");
    return REANN_OK;
}
// the forward LA -> GA message of layer t for the periodic images held by this handle
static void enqueue_image_gather(reann *h, const LaunchCtx &ctx, Marks &mk, int t) {
    const LayerPtrs p = layer_ptrs(h);
    mk.mark(4);
    launch_ghost_gather(ctx, p.c_ext + t * p.cstride, (const XRec *)h->xrec.p, h->N, h->n_ext, h->md.nphip);
}

__global__ void k_zero_halo_rows(float *__restrict__ bbar, int nb, int64_t N, const int32_t *__restrict__ perm,
                                 const uint8_t *__restrict__ halo_caller) {
    const int64_t k = blockIdx.x;                       // internal atom index
    if (k >= N || !halo_caller[perm[k]]) return;
    for (int q = threadIdx.x; q < nb; q += blockDim.x) bbar[k * nb + q] = 0.f;
}

// layer t of the reverse pass (Eqs. 3-5): bbar^t from dE/dc^{t+1} (or from E_i), per-edge g_e / kappa_e, reverse gather
static int enqueue_backward_layer(reann *h, const LaunchCtx &ctx, Marks &mk, int t, bool want_vir,
                                  const std::vector<int64_t> &ch_atom, const std::vector<int64_t> &ch_edge) {
    const ModelDims &md = h->md;
    const int64_t N = h->N;
    const LayerPtrs p = layer_ptrs(h);
    const int C = (int)ch_atom.size() - 1;
    mk.mark(5);
    const bool last = t == md.T - 1;
    int rcode = h->dense_tc
                    ? launch_dense_tc_bwd(ctx, md, h->ld[t], p.wttab + (size_t)t * md.S, (const DenseTile *)h->tiles.p, h->n_tiles,
                                          (const int32_t *)h->sp_list.p, p.zst + t * p.zstride, h->zs,
                                          last ? nullptr : (const float *)h->cbar.p, md.nphip, (float *)h->Qbuf.p, h->mlp_tf32)
                    : launch_dense_bwd(ctx, md, h->ld[t], p.wtab + (size_t)t * md.S, (const DenseTile *)h->tiles.p, h->n_tiles,
                                       (const int32_t *)h->sp_list.p, p.zst + t * p.zstride, h->zs,
                                       last ? nullptr : (const float *)h->cbar.p, md.nphip, (float *)h->Qbuf.p);
    if (rcode) return set_err(h, rcode, "dense backward: unsupported MLP shape or shared-memory size");
    launch_gram_bwd(ctx, md, N, (const int32_t *)h->sp_list.p, p.gram_tiles, h->n_tiles, p.b + t * p.bstride, (const float *)h->Qbuf.p,
                    (float *)h->bbar.p);
    // ghost atoms of a decomposed run are not centres on this rank: their rows of bbar are zero (their edges belong
    // to the owning rank, "local parts computed in place")
    if (h->have_halo && N > 0)
        LAUNCH(ctx, k_zero_halo_rows, (unsigned)N, 64, 0, (float *)h->bbar.p, md.NB, N, (const int32_t *)h->perm.p,
               (const uint8_t *)h->halo_caller.p);
    mk.mark(6);
    for (int c = 0; c < C; ++c) {
        if (c > 0) mk.mark(6);
        rcode = launch_edge_bwd(ctx, md, t, N, (const int64_t *)h->rc_ptr.p, (const uint32_t *)h->col_rc.p,
                                (const float4 *)h->geom.p, p.c_ext + t * p.cstride, (const float *)h->rcen.p,
                                (const float *)h->alpha.p, (const float *)h->bbar.p, (float *)h->kappa.p,
                                (float4 *)h->gst.p, want_vir ? (double *)h->vir_part.p : nullptr, ch_atom[(size_t)c],
                                ch_atom[(size_t)c + 1], ch_edge[(size_t)c], !last);
        if (rcode) return set_err(h, rcode, "edge backward: unsupported (n_gauss, L) combination");
        mk.mark(t >= 1 ? 7 : 9);
        // the top layer stores g_e, the layers below add theirs to it, so the stash holds the sum over the layers after
        // layer 0 and the forces are gathered once, there, with its last chunk; cbar: = for the first chunk, += after
        if (t >= 1 || c == C - 1)
            launch_rev_gather(ctx, N, (const int64_t *)h->rc_ptr.p, (const uint32_t *)h->rev_rc.p, (const float *)h->kappa.p,
                              (const float4 *)h->gst.p, md.nphip, t >= 1, (float *)h->cbar.p, (double *)h->Fc.p,
                              ch_edge[(size_t)c], ch_edge[(size_t)c + 1], t == 0 && c == C - 1, c > 0);
    }
    return REANN_OK;
}

static int enqueue_zero_accumulators(reann *h) {
    if (h->N > 0) {
        CU(h, cudaMemsetAsync(h->Fc.p, 0, sizeof(double) * 3 * (size_t)h->N, h->stream));
        CU(h, cudaMemsetAsync(h->vir_part.p, 0, sizeof(double) * 9 * (size_t)h->n_vir_blocks, h->stream));
    }
    return REANN_OK;
}

static void enqueue_output(reann *h, const LaunchCtx &ctx, Marks &mk, const OutPtrs &o) {
    mk.mark(8);
    launch_output(ctx, h->N, (const int32_t *)h->inv_perm.p, (const double *)h->Fc.p, (const float *)h->Ei.p,
                  (const double *)h->vir_part.p, h->N > 0 ? h->n_vir_blocks : 0, o.dE, o.dF, o.dV, (double *)h->Ei_caller.p,
                  (double *)h->red_scratch.p, h->have_halo ? (const uint8_t *)h->halo_caller.p : nullptr);
}

// everything after the prep: compact list, T forward layers, reverse pass, outputs. ch_atom / ch_edge: stash chunks.
static int enqueue_layers(reann *h, Marks &mk, const OutPtrs &o, bool want_vir, const std::vector<int64_t> &ch_atom,
                          const std::vector<int64_t> &ch_edge, bool guarded) {
    const ModelDims &md = h->md;
    LaunchCtx ctx = h->ctx();
    if (guarded) ctx.skip = (const int32_t *)h->flags.p;
    enqueue_filter_fill(h, ctx);
    for (int t = 0; t < md.T; ++t) {
        RC(enqueue_forward_layer(h, ctx, mk, t));
        if (t + 1 < md.T) enqueue_image_gather(h, ctx, mk, t + 1);
    }
    RC(enqueue_zero_accumulators(h));
    for (int t = md.T - 1; t >= 0; --t) RC(enqueue_backward_layer(h, ctx, mk, t, want_vir, ch_atom, ch_edge));
    enqueue_output(h, ctx, mk, o);
    return REANN_OK;
}

extern "C" int reann_energy_forces(reann_t *h, const double *pos, const double *box9, double *E, double *F,
                                   double *virial) {
    if (!h) return REANN_ERR_ARG;
    if (!h->have_list) return set_err(h, REANN_ERR_NO_NEIGHBORS, "call reann_build_neighbors first");
    RC(check_box(h, box9));
    const ModelDims &md = h->md;
    const int64_t N = h->N;
    const double *d_pos = nullptr;
    RC(device_positions(h, pos, &d_pos));
    h->n_calls++;
    Marks mk{h, {}};
    mk.mark(1);

    const bool E_dev = is_device_ptr(E), F_dev = is_device_ptr(F), V_dev = is_device_ptr(virial);
    double *stage = (double *)h->out_stage.p;
    OutPtrs o;
    o.dE = E ? (E_dev ? E : stage) : stage;
    o.dV = virial ? (V_dev ? virial : stage + 1) : nullptr;
    o.dF = F ? (F_dev ? F : stage + 16) : nullptr;
    o.E_host = E && !E_dev; o.F_host = F && !F_dev && N > 0; o.V_host = virial && !V_dev;

    if (memcmp(box9, h->box_build, sizeof(double) * 9) != 0 && N > 0) RC(do_build(h, d_pos, box9));   // box changed

    // One pass = the whole evaluation enqueued on the current list with NO host round trip in the middle: the skin
    // criterion and the capacity of the compact-edge buffers are checked on the device, the kernels that follow
    // return at once when either fails, and the host looks at the flag word after the evaluation (one stream
    // synchronisation per call) and redoes the step after a rebuild / after growing the buffers. Systems whose
    // kappa stash is held in chunks (config 5) need the chunk boundaries on the host and synchronise once more.
    for (int attempt = 0; attempt < 4; ++attempt) {
        if (N == 0) {
            std::vector<int64_t> ca{0, 0}, ce{0, 0};
            RC(enqueue_layers(h, mk, o, virial != nullptr, ca, ce, false));
            break;
        }
        const bool chunked = h->stash_chunks > 1 || h->cap_rc == 0;
        int32_t flag = 0;
        int64_t n_rc = 0;
        if (!chunked) {
            // ---------------- fast path: a CUDA graph of the steady-state launch sequence (replayed while the list, the
            // buffers and the device addresses the kernels work on stay the same) ----------------
            // host pointers too: the kernels then work on the handle's staging buffers (fixed device addresses), the copies
            // to and from the caller's memory are enqueued around the graph launch
            const bool graphable = h->use_graph && !h->profiling;
            const reann::GraphKey key{d_pos, o.dE, o.dF, o.dV, h->n_rebuilds, h->cap_rc, h->stream};
            if (graphable && h->gexec && memcmp(&key, &h->gkey, sizeof(key)) == 0) {
                CU(h, cudaGraphLaunch(h->gexec, h->stream));
                h->n_launches += h->g_kernels;
            } else {
                const bool capture = graphable;
                const int64_t launches0 = h->n_launches;
                if (capture) { graph_drop(h); CU(h, cudaStreamBeginCapture(h->stream, cudaStreamCaptureModeThreadLocal)); }
                int rcode = enqueue_prep(h, d_pos);
                const std::vector<int64_t> ca{0, N}, ce{0, INT64_MAX};   // one chunk: every edge (the count stays on the device)
                if (rcode == REANN_OK) rcode = enqueue_layers(h, mk, o, virial != nullptr, ca, ce, true);
                if (rcode == REANN_OK && cudaMemcpyAsync(h->h_flags, h->flags.p, 16, cudaMemcpyDeviceToHost, h->stream) != cudaSuccess)
                    rcode = set_err(h, REANN_ERR_CUDA, "copy of the flag word failed");
                if (capture) {
                    cudaGraph_t g = nullptr;
                    const cudaError_t e1 = cudaStreamEndCapture(h->stream, &g);
                    if (rcode != REANN_OK) { if (g) cudaGraphDestroy(g); cudaGetLastError(); return rcode; }
                    if (e1 != cudaSuccess || !g) { cudaGetLastError(); return set_err(h, REANN_ERR_CUDA, "stream capture failed: %s", cudaGetErrorString(e1)); }
                    const cudaError_t e2 = cudaGraphInstantiate(&h->gexec, g, 0);
                    cudaGraphDestroy(g);
                    if (e2 != cudaSuccess) { h->gexec = nullptr; cudaGetLastError(); return set_err(h, REANN_ERR_CUDA, "graph instantiation failed: %s", cudaGetErrorString(e2)); }
                    h->gkey = key;
                    h->g_kernels = h->n_launches - launches0;
                    CU(h, cudaGraphLaunch(h->gexec, h->stream));
                } else if (rcode != REANN_OK) return rcode;
            }
            if (o.E_host) CU(h, cudaMemcpyAsync(E, stage, 8, cudaMemcpyDeviceToHost, h->stream));
            if (o.V_host) CU(h, cudaMemcpyAsync(virial, stage + 1, 72, cudaMemcpyDeviceToHost, h->stream));
            if (o.F_host) CU(h, cudaMemcpyAsync(F, stage + 16, sizeof(double) * 3 * (size_t)N, cudaMemcpyDeviceToHost, h->stream));
            mk.mark(8);
            CU(h, cudaStreamSynchronize(h->stream));
            flag = h->h_flags[0];
            memcpy(&n_rc, h->h_flags + 2, 8);
        } else {
            // ---------------- chunked / first-call path: read the compact edge count and the chunk boundaries first ----------------
            RC(enqueue_prep(h, d_pos));
            CU(h, cudaMemcpyAsync(h->h_flags, h->flags.p, 16, cudaMemcpyDeviceToHost, h->stream));
            CU(h, cudaStreamSynchronize(h->stream));
            flag = h->h_flags[0];
            memcpy(&n_rc, h->h_flags + 2, 8);
            if (!(flag & FLAG_REBUILD)) {
                RC(ensure_rc_capacity(h, n_rc));
                flag &= ~FLAG_OVERFLOW;
                const int C = h->stash_chunks;
                std::vector<int64_t> ch_atom((size_t)C + 1, 0), ch_edge((size_t)C + 1, 0);
                ch_atom[(size_t)C] = N; ch_edge[(size_t)C] = n_rc;
                if (C > 1) {
                    for (int c = 1; c < C; ++c) ch_atom[(size_t)c] = ((N * c / C) + 3) & ~(int64_t)3;
                    for (int c = 1; c < C; ++c)
                        CU(h, cudaMemcpyAsync(&ch_edge[(size_t)c], (const int64_t *)h->rc_ptr.p + ch_atom[(size_t)c], 8, cudaMemcpyDeviceToHost, h->stream));
                    CU(h, cudaStreamSynchronize(h->stream));
                    int64_t widest = 0;
                    for (int c = 0; c < C; ++c) widest = std::max(widest, ch_edge[(size_t)c + 1] - ch_edge[(size_t)c]);
                    RC(dev_ensure(h, h->kappa, sizeof(float) * (size_t)widest * md.nphip));
                }
                RC(enqueue_layers(h, mk, o, virial != nullptr, ch_atom, ch_edge, false));
                if (o.E_host) CU(h, cudaMemcpyAsync(E, stage, 8, cudaMemcpyDeviceToHost, h->stream));
                if (o.V_host) CU(h, cudaMemcpyAsync(virial, stage + 1, 72, cudaMemcpyDeviceToHost, h->stream));
                if (o.F_host) CU(h, cudaMemcpyAsync(F, stage + 16, sizeof(double) * 3 * (size_t)N, cudaMemcpyDeviceToHost, h->stream));
                mk.mark(8);
                CU(h, cudaStreamSynchronize(h->stream));
            }
        }
        if (flag & FLAG_REBUILD) { RC(do_build(h, d_pos, box9)); mk.m.clear(); mk.mark(1); continue; }   // A4: rebuild, redo
        if (flag & FLAG_OVERFLOW) { RC(ensure_rc_capacity(h, n_rc)); graph_drop(h); mk.m.clear(); mk.mark(1); continue; }
        h->E_rc = n_rc;
        break;
    }
    mk.finish();
    CU(h, cudaGetLastError());
    return REANN_OK;
}

// =============================================================================================
// NEXT-1 groundwork: one rank of a spatially decomposed run (Fig. 3-4). The handle holds the rank's
// local atoms and copies of the other ranks' atoms within rc + skin of its domain (ghost atoms, reann_set_halo); the
// caller drives the layers and moves the two messages of the paper between ranks: forward, c^{t+1} of the ghost
// atoms from their owners; backward, dE/dc^t of the ghost atoms to their owners.
__global__ void k_rows_get(const float *__restrict__ base, int stride, int ncol, const int32_t *__restrict__ inv_perm,
                           const int64_t *__restrict__ idx, int64_t n, float *__restrict__ out) {
    const int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= n * ncol) return;
    const int64_t r = q / ncol; const int c = (int)(q - r * ncol);
    out[q] = base[(int64_t)inv_perm[idx[r]] * stride + c];
}
__global__ void k_rows_put(float *__restrict__ base, int stride, int ncol, const int32_t *__restrict__ inv_perm,
                           const int64_t *__restrict__ idx, int64_t n, const float *__restrict__ in, int add) {
    const int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= n * ncol) return;
    const int64_t r = q / ncol; const int c = (int)(q - r * ncol);
    float *dst = base + (int64_t)inv_perm[idx[r]] * stride + c;      // distinct rows: the caller's indices are unique
    *dst = add ? *dst + in[q] : in[q];
}

static int rows_xfer(reann *h, float *base, int64_t n, const int64_t *idx, float *host, int mode /*0 get, 1 set, 2 add*/) {
    if (n < 0 || (n > 0 && (!idx || !host))) return set_err(h, REANN_ERR_ARG, "bad argument");
    if (n == 0) return REANN_OK;
    for (int64_t k = 0; k < n; ++k)
        if (idx[k] < 0 || idx[k] >= h->N) return set_err(h, REANN_ERR_ARG, "atom index out of range");
    const int nphi = h->md.nphi, stride = h->md.nphip;
    RC(dev_ensure(h, h->xch_idx, sizeof(int64_t) * (size_t)n));
    RC(dev_ensure(h, h->xch_val, sizeof(float) * (size_t)n * nphi));
    LaunchCtx ctx = h->ctx();
    CU(h, cudaMemcpyAsync(h->xch_idx.p, idx, sizeof(int64_t) * (size_t)n, cudaMemcpyHostToDevice, h->stream));
    if (mode == 0) {
        LAUNCH(ctx, k_rows_get, div_up(n * nphi, 256), 256, 0, (const float *)base, stride, nphi, (const int32_t *)h->inv_perm.p,
               (const int64_t *)h->xch_idx.p, n, (float *)h->xch_val.p);
        CU(h, cudaMemcpyAsync(host, h->xch_val.p, sizeof(float) * (size_t)n * nphi, cudaMemcpyDeviceToHost, h->stream));
    } else {
        CU(h, cudaMemcpyAsync(h->xch_val.p, host, sizeof(float) * (size_t)n * nphi, cudaMemcpyHostToDevice, h->stream));
        LAUNCH(ctx, k_rows_put, div_up(n * nphi, 256), 256, 0, base, stride, nphi, (const int32_t *)h->inv_perm.p,
               (const int64_t *)h->xch_idx.p, n, (const float *)h->xch_val.p, mode == 2 ? 1 : 0);
    }
    CU(h, cudaStreamSynchronize(h->stream));
    return REANN_OK;
}

extern "C" int reann_set_halo(reann_t *h, const uint8_t *is_halo) {
    if (!h) return REANN_ERR_ARG;
    if (!is_halo || h->N == 0) { h->have_halo = false; return REANN_OK; }
    RC(dev_ensure(h, h->halo_caller, (size_t)h->N));
    CU(h, cudaMemcpyAsync(h->halo_caller.p, is_halo, (size_t)h->N, cudaMemcpyHostToDevice, h->stream));
    CU(h, cudaStreamSynchronize(h->stream));
    h->have_halo = true;
    return REANN_OK;
}

extern "C" int reann_step_begin(reann_t *h, const double *pos, const double *box9, int want_virial) {
    if (!h) return REANN_ERR_ARG;
    if (!h->have_list) return set_err(h, REANN_ERR_NO_NEIGHBORS, "call reann_build_neighbors first");
    RC(check_box(h, box9));
    const double *d_pos = nullptr;
    RC(device_positions(h, pos, &d_pos));
    h->n_calls++;
    h->step_state = 0;
    if (memcmp(box9, h->box_build, sizeof(double) * 9) != 0 && h->N > 0) RC(do_build(h, d_pos, box9));
    for (int attempt = 0; attempt < 3 && h->N > 0; ++attempt) {
        RC(enqueue_prep(h, d_pos));
        CU(h, cudaMemcpyAsync(h->h_flags, h->flags.p, 16, cudaMemcpyDeviceToHost, h->stream));
        CU(h, cudaStreamSynchronize(h->stream));
        if (h->h_flags[0] & FLAG_REBUILD) { RC(do_build(h, d_pos, box9)); continue; }
        int64_t n_rc = 0;
        memcpy(&n_rc, h->h_flags + 2, 8);
        RC(ensure_rc_capacity(h, n_rc));
        h->E_rc = n_rc;
        break;
    }
    if (h->stash_chunks > 1) return set_err(h, REANN_ERR_UNSUPPORTED, "layer-by-layer calls need the whole per-edge stash in memory");
    enqueue_filter_fill(h, h->ctx());
    RC(enqueue_zero_accumulators(h));
    h->step_state = 1;
    h->step_vir = want_virial != 0;
    CU(h, cudaGetLastError());
    return REANN_OK;
}

extern "C" int reann_step_forward(reann_t *h, int t) {
    if (!h) return REANN_ERR_ARG;
    if (h->step_state != 1 || t < 0 || t >= h->md.T) return set_err(h, REANN_ERR_ARG, "reann_step_forward: out of sequence or bad layer");
    Marks mk{h, {}};
    const LaunchCtx ctx = h->ctx();
    if (t >= 1) enqueue_image_gather(h, ctx, mk, t);      // periodic images follow the (possibly just received) c^t rows
    RC(enqueue_forward_layer(h, ctx, mk, t));
    CU(h, cudaGetLastError());
    return REANN_OK;
}

extern "C" int reann_coeff_get(reann_t *h, int t, int64_t n, const int64_t *idx, float *out) {
    if (!h) return REANN_ERR_ARG;
    if (h->step_state == 0 || t < 0 || t >= h->md.T) return set_err(h, REANN_ERR_ARG, "reann_coeff_get: out of sequence or bad layer");
    return rows_xfer(h, (float *)h->c_ext.p + (size_t)t * h->n_ext * h->md.nphip, n, idx, out, 0);
}
extern "C" int reann_coeff_set(reann_t *h, int t, int64_t n, const int64_t *idx, const float *in) {
    if (!h) return REANN_ERR_ARG;
    if (h->step_state != 1 || t < 1 || t >= h->md.T) return set_err(h, REANN_ERR_ARG, "reann_coeff_set: out of sequence or bad layer");
    return rows_xfer(h, (float *)h->c_ext.p + (size_t)t * h->n_ext * h->md.nphip, n, idx, const_cast<float *>(in), 1);
}

extern "C" int reann_step_backward(reann_t *h, int t) {
    if (!h) return REANN_ERR_ARG;
    if (h->step_state == 0 || t < 0 || t >= h->md.T) return set_err(h, REANN_ERR_ARG, "reann_step_backward: out of sequence or bad layer");
    h->step_state = 2;
    Marks mk{h, {}};
    const std::vector<int64_t> ca{0, h->N}, ce{0, INT64_MAX};
    RC(enqueue_backward_layer(h, h->ctx(), mk, t, h->step_vir, ca, ce));
    CU(h, cudaGetLastError());
    return REANN_OK;
}

extern "C" int reann_cbar_get(reann_t *h, int64_t n, const int64_t *idx, float *out) {
    if (!h) return REANN_ERR_ARG;
    if (h->step_state != 2) return set_err(h, REANN_ERR_ARG, "reann_cbar_get: no reverse layer evaluated yet");
    return rows_xfer(h, (float *)h->cbar.p, n, idx, out, 0);
}
extern "C" int reann_cbar_add(reann_t *h, int64_t n, const int64_t *idx, const float *in) {
    if (!h) return REANN_ERR_ARG;
    if (h->step_state != 2) return set_err(h, REANN_ERR_ARG, "reann_cbar_add: no reverse layer evaluated yet");
    return rows_xfer(h, (float *)h->cbar.p, n, idx, const_cast<float *>(in), 2);
}

extern "C" int reann_step_end(reann_t *h, double *E, double *F, double *virial) {
    if (!h) return REANN_ERR_ARG;
    if (h->step_state == 0) return set_err(h, REANN_ERR_ARG, "reann_step_end: no evaluation in progress");
    const int64_t N = h->N;
    const bool E_dev = is_device_ptr(E), F_dev = is_device_ptr(F), V_dev = is_device_ptr(virial);
    double *stage = (double *)h->out_stage.p;
    OutPtrs o;
    o.dE = E ? (E_dev ? E : stage) : stage;
    o.dV = (virial && h->step_vir) ? (V_dev ? virial : stage + 1) : nullptr;
    o.dF = F ? (F_dev ? F : stage + 16) : nullptr;
    Marks mk{h, {}};
    enqueue_output(h, h->ctx(), mk, o);
    if (E && !E_dev) CU(h, cudaMemcpyAsync(E, stage, 8, cudaMemcpyDeviceToHost, h->stream));
    if (o.dV && !V_dev) CU(h, cudaMemcpyAsync(virial, stage + 1, 72, cudaMemcpyDeviceToHost, h->stream));
    if (F && !F_dev && N > 0) CU(h, cudaMemcpyAsync(F, stage + 16, sizeof(double) * 3 * (size_t)N, cudaMemcpyDeviceToHost, h->stream));
    CU(h, cudaStreamSynchronize(h->stream));
    h->step_state = 0;
    CU(h, cudaGetLastError());
    return REANN_OK;
}

extern "C" int reann_get_neighbors(reann_t *h, int64_t *n_edges, int64_t *row_ptr, int32_t *j, int8_t *shift) {
    if (!h) return REANN_ERR_ARG;
    if (h->N == 0) { if (n_edges) *n_edges = 0; if (row_ptr) row_ptr[0] = 0; return REANN_OK; }
    return neighbor_export(h, n_edges, row_ptr, j, shift);
}

extern "C" int reann_get_neighbor_rows(reann_t *h, int64_t n_sel, const int64_t *atoms, int64_t *row_ptr, int32_t *j,
                                       int8_t *shift) {
    if (!h) return REANN_ERR_ARG;
    return neighbor_export_rows(h, n_sel, atoms, row_ptr, j, shift);
}

extern "C" int reann_get_stats(reann_t *h, reann_stats_t *out) {
    if (!h || !out) return REANN_ERR_ARG;
    memset(out, 0, sizeof(*out));
    out->n_atoms = h->N; out->n_ext = h->n_ext; out->n_edges_list = h->E_list; out->n_edges_rc = h->E_rc;
    out->n_rebuilds = h->n_rebuilds; out->n_calls = h->n_calls; out->n_launches = h->n_launches;
    out->ms_build = h->ms[0]; out->ms_prep = h->ms[1]; out->ms_edge_fwd = h->ms[2]; out->ms_dense_fwd = h->ms[3];
    out->ms_gather = h->ms[4]; out->ms_dense_bwd = h->ms[5]; out->ms_edge_bwd = h->ms[6]; out->ms_rev_gather = h->ms[7];
    out->ms_output = h->ms[8]; out->n_profiled_calls = h->n_prof_calls; out->bytes_device = h->bytes_device;
    out->ms_rev_gather_t0 = h->ms[9]; out->stash_chunks = h->stash_chunks;
    return REANN_OK;
}

extern "C" int reann_get_atomic_energies(reann_t *h, double *Ei) {
    if (!h || !Ei) return REANN_ERR_ARG;
    if (!h->have_list || h->n_calls == 0) return set_err(h, REANN_ERR_NO_NEIGHBORS, "no evaluation yet");
    if (h->N == 0) return REANN_OK;
    CU(h, cudaMemcpyAsync(Ei, h->Ei_caller.p, sizeof(double) * (size_t)h->N,
                          is_device_ptr(Ei) ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, h->stream));
    CU(h, cudaStreamSynchronize(h->stream));
    return REANN_OK;
}

extern "C" int reann_verlet(reann_t *h, double *pos, double *vel, const double *F, const double *inv_mass, double dt,
                            double acc_unit, int drift) {
    if (!h || !pos || !vel || !F || !inv_mass) return REANN_ERR_ARG;
    if (!is_device_ptr(pos) || !is_device_ptr(vel) || !is_device_ptr(F) || !is_device_ptr(inv_mass))
        return set_err(h, REANN_ERR_ARG, "reann_verlet takes device pointers");
    launch_verlet(h->ctx(), h->N, pos, vel, F, inv_mass, dt, acc_unit, drift);
    CU(h, cudaGetLastError());
    return REANN_OK;
}

// NEXT-3 (SURVEY.md 8(f); PAPER.md:110-116 NVT MD, :122): n_steps of velocity Verlet (+ Nose-Hoover thermostat) with
// positions, velocities, forces and the thermostat state on the device throughout; see md.cu for the scheme.
extern "C" int reann_md_run(reann_t *h, double *pos, double *vel, const double *inv_mass, const double *box9,
                            int64_t n_steps, double dt, double acc_unit, double kT, double tau, double *F, double *virial,
                            reann_md_state_t *st) {
    if (!h || !st || !pos || !vel || !inv_mass || !F || n_steps < 0 || !(dt > 0.0) || !(acc_unit > 0.0)) return REANN_ERR_ARG;
    if (!is_device_ptr(pos) || !is_device_ptr(vel) || !is_device_ptr(inv_mass) || !is_device_ptr(F) ||
        (virial && !is_device_ptr(virial)))
        return set_err(h, REANN_ERR_ARG, "reann_md_run takes device pointers (pos, vel, inv_mass, F, virial)");
    const bool nvt = kT > 0.0;
    if (nvt && !(tau > 0.0)) return set_err(h, REANN_ERR_ARG, "thermostat time constant tau must be > 0");
    const int64_t N = h->N;
    const double g = 3.0 * (double)N, g_kT = g * kT, Q = nvt ? g_kT * tau * tau : 1.0;
    RC(dev_ensure(h, h->md_state, sizeof(double) * 8));
    RC(dev_ensure(h, h->md_partial, sizeof(double) * (size_t)(md_blocks(N) + 1)));
    RC(dev_ensure(h, h->md_E, sizeof(double)));
    double *state = (double *)h->md_state.p, *part = (double *)h->md_partial.p, *dE = (double *)h->md_E.p;
    const double init[8] = {st->xi, st->vxi, 1.0, 0.0, 1.0, 0.0, 0.0, 0.0};
    CU(h, cudaMemcpyAsync(state, init, sizeof(init), cudaMemcpyHostToDevice, h->stream));
    const int64_t rebuilds0 = h->n_rebuilds;
    if (!h->have_list) RC(reann_build_neighbors(h, pos, box9));
    if (!st->forces_valid) RC(reann_energy_forces(h, pos, box9, dE, F, virial));   // forces at the initial positions
    LaunchCtx ctx = h->ctx();
    launch_md_kick(ctx, N, pos, vel, F, inv_mass, 0.0, acc_unit, 0, nullptr, part);      // sum m v^2 of the initial velocities
    launch_nh_update(ctx, N, part, state, 0.5 * dt, g_kT, Q, acc_unit, n_steps > 0 ? 0 : 2, nvt && n_steps > 0);
    for (int64_t k = 0; k < n_steps; ++k) {
        launch_md_kick(ctx, N, pos, vel, F, inv_mass, dt, acc_unit, 1, state, nullptr);  // (pending scale) half kick + drift
        RC(reann_energy_forces(h, pos, box9, dE, F, virial));
        launch_md_kick(ctx, N, pos, vel, F, inv_mass, dt, acc_unit, 0, nullptr, part);   // half kick + sum m v^2
        launch_nh_update(ctx, N, part, state, 0.5 * dt, g_kT, Q, acc_unit, k + 1 < n_steps ? 1 : 2, nvt);
    }
    launch_md_scale(ctx, N, vel, state);
    double hs[8], pe = 0.0;
    CU(h, cudaMemcpyAsync(hs, state, sizeof(hs), cudaMemcpyDeviceToHost, h->stream));
    CU(h, cudaMemcpyAsync(&pe, dE, sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    CU(h, cudaStreamSynchronize(h->stream));
    st->xi = hs[0]; st->vxi = hs[1];
    st->kinetic = 0.5 * hs[3]; st->potential = pe;
    st->conserved = st->kinetic + pe + (nvt ? 0.5 * Q * hs[1] * hs[1] + g_kT * hs[0] : 0.0);
    st->n_steps_done = n_steps;
    st->n_rebuilds = h->n_rebuilds - rebuilds0;
    CU(h, cudaGetLastError());
    return REANN_OK;
}
