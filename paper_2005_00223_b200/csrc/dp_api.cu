// C-ABI entry points (include/dp.h): model creation (weight conversion + re-layout into MMA fragment order),
// workspace carve-up (the caller-owned "trunk"), kernel sequencing on the caller's stream.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "embed_mix.cuh"
#include "embed_tc.cuh"
#include "embed_tc2.cuh"

namespace {

inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

long ncell_max_for(long N) { return N < 512 ? 512 : N; }

// NE: capacity of the arrays that a neighbour index can address (NE = N without ghosts, Grid3::cap_ext in ghost mode)
WsLayout ws_layout(const dp_model *m, long N, long NE) {
    WsLayout L{};
    size_t o = 0;
    auto take = [&](size_t bytes) { size_t r = o; o = align256(o + bytes); return r; };
    const bool ghost = NE > N;
    const size_t nbins = (ghost ? 2 : 1) * (size_t)m->T * (size_t)ncell_max_for(N);
    L.status = take(64);
    L.bin_count = take(sizeof(int) * (nbins + 1));
    L.bin_start = take(sizeof(int) * (nbins + 1));
    L.bin_cursor = take(sizeof(int) * nbins);
    L.atom_bin = take(sizeof(int) * (size_t)NE);
    L.tmp_order = take(sizeof(int) * (size_t)NE);
    L.perm = take(sizeof(int) * (size_t)NE);
    L.inv = take(sizeof(int) * (size_t)N);
    L.xs = take(sizeof(double) * 3 * (size_t)NE);
    L.xsf = take(sizeof(float) * 4 * (size_t)N);
    L.scan_tmp = take(sizeof(int) * 2 * ((nbins > (size_t)N ? nbins : (size_t)N) / 4096 + 4));
    L.xw = take(sizeof(double) * 3 * (size_t)NE);
    if (ghost) {
        L.ext_owner = take(sizeof(int) * (size_t)NE);
        L.ext_code = take(sizeof(int) * (size_t)NE);
        L.ext_base = take(sizeof(int) * (size_t)NE);
        L.ext_scode = take(sizeof(int) * (size_t)NE);
        L.gcnt = take(sizeof(int) * (size_t)N);
        L.gstart = take(sizeof(int) * ((size_t)N + 1));
    }
    L.nlist = take(sizeof(int) * (size_t)N * m->Nm);
    L.nreal = take(sizeof(int) * (size_t)N * m->T);
    if (dp_uses_rows(m)) {
        L.rowcnt = take(sizeof(int) * (size_t)N * m->T);
        L.rowstart = take(sizeof(int) * ((size_t)N + 1) * m->T);
        L.rows_rh = take(m->wide_gen ? 0 : sizeof(float) * 4 * (size_t)N * m->Nm);     // block b starts at row offset N*off[b]
        L.rows_id = take(sizeof(int) * 2 * (size_t)N * m->Nm);
        if (m->prec == DP_MIX16) {
            L.rows_g = take(sizeof(float) * 4 * (size_t)N * m->Nm);
            L.fj32 = take(sizeof(float) * 4 * (size_t)NE);
            L.multi_cnt = take(sizeof(int) * DP_MAX_TYPES * DP_MAX_TYPES);
        }
    }
    const size_t esz = m->prec == DP_FP64 ? sizeof(double) : sizeof(float);
    const int nt3 = 2 * ((m->m0 + 3) / 4);          // EmbW<W>::NT3
    L.A = take(esz * (size_t)N * 4 * m->m2);
    if (m->wide) L.gAf = take(m->prec == DP_FP64 ? sizeof(double) * (size_t)N * 4 * m->m2 : 0);      // the wide paths read gA itself
    else if (m->prec == DP_FP64) L.gAf = take(sizeof(double) * (size_t)N * 3 * nt3 * 32);
    else L.gAf = take(sizeof(uint32_t) * (size_t)N * 2 * (2 * nt3) * 32);     // MIX-32 fragments / MIX-16 operand image (smaller)
    L.gscale = take(sizeof(float) * (size_t)N);
    // (MIX-16: buffers 2..6 also hold the gz1 operand images, one per 128-row tile and at least one per type: the pad
    // covers systems with fewer rows than a tile)
    L.fit_act = take(esz * (size_t)N * 240 * 7 + (m->prec == DP_MIX16 ? ((size_t)m->T + 1) * FIT_GZ_TILE_BYTES : 0));
    L.gD = take(esz * (size_t)N * m->m2 * 16);
    L.eatom = take(sizeof(double) * (size_t)N);
    L.fsorted = take(sizeof(double) * 3 * (size_t)NE);
    L.virial = take(sizeof(double) * 16);
    if (m->wide_gen) {  // FP64 / MIX-32 wide nets (wide_gen.cu): row-major activations and per-row vectors over the compact rows
        const size_t rows = (size_t)N * m->Nm;
        L.wide_tab = take(sizeof(int) * 4 * ((size_t)m->T * m->T + 1));
        L.wide_rh = take(esz * 4 * rows);
        L.wide_gr = take(esz * 4 * rows);
        L.wide_t1 = take(esz * rows * m->m0);
        L.wide_y2 = take(esz * rows * m->m1);
        L.wide_t2 = take(esz * rows * m->m1);
        L.wide_t3 = take(esz * rows * m->m2);
    } else if (m->wide) {      // activation images of the wide-network path: 128 rows x 9 W fp16 per tile (wide.cu)
        const size_t tiles = (size_t)wide_tiles_cap(m, N), chunk = 2048;
        L.wide_tab = take(sizeof(int) * 4 * ((size_t)m->T * m->T + 1));
        L.wide_t1 = take(tiles * (m->m0 / 8) * chunk);
        L.wide_y2 = take(tiles * (m->m1 / 8) * chunk);
        L.wide_t2 = take(tiles * (m->m1 / 8) * chunk);
        L.wide_t3 = take(tiles * (m->m2 / 8) * chunk);
    }
    L.total = o;
    return L;
}

// row offsets (N * off[b] + prefix sums of the rows per atom) are 32-bit: natoms * max(sel) must stay below 2^31
bool rows_fit_int32(const dp_model *m, long N) {
    for (int b = 0; b < m->T; ++b) if ((long)N * m->sel[b] >= (1L << 31)) return false;
    return true;
}

// Cell grid of one evaluation.  Orthorhombic boxes with every length >= 2 rc take the minimum-image path (nlist.cu);
// everything else (a general cell, or an edge shorter than 2 rc) takes the ghost path (ghost.cu).  false: degenerate box.
// (32, 64, 128) networks: which precision modes have kernels for them
bool paper_shape_supported(dp_precision prec) { return prec == DP_FP64 || prec == DP_MIX16 || prec == DP_MIX32; }

bool make_grid(const dp_model *m, long N, const double *box, Grid3 *g) {
    *g = Grid3{};
    const bool ortho = !(box[1] != 0 || box[2] != 0 || box[3] != 0 || box[5] != 0 || box[6] != 0 || box[7] != 0);
    const double Ls[3] = {box[0], box[4], box[8]};
    const long cap = ncell_max_for(N);
    bool small = false;
    if (ortho)
        for (int a = 0; a < 3; ++a) {
            if (!(Ls[a] > 0.0)) return false;
            if (!(Ls[a] >= 2.0 * m->rc)) small = true;
        }
    if (!ortho || small) {
        // ---- ghost mode.  Inverse by cofactors, one expression per entry: the same expressions as the oracle (reading N2t)
        const double *H = box;
        double *Hi = g->Hinv;
        const double c00 = H[4] * H[8] - H[5] * H[7], c01 = H[5] * H[6] - H[3] * H[8], c02 = H[3] * H[7] - H[4] * H[6];
        const double det = H[0] * c00 + H[1] * c01 + H[2] * c02;
        if (!(std::fabs(det) > 0.0) || !std::isfinite(det)) return false;
        Hi[0] = c00 / det; Hi[1] = (H[2] * H[7] - H[1] * H[8]) / det; Hi[2] = (H[1] * H[5] - H[2] * H[4]) / det;
        Hi[3] = c01 / det; Hi[4] = (H[0] * H[8] - H[2] * H[6]) / det; Hi[5] = (H[2] * H[3] - H[0] * H[5]) / det;
        Hi[6] = c02 / det; Hi[7] = (H[1] * H[6] - H[0] * H[7]) / det; Hi[8] = (H[0] * H[4] - H[1] * H[3]) / det;
        g->ghost = 1; g->ortho = ortho ? 1 : 0; g->reach = 1;
        double images = 1.0, ratio = 1.0;
        for (int k = 0; k < 3; ++k) {
            // h_k: height of the cell perpendicular to the other two edges (= L_k for a diagonal box)
            const double h = ortho ? Ls[k] : 1.0 / std::sqrt(Hi[k] * Hi[k] + Hi[3 + k] * Hi[3 + k] + Hi[6 + k] * Hi[6 + k]);
            const int ni = (int)std::ceil(m->rc / h);
            if (ni > 7) return false;                       // image shifts are packed in 4 bits
            g->nimg[k] = ni;
            const double mk = m->rc / h * (1.0 + 1e-9) + 1e-12;     // slab width in fractional units, with margin
            g->flo[k] = -mk;
            g->nc[k] = (int)std::floor((1.0 + 2.0 * mk) / mk);     // cells of fractional width >= mk: neighbours within +-1 cell
            if (g->nc[k] < 1) g->nc[k] = 1;
            images *= 2.0 * ni + 1.0;
            ratio *= 1.0 + 2.0 * mk;
            g->L[k] = 1e300;                                 // downstream kernels: no minimum-image step
            g->inv_cw[k] = 0.0;
        }
        for (int k = 0; k < 9; ++k) g->H[k] = box[k];
        while ((long)g->nc[0] * g->nc[1] * g->nc[2] > cap) {
            int big = 0;
            for (int a = 1; a < 3; ++a) if (g->nc[a] > g->nc[big]) big = a;
            g->nc[big] -= 1;
        }
        for (int k = 0; k < 3; ++k) g->fcw[k] = (double)g->nc[k] / (1.0 - 2.0 * g->flo[k]);
        g->ncell = g->nc[0] * g->nc[1] * g->nc[2];
        // capacity of the extended arrays: never more than every image of every atom; twice the uniform-density expectation
        // otherwise (an overflow is detected on the device and reported as DP_ENOMEM by dp_status)
        const double all = (double)N * images, est = 2.0 * (double)N * ratio + 1024.0;
        const double ce = all < est ? all : est;
        if (ce > 16777216.0) return false;
        g->cap_ext = (long)ce > N ? (long)ce : N + 1;
        return true;
    }
    // half-width cells (edge >= rc/2, 5 x 5 x 5 neighbourhood: 58 % of the candidates of the 3 x 3 x 3 search) when the grid
    // then has at least 5 cells per axis and fits the bin arrays; else cells of edge >= rc
    // the MD loop's buffered list searches rc + skin (every call of one dp_md_run uses the same grid)
    const double rl = m->rc + (m->list_mode ? m->md_skin : 0.0);
    g->reach = 2;
    g->cap_ext = N;
    for (int a = 0; a < 3; ++a) {
        g->L[a] = Ls[a];
        g->nc[a] = (int)std::floor(Ls[a] / (0.5 * rl * (1.0 + 1e-9)));
        if (g->nc[a] < 5) g->reach = 1;
    }
    if ((long)g->nc[0] * g->nc[1] * g->nc[2] > cap) g->reach = 1;
    if (g->reach == 1)
        for (int a = 0; a < 3; ++a) {
            int nc = (int)std::floor(Ls[a] / (rl * (1.0 + 1e-9)));
            g->nc[a] = nc < 1 ? 1 : nc;
        }
    while ((long)g->nc[0] * g->nc[1] * g->nc[2] > cap) {
        int big = 0;
        for (int a = 1; a < 3; ++a) if (g->nc[a] > g->nc[big]) big = a;
        g->nc[big] -= 1;
    }
    for (int a = 0; a < 3; ++a) g->inv_cw[a] = (double)g->nc[a] / Ls[a];
    g->ncell = g->nc[0] * g->nc[1] * g->nc[2];
    return true;
}

// logical feature maps of the register-chained embedding net (dp_internal.h)
template <typename TW, int W>
void build_embed_frag(const double *net, EmbedNetFrag<TW, W> *out) {
    constexpr int M0 = EmbW<W>::M0, M1 = EmbW<W>::M1, M2E = EmbW<W>::M2E, KC1 = EmbW<W>::KC1, NT2 = EmbW<W>::NT2, NT3 = EmbW<W>::NT3, NT1 = EmbW<W>::NT1;
    auto f2map = [](int nt, int r, int j) { int e = 4 * nt + r; return e < M0 ? e + M0 * j : -1; };
    auto f3map = [&](int nt3, int r, int j3) { int f = f2map(nt3 >> 1, r, nt3 & 1); return f < 0 ? -1 : f + M1 * j3; };
    const double *W1 = net, *b1 = W1 + M0, *W2 = b1 + M0, *b2 = W2 + M0 * M1, *W3 = b2 + M1, *b3 = W3 + M1 * M2E;
    std::memset(out, 0, sizeof(*out));
    for (int kc = 0; kc < KC1; ++kc)
        for (int r = 0; r < 4; ++r) {
            int e = 4 * kc + r;
            if (e < M0) { out->w1[4 * kc + r] = (TW)W1[e]; out->b1[4 * kc + r] = (TW)b1[e]; }
        }
    for (int nt = 0; nt < NT2; ++nt)
        for (int r = 0; r < 4; ++r)
            for (int j = 0; j < 2; ++j) { int f = f2map(nt, r, j); if (f >= 0) out->b2[nt * 8 + 2 * r + j] = (TW)b2[f]; }
    for (int nt = 0; nt < NT3; ++nt)
        for (int r = 0; r < 4; ++r)
            for (int j = 0; j < 2; ++j) { int f = f3map(nt, r, j); if (f >= 0) out->b3[nt * 8 + 2 * r + j] = (TW)b3[f]; }
    for (int kc = 0; kc < KC1; ++kc)
        for (int nt = 0; nt < NT2; ++nt)
            for (int l = 0; l < 32; ++l) {
                int ein = 4 * kc + (l & 3), n = l >> 2, fo = f2map(nt, n >> 1, n & 1);
                if (ein < M0 && fo >= 0) out->W2f[(kc * NT2 + nt) * 32 + l] = (TW)W2[ein * M1 + fo];
            }
    for (int kc = 0; kc < 2 * NT2; ++kc)
        for (int nt3 = 0; nt3 < NT3; ++nt3)
            for (int l = 0; l < 32; ++l) {
                int fin = f2map(kc >> 1, l & 3, kc & 1), n = l >> 2, fo = f3map(nt3, n >> 1, n & 1);
                if (fin >= 0 && fo >= 0) out->W3f[(kc * NT3 + nt3) * 32 + l] = (TW)W3[fin * M2E + fo];
            }
    for (int kc = 0; kc < 2 * NT3; ++kc)
        for (int nt2 = 0; nt2 < NT2; ++nt2)
            for (int l = 0; l < 32; ++l) {
                int fo = f3map(kc >> 1, l & 3, kc & 1), n = l >> 2, fin = f2map(nt2, n >> 1, n & 1);
                if (fin >= 0 && fo >= 0) out->W3Tf[(kc * NT2 + nt2) * 32 + l] = (TW)W3[fin * M2E + fo];
            }
    for (int kc = 0; kc < 2 * NT2; ++kc)
        for (int nt1 = 0; nt1 < NT1; ++nt1)
            for (int l = 0; l < 32; ++l) {
                int fo = f2map(kc >> 1, l & 3, kc & 1), n = l >> 2;
                int kc1 = 2 * nt1 + (n & 1), e = 4 * kc1 + (n >> 1);
                if (kc1 < KC1 && e < M0 && fo >= 0) out->W2Tf[(kc * NT1 + nt1) * 32 + l] = (TW)W2[e * M1 + fo];
            }
}

inline uint32_t hbits2(float x, float y) {
    return (uint32_t)__half_as_ushort(__float2half_rn(x)) | ((uint32_t)__half_as_ushort(__float2half_rn(y)) << 16);
}
// part 0: fp16(x); part 1: fp16(x - fp16(x))
inline float hpart(double x, int part) {
    float xf = (float)x;
    float hi = __half2float(__float2half_rn(xf));
    return part == 0 ? hi : xf - hi;
}

template <int NSW, int W>
void build_embed_frag_h(const double *net, EmbedNetFragH<NSW, W> *out) {
    constexpr int M0 = HW<W>::M0, M1 = HW<W>::M1, M2E = HW<W>::M2E, HNT2 = HW<W>::HNT2, HNT3 = HW<W>::HNT3;
    auto h_f2 = [](int nt, int r, int j) { return ::h_f2<W>(nt, r, j); };
    auto h_f3 = [](int nt3, int r, int j3) { return ::h_f3<W>(nt3, r, j3); };
    const double *W1 = net, *b1 = W1 + M0, *W2 = b1 + M0, *b2 = W2 + M0 * M1, *W3 = b2 + M1, *b3 = W3 + M1 * M2E;
    std::memset(out, 0, sizeof(*out));
    for (int e = 0; e < M0; ++e) { out->w1[e] = (float)W1[e]; out->b1[e] = (float)b1[e]; }
    for (int nt = 0; nt < HNT2; ++nt)
        for (int r = 0; r < 4; ++r)
            for (int j = 0; j < 2; ++j) { int f = h_f2(nt, r, j); if (f >= 0) out->b2[nt * 8 + 2 * r + j] = (float)b2[f]; }
    for (int nt = 0; nt < HNT3; ++nt)
        for (int r = 0; r < 4; ++r)
            for (int j = 0; j < 2; ++j) { int f = h_f3(nt, r, j); if (f >= 0) out->b3[nt * 8 + 2 * r + j] = (float)b3[f]; }
    auto w2 = [&](int e, int f) { return (e >= 0 && e < M0 && f >= 0) ? W2[e * M1 + f] : 0.0; };
    auto w3 = [&](int fi, int fo) { return (fi >= 0 && fo >= 0) ? W3[fi * M2E + fo] : 0.0; };
    for (int p = 0; p < NSW; ++p)
        for (int l = 0; l < 32; ++l) {
            const int r = l & 3, g = l >> 2;
            // layer 2 forward: K natural e = 16 s + 8 h + 2r + {0,1}; N position (nt, g/2, g%2)
            for (int s = 0; s < 2; ++s)
                for (int nt = 0; nt < HNT2; ++nt)
                    for (int h = 0; h < 2; ++h) {
                        int e0 = 16 * s + 8 * h + 2 * r, fo = h_f2(nt, g >> 1, g & 1);
                        out->W2f[p][s][nt][l][h] = hbits2(hpart(w2(e0, fo), p), hpart(w2(e0 + 1, fo), p));
                    }
            // layer 3 forward: K positions of y2 (tile 2s + h, r, j); N position (nt3, g/2, g%2)
            for (int s = 0; s < 4; ++s)
                for (int nt3 = 0; nt3 < HNT3; ++nt3)
                    for (int h = 0; h < 2; ++h) {
                        int t = 2 * s + h;
                        if (t >= HNT2) continue;
                        int fo = h_f3(nt3, g >> 1, g & 1);
                        out->W3f[p][s][nt3][l][h] = hbits2(hpart(w3(h_f2(t, r, 0), fo), p), hpart(w3(h_f2(t, r, 1), fo), p));
                    }
            // layer 3 backward: K positions of G (tile 2s + h, r, j3); N position of y2 (nt2, g/2, g%2)
            for (int s = 0; s < HNT3 / 2; ++s)
                for (int nt2 = 0; nt2 < HNT2; ++nt2)
                    for (int h = 0; h < 2; ++h) {
                        int t = 2 * s + h, fi = h_f2(nt2, g >> 1, g & 1);
                        out->W3Tf[p][s][nt2][l][h] = hbits2(hpart(w3(fi, h_f3(t, r, 0)), p), hpart(w3(fi, h_f3(t, r, 1)), p));
                    }
            // layer 2 backward: K positions of y2 (tile 2s + h, r, j2); N natural e = 8 t1 + g
            for (int s = 0; s < 4; ++s)
                for (int t1 = 0; t1 < 4; ++t1)
                    for (int h = 0; h < 2; ++h) {
                        int t = 2 * s + h;
                        if (t >= HNT2) continue;
                        int e = 8 * t1 + g;
                        out->W2Tf[p][s][t1][l][h] = hbits2(hpart(w2(e, h_f2(t, r, 0)), p), hpart(w2(e, h_f2(t, r, 1)), p));
                    }
        }
}

template <int NSW, int W>
void build_embed_tc(const double *net, EmbedNetTC<NSW> *out) {
    constexpr int M0 = W, M1 = 2 * W, M2E = 4 * W;
    auto tc_e_of_p1 = [](int p1) { return ::tc_e_of_p1<W>(p1); };
    auto tc_f_of_n = [](int n) { return ::tc_f_of_n<W>(n); };
    auto tc_m_of_c3 = [](int c) { return ::tc_m_of_c3<W>(c); };
    const double *W1 = net, *b1 = W1 + M0, *W2 = b1 + M0, *b2 = W2 + M0 * M1, *W3 = b2 + M1, *b3 = W3 + M1 * M2E;
    std::memset(out, 0, sizeof(*out));
    for (int p1 = 0; p1 < TC_K1; ++p1) { int e = tc_e_of_p1(p1); if (e >= 0) { out->w1[p1] = (float)W1[e]; out->b1[p1] = (float)b1[e]; } }
    for (int n = 0; n < TC_N2; ++n) { int f = tc_f_of_n(n); if (f >= 0) out->b2[n] = (float)b2[f]; }
    for (int c = 0; c < TC_N3; ++c) { int m = tc_m_of_c3(c); if (m >= 0) out->b3[c] = (float)b3[m]; }
    auto w2 = [&](int p1, int n) { int e = tc_e_of_p1(p1), f = tc_f_of_n(n); return (e >= 0 && f >= 0) ? W2[e * M1 + f] : 0.0; };
    auto w3 = [&](int n, int c) { int f = tc_f_of_n(n), m = tc_m_of_c3(c); return (f >= 0 && m >= 0) ? W3[f * M2E + m] : 0.0; };
    for (int p = 0; p < NSW; ++p) {
        for (int k = 0; k < TC_K1; ++k) for (int n = 0; n < TC_N2; ++n) out->W2[p][k >> 3][n][k & 7] = __float2half_rn(hpart(w2(k, n), p));
        for (int k = 0; k < TC_N2; ++k) for (int c = 0; c < TC_N3; ++c) out->W3[p][k >> 3][c][k & 7] = __float2half_rn(hpart(w3(k, c), p));
        for (int k = 0; k < TC_N3; ++k) for (int n = 0; n < TC_N2; ++n) out->W3T[p][k >> 3][n][k & 7] = __float2half_rn(hpart(w3(n, k), p));
        for (int k = 0; k < TC_N2; ++k) for (int q = 0; q < TC_K1; ++q) out->W2T[p][k >> 3][q][k & 7] = __float2half_rn(hpart(w2(q, k), p));
    }
}

// MIX-16 operand images of the warpgroup-per-tile kernels (embed_tc2.cuh): fp16 weights ("stored in half precision",
// PAPER.md:125), biases as hi + lo rows multiplied by constant-one columns, residual folds pre-summed in fp64.
template <int W>
void build_embed_tc2(const double *net, EmbedNetTC2<W> *out) {
    constexpr int M0 = T2<W>::M0, M1 = T2<W>::M1, M2E = T2<W>::M2E;
    const double *W1 = net, *b1 = W1 + M0, *W2 = b1 + M0, *b2 = W2 + M0 * M1, *W3 = b2 + M1, *b3 = W3 + M1 * M2E;
    std::memset(out, 0, sizeof(*out));
    for (int e = 0; e < M0; ++e) { out->w1[e] = (float)W1[e]; out->b1[e] = (float)b1[e]; }
    auto h = [](double x) { return __float2half_rn((float)x); };
    for (int k = 0; k < T2_K1; ++k)
        for (int n = 0; n < M1; ++n) {
            double v = 0.0;
            if (k < M0) v = W2[k * M1 + n];
            else if (!T2<W>::ONES_STEP && k == T2_ONE_HI) v = hpart(b2[n], 0);
            else if (!T2<W>::ONES_STEP && k == T2_ONE_LO) v = hpart(b2[n], 1);
            out->W2[k >> 3][n][k & 7] = h(v);
        }
    for (int k = 0; k < T2_K2 + T2_K1; ++k)
        for (int m = 0; m < M2E; ++m) {
            double v = 0.0;
            if (k < M1) v = W3[k * M2E + m];
            else if (k >= T2_K2) {
                const int e = k - T2_K2;
                if (e < M0) v = W3[e * M2E + m] + W3[(e + M0) * M2E + m];
                else if (!T2<W>::ONES_STEP && e == T2_ONE_HI) v = hpart(b3[m], 0);
                else if (!T2<W>::ONES_STEP && e == T2_ONE_LO) v = hpart(b3[m], 1);
            }
            out->W3[k >> 3][m][k & 7] = h(v);
        }
    for (int k = 0; k < M2E; ++k) {          // k = layer-3 feature m
        for (int e = 0; e < M0; ++e) out->W3T[k >> 3][e][k & 7] = h(W3[e * M2E + k] + W3[(e + M0) * M2E + k]);
        for (int f = 0; f < M1; ++f) out->W3T[k >> 3][32 + f][k & 7] = h(W3[f * M2E + k]);
    }
    for (int k = 0; k < M1; ++k)             // k = layer-2 feature f
        for (int e = 0; e < M0; ++e) out->W2T[k >> 3][e][k & 7] = h(W2[e * M1 + k]);
    if (T2<W>::ONES_STEP) {                  // bias rows of the ones step: k = 0 hi part, k = 1 lo part
        for (int n = 0; n < M1; ++n) { out->Bb2[n][0] = h(hpart(b2[n], 0)); out->Bb2[n][1] = h(hpart(b2[n], 1)); }
        for (int m = 0; m < M2E; ++m) { out->Bb3[m][0] = h(hpart(b3[m], 0)); out->Bb3[m][1] = h(hpart(b3[m], 1)); }
    }
}

template <typename Tp>
cudaError_t upload(const std::vector<Tp> &h, void **dev) {
    cudaError_t e = cudaMalloc(dev, h.size() * sizeof(Tp));
    if (e != cudaSuccess) return e;
    return cudaMemcpy(*dev, h.data(), h.size() * sizeof(Tp), cudaMemcpyHostToDevice);
}

__global__ void k_finalize(long N, const int *__restrict__ perm, const double *__restrict__ fsorted,
                           const double *__restrict__ eatom, const double *__restrict__ vir_ws,
                           double *__restrict__ energy, double *__restrict__ eatom_out, double *__restrict__ forces,
                           double *__restrict__ virial) {
    __shared__ double red[8];
    const long s = blockIdx.x * (long)blockDim.x + threadIdx.x;
    double e = 0.0;
    if (s < N) {
        const int u = perm[s];
        e = eatom[s];
        if (eatom_out) eatom_out[u] = e;
        forces[3L * u] = fsorted[3 * s];
        forces[3L * u + 1] = fsorted[3 * s + 1];
        forces[3L * u + 2] = fsorted[3 * s + 2];
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) e += __shfl_xor_sync(0xffffffffu, e, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = e;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) t += red[w];
        atomicAdd(energy, t);
    }
    if (virial && blockIdx.x == 0 && threadIdx.x < 9) virial[threadIdx.x] = vir_ws[threadIdx.x];
}

}  // namespace

cudaError_t launch_finalize(const dp_model *m, long N, char *ws, const WsLayout &L, double *energy, double *eatom,
                            double *forces, double *virial, cudaStream_t st) {
    (void)m;
    k_finalize<<<(unsigned)((N + 255) / 256), 256, 0, st>>>(N, (int *)(ws + L.perm), (double *)(ws + L.fsorted),
                                                           (double *)(ws + L.eatom), (double *)(ws + L.virial), energy,
                                                           eatom, forces, virial);
    return cudaGetLastError();
}

extern "C" {

const char *dp_strerror(int code) {
    switch (code) {
        case DP_OK: return "ok";
        case DP_EINVAL: return "invalid argument";
        case DP_EBOX: return "degenerate box (zero volume, or more than 7 periodic images per axis inside rc)";
        case DP_ENOMEM: return "workspace too small";
        case DP_ETYPE: return "atom type outside type_map";
        case DP_ECUDA: return "CUDA error or no device";
        case DP_ENEIGH: return "too many neighbour candidates for the sort buffer";
        case DP_EUNSUPPORTED: return "precision mode or shape not supported by this build";
        case DP_ESKIN: return "an atom moved more than skin/2 since the buffered neighbour list was built";
        default: return "unknown error";
    }
}

int dp_create(dp_model **out, const dp_weights *w, const int *type_map, int n_type_map, double rc, double rc_smth,
              const int *sel, dp_precision prec) {
    if (!out || !w || !type_map || !sel || n_type_map <= 0) return DP_EINVAL;
    if (!w->embed || !w->fit || !w->ebias || !w->avg || !w->std) return DP_EINVAL;
    const int T = w->ntypes;
    if (T < 1 || T > DP_MAX_TYPES) return DP_EINVAL;
    if (!(rc > 0) || !(rc_smth >= 0) || !(rc_smth < rc) || !(rc * rc < 128.0)) return DP_EINVAL;
    // embedding widths (W, 2 W, 4 W) with W = 25 (BASELINE configs) or W = 32 (the paper's own networks)
    // or the wide nets of the network-size study W = 64, 128, 256, 512 (MIX-16: wide.cu, FP64 / MIX-32: wide_gen.cu)
    const int W0 = w->embed_widths[0];
    const bool wide = W0 == 64 || W0 == 128 || W0 == 256 || W0 == 512;
    if ((W0 != 25 && W0 != 32 && !wide) || w->embed_widths[1] != 2 * W0 || w->embed_widths[2] != 4 * W0 || w->axis != 16 ||
        w->fit_widths[0] != 240 || w->fit_widths[1] != 240 || w->fit_widths[2] != 240)
        return DP_EUNSUPPORTED;
    if (W0 == 32 && !paper_shape_supported(prec)) return DP_EUNSUPPORTED;
    if (prec != DP_FP64 && prec != DP_MIX32 && prec != DP_MIX16) return DP_EINVAL;
    int maxsel = 0, Nm = 0;
    for (int b = 0; b < T; ++b) { if (sel[b] <= 0) return DP_EINVAL; Nm += sel[b]; if (sel[b] > maxsel) maxsel = sel[b]; }
    for (int k = 0; k < n_type_map; ++k) if (type_map[k] >= T) return DP_EINVAL;
    for (int a = 0; a < T; ++a) for (int c = 0; c < 4; ++c) if (!(w->std[4 * a + c] > 0)) return DP_EINVAL;
    int dev = 0, ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return DP_ECUDA;
    if (cudaGetDevice(&dev) != cudaSuccess) return DP_ECUDA;
    dp_model *m = new (std::nothrow) dp_model();
    if (!m) return DP_EINVAL;
    std::memset(m, 0, sizeof(*m));
    m->device = dev;
    m->T = T; m->Nm = Nm; m->axis = 16; m->F = 240; m->rc = rc; m->rc_smth = rc_smth; m->prec = prec;
    m->m0 = W0; m->m1 = 2 * W0; m->m2 = 4 * W0;
    m->wide = wide ? 1 : 0;
    m->wide_gen = (wide && prec != DP_MIX16) ? 1 : 0;
    m->n_type_map = n_type_map;
    for (int b = 0; b < T; ++b) { m->sel[b] = sel[b]; m->off[b + 1] = m->off[b] + sel[b]; }
    int cap = 256;
    while (cap < 2 * maxsel) cap <<= 1;
    if (cap > 4096) cap = 4096;
    if (cap < maxsel) { delete m; return DP_EINVAL; }
    m->sort_cap = cap;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess) { delete m; return DP_ECUDA; }
    m->num_sms = prop.multiProcessorCount;

    cudaError_t e = cudaSuccess;
    auto ok = [&](cudaError_t x) { if (e == cudaSuccess) e = x; };
    std::vector<int> tm(type_map, type_map + n_type_map);
    ok(upload(tm, (void **)&m->type_map_dev));
    const size_t ensz = (size_t)W0 + W0 + (size_t)W0 * 2 * W0 + 2 * W0 + (size_t)2 * W0 * 4 * W0 + 4 * W0;
    if (wide && prec != DP_MIX16) {     // wide nets in FP64 / MIX-32: row-major weights and their transposes (wide_gen.cu)
        const size_t ne = wide_gen_net_elems(W0, prec == DP_FP64), esz = prec == DP_FP64 ? 8 : 4;
        std::vector<char> blk((size_t)T * T * ne * esz);
        for (int ab = 0; ab < T * T; ++ab) wide_gen_build_net(W0, prec == DP_FP64, w->embed + ab * ensz, &blk[(size_t)ab * ne * esz]);
        ok(upload(blk, &m->wide_vec_dev));
    } else if (prec == DP_FP64 && W0 == 32) {
        std::vector<EmbedNetFrag<double, 32>> frags((size_t)T * T);
        for (int ab = 0; ab < T * T; ++ab) build_embed_frag<double, 32>(w->embed + ab * ensz, &frags[ab]);
        ok(upload(frags, &m->embed_frag_dev));
    } else if (prec == DP_FP64) {
        std::vector<EmbedNetFrag<double, 25>> frags((size_t)T * T);
        for (int ab = 0; ab < T * T; ++ab) build_embed_frag<double, 25>(w->embed + ab * ensz, &frags[ab]);
        ok(upload(frags, &m->embed_frag_dev));
    } else if (prec == DP_MIX32) {      // tcgen05 forward (embed_tc.cu), mma.sync backward (embed_mix.cu): weights as hi + lo fp16
        std::vector<EmbedNetTC<2>> nets((size_t)T * T);
        if (W0 == 32) {
            std::vector<EmbedNetFragH<2, 32>> frags((size_t)T * T);
            for (int ab = 0; ab < T * T; ++ab) build_embed_frag_h<2, 32>(w->embed + ab * ensz, &frags[ab]);
            ok(upload(frags, &m->embed_frag_dev));
            for (int ab = 0; ab < T * T; ++ab) build_embed_tc<2, 32>(w->embed + ab * ensz, &nets[ab]);
        } else {
            std::vector<EmbedNetFragH<2, 25>> frags((size_t)T * T);
            for (int ab = 0; ab < T * T; ++ab) build_embed_frag_h<2, 25>(w->embed + ab * ensz, &frags[ab]);
            ok(upload(frags, &m->embed_frag_dev));
            for (int ab = 0; ab < T * T; ++ab) build_embed_tc<2, 25>(w->embed + ab * ensz, &nets[ab]);
        }
        ok(upload(nets, &m->embed_tc_dev));
    } else if (wide) {                  // MIX-16, wide nets: one tcgen05 GEMM per layer (wide.cu)
        const size_t ie = wide_net_img_elems(W0);
        std::vector<float> vec((size_t)T * T * 8 * W0);
        std::vector<__half> img((size_t)T * T * ie);
        for (int ab = 0; ab < T * T; ++ab) wide_build_net(W0, w->embed + ab * ensz, &vec[(size_t)ab * 8 * W0], &img[(size_t)ab * ie]);
        ok(upload(vec, &m->wide_vec_dev));
        ok(upload(img, &m->wide_img_dev));
    } else {                            // MIX-16: warpgroup-per-tile tcgen05 kernels (embed_tc2*.cu)
        if (W0 == 32) {
            std::vector<EmbedNetTC2<32>> nets((size_t)T * T);
            for (int ab = 0; ab < T * T; ++ab) build_embed_tc2<32>(w->embed + ab * ensz, &nets[ab]);
            ok(upload(nets, &m->embed_tc2_dev));
        } else {
            std::vector<EmbedNetTC2<25>> nets((size_t)T * T);
            for (int ab = 0; ab < T * T; ++ab) build_embed_tc2<25>(w->embed + ab * ensz, &nets[ab]);
            ok(upload(nets, &m->embed_tc2_dev));
        }
        // short neighbour rows: the forward's rounding of the activations to one fp16 value averages over too few rows to
        // hold the MIX-16 force tolerance (measured): carry them as hi + lo pairs there
        m->fwd_split = (Nm < 128 && W0 == 25) ? 1 : 0;
        if (m->fwd_split) {
            std::vector<EmbedNetTC<1>> n1((size_t)T * T);
            for (int ab = 0; ab < T * T; ++ab) build_embed_tc<1, 25>(w->embed + ab * ensz, &n1[ab]);
            ok(upload(n1, &m->embed_tc_dev));
        }
    }
    const int ND = m->m2 * 16, F = 240;
    const size_t fnsz = (size_t)ND * F + F + (size_t)F * F + F + (size_t)F * F + F + F + 1;
    std::vector<double> V1((size_t)T * ND * F), V2((size_t)T * F * F), V3((size_t)T * F * F), c1(T * F), c2(T * F),
        c3(T * F), v4(T * F), c4(T);
    for (int a = 0; a < T; ++a) {
        const double *p = w->fit + a * fnsz;
        std::memcpy(&V1[(size_t)a * ND * F], p, sizeof(double) * ND * F); p += (size_t)ND * F;
        std::memcpy(&c1[a * F], p, sizeof(double) * F); p += F;
        std::memcpy(&V2[(size_t)a * F * F], p, sizeof(double) * F * F); p += (size_t)F * F;
        std::memcpy(&c2[a * F], p, sizeof(double) * F); p += F;
        std::memcpy(&V3[(size_t)a * F * F], p, sizeof(double) * F * F); p += (size_t)F * F;
        std::memcpy(&c3[a * F], p, sizeof(double) * F); p += F;
        std::memcpy(&v4[a * F], p, sizeof(double) * F); p += F;
        c4[a] = p[0];
    }
    if (prec == DP_FP64) {
        ok(upload(V1, &m->fitV1_dev)); ok(upload(V2, &m->fitV2_dev)); ok(upload(V3, &m->fitV3_dev));
        ok(upload(c1, &m->fitc1_dev)); ok(upload(c2, &m->fitc2_dev)); ok(upload(c3, &m->fitc3_dev));
        ok(upload(v4, &m->fitv4_dev)); ok(upload(c4, &m->fitc4_dev));
    } else {   // "trained in double precision, and cast": fp32 copies, fp16 rounding happens per MMA operand
        auto f32 = [](const std::vector<double> &v) { return std::vector<float>(v.begin(), v.end()); };
        ok(upload(f32(V1), &m->fitV1_dev)); ok(upload(f32(V2), &m->fitV2_dev)); ok(upload(f32(V3), &m->fitV3_dev));
        ok(upload(f32(c1), &m->fitc1_dev)); ok(upload(f32(c2), &m->fitc2_dev)); ok(upload(f32(c3), &m->fitc3_dev));
        ok(upload(f32(v4), &m->fitv4_dev)); ok(upload(f32(c4), &m->fitc4_dev));
    }
    // MIX-16: tcgen05 fitting GEMMs (fit_tc.cu) take fp16 weight images; activations are carried as hi + lo fp16 pairs
    if (prec == DP_MIX16) {
        std::vector<__half> img((size_t)T * fit_tc_type_elems(ND));
        for (int a = 0; a < T; ++a)
            fit_tc_build_type(ND, &V1[(size_t)a * ND * F], &V2[(size_t)a * F * F], &V3[(size_t)a * F * F], &img[(size_t)a * fit_tc_type_elems(ND)]);
        ok(upload(img, &m->fit_tc_img_dev));
    }
    // MIX-32: the two large fitting products run on the tcgen05 kernels with hi + lo weight images (fit_tc.cu)
    if (prec == DP_MIX32) {
        std::vector<__half> img((size_t)T * fit_tc32_type_elems(ND));
        for (int a = 0; a < T; ++a) fit_tc32_build_type(ND, &V1[(size_t)a * ND * F], &img[(size_t)a * fit_tc32_type_elems(ND)]);
        ok(upload(img, &m->fit_tc_img_dev));
    }
    std::vector<double> avg(w->avg, w->avg + 4 * T), sd(w->std, w->std + 4 * T), eb(w->ebias, w->ebias + T);
    ok(upload(avg, (void **)&m->avg_dev)); ok(upload(sd, (void **)&m->std_dev)); ok(upload(eb, (void **)&m->ebias_dev));
    if (e != cudaSuccess) { dp_destroy(m); return DP_ECUDA; }
    *out = m;
    return DP_OK;
}

void dp_destroy(dp_model *m) {
    if (!m) return;
    void *ptrs[] = {m->wide_vec_dev, m->wide_img_dev, m->type_map_dev, m->embed_frag_dev, m->embed_tc_dev, m->embed_tc2_dev, m->fit_tc_img_dev, m->avg_dev, m->std_dev, m->ebias_dev, m->fitV1_dev, m->fitV2_dev,
                    m->fitV3_dev, m->fitc1_dev, m->fitc2_dev, m->fitc3_dev, m->fitv4_dev, m->fitc4_dev};
    for (void *p : ptrs) if (p) cudaFree(p);
    if (m->ev[0]) for (int k = 0; k < DP_NEVENTS; ++k) cudaEventDestroy(m->ev[k]);
    delete m;
}

size_t dp_workspace_bytes(const dp_model *m, long natoms, const double *box_host) {
    if (!m || natoms <= 0 || natoms > 16777216 || !rows_fit_int32(m, natoms)) return 0;
    if (!box_host) return ws_layout(m, natoms, natoms).total;
    Grid3 g;
    if (!make_grid(m, natoms, box_host, &g)) return 0;
    return ws_layout(m, natoms, g.cap_ext).total;
}

int dp_launches_per_compute(const dp_model *m) {
    if (!m) return 0;
    int n = 6 + 1;                                   // wrap, 3-launch bin scan, scatter, bin sort; list
    if (m->wide_gen) {                               // wide_gen.cu
        n += 3 * m->T;                               // row prefix sums
        n += 6;                                      // environment rows, tile table, layer 1, two GEMMs, contraction
        n += m->prec == DP_FP64 ? 9 : 7;             // FP64: descriptor, 6 GEMMs, energy, gA; MIX-32: first (tcgen05), 4 GEMMs, energy, last (tcgen05)
        if (m->prec == DP_FP64 && m->last_natoms > 0 && fit_f64_splitk(m, m->last_natoms)) n += 1;
        n += 4 + m->T;                               // backward head, two GEMMs, layer 1 + normalisation, force + virial per neighbour type
    } else if (m->prec == DP_FP64) {
        n += 1 + 9 + 1;                              // forward; descriptor, 6 GEMMs, energy, gA; backward (with S8, S9)
        if (m->last_natoms > 0 && fit_f64_splitk(m, m->last_natoms)) n += 1;     // small systems: split-K first layer + bias / tanh
    } else {
        n += 3 * m->T;                               // row prefix sums, one 3-launch scan per neighbour type
        n += 2;                                      // environment rows + tcgen05 forward
        if (m->wide) n += 4 + 3 + 6;                 // tile table, layer 1, two GEMMs, contraction; fitting (3); scale, head, two GEMMs, force + virial, fp32 shares
        else if (m->prec == DP_MIX16) n += 3 + 6;    // first layer, fused 240 x 240 chain, last product; gA fold, tile classes, backward (two launches), force + virial, fp32 shares
        else n += 8 + 1;                             // first layer (tcgen05), 4 GEMMs, energy, last product (tcgen05), gA fragments; backward (with S8, S9)
    }
    return n + 1;                                    // finalize
}

int dp_compute(dp_model *m, long natoms, const double *coords_dev, const int *types_dev, const double *box_host,
               void *workspace_dev, size_t workspace_bytes, void *cuda_stream, double *energy_dev,
               double *atom_energy_dev, double *forces_dev, double *virial_dev) {
    if (!m || natoms <= 0 || natoms > 16777216 || !coords_dev || !types_dev || !box_host || !workspace_dev ||
        !energy_dev || !forces_dev)
        return DP_EINVAL;
    if (((uintptr_t)workspace_dev & 255) != 0) return DP_EINVAL;
    if (!rows_fit_int32(m, natoms)) return DP_EINVAL;
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != m->device) return DP_ECUDA;    // weights live on the device of dp_create
    Grid3 g;
    if (!make_grid(m, natoms, box_host, &g)) return DP_EBOX;
    if (g.ghost && m->list_mode) return DP_EUNSUPPORTED;        // the buffered list of dp_md_run needs the minimum-image path
    const WsLayout L = ws_layout(m, natoms, g.cap_ext);
    if (workspace_bytes < L.total) return DP_ENOMEM;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    char *ws = (char *)workspace_dev;
    cudaError_t e = cudaSuccess;
    int step = 0;
    auto ok = [&](cudaError_t x) { ++step; if (e == cudaSuccess && x != cudaSuccess) { e = x; m->last_cuda_error = (int)x; m->last_cuda_step = step; } };
    // status word 0 = error flags: cleared per call, except inside one dp_md_run, where they accumulate (dp_status then
    // reports the whole run); the counters behind it are per evaluation
    ok(m->keep_flags ? cudaMemsetAsync(ws + L.status + 4, 0, 60, st) : cudaMemsetAsync(ws + L.status, 0, 64, st));
    ok(cudaMemsetAsync(ws + L.fsorted, 0, sizeof(double) * 3 * (size_t)g.cap_ext, st));
    ok(cudaMemsetAsync(ws + L.virial, 0, sizeof(double) * 16, st));
    ok(cudaMemsetAsync(energy_dev, 0, sizeof(double), st));
    auto mark = [&](int k) { if (m->profile) ok(cudaEventRecord(m->ev[k], st)); };
    mark(0);
    if (g.ghost) {
        ok(launch_build_ghost(m, natoms, coords_dev, types_dev, g, ws, L, st));
        ok(launch_nlist_ghost(m, natoms, g, ws, L, st));
    } else {
        ok(m->list_mode == 2 ? launch_regather(m, natoms, coords_dev, g, ws, L, st)
                             : launch_build_cells(m, natoms, coords_dev, types_dev, g, ws, L, st));
        ok(launch_nlist(m, natoms, g, ws, L, st));
    }
    mark(1);
    const bool f64 = m->prec == DP_FP64;
    const bool m16 = m->prec == DP_MIX16;
    ok(m->wide_gen ? launch_embed_fwd_wide_gen(m, natoms, g, ws, L, st)
           : f64 ? launch_embed_fwd_f64(m, natoms, g, ws, L, st)
           : m->wide ? launch_embed_fwd_wide(m, natoms, g, ws, L, st)
           : (m16 && !m->fwd_split ? launch_embed_fwd_tc2(m, natoms, g, ws, L, st) : launch_embed_fwd_tc(m, natoms, g, ws, L, st)));
    mark(2);
    ok(f64 ? launch_fit_f64(m, natoms, g, ws, L, st) : (m16 ? launch_fit_tc(m, natoms, g, ws, L, st) : launch_fit_mix(m, natoms, g, ws, L, st)));
    mark(3);
    ok(m->wide_gen ? launch_embed_bwd_wide_gen(m, natoms, g, ws, L, st)
           : f64 ? launch_embed_bwd_f64(m, natoms, g, ws, L, st)
           : m->wide ? launch_embed_bwd_wide(m, natoms, g, ws, L, st)
           : (m16 ? launch_embed_bwd_tc2(m, natoms, g, ws, L, st) : launch_embed_bwd_mix(m, natoms, g, ws, L, st)));
    if (g.ghost) ok(launch_fold_ghost(m, natoms, g, ws, L, st));
    mark(4);
    ok(launch_finalize(m, natoms, ws, L, energy_dev, atom_energy_dev, forces_dev, virial_dev, st));
    mark(5);
    m->last_natoms = natoms; m->last_next = g.cap_ext; m->last_ws = workspace_dev; m->last_stream = st;
    return e == cudaSuccess ? DP_OK : DP_ECUDA;
}

const char *dp_last_cuda_error(const dp_model *m, int *step) {
    if (!m) return "no model";
    if (step) *step = m->last_cuda_step;
    return cudaGetErrorString((cudaError_t)m->last_cuda_error);
}

int dp_profile_enable(dp_model *m, int on) {
    if (!m) return DP_EINVAL;
    if (on && !m->ev[0]) {
        for (int k = 0; k < DP_NEVENTS; ++k)
            if (cudaEventCreate(&m->ev[k]) != cudaSuccess) return DP_ECUDA;
    }
    m->profile = on ? 1 : 0;
    return DP_OK;
}

int dp_profile_read(dp_model *m, double *ms_host) {
    if (!m || !ms_host || !m->profile || !m->last_ws) return DP_EINVAL;
    if (cudaEventSynchronize(m->ev[5]) != cudaSuccess) return DP_ECUDA;
    for (int k = 0; k < 5; ++k) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, m->ev[k], m->ev[k + 1]) != cudaSuccess) return DP_ECUDA;
        ms_host[k] = ms;
    }
    ms_host[5] = ms_host[3];
    if (m->prec == DP_MIX16 || m->wide_gen) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, m->ev[6], m->ev[7]) != cudaSuccess) return DP_ECUDA;
        ms_host[5] = ms;
    }
    return DP_OK;
}

int dp_get_nlist(dp_model *m, int *nlist_dev, void *cuda_stream) {
    if (!m || !nlist_dev || !m->last_ws) return DP_EINVAL;
    const WsLayout L = ws_layout(m, m->last_natoms, m->last_next);
    cudaError_t e = launch_get_nlist(m, m->last_natoms, (char *)m->last_ws, L, nlist_dev, (cudaStream_t)cuda_stream);
    return e == cudaSuccess ? DP_OK : DP_ECUDA;
}

int dp_status(dp_model *m, long *n_truncated_atoms) {
    if (!m || !m->last_ws) return DP_EINVAL;
    if (cudaStreamSynchronize(m->last_stream) != cudaSuccess) return DP_ECUDA;
    int st[2] = {0, 0};
    const WsLayout L = ws_layout(m, m->last_natoms, m->last_next);
    if (cudaMemcpy(st, (char *)m->last_ws + L.status, sizeof(st), cudaMemcpyDeviceToHost) != cudaSuccess) return DP_ECUDA;
    if (n_truncated_atoms) *n_truncated_atoms = st[1];
    if (st[0] & 1) return DP_ETYPE;
    if (st[0] & 8) return DP_ENOMEM;         // ghost mode: more periodic images than the extended arrays hold
    if (st[0] & 2) return DP_ENEIGH;
    if (st[0] & 4) return DP_ESKIN;
    return DP_OK;
}

int dp_last_row_counts(dp_model *m, long *rows_forward, long *rows_backward) {
    if (!m || !m->last_ws) return DP_EINVAL;
    if (cudaStreamSynchronize(m->last_stream) != cudaSuccess) return DP_ECUDA;
    unsigned long long c[2] = {0, 0};
    const WsLayout L = ws_layout(m, m->last_natoms, m->last_next);
    if (cudaMemcpy(c, (char *)m->last_ws + L.status + 8, sizeof(c), cudaMemcpyDeviceToHost) != cudaSuccess) return DP_ECUDA;
    if (rows_forward) *rows_forward = (long)c[0];
    if (rows_backward) *rows_backward = (long)c[1];
    return DP_OK;
}

}  // extern "C"
