/*
 * dp_oracle.c -- plain CPU fp64 ORACLE for the Deep Potential (se_a) energy / force / virial path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may build, load or call it.  It shares no code,
 * header, table or helper with the CUDA path (paper_2005_00223_b200/csrc); both sides receive the
 * same seeded input arrays from paper_2005_00223_b200/synth.py and nothing else.
 *
 * What it computes, and the passages it follows (PAPER.md = /root/reference/PAPER.md, SC'20
 * "Pushing the limit of molecular dynamics with ab initio accuracy to 100 million atoms with machine
 * learning"; the paper gives the structure in prose only, every formula it omits is the reading listed
 * in DESIGN.md section "Readings" = SURVEY.md section 8(c) N1..N10 / Q1..Q23):
 *
 *   E = sum_i E_i, E_i = fitting_net(D_i), D_i = "product of terms involving the environment matrix
 *   R~ and the embedding matrix G"                                   PAPER.md:51 (section III-B), Fig.1
 *   neighbour list sorted by type, then by distance, each type block padded to its capacity, nearest
 *   N_max kept on overflow                                           PAPER.md:109 (section V-B1)
 *   one 64-bit key per list element (type | distance | index)       PAPER.md:113 (section V-B2)
 *   Environment / ProdForce / ProdViral: env matrix, force, virial
 *   positions and environment matrix in double precision
 *   y = x W + b ; skip (x,x) + ... ; grad tanh = 1 - tanh^2          PAPER.md:133-137 (section V-C)
 *
 * The DP evaluation is an exact function, so the oracle is the plain definition written out with plain
 * loops, in the order N1..N10, fp64 throughout, libm tanh/sqrt, no blocking, no fusion, no BLAS.
 * OpenMP over centre atoms only (each centre is independent).  Compile: gcc -O2 -ffp-contract=off
 * -fopenmp -shared -fPIC (see oracle/build.py).
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): ideal-FCC shell census and per-shell s(r) closed forms
 * (tests/golden/fcc_shells.txt), switch end-point/continuity values, zero-weight closed form
 * E = N*ebias, forces = -grad E by central finite differences, sum F = 0, translation / rotation /
 * permutation invariance, virial = -dE/d(strain) by finite differences and = sum F (x) r for an
 * isolated cluster, continuity of E across rc, an independent numpy (matmul/einsum) evaluation of E on
 * tiny systems, key order == lexicographic order, overflow keeps the nearest.
 * Unpinned: absolute E/F values of the paper's trained models (the paper prints none) and the MIX-32 /
 * MIX-16 deviations of PAPER.md:127 (weights absent) -- "parity unpinned" for those two items only.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int type;           /* model type of neighbour j                        */
    uint64_t q;         /* floor(r2 * 2^29)                                  */
    int j;              /* user index of neighbour                           */
    int shift;          /* image code, only a tie-break between images of j  */
    double d[3];        /* r_j - r_i + image shift                           */
    double r2;
} nb_t;

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* N3: key = type * 2^60 | q * 2^24 | j   (4 / 36 / 24 bits), the binary restatement of the paper's
 * decimal packing type*10^16 + floor(|r|*10^8)*10^6 + j (reading Q11). */
uint64_t oracle_key(int type, double r2, int j) {
    uint64_t q = (uint64_t)floor(r2 * 536870912.0);
    return ((uint64_t)type << 60) | (q << 24) | (uint64_t)j;
}

static int nb_cmp(const void *pa, const void *pb) {
    const nb_t *a = (const nb_t *)pa, *b = (const nb_t *)pb;
    if (a->type != b->type) return a->type < b->type ? -1 : 1;
    if (a->q != b->q) return a->q < b->q ? -1 : 1;
    if (a->j != b->j) return a->j < b->j ? -1 : 1;
    if (a->shift != b->shift) return a->shift < b->shift ? -1 : 1;
    return 0;
}

/* N2: canonical wrap of one coordinate into [0, L). */
double oracle_wrap(double x, double L) {
    double t = x / L;
    double f = floor(t);
    double xw = fma(-f, L, x);
    if (xw >= L) xw -= L;
    if (xw < 0.0) xw += L;
    return xw;
}

/* N4 / N9 (Q2): quintic switch.  w = 1 (r < rc_smth); u^3(-6u^2+15u-10)+1 (rc_smth <= r < rc); 0 beyond.
 * dw = dw/dr. */
double oracle_switch(double r, double rc_smth, double rc, double *dw) {
    if (r < rc_smth) { if (dw) *dw = 0.0; return 1.0; }
    if (r >= rc) { if (dw) *dw = 0.0; return 0.0; }
    double u = (r - rc_smth) / (rc - rc_smth);
    double w = u * u * u * (-6.0 * u * u + 15.0 * u - 10.0) + 1.0;
    if (dw) *dw = -30.0 * u * u * (u - 1.0) * (u - 1.0) / (rc - rc_smth);
    return w;
}

/* N4 / N9 (Q1): env row R~ = s(r) (1, dx/r, dy/r, dz/r), s = w/r, and dR~_c/dd_b. */
void oracle_env_row(const double d[3], double rc_smth, double rc, double Rt[4], double dRt[12]) {
    double r2 = fma(d[2], d[2], fma(d[1], d[1], d[0] * d[0]));
    double r = sqrt(r2);
    double dw, w = oracle_switch(r, rc_smth, rc, &dw);
    double s = w / r;
    double sp = dw / r - w / (r * r);              /* s' */
    Rt[0] = s;
    for (int c = 0; c < 3; ++c) Rt[1 + c] = s * d[c] / r;
    if (dRt) {
        for (int b = 0; b < 3; ++b) dRt[0 * 3 + b] = sp * d[b] / r;
        for (int c = 0; c < 3; ++c)
            for (int b = 0; b < 3; ++b)
                dRt[(1 + c) * 3 + b] = (sp / r - s / (r * r)) * (d[b] / r) * d[c] + (b == c ? s / r : 0.0);
    }
}

/* One dense layer, N5 / N7 layer rule (Q9): z = x W + b, t = tanh(z);
 *   nout == 2 nin : y = (x,x) + t ;  nout == nin : y = x + t ;  else y = t.      W row-major [nin][nout]. */
static void layer_fwd(const double *x, int nin, const double *W, const double *b, int nout,
                      double *t, double *y) {
    for (int o = 0; o < nout; ++o) {
        double z = b[o];
        for (int i = 0; i < nin; ++i) z += x[i] * W[i * nout + o];
        t[o] = tanh(z);
    }
    for (int o = 0; o < nout; ++o) {
        if (nout == 2 * nin) y[o] = x[o % nin] + t[o];
        else if (nout == nin) y[o] = x[o] + t[o];
        else y[o] = t[o];
    }
}

/* Backward of the same layer: given gy = dE/dy and the stored t, return gx = dE/dx. */
static void layer_bwd(const double *gy, const double *t, int nin, const double *W, int nout, double *gx) {
    for (int i = 0; i < nin; ++i) {
        double g = 0.0;
        for (int o = 0; o < nout; ++o) g += gy[o] * (1.0 - t[o] * t[o]) * W[i * nout + o];
        if (nout == 2 * nin) g += gy[i] + gy[i + nin];
        else if (nout == nin) g += gy[i];
        gx[i] = g;
    }
}

/* N5: embedding net of one scalar s -> G[m2].  net = W1 b1 W2 b2 W3 b3.  Exposed for the pins. */
void oracle_embed_net(const double *net, int m0, int m1, int m2, double s, double *G) {
    const double *W1 = net, *b1 = W1 + m0, *W2 = b1 + m0, *b2 = W2 + m0 * m1, *W3 = b2 + m1, *b3 = W3 + m1 * m2;
    double *t = (double *)malloc(sizeof(double) * (size_t)(m0 + m1 + m2 + m0 + m1));
    double *t1 = t, *t2 = t1 + m0, *t3 = t2 + m1, *y1 = t3 + m2, *y2 = y1 + m0;
    layer_fwd(&s, 1, W1, b1, m0, t1, y1);
    layer_fwd(y1, m0, W2, b2, m1, t2, y2);
    layer_fwd(y2, m1, W3, b3, m2, t3, G);
    free(t);
}

/* N7: fitting net of one descriptor D[nd] -> scalar (without ebias).  Exposed for the pins. */
double oracle_fit_net(const double *net, int nd, int f0, int f1, int f2, const double *D) {
    const double *V1 = net, *c1 = V1 + (size_t)nd * f0, *V2 = c1 + f0, *c2 = V2 + f0 * f1, *V3 = c2 + f1,
                 *c3 = V3 + f1 * f2, *v4 = c3 + f2, *c4 = v4 + f2;
    double *buf = (double *)malloc(sizeof(double) * (size_t)(2 * (f0 + f1 + f2)));
    double *t1 = buf, *h1 = t1 + f0, *t2 = h1 + f0, *h2 = t2 + f1, *t3 = h2 + f1, *h3 = t3 + f2;
    layer_fwd(D, nd, V1, c1, f0, t1, h1);
    layer_fwd(h1, f0, V2, c2, f1, t2, h2);
    layer_fwd(h2, f1, V3, c3, f2, t3, h3);
    double e = c4[0];
    for (int o = 0; o < f2; ++o) e += h3[o] * v4[o];
    free(buf);
    return e;
}

/* N2t: general (triclinic) cell, rows a, b, c of the row-major 3 x 3 box H.  Inverse by cofactors, each entry one
 * expression (compiled without contraction), so that any implementation that writes the same expressions gets the same bits. */
static void box_inverse(const double *H, double *Hi, double *vol) {
    const double c00 = H[4] * H[8] - H[5] * H[7], c01 = H[5] * H[6] - H[3] * H[8], c02 = H[3] * H[7] - H[4] * H[6];
    const double det = H[0] * c00 + H[1] * c01 + H[2] * c02;
    Hi[0] = c00 / det; Hi[1] = (H[2] * H[7] - H[1] * H[8]) / det; Hi[2] = (H[1] * H[5] - H[2] * H[4]) / det;
    Hi[3] = c01 / det; Hi[4] = (H[0] * H[8] - H[2] * H[6]) / det; Hi[5] = (H[2] * H[3] - H[0] * H[5]) / det;
    Hi[6] = c02 / det; Hi[7] = (H[1] * H[6] - H[0] * H[7]) / det; Hi[8] = (H[0] * H[4] - H[1] * H[3]) / det;
    *vol = fabs(det);
}

/* N2t canonical wrap of a point into the cell: fractional coordinates t_k = x . Hinv[:,k] (fma chain, x0 first),
 * n_k = floor(t_k), xw = x - n_0 a - n_1 b - n_2 c (fma chain, a first).  Exposed for the pins. */
void oracle_wrap_triclinic(const double *H, const double *x, double *xw) {
    double Hi[9], vol;
    box_inverse(H, Hi, &vol);
    double n[3];
    for (int k = 0; k < 3; ++k) n[k] = floor(fma(x[2], Hi[6 + k], fma(x[1], Hi[3 + k], x[0] * Hi[k])));
    for (int c = 0; c < 3; ++c) xw[c] = fma(-n[2], H[6 + c], fma(-n[1], H[3 + c], fma(-n[0], H[c], x[c])));
}

/* N1-N3: formatted neighbour rows of the listed centres by brute force over all atoms and all images.
 * box: row-major 3 x 3, rows a, b, c.  Orthorhombic (zero off-diagonals): wrap N2 per axis, shift s * L per axis.
 * General cell (reading N2t, the multi-component / arbitrary-cell systems of PAPER.md:107 and the ghost region of
 * Fig. 1(a)): wrap N2t, shift vector v_c = fma(s_2, c_c, fma(s_1, b_c, s_0 * a_c)), image range per axis
 * ceil(rc / h_k) with h_k the height of the cell perpendicular to the other two edges; d = (xw_j - xw_i) + v as in N2.
 * types: MODEL types in [0,T).  nlist_out [ncenters][Nm] user indices, -1 pad.  dvec_out [ncenters][Nm][3]
 * (may be NULL).  ntrunc_out (may be NULL): number of listed centres with at least one over-full block.
 * The only pruning (orthorhombic path) is per axis, |d_axis| >= rc => r2 >= rc*rc, which cannot change the result. */
int oracle_nlist(long N, const double *coords, const int *types, const double *box, double rc, int T,
                 const int *sel, long ncenters, const long *centers, int *nlist_out, double *dvec_out,
                 long *ntrunc_out) {
    const int ortho = !(box[1] != 0 || box[2] != 0 || box[3] != 0 || box[5] != 0 || box[6] != 0 || box[7] != 0);
    const double L[3] = {box[0], box[4], box[8]};
    if (!(rc * rc < 128.0) || T < 1 || T > 16 || N > 16777216) return -1;
    if (ortho && !(L[0] > 0 && L[1] > 0 && L[2] > 0)) return -1;
    int Nm = 0;
    int off[17];
    for (int b = 0; b < T; ++b) { off[b] = Nm; Nm += sel[b]; }
    off[T] = Nm;
    int nimg[3];
    double *xw = (double *)malloc(sizeof(double) * 3 * (size_t)N);
    if (ortho) {
        for (int a = 0; a < 3; ++a) nimg[a] = (int)ceil(rc / L[a]);
        for (long i = 0; i < N; ++i)
            for (int a = 0; a < 3; ++a) xw[3 * i + a] = oracle_wrap(coords[3 * i + a], L[a]);
    } else {
        double Hi[9], vol;
        box_inverse(box, Hi, &vol);
        if (!(vol > 0)) { free(xw); return -2; }
        for (int k = 0; k < 3; ++k) {       /* h_k = V / |e_{k+1} x e_{k+2}| = 1 / |column k of Hinv| */
            const double h = 1.0 / sqrt(Hi[k] * Hi[k] + Hi[3 + k] * Hi[3 + k] + Hi[6 + k] * Hi[6 + k]);
            nimg[k] = (int)ceil(rc / h);
        }
        for (long i = 0; i < N; ++i) oracle_wrap_triclinic(box, coords + 3 * i, xw + 3 * i);
    }
    const double rc2 = rc * rc;
    long ntrunc = 0;
#pragma omp parallel for schedule(dynamic, 4) reduction(+ : ntrunc)
    for (long ic = 0; ic < ncenters; ++ic) {
        const long i = centers ? centers[ic] : ic;
        size_t cap = 1024, n = 0;
        nb_t *nb = (nb_t *)malloc(cap * sizeof(nb_t));
        for (long j = 0; j < N; ++j) {
            for (int sx = -nimg[0]; sx <= nimg[0]; ++sx) {
                double dx = 0.0;
                if (ortho) {
                    dx = (xw[3 * j + 0] - xw[3 * i + 0]) + (double)sx * L[0];
                    if (fabs(dx) >= rc) continue;
                }
                for (int sy = -nimg[1]; sy <= nimg[1]; ++sy) {
                    double dy = 0.0;
                    if (ortho) {
                        dy = (xw[3 * j + 1] - xw[3 * i + 1]) + (double)sy * L[1];
                        if (fabs(dy) >= rc) continue;
                    }
                    for (int sz = -nimg[2]; sz <= nimg[2]; ++sz) {
                        if (j == i && sx == 0 && sy == 0 && sz == 0) continue;
                        double dz;
                        if (ortho) {
                            dz = (xw[3 * j + 2] - xw[3 * i + 2]) + (double)sz * L[2];
                        } else {
                            double v[3];
                            for (int c = 0; c < 3; ++c)
                                v[c] = fma((double)sz, box[6 + c], fma((double)sy, box[3 + c], (double)sx * box[c]));
                            dx = (xw[3 * j + 0] - xw[3 * i + 0]) + v[0];
                            dy = (xw[3 * j + 1] - xw[3 * i + 1]) + v[1];
                            dz = (xw[3 * j + 2] - xw[3 * i + 2]) + v[2];
                        }
                        double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
                        if (!(r2 < rc2)) continue;
                        if (n == cap) { cap *= 2; nb = (nb_t *)realloc(nb, cap * sizeof(nb_t)); }
                        nb[n].type = types[j];
                        nb[n].q = (uint64_t)floor(r2 * 536870912.0);
                        nb[n].j = (int)j;
                        nb[n].shift = ((sx + nimg[0]) * (2 * nimg[1] + 1) + (sy + nimg[1])) * (2 * nimg[2] + 1) + (sz + nimg[2]);
                        nb[n].d[0] = dx; nb[n].d[1] = dy; nb[n].d[2] = dz;
                        nb[n].r2 = r2;
                        ++n;
                    }
                }
            }
        }
        qsort(nb, n, sizeof(nb_t), nb_cmp);
        int *row = nlist_out + (size_t)ic * Nm;
        double *drow = dvec_out ? dvec_out + (size_t)ic * Nm * 3 : NULL;
        for (int k = 0; k < Nm; ++k) row[k] = -1;
        if (drow) memset(drow, 0, sizeof(double) * 3 * (size_t)Nm);
        int filled[16] = {0};
        int over = 0;
        for (size_t p = 0; p < n; ++p) {
            int b = nb[p].type;
            if (filled[b] < sel[b]) {
                int k = off[b] + filled[b]++;
                row[k] = nb[p].j;
                if (drow) { drow[3 * k] = nb[p].d[0]; drow[3 * k + 1] = nb[p].d[1]; drow[3 * k + 2] = nb[p].d[2]; }
            } else over = 1;
        }
        ntrunc += over;
        free(nb);
    }
    free(xw);
    if (ntrunc_out) *ntrunc_out = ntrunc;
    return 0;
}

/* N4-N9 for the listed centres, given their formatted rows (nlist, dvec from oracle_nlist).
 * Outputs: atom_energy_out [ncenters]; gslot_out [ncenters][Nm][3] = dE_i/dd_k (0 for padded slots);
 * optional descr_out [ncenters][m2*axis] (D_i) and amat_out [ncenters][4][m2] (A_i) for the pins. */
int oracle_eval_centers(int T, const int *sel, int m0, int m1, int m2, int axis, int f0, int f1, int f2,
                        const double *embed, const double *fit, const double *ebias, const double *avg,
                        const double *std, double rc, double rc_smth, const int *types, long ncenters,
                        const long *centers, const int *nlist, const double *dvec, double *atom_energy_out,
                        double *gslot_out, double *descr_out, double *amat_out) {
    int Nm = 0;
    int off[17];
    for (int b = 0; b < T; ++b) { off[b] = Nm; Nm += sel[b]; }
    off[T] = Nm;
    const int nd = m2 * axis;
    const size_t ensz = (size_t)m0 + m0 + (size_t)m0 * m1 + m1 + (size_t)m1 * m2 + m2;
    const size_t fnsz = (size_t)nd * f0 + f0 + (size_t)f0 * f1 + f1 + (size_t)f1 * f2 + f2 + f2 + 1;
    const double inv_nm = 1.0 / (double)Nm;
#pragma omp parallel for schedule(dynamic, 1)
    for (long ic = 0; ic < ncenters; ++ic) {
        const long i = centers ? centers[ic] : ic;
        const int a = types[i];
        const int *row = nlist + (size_t)ic * Nm;
        const double *drow = dvec + (size_t)ic * Nm * 3;
        const double *av = avg + 4 * a, *sd = std + 4 * a;
        /* per-row storage */
        double *Rh = (double *)calloc((size_t)Nm * 4, sizeof(double));        /* R^            */
        double *dRt = (double *)calloc((size_t)Nm * 12, sizeof(double));      /* dR~_c / dd_b  */
        double *T1 = (double *)malloc(sizeof(double) * (size_t)Nm * m0), *Y1 = (double *)malloc(sizeof(double) * (size_t)Nm * m0);
        double *T2 = (double *)malloc(sizeof(double) * (size_t)Nm * m1), *Y2 = (double *)malloc(sizeof(double) * (size_t)Nm * m1);
        double *T3 = (double *)malloc(sizeof(double) * (size_t)Nm * m2), *G = (double *)malloc(sizeof(double) * (size_t)Nm * m2);
        double *A = (double *)calloc((size_t)4 * m2, sizeof(double));
        double *D = (double *)malloc(sizeof(double) * (size_t)nd);
        /* N4 + N5, every slot (padded slots have R~ = 0; Q4) */
        for (int b = 0; b < T; ++b) {
            const double *net = embed + ((size_t)a * T + b) * ensz;
            const double *W1 = net, *b1 = W1 + m0, *W2 = b1 + m0, *b2 = W2 + (size_t)m0 * m1, *W3 = b2 + m1, *b3 = W3 + (size_t)m1 * m2;
            for (int k = off[b]; k < off[b + 1]; ++k) {
                double Rt[4] = {0, 0, 0, 0};
                if (row[k] >= 0) oracle_env_row(drow + 3 * k, rc_smth, rc, Rt, dRt + 12 * (size_t)k);
                for (int c = 0; c < 4; ++c) Rh[4 * k + c] = (Rt[c] - av[c]) / sd[c];
                double s = Rh[4 * k];
                layer_fwd(&s, 1, W1, b1, m0, T1 + (size_t)k * m0, Y1 + (size_t)k * m0);
                layer_fwd(Y1 + (size_t)k * m0, m0, W2, b2, m1, T2 + (size_t)k * m1, Y2 + (size_t)k * m1);
                layer_fwd(Y2 + (size_t)k * m1, m1, W3, b3, m2, T3 + (size_t)k * m2, G + (size_t)k * m2);
            }
        }
        /* N6 */
        for (int c = 0; c < 4; ++c)
            for (int m = 0; m < m2; ++m) {
                double acc = 0.0;
                for (int k = 0; k < Nm; ++k) acc += Rh[4 * k + c] * G[(size_t)k * m2 + m];
                A[c * m2 + m] = inv_nm * acc;
            }
        for (int m = 0; m < m2; ++m)
            for (int p = 0; p < axis; ++p) {
                double acc = 0.0;
                for (int c = 0; c < 4; ++c) acc += A[c * m2 + m] * A[c * m2 + p];
                D[m * axis + p] = acc;
            }
        /* N7 */
        const double *net = fit + (size_t)a * fnsz;
        const double *V1 = net, *c1 = V1 + (size_t)nd * f0, *V2 = c1 + f0, *c2 = V2 + (size_t)f0 * f1, *V3 = c2 + f1,
                     *c3 = V3 + (size_t)f1 * f2, *v4 = c3 + f2, *c4 = v4 + f2;
        double *fb = (double *)malloc(sizeof(double) * (size_t)(2 * (f0 + f1 + f2) + f0 + f1 + f2 + nd));
        double *t1 = fb, *h1 = t1 + f0, *t2 = h1 + f0, *h2 = t2 + f1, *t3 = h2 + f1, *h3 = t3 + f2;
        double *g3 = h3 + f2, *g2 = g3 + f2, *g1 = g2 + f1, *gD = g1 + f0;
        layer_fwd(D, nd, V1, c1, f0, t1, h1);
        layer_fwd(h1, f0, V2, c2, f1, t2, h2);
        layer_fwd(h2, f1, V3, c3, f2, t3, h3);
        double e = c4[0];
        for (int o = 0; o < f2; ++o) e += h3[o] * v4[o];
        atom_energy_out[ic] = e + ebias[a];
        if (descr_out) memcpy(descr_out + (size_t)ic * nd, D, sizeof(double) * (size_t)nd);
        if (amat_out) memcpy(amat_out + (size_t)ic * 4 * m2, A, sizeof(double) * 4 * (size_t)m2);
        /* N8 backward: fitting net */
        for (int o = 0; o < f2; ++o) g3[o] = v4[o];
        layer_bwd(g3, t3, f1, V3, f2, g2);
        layer_bwd(g2, t2, f0, V2, f1, g1);
        layer_bwd(g1, t1, nd, V1, f0, gD);
        /* gA[c][m] = sum_p gD[m][p] A[c][p] + [m < axis] sum_m' gD[m'][m] A[c][m'] */
        double *gA = (double *)malloc(sizeof(double) * 4 * (size_t)m2);
        for (int c = 0; c < 4; ++c)
            for (int m = 0; m < m2; ++m) {
                double acc = 0.0;
                for (int p = 0; p < axis; ++p) acc += gD[m * axis + p] * A[c * m2 + p];
                if (m < axis)
                    for (int mp = 0; mp < m2; ++mp) acc += gD[mp * axis + m] * A[c * m2 + mp];
                gA[c * m2 + m] = acc;
            }
        /* N8 per row + N9 */
        double *dG = (double *)malloc(sizeof(double) * (size_t)(m2 + m1 + m0 + 1));
        double *dy2 = dG + m2, *dy1 = dy2 + m1, *ds = dy1 + m0;
        double *gs = gslot_out + (size_t)ic * Nm * 3;
        for (int b = 0; b < T; ++b) {
            const double *en = embed + ((size_t)a * T + b) * ensz;
            const double *W1 = en, *W2 = W1 + 2 * m0, *W3 = W2 + (size_t)m0 * m1 + m1;
            for (int k = off[b]; k < off[b + 1]; ++k) {
                gs[3 * k] = gs[3 * k + 1] = gs[3 * k + 2] = 0.0;
                if (row[k] < 0) continue;       /* padded slot: gradient has no coordinate to act on */
                double dRh[4];
                for (int c = 0; c < 4; ++c) {
                    double acc = 0.0;
                    for (int m = 0; m < m2; ++m) acc += gA[c * m2 + m] * G[(size_t)k * m2 + m];
                    dRh[c] = inv_nm * acc;
                }
                for (int m = 0; m < m2; ++m) {
                    double acc = 0.0;
                    for (int c = 0; c < 4; ++c) acc += gA[c * m2 + m] * Rh[4 * k + c];
                    dG[m] = inv_nm * acc;
                }
                layer_bwd(dG, T3 + (size_t)k * m2, m1, W3, m2, dy2);
                layer_bwd(dy2, T2 + (size_t)k * m1, m0, W2, m1, dy1);
                layer_bwd(dy1, T1 + (size_t)k * m0, 1, W1, m0, ds);
                dRh[0] += ds[0];
                double gRt[4];
                for (int c = 0; c < 4; ++c) gRt[c] = dRh[c] / sd[c];
                for (int bb = 0; bb < 3; ++bb) {
                    double acc = 0.0;
                    for (int c = 0; c < 4; ++c) acc += gRt[c] * dRt[12 * (size_t)k + c * 3 + bb];
                    gs[3 * k + bb] = acc;
                }
            }
        }
        free(dG); free(gA); free(fb); free(D); free(A); free(G); free(T3); free(Y2); free(T2); free(Y1); free(T1);
        free(dRt); free(Rh);
    }
    return 0;
}

/* N10: F_i += g_k ; F_j -= g_k ; Xi_ab -= d_k,a g_k,b.  forces_out [N][3] and virial_out [9] are
 * accumulated into (caller zeroes them).  Serial on purpose. */
void oracle_assemble(long ncenters, const long *centers, int Nm, const int *nlist, const double *dvec,
                     const double *gslot, double *forces_out, double *virial_out) {
    for (long ic = 0; ic < ncenters; ++ic) {
        const long i = centers ? centers[ic] : ic;
        for (int k = 0; k < Nm; ++k) {
            const int j = nlist[(size_t)ic * Nm + k];
            if (j < 0) continue;
            const double *g = gslot + ((size_t)ic * Nm + k) * 3;
            const double *d = dvec + ((size_t)ic * Nm + k) * 3;
            for (int b = 0; b < 3; ++b) {
                forces_out[3 * i + b] += g[b];
                forces_out[3 * (size_t)j + b] -= g[b];
            }
            for (int a = 0; a < 3; ++a)
                for (int b = 0; b < 3; ++b) virial_out[3 * a + b] -= d[a] * g[b];
        }
    }
}
