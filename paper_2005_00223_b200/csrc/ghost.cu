// S1 + S2 for general cells: a triclinic box, or a box with an edge shorter than 2 rc (the "ghost region"
// of Fig. 1(a), which the paper takes from LAMMPS; multi-component systems in arbitrary cells).
//
// The minimum image is not unique in such cells, so the periodic images become explicit GHOST atoms: every image of a local
// atom that lies in the slab of fractional width rc / h_k around the cell is appended to the atom arrays (locals first, in
// the usual (type, cell) order; ghosts behind them, binned on the same cell grid).  The list kernel searches the 27 cells
// around a local atom among locals and ghosts.  Everything downstream (environment matrix, embedding, ProdForce) indexes
// the extended arrays and needs no image arithmetic (the box lengths it sees are 1e300: the minimum-image step is a no-op);
// forces that land on ghosts are folded back onto their owners at the end (the reverse ghost exchange of PAPER.md:141-143,
// inside one GPU).
//
// Bit-exact against the oracle: membership and order are decided with the oracle's arithmetic, d = (xw_j - xw_i) + shift on
// the WRAPPED owner coordinates (reading N2 / N2t of DESIGN.md), not on the pre-added ghost positions.
#include "dp_internal.h"

namespace {

constexpr int CODE_CENTER = 8 | (8 << 4) | (8 << 8);       // shift (0, 0, 0); each component is stored as s + 8, |s| <= 7

__device__ __forceinline__ int pack_code(int sa, int sb, int sc) { return (sa + 8) | ((sb + 8) << 4) | ((sc + 8) << 8); }

// N2 (orthorhombic) / N2t (general cell) canonical wrap; also returns the fractional coordinates of the wrapped point
__device__ __forceinline__ void wrap_point(const Grid3 &g, const double *x, double *xw, double *f) {
    if (g.ortho) {
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const double L = g.H[4 * a];
            const double t = __ddiv_rn(x[a], L);
            const double fl = floor(t);
            double w = __fma_rn(-fl, L, x[a]);
            if (w >= L) w = __dsub_rn(w, L);
            if (w < 0.0) w = __dadd_rn(w, L);
            xw[a] = w;
            f[a] = w / L;
        }
    } else {
        double n[3];
#pragma unroll
        for (int k = 0; k < 3; ++k) n[k] = floor(__fma_rn(x[2], g.Hinv[6 + k], __fma_rn(x[1], g.Hinv[3 + k], __dmul_rn(x[0], g.Hinv[k]))));
#pragma unroll
        for (int c = 0; c < 3; ++c) xw[c] = __fma_rn(-n[2], g.H[6 + c], __fma_rn(-n[1], g.H[3 + c], __fma_rn(-n[0], g.H[c], x[c])));
#pragma unroll
        for (int k = 0; k < 3; ++k) f[k] = xw[0] * g.Hinv[k] + xw[1] * g.Hinv[3 + k] + xw[2] * g.Hinv[6 + k];
    }
}

// shift vector of an image: orthorhombic s * L per axis, general v_c = fma(s_2, c_c, fma(s_1, b_c, s_0 * a_c))  (oracle N2t)
__device__ __forceinline__ void shift_vec(const Grid3 &g, int sa, int sb, int sc, double *v) {
    if (g.ortho) {
        v[0] = __dmul_rn((double)sa, g.H[0]); v[1] = __dmul_rn((double)sb, g.H[4]); v[2] = __dmul_rn((double)sc, g.H[8]);
    } else {
#pragma unroll
        for (int c = 0; c < 3; ++c) v[c] = __fma_rn((double)sc, g.H[6 + c], __fma_rn((double)sb, g.H[3 + c], __dmul_rn((double)sa, g.H[c])));
    }
}

__device__ __forceinline__ bool in_region(const Grid3 &g, const double *f) {
    return f[0] > g.flo[0] && f[0] < 1.0 - g.flo[0] && f[1] > g.flo[1] && f[1] < 1.0 - g.flo[1] && f[2] > g.flo[2] && f[2] < 1.0 - g.flo[2];
}

__device__ __forceinline__ int cell_index(const Grid3 &g, const double *f) {
    int c[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        int v = (int)floor((f[k] - g.flo[k]) * g.fcw[k]);
        c[k] = v < 0 ? 0 : (v >= g.nc[k] ? g.nc[k] - 1 : v);
    }
    return (c[0] * g.nc[1] + c[1]) * g.nc[2] + c[2];
}

// pass 1: wrap, count the images of every atom that fall into the extended region
__global__ void k_gwrap(long N, const double *__restrict__ coords, const __grid_constant__ Grid3 g, double *__restrict__ xw,
                        int *__restrict__ gcnt) {
    const long i = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (i >= N) return;
    const double x[3] = {coords[3 * i], coords[3 * i + 1], coords[3 * i + 2]};
    double w[3], f[3];
    wrap_point(g, x, w, f);
    xw[3 * i] = w[0]; xw[3 * i + 1] = w[1]; xw[3 * i + 2] = w[2];
    int n = 0;
    for (int sa = -g.nimg[0]; sa <= g.nimg[0]; ++sa)
        for (int sb = -g.nimg[1]; sb <= g.nimg[1]; ++sb)
            for (int sc = -g.nimg[2]; sc <= g.nimg[2]; ++sc) {
                if (sa == 0 && sb == 0 && sc == 0) continue;
                const double fs[3] = {f[0] + sa, f[1] + sb, f[2] + sc};
                n += in_region(g, fs) ? 1 : 0;
            }
    gcnt[i] = n;
}

// pass 2: local items u = i and ghost items u = N + gstart[i] + k: position, owner, image code, bin
__global__ void k_gfill(long N, int T, const int *__restrict__ types, const int *__restrict__ type_map, int n_type_map,
                        const __grid_constant__ Grid3 g, const int *__restrict__ gstart, double *__restrict__ xw,
                        int *__restrict__ owner, int *__restrict__ code, int *__restrict__ atom_bin, int *__restrict__ bin_count,
                        int *__restrict__ status) {
    const long i = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (i == 0) {
        const long tot = N + gstart[N];
        status[6] = (int)(tot < g.cap_ext ? tot : g.cap_ext);
        if (tot > g.cap_ext) atomicOr(&status[0], 8);
    }
    if (i >= N) return;
    const int ut = types[i];
    int mt = (ut >= 0 && ut < n_type_map) ? type_map[ut] : -1;
    if (mt < 0) { atomicOr(&status[0], 1); mt = 0; }
    const double w[3] = {xw[3 * i], xw[3 * i + 1], xw[3 * i + 2]};
    double f[3];
    if (g.ortho) { f[0] = w[0] / g.H[0]; f[1] = w[1] / g.H[4]; f[2] = w[2] / g.H[8]; }
    else {
#pragma unroll
        for (int k = 0; k < 3; ++k) f[k] = w[0] * g.Hinv[k] + w[1] * g.Hinv[3 + k] + w[2] * g.Hinv[6 + k];
    }
    owner[i] = (int)i;
    code[i] = CODE_CENTER;
    int bin = mt * g.ncell + cell_index(g, f);
    atom_bin[i] = bin;
    atomicAdd(&bin_count[bin], 1);
    long u = N + gstart[i];
    for (int sa = -g.nimg[0]; sa <= g.nimg[0]; ++sa)
        for (int sb = -g.nimg[1]; sb <= g.nimg[1]; ++sb)
            for (int sc = -g.nimg[2]; sc <= g.nimg[2]; ++sc) {
                if (sa == 0 && sb == 0 && sc == 0) continue;
                const double fs[3] = {f[0] + sa, f[1] + sb, f[2] + sc};
                if (!in_region(g, fs)) continue;
                if (u < g.cap_ext) {
                    double v[3];
                    shift_vec(g, sa, sb, sc, v);
                    xw[3 * u] = w[0] + v[0]; xw[3 * u + 1] = w[1] + v[1]; xw[3 * u + 2] = w[2] + v[2];
                    owner[u] = (int)i;
                    code[u] = pack_code(sa, sb, sc);
                    bin = (T + mt) * g.ncell + cell_index(g, fs);
                    atom_bin[u] = bin;
                    atomicAdd(&bin_count[bin], 1);
                }
                ++u;
            }
}

__global__ void k_gscatter(const int *__restrict__ n_ext, const int *__restrict__ atom_bin, const int *__restrict__ bin_start,
                           int *__restrict__ cursor, int *__restrict__ tmp_order) {
    const long u = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (u >= *n_ext) return;
    const int bin = atom_bin[u];
    tmp_order[bin_start[bin] + atomicAdd(&cursor[bin], 1)] = (int)u;
}

// order every bin by item index (reproducible internal order), write the sorted arrays
__global__ void k_gsort(long N, const int *__restrict__ n_ext, const int *__restrict__ atom_bin, const int *__restrict__ bin_start,
                        const int *__restrict__ tmp_order, const double *__restrict__ xw, const int *__restrict__ owner,
                        const int *__restrict__ code, int *__restrict__ perm, int *__restrict__ inv, double *__restrict__ xs,
                        int *__restrict__ scode) {
    const long s = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (s >= *n_ext) return;
    const int u = tmp_order[s];
    const int bin = atom_bin[u];
    const int b0 = bin_start[bin], b1 = bin_start[bin + 1];
    int rank = 0;
    for (int t = b0; t < b1; ++t) rank += tmp_order[t] < u;
    const int dst = b0 + rank;
    perm[dst] = owner[u];                  // sorted item -> USER index of its owner
    scode[dst] = code[u];
    if (u < N) inv[u] = dst;
    xs[3 * (long)dst] = xw[3 * (long)u]; xs[3 * (long)dst + 1] = xw[3 * (long)u + 1]; xs[3 * (long)dst + 2] = xw[3 * (long)u + 2];
}

__global__ void k_gbase(const int *__restrict__ n_ext, const int *__restrict__ perm, const int *__restrict__ inv, int *__restrict__ base) {
    const long e = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (e >= *n_ext) return;
    base[e] = inv[perm[e]];
}

// One warp per local (sorted) atom: exact fp64 test of every item in the 27 cells around it (locals and ghosts of each type),
// 64-bit key, bitonic sort of (key, item) pairs in shared memory, nearest sel[b] kept, -1 padded.
__global__ void __launch_bounds__(128)
k_nlist_ghost(long N, int T, const __grid_constant__ Grid3 g, double rc2, int cap, const int *__restrict__ bin_start,
              const double *__restrict__ xs, const int *__restrict__ perm, const int *__restrict__ base,
              const int *__restrict__ scode, int Nm, const __grid_constant__ TypeTab tt, int *__restrict__ nlist,
              int *__restrict__ nreal, int *__restrict__ rowcnt, int *__restrict__ status) {
    extern __shared__ unsigned long long gk_all[];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const long i = blockIdx.x * 4L + wid;
    if (i >= N) return;
    unsigned long long *keys = gk_all + (size_t)wid * cap;
    int *vals = reinterpret_cast<int *>(gk_all + (size_t)4 * cap) + (size_t)wid * cap;
    const double xi = xs[3 * i], yi = xs[3 * i + 1], zi = xs[3 * i + 2];
    double fi[3];
    if (g.ortho) { fi[0] = xi / g.H[0]; fi[1] = yi / g.H[4]; fi[2] = zi / g.H[8]; }
    else {
#pragma unroll
        for (int k = 0; k < 3; ++k) fi[k] = xi * g.Hinv[k] + yi * g.Hinv[3 + k] + zi * g.Hinv[6 + k];
    }
    const int ci = cell_index(g, fi);
    const int cz = ci % g.nc[2], cy = (ci / g.nc[2]) % g.nc[1], cx = ci / (g.nc[2] * g.nc[1]);
    const unsigned lt = (1u << lane) - 1u;
    bool truncated = false;
    int off = 0;
    for (int b = 0; b < T; ++b) {
        int n = 0;
        for (int ox = -1; ox <= 1; ++ox) {
            const int ax = cx + ox;
            if (ax < 0 || ax >= g.nc[0]) continue;
            for (int oy = -1; oy <= 1; ++oy) {
                const int ay = cy + oy;
                if (ay < 0 || ay >= g.nc[1]) continue;
                for (int oz = -1; oz <= 1; ++oz) {
                    const int az = cz + oz;
                    if (az < 0 || az >= g.nc[2]) continue;
                    const int cell = (ax * g.nc[1] + ay) * g.nc[2] + az;
                    for (int kind = 0; kind < 2; ++kind) {
                        const int bin = (kind * T + b) * g.ncell + cell;
                        const int s0 = bin_start[bin], s1 = bin_start[bin + 1];
                        for (int sb_ = s0; sb_ < s1; sb_ += 32) {
                            const int e = sb_ + lane;
                            bool ok = false;
                            unsigned long long key = 0;
                            if (e < s1 && e != i) {
                                const int o = base[e], cd = scode[e];
                                double v[3];
                                shift_vec(g, (cd & 15) - 8, ((cd >> 4) & 15) - 8, ((cd >> 8) & 15) - 8, v);
                                const double dx = __dadd_rn(__dsub_rn(xs[3 * (long)o], xi), v[0]);
                                const double dy = __dadd_rn(__dsub_rn(xs[3 * (long)o + 1], yi), v[1]);
                                const double dz = __dadd_rn(__dsub_rn(xs[3 * (long)o + 2], zi), v[2]);
                                const double r2 = __fma_rn(dz, dz, __fma_rn(dy, dy, __dmul_rn(dx, dx)));
                                if (r2 < rc2) {
                                    ok = true;
                                    key = (__double2ull_rd(r2 * 536870912.0) << 24) | (unsigned long long)perm[e];
                                }
                            }
                            const unsigned mask = __ballot_sync(0xffffffffu, ok);
                            const int pos = n + __popc(mask & lt);
                            if (ok && pos < cap) { keys[pos] = key; vals[pos] = e; }
                            n += __popc(mask);
                        }
                    }
                }
            }
        }
        if (n > cap) { if (lane == 0) atomicOr(&status[0], 2); n = cap; }
        int P = 32;
        while (P < n) P <<= 1;
        for (int k = n + lane; k < P; k += 32) { keys[k] = ~0ull; vals[k] = -1; }
        __syncwarp();
        for (int k = 2; k <= P; k <<= 1) {
            for (int j = k >> 1; j > 0; j >>= 1) {
                for (int idx = lane; idx < P; idx += 32) {
                    const int ixj = idx ^ j;
                    if (ixj > idx) {
                        const unsigned long long a = keys[idx], c = keys[ixj];
                        const bool asc = (idx & k) == 0;
                        // images of one atom at exactly the same quantised distance share a key: order them by item index
                        const int va = vals[idx], vc = vals[ixj];
                        const bool gt = a > c || (a == c && va > vc);
                        if (gt == asc) { keys[idx] = c; keys[ixj] = a; vals[idx] = vc; vals[ixj] = va; }
                    }
                }
                __syncwarp();
            }
        }
        const int selb = tt.sel[b];
        const int nkeep = n < selb ? n : selb;
        for (int k = lane; k < selb; k += 32) nlist[i * Nm + off + k] = k < nkeep ? vals[k] : -1;
        if (lane == 0) {
            nreal[i * T + b] = nkeep;
            if (rowcnt) rowcnt[(long)b * N + i] = nkeep + (nkeep < selb ? 1 : 0);
        }
        truncated |= n > selb;
        off += selb;
        __syncwarp();
    }
    if (truncated && lane == 0) atomicAdd(&status[1], 1);
}

// forces that landed on ghost items go back to their owners (fp64 atomics; a ghost has exactly one owner)
__global__ void k_gfold(long N, const int *__restrict__ n_ext, const int *__restrict__ base, double *__restrict__ fsorted) {
    const long e = N + blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (e >= *n_ext) return;
    const long o = base[e];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const double v = fsorted[3 * e + c];
        if (v != 0.0) atomicAdd(&fsorted[3 * o + c], v);
    }
}

}  // namespace

cudaError_t launch_build_ghost(const dp_model *m, long N, const double *coords, const int *types, const Grid3 &g, char *ws,
                               const WsLayout &L, cudaStream_t st) {
    const int nbins = 2 * m->T * g.ncell;
    int *status = (int *)(ws + L.status);
    int *cnt = (int *)(ws + L.bin_count), *start = (int *)(ws + L.bin_start), *cursor = (int *)(ws + L.bin_cursor);
    int *gcnt = (int *)(ws + L.gcnt), *gstart = (int *)(ws + L.gstart);
    const int *n_ext = status + 6;
    cudaMemsetAsync(cnt, 0, sizeof(int) * (size_t)(nbins + 1), st);
    cudaMemsetAsync(cursor, 0, sizeof(int) * (size_t)nbins, st);
    const unsigned nb = (unsigned)((N + 255) / 256), nbe = (unsigned)((g.cap_ext + 255) / 256);
    k_gwrap<<<nb, 256, 0, st>>>(N, coords, g, (double *)(ws + L.xw), gcnt);
    dp_launch_scan((int)N, gcnt, gstart, (int *)(ws + L.scan_tmp), st);
    k_gfill<<<nb, 256, 0, st>>>(N, m->T, types, m->type_map_dev, m->n_type_map, g, gstart, (double *)(ws + L.xw),
                                (int *)(ws + L.ext_owner), (int *)(ws + L.ext_code), (int *)(ws + L.atom_bin), cnt, status);
    dp_launch_scan(nbins, cnt, start, (int *)(ws + L.scan_tmp), st);
    k_gscatter<<<nbe, 256, 0, st>>>(n_ext, (int *)(ws + L.atom_bin), start, cursor, (int *)(ws + L.tmp_order));
    k_gsort<<<nbe, 256, 0, st>>>(N, n_ext, (int *)(ws + L.atom_bin), start, (int *)(ws + L.tmp_order), (double *)(ws + L.xw),
                                 (int *)(ws + L.ext_owner), (int *)(ws + L.ext_code), (int *)(ws + L.perm), (int *)(ws + L.inv),
                                 (double *)(ws + L.xs), (int *)(ws + L.ext_scode));
    k_gbase<<<nbe, 256, 0, st>>>(n_ext, (int *)(ws + L.perm), (int *)(ws + L.inv), (int *)(ws + L.ext_base));
    return cudaGetLastError();
}

cudaError_t launch_nlist_ghost(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st) {
    const int cap = m->sort_cap;
    const size_t smem = (size_t)4 * cap * (sizeof(unsigned long long) + sizeof(int));
    DP_SMEM_OPTIN(k_nlist_ghost, 4 * 4096 * 12);
    const TypeTab tt = make_typetab(m);
    k_nlist_ghost<<<(unsigned)((N + 3) / 4), 128, smem, st>>>(N, m->T, g, m->rc * m->rc, cap, (int *)(ws + L.bin_start),
                                                            (double *)(ws + L.xs), (int *)(ws + L.perm), (int *)(ws + L.ext_base),
                                                            (int *)(ws + L.ext_scode), m->Nm, tt, (int *)(ws + L.nlist),
                                                            (int *)(ws + L.nreal), !dp_uses_rows(m) ? nullptr : (int *)(ws + L.rowcnt),
                                                            (int *)(ws + L.status));
    if (dp_uses_rows(m))
        for (int b = 0; b < m->T; ++b)
            dp_launch_scan((int)N, (int *)(ws + L.rowcnt) + (long)b * N, (int *)(ws + L.rowstart) + (long)b * (N + 1), (int *)(ws + L.scan_tmp), st);
    return cudaGetLastError();
}

cudaError_t launch_fold_ghost(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st) {
    (void)m;
    const long ng = g.cap_ext - N;
    if (ng <= 0) return cudaSuccess;
    k_gfold<<<(unsigned)((ng + 255) / 256), 256, 0, st>>>(N, (int *)(ws + L.status) + 6, (int *)(ws + L.ext_base), (double *)(ws + L.fsorted));
    return cudaGetLastError();
}
