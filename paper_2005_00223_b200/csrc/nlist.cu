// S1 + S2 of SURVEY.md section 8(a): canonical wrap, (type, cell) binning, and the formatted neighbour list
// "sorted by type, then by distance, padded to the cut-off number, nearest N_max kept" with one
// 64-bit key per element (binary restatement, reading Q11).  Bit-exact against the
// oracle: the arithmetic that decides list membership and order uses explicit round-to-nearest intrinsics so
// that nvcc cannot contract it differently from the reading N2 of DESIGN.md.
#include "dp_internal.h"

namespace {

__device__ __forceinline__ double wrap_coord(double x, double L) {
    double t = __ddiv_rn(x, L);
    double f = floor(t);
    double xw = __fma_rn(-f, L, x);
    if (xw >= L) xw = __dsub_rn(xw, L);
    if (xw < 0.0) xw = __dadd_rn(xw, L);
    return xw;
}

__device__ __forceinline__ int cell_of(double xw, double inv_cw, int nc) {
    int c = (int)(xw * inv_cw);
    return c < 0 ? 0 : (c >= nc ? nc - 1 : c);
}

__global__ void k_wrap_bin(long N, const double *__restrict__ coords, const int *__restrict__ types,
                           const int *__restrict__ type_map, int n_type_map, Grid3 g, double *__restrict__ xw,
                           int *__restrict__ atom_bin, int *__restrict__ bin_count, int *__restrict__ status) {
    long i = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (i >= N) return;
    int c[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        double w = wrap_coord(coords[3 * i + a], g.L[a]);
        xw[3 * i + a] = w;
        c[a] = cell_of(w, g.inv_cw[a], g.nc[a]);
    }
    int ut = types[i];
    int mt = (ut >= 0 && ut < n_type_map) ? type_map[ut] : -1;
    if (mt < 0) { atomicOr(&status[0], 1); mt = 0; }
    int bin = mt * g.ncell + (c[0] * g.nc[1] + c[1]) * g.nc[2] + c[2];
    atom_bin[i] = bin;
    atomicAdd(&bin_count[bin], 1);
}

// exclusive scan of cnt[0..n) -> start[0..n]; one block, 4 elements per thread per pass.
__global__ void k_scan(int n, const int *__restrict__ cnt, int *__restrict__ start) {
    __shared__ int warp_sums[32];
    __shared__ int carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    for (int base = 0; base < n; base += 4 * blockDim.x) {
        const int i0 = base + 4 * threadIdx.x;
        int v[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) v[k] = i0 + k < n ? cnt[i0 + k] : 0;
        const int tsum = v[0] + v[1] + v[2] + v[3];
        int x = tsum;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int y = __shfl_up_sync(0xffffffffu, x, o);
            if (lane >= o) x += y;
        }
        if (lane == 31) warp_sums[wid] = x;
        __syncthreads();
        if (wid == 0) {
            int s = lane < nw ? warp_sums[lane] : 0;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                int y = __shfl_up_sync(0xffffffffu, s, o);
                if (lane >= o) s += y;
            }
            warp_sums[lane] = s;
        }
        __syncthreads();
        int prefix = carry + (wid ? warp_sums[wid - 1] : 0) + x - tsum;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            if (i0 + k < n) start[i0 + k] = prefix;
            prefix += v[k];
        }
        __syncthreads();
        if (threadIdx.x == blockDim.x - 1) carry = prefix;
        __syncthreads();
    }
    if (threadIdx.x == 0) start[n] = carry;
}

// Two-level scan for long arrays: tile sums, the single-block scan above over the sums, then each tile scans itself.
constexpr int SCAN_TILE = 4096;        // 1024 threads x 4 elements
__global__ void __launch_bounds__(1024) k_scan_sums(int n, const int *__restrict__ cnt, int *__restrict__ sums) {
    __shared__ int ws[32];
    const int i0 = blockIdx.x * SCAN_TILE + 4 * threadIdx.x;
    int v = 0;
#pragma unroll
    for (int k = 0; k < 4; ++k) v += i0 + k < n ? cnt[i0 + k] : 0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x < 32) {
        v = ws[threadIdx.x];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (threadIdx.x == 0) sums[blockIdx.x] = v;
    }
}
__global__ void __launch_bounds__(1024) k_scan_tiles(int n, const int *__restrict__ cnt, const int *__restrict__ tile_start,
                                                      int *__restrict__ start) {
    __shared__ int warp_sums[32];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int i0 = blockIdx.x * SCAN_TILE + 4 * threadIdx.x;
    int v[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) v[k] = i0 + k < n ? cnt[i0 + k] : 0;
    const int tsum = v[0] + v[1] + v[2] + v[3];
    int x = tsum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int y = __shfl_up_sync(0xffffffffu, x, o);
        if (lane >= o) x += y;
    }
    if (lane == 31) warp_sums[wid] = x;
    __syncthreads();
    if (wid == 0) {
        int s = warp_sums[lane];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int y = __shfl_up_sync(0xffffffffu, s, o);
            if (lane >= o) s += y;
        }
        warp_sums[lane] = s;
    }
    __syncthreads();
    int prefix = tile_start[blockIdx.x] + (wid ? warp_sums[wid - 1] : 0) + x - tsum;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        if (i0 + k < n) start[i0 + k] = prefix;
        prefix += v[k];
    }
    if (blockIdx.x == gridDim.x - 1 && threadIdx.x == 0) start[n] = tile_start[gridDim.x];
}
// exclusive scan of cnt[0..n) -> start[0..n] (three launches; tmp holds 2 * (n / SCAN_TILE + 2) ints)
inline void launch_scan(int n, const int *cnt, int *start, int *tmp, cudaStream_t st) {
    const int nt = (n + SCAN_TILE - 1) / SCAN_TILE;
    int *sums = tmp, *tile_start = tmp + nt + 1;
    k_scan_sums<<<nt, 1024, 0, st>>>(n, cnt, sums);
    k_scan<<<1, 1024, 0, st>>>(nt, sums, tile_start);
    k_scan_tiles<<<nt, 1024, 0, st>>>(n, cnt, tile_start, start);
}

__global__ void k_scatter(long N, const int *__restrict__ atom_bin, const int *__restrict__ bin_start,
                          int *__restrict__ cursor, int *__restrict__ tmp_order) {
    long i = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (i >= N) return;
    int bin = atom_bin[i];
    int slot = bin_start[bin] + atomicAdd(&cursor[bin], 1);
    tmp_order[slot] = (int)i;
}

// order every bin by user index (makes the internal order, hence every later summation order, reproducible)
__global__ void k_bin_sort(long N, const int *__restrict__ atom_bin, const int *__restrict__ bin_start,
                           const int *__restrict__ tmp_order, const double *__restrict__ xw, int *__restrict__ perm,
                           int *__restrict__ inv, double *__restrict__ xs, float4 *__restrict__ xsf) {
    long s = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (s >= N) return;
    int u = tmp_order[s];
    int bin = atom_bin[u];
    int b0 = bin_start[bin], b1 = bin_start[bin + 1];
    int rank = 0;
    for (int t = b0; t < b1; ++t) rank += tmp_order[t] < u;
    int dst = b0 + rank;
    perm[dst] = u;
    inv[u] = dst;
    xs[3 * (long)dst + 0] = xw[3 * (long)u + 0];
    xs[3 * (long)dst + 1] = xw[3 * (long)u + 1];
    xs[3 * (long)dst + 2] = xw[3 * (long)u + 2];
    xsf[dst] = make_float4((float)xw[3 * (long)u + 0], (float)xw[3 * (long)u + 1], (float)xw[3 * (long)u + 2], 0.f);
}

__device__ __forceinline__ double min_image(double t, double L, double halfL) {
    double s = t > halfL ? -1.0 : (t < -halfL ? 1.0 : 0.0);
    return __dadd_rn(t, __dmul_rn(s, L));
}

// ---- list kernel ------------------------------------------------------------------------------------------------------
// Bitonic sort of 32 R keys held R per lane (element index = lane * R + r), every merge ascending: the first stage of a
// merge of width k pairs idx with idx ^ (k - 1), the following ones idx with idx ^ j.  Strides below R are register
// exchanges, larger ones warp shuffles; the smaller key always goes to the smaller index (one 64-bit compare per element).
template <int R, typename K>
__device__ __forceinline__ void warp_sort_regs(K (&key)[R], int lane) {
#pragma unroll
    for (int k = 2; k <= 32 * R; k <<= 1) {
        // flip stage
        if (k <= R) {
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const int q = r ^ (k - 1);
                if (q > r) {
                    const K a = key[r], c = key[q];
                    const bool sw = a > c;
                    key[r] = sw ? c : a;
                    key[q] = sw ? a : c;
                }
            }
        } else {
            const int jl = k / R - 1;
            const bool lower = (lane & (k / (2 * R))) == 0;
            K o[R];
#pragma unroll
            for (int r = 0; r < R; ++r) o[r] = __shfl_xor_sync(0xffffffffu, key[R - 1 - r], jl);
#pragma unroll
            for (int r = 0; r < R; ++r) key[r] = ((key[r] < o[r]) == lower) ? key[r] : o[r];
        }
#pragma unroll
        for (int j = k >> 2; j > 0; j >>= 1) {
            if (j < R) {
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const int q = r ^ j;
                    if (q > r) {
                        const K a = key[r], c = key[q];
                        const bool sw = a > c;
                        key[r] = sw ? c : a;
                        key[q] = sw ? a : c;
                    }
                }
            } else {
                const int jl = j / R;
                const bool lower = (lane & jl) == 0;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const K a = key[r];
                    const K o = __shfl_xor_sync(0xffffffffu, a, jl);
                    key[r] = ((a < o) == lower) ? a : o;
                }
            }
        }
    }
}

template <int R>
__device__ __forceinline__ void sort_and_emit(const unsigned long long *keys, const int *sidx, int n, int lane, int selb,
                                              const int *__restrict__ inv, int *__restrict__ out) {
    // Sort 32-bit proxies {top 24 bits of the quantised r^2, position in keys[]} with min / max, fetch the 64-bit keys in
    // that order and verify it; only a warp whose proxies tie (equal r^2 to 2^-17 A^2, e.g. a perfect lattice)
    // re-sorts the 64-bit keys.  The emitted order is always the exact key order.
    unsigned long long key[R];
    uint32_t pk[R];
    bool resorted;
    {
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int idx = lane * R + r;
            pk[r] = idx < n ? (((uint32_t)(keys[idx] >> 36) << 8) | (uint32_t)idx) : 0xFFFFFFFFu;   // key = q << 24 | j, q < 2^36
        }
        warp_sort_regs<R>(pk, lane);
        bool bad = false;
#pragma unroll
        for (int r = 0; r < R; ++r) key[r] = pk[r] != 0xFFFFFFFFu ? keys[pk[r] & 255u] : ~0ull;
#pragma unroll
        for (int r = 0; r + 1 < R; ++r) bad |= key[r] > key[r + 1];
        const unsigned long long nxt = __shfl_down_sync(0xffffffffu, key[0], 1);
        bad |= lane < 31 && key[R - 1] > nxt;
        resorted = __any_sync(0xffffffffu, bad);
        if (resorted) warp_sort_regs<R>(key, lane);
    }
    const int nkeep = n < selb ? n : selb;
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int rank = lane * R + r;
        // sorted-space index of the neighbour: kept beside the key by pass 2 (proxy order), or through inv after a re-sort
        if (rank < selb) out[rank] = rank < nkeep ? (resorted ? inv[(int)(key[r] & 0xFFFFFFull)] : sidx[pk[r] & 255u]) : -1;
    }
    for (int k = 32 * R + lane; k < selb; k += 32) out[k] = -1;
}

// One warp per (sorted) atom.  Pass 1: fp32 distances on the fp32 copy of the coordinates select candidates conservatively
// (margin covers the rounding of the copy), ballot-compacted into shared memory.  Pass 2: the exact test and the 64-bit key
// (canonical fp64 arithmetic of DESIGN.md reading N2) on the few survivors only.  Sort in registers.
//
// Pass 1 walks one flat candidate range: the z cells of an (x, y) column are consecutive bins, so a column is one run of
// sorted atoms (two when it wraps around the box); lane c < 25 looks up the runs of column c, a warp scan turns the run
// lengths into a table {end of the run in the flat range, first atom - start in the flat range}, and the warp then
// tests 32 consecutive flat positions per iteration with every lane busy.
struct NlistF32 {
    float L[3], invL[3];
    float rc2_margin;        // pass-1 radius of the cell search (rc, or rc + skin when the candidates are stored), with margin
    float rc2_margin_rc;     // rc with margin: pass 1 over stored candidates (MODE 2)
};
// conservative fp32 test of sorted atom s against the centre pf (minimum image: d - L rint(d / L), rint through the 1.5 * 2^23 shift)
// WRAP = false: the caller knows that the plain difference is the minimum image (interior centre, see k_nlist2)
template <bool WRAP = true>
__device__ __forceinline__ bool near_f32(const float4 *__restrict__ xsf, int s, const float4 &pf, const NlistF32 &gf, float r2m) {
    const float4 q = __ldg(&xsf[s]);
    float dx = q.x - pf.x, dy = q.y - pf.y, dz = q.z - pf.z;
    if (WRAP) {
        const float tx = fmaf(dx, gf.invL[0], 12582912.f) - 12582912.f;
        const float ty = fmaf(dy, gf.invL[1], 12582912.f) - 12582912.f;
        const float tz = fmaf(dz, gf.invL[2], 12582912.f) - 12582912.f;
        dx = fmaf(-tx, gf.L[0], dx); dy = fmaf(-ty, gf.L[1], dy); dz = fmaf(-tz, gf.L[2], dz);
    }
    return fmaf(dz, dz, fmaf(dy, dy, dx * dx)) < r2m;
}
__device__ __forceinline__ int warp_incl_scan(int v, int lane) {
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const int o = __shfl_up_sync(0xffffffffu, v, d);
        v += lane >= d ? o : 0;
    }
    return v;
}
// MODE 0: every call searches the cells.  MODE 1 / 2: the MD loop's buffered list ("neighbor list with a 2 A
// buffer region ... updated every 50 steps"): MODE 1 searches the cells with rc + skin in pass 1 and also stores the
// survivors (sorted-space atom indices, cap per atom and type); MODE 2 skips the cells and pass 1 and starts from the
// stored candidates.  Pass 2 (exact test, key), sort and truncation are the same every step, so the list stays bit-exact.
template <int MODE>
__global__ void __launch_bounds__(128, 8)
k_nlist2(long N, int T, Grid3 g, double rc2, NlistF32 gf, int cap, const int *__restrict__ bin_start,
         const double *__restrict__ xs, const float4 *__restrict__ xsf, const int *__restrict__ perm,
         const int *__restrict__ inv, int Nm, const __grid_constant__ TypeTab tt, int *__restrict__ nlist, int *__restrict__ nreal,
         int *__restrict__ rowcnt, int *__restrict__ status, int *__restrict__ cand, int *__restrict__ candcnt) {
    extern __shared__ unsigned long long keys_all[];
    __shared__ int2 runtab_all[4][66];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const long i = blockIdx.x * 4L + wid;
    if (i >= N) return;
    unsigned long long *keys = keys_all + (size_t)wid * cap;
    int *sidx = reinterpret_cast<int *>(keys_all + (size_t)4 * cap) + (size_t)wid * cap;   // sorted-space index beside every key
    int2 *runtab = runtab_all[wid];
    const int *sel = tt.sel;
    const double xi = xs[3 * i], yi = xs[3 * i + 1], zi = xs[3 * i + 2];
    const float4 pf = xsf[i];
    const int ii = (int)i;
    const int cx = cell_of(xi, g.inv_cw[0], g.nc[0]), cy = cell_of(yi, g.inv_cw[1], g.nc[1]),
              cz = cell_of(zi, g.inv_cw[2], g.nc[2]);
    const int R_ = g.reach;       // reach 2 is only chosen for grids with >= 5 cells per axis
    const int lo0 = R_ == 2 ? -2 : (g.nc[0] >= 3 ? -1 : 0), hi0 = R_ == 2 ? 2 : (g.nc[0] >= 2 ? 1 : 0);
    const int lo1 = R_ == 2 ? -2 : (g.nc[1] >= 3 ? -1 : 0), hi1 = R_ == 2 ? 2 : (g.nc[1] >= 2 ? 1 : 0);
    const int lo2 = R_ == 2 ? -2 : (g.nc[2] >= 3 ? -1 : 0), hi2 = R_ == 2 ? 2 : (g.nc[2] >= 2 ? 1 : 0);
    const double hx = 0.5 * g.L[0], hy = 0.5 * g.L[1], hz = 0.5 * g.L[2];
    // this lane's column (first z bin of it, relative to the type's bins) and the z cell ranges A (in the box) and B (wrapped)
    const int ny = hi1 - lo1 + 1, ncol = (hi0 - lo0 + 1) * ny;       // <= 25
    int colrel = 0;
    if (lane < ncol) {
        int ax = cx + lo0 + lane / ny; ax += ax < 0 ? g.nc[0] : 0; ax -= ax >= g.nc[0] ? g.nc[0] : 0;
        int ay = cy + lo1 + lane % ny; ay += ay < 0 ? g.nc[1] : 0; ay -= ay >= g.nc[1] ? g.nc[1] : 0;
        colrel = (ax * g.nc[1] + ay) * g.nc[2];
    }
    const int zlo = cz + lo2, zhi = cz + hi2;
    const int za0 = zlo < 0 ? 0 : zlo, za1 = zhi >= g.nc[2] ? g.nc[2] - 1 : zhi;
    int zb0 = 0, zb1 = -1;
    if (zlo < 0) { zb0 = zlo + g.nc[2]; zb1 = g.nc[2] - 1; }
    else if (zhi >= g.nc[2]) { zb0 = 0; zb1 = zhi - g.nc[2]; }
    const unsigned lt = (1u << lane) - 1u;
    // Interior centre: the searched cells do not wrap on any axis and span less than half the box ((reach + 1) cell widths
    // < L / 2), so the plain coordinate difference of every candidate is its minimum image: pass 1 skips the wrap arithmetic.
    const bool interior = cx + lo0 >= 0 && cx + hi0 < g.nc[0] && cy + lo1 >= 0 && cy + hi1 < g.nc[1] && zlo >= 0 && zhi < g.nc[2] &&
                          g.nc[0] > 2 * (R_ + 1) && g.nc[1] > 2 * (R_ + 1) && g.nc[2] > 2 * (R_ + 1);
    bool truncated = false;
    int off = 0;
    for (int b = 0; b < T; ++b) {
        int n1 = 0;
        if (MODE == 2) {
            // ---- pass 1 over the stored candidates (they were within rc + skin at the last cell search) ----
            const int total = candcnt[(long)b * N + i];
            const int *cs = cand + ((long)b * N + i) * cap;
            for (int base = 0; base < total; base += 128) {       // four candidates per lane and iteration, as in the cell search
                int sv[4];
                bool okv[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) { const int idx = base + 32 * u + lane; sv[u] = idx < total ? cs[idx] : ii; }
#pragma unroll
                for (int u = 0; u < 4; ++u) okv[u] = near_f32(xsf, sv[u], pf, gf, gf.rc2_margin_rc);
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const bool ok = okv[u] && sv[u] != ii;
                    const unsigned mask = __ballot_sync(0xffffffffu, ok);
                    if (ok) keys[n1 + __popc(mask & lt)] = (unsigned long long)sv[u];
                    n1 += __popc(mask);
                }
            }
        } else {
        // ---- run table ----
        int sA = 0, lenA = 0, sB = 0, lenB = 0;
        if (lane < ncol) {
            const int *bs = bin_start + b * g.ncell + colrel;
            sA = bs[za0]; lenA = bs[za1 + 1] - sA;
            if (zb1 >= zb0) { sB = bs[zb0]; lenB = bs[zb1 + 1] - sB; }
        }
        const unsigned mA = __ballot_sync(0xffffffffu, lenA > 0), mB = __ballot_sync(0xffffffffu, lenB > 0);
        const int inA = warp_incl_scan(lenA, lane);
        const int totA = __shfl_sync(0xffffffffu, inA, 31);
        int total = totA;
        if (lenA > 0) runtab[__popc(mA & lt)] = make_int2(inA, sA - (inA - lenA));
        int nrun = __popc(mA);
        if (mB) {
            const int inB = warp_incl_scan(lenB, lane);
            if (lenB > 0) runtab[nrun + __popc(mB & lt)] = make_int2(totA + inB, sB - (totA + inB - lenB));
            total += __shfl_sync(0xffffffffu, inB, 31);
            nrun += __popc(mB);
        }
        if (lane == 0) runtab[nrun] = make_int2(0x7fffffff, 0);
        __syncwarp();
        // ---- pass 1: conservative fp32 filter ----
        int r = 0;
        int2 e = runtab[0];
        // PU candidates per lane and iteration (their gathers in flight together); a position past the range tests the centre itself
        constexpr int PU = 4;
        for (int base = 0; base < total; base += 32 * PU) {
            int sv[PU];
            bool okv[PU];
#pragma unroll
            for (int u = 0; u < PU; ++u) {
                const int idx = base + 32 * u + lane;
                while (idx >= e.x) e = runtab[++r];
                sv[u] = idx < total ? idx + e.y : ii;
            }
            if (interior) {
#pragma unroll
                for (int u = 0; u < PU; ++u) okv[u] = near_f32<false>(xsf, sv[u], pf, gf, gf.rc2_margin);
            } else {
#pragma unroll
                for (int u = 0; u < PU; ++u) okv[u] = near_f32<true>(xsf, sv[u], pf, gf, gf.rc2_margin);
            }
#pragma unroll
            for (int u = 0; u < PU; ++u) {
                const bool ok = okv[u] && sv[u] != ii;
                const unsigned mask = __ballot_sync(0xffffffffu, ok);
                const int pos = n1 + __popc(mask & lt);
                if (ok && pos < cap) keys[pos] = (unsigned long long)sv[u];
                n1 += __popc(mask);
            }
        }
        if (n1 > cap) { if (lane == 0) atomicOr(&status[0], 2); n1 = cap; }
        __syncwarp();
        if (MODE == 1) {
            int *cs = cand + ((long)b * N + i) * cap;
            for (int k = lane; k < n1; k += 32) cs[k] = (int)keys[k];
            if (lane == 0) candcnt[(long)b * N + i] = n1;
        }
        }
        __syncwarp();
        // ---- pass 2: exact test + key on the survivors, compacted in place; two entries per lane and iteration with
        // unconditional gathers (an entry past the end tests the centre itself and is dropped) ----
        int n = 0;
        for (int base = 0; base < n1; base += 64) {
            int sv[2];
            double r2v[2];
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                const int k = base + 32 * u + lane;
                sv[u] = k < n1 ? (int)keys[k] : ii;
            }
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                const long s3 = 3 * (long)sv[u];
                const double dx = min_image(__dsub_rn(xs[s3], xi), g.L[0], hx);
                const double dy = min_image(__dsub_rn(xs[s3 + 1], yi), g.L[1], hy);
                const double dz = min_image(__dsub_rn(xs[s3 + 2], zi), g.L[2], hz);
                r2v[u] = __fma_rn(dz, dz, __fma_rn(dy, dy, __dmul_rn(dx, dx)));
            }
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                const bool ok = r2v[u] < rc2 && sv[u] != ii;
                unsigned long long key = 0;
                if (ok) key = (__double2ull_rd(r2v[u] * 536870912.0) << 24) | (unsigned long long)perm[sv[u]];
                // every lane has read both of its entries, and this batch writes below the entries of the next one
                const unsigned mask = __ballot_sync(0xffffffffu, ok);
                if (ok) { const int p = n + __popc(mask & lt); keys[p] = key; sidx[p] = sv[u]; }
                n += __popc(mask);
            }
        }
        __syncwarp();
        int *out = nlist + i * Nm + off;
        if (n <= 32) sort_and_emit<1>(keys, sidx, n, lane, sel[b], inv, out);
        else if (n <= 64) sort_and_emit<2>(keys, sidx, n, lane, sel[b], inv, out);
        else if (n <= 128) sort_and_emit<4>(keys, sidx, n, lane, sel[b], inv, out);
        else if (n <= 256) sort_and_emit<8>(keys, sidx, n, lane, sel[b], inv, out);
        else {
            int P = 512;
            while (P < n) P <<= 1;
            for (int k = n + lane; k < P; k += 32) keys[k] = ~0ull;
            __syncwarp();
            for (int k = 2; k <= P; k <<= 1) {
                for (int j = k >> 1; j > 0; j >>= 1) {
                    for (int idx = lane; idx < P; idx += 32) {
                        const int ixj = idx ^ j;
                        if (ixj > idx) {
                            const unsigned long long a = keys[idx], c = keys[ixj];
                            const bool asc = (idx & k) == 0;
                            if ((a > c) == asc) { keys[idx] = c; keys[ixj] = a; }
                        }
                    }
                    __syncwarp();
                }
            }
            const int nkeep = n < sel[b] ? n : sel[b];
            for (int k = lane; k < sel[b]; k += 32) out[k] = k < nkeep ? inv[(int)(keys[k] & 0xFFFFFFull)] : -1;
        }
        const int nkeep = n < sel[b] ? n : sel[b];
        if (lane == 0) {
            nreal[i * T + b] = nkeep;
            if (rowcnt) rowcnt[(long)b * N + i] = nkeep + (nkeep < sel[b] ? 1 : 0);
        }
        truncated |= n > sel[b];
        off += sel[b];
        __syncwarp();
    }
    if (truncated && lane == 0) atomicAdd(&status[1], 1);
}

__global__ void k_get_nlist(long N, int Nm, const int *__restrict__ nlist, const int *__restrict__ perm,
                            int *__restrict__ out) {
    long t = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (t >= N * Nm) return;
    long i = t / Nm;
    int k = (int)(t - i * Nm);
    int v = nlist[t];
    out[(long)perm[i] * Nm + k] = v >= 0 ? perm[v] : -1;
}

// Reuse step of the buffered list: the sorted order of the last cell build is kept, only the coordinates are refreshed
// (canonical wrap as k_wrap_bin).  An atom that moved more than skin / 2 since the build breaks the superset guarantee.
__global__ void k_regather(long N, const double *__restrict__ coords, const int *__restrict__ perm, Grid3 g,
                           const double *__restrict__ xref, double half_skin2, double *__restrict__ xs,
                           float4 *__restrict__ xsf, int *__restrict__ status) {
    long s = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (s >= N) return;
    const long u = perm[s];
    double w[3], d2 = 0.0;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const double x = coords[3 * u + a], d = x - xref[3 * u + a];
        w[a] = wrap_coord(x, g.L[a]);
        d2 += d * d;
        xs[3 * s + a] = w[a];
    }
    xsf[s] = make_float4((float)w[0], (float)w[1], (float)w[2], 0.f);
    if (d2 > half_skin2) atomicOr(&status[0], 4);
}

}  // namespace

void dp_launch_scan(int n, const int *cnt, int *start, int *tmp, cudaStream_t st) { launch_scan(n, cnt, start, tmp, st); }

cudaError_t launch_regather(const dp_model *m, long N, const double *coords, const Grid3 &g, char *ws, const WsLayout &L,
                            cudaStream_t st) {
    k_regather<<<(unsigned)((N + 255) / 256), 256, 0, st>>>(N, coords, (int *)(ws + L.perm), g, m->md_xref,
                                                           0.25 * m->md_skin * m->md_skin, (double *)(ws + L.xs),
                                                           (float4 *)(ws + L.xsf), (int *)(ws + L.status));
    return cudaGetLastError();
}

cudaError_t launch_build_cells(const dp_model *m, long N, const double *coords, const int *types, const Grid3 &g,
                               char *ws, const WsLayout &L, cudaStream_t st) {
    const int nbins = m->T * g.ncell;
    int *status = (int *)(ws + L.status);
    int *cnt = (int *)(ws + L.bin_count), *start = (int *)(ws + L.bin_start), *cursor = (int *)(ws + L.bin_cursor);
    cudaMemsetAsync(cnt, 0, sizeof(int) * (size_t)(nbins + 1), st);
    cudaMemsetAsync(cursor, 0, sizeof(int) * (size_t)nbins, st);
    const int nb = (int)((N + 255) / 256);
    k_wrap_bin<<<nb, 256, 0, st>>>(N, coords, types, m->type_map_dev, m->n_type_map, g, (double *)(ws + L.xw),
                                   (int *)(ws + L.atom_bin), cnt, status);
    launch_scan(nbins, cnt, start, (int *)(ws + L.scan_tmp), st);
    k_scatter<<<nb, 256, 0, st>>>(N, (int *)(ws + L.atom_bin), start, cursor, (int *)(ws + L.tmp_order));
    k_bin_sort<<<nb, 256, 0, st>>>(N, (int *)(ws + L.atom_bin), start, (int *)(ws + L.tmp_order),
                                   (double *)(ws + L.xw), (int *)(ws + L.perm), (int *)(ws + L.inv),
                                   (double *)(ws + L.xs), (float4 *)(ws + L.xsf));
    return cudaGetLastError();
}

cudaError_t launch_nlist(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st) {
    const int cap = m->sort_cap;
    const size_t smem = (size_t)4 * cap * (sizeof(unsigned long long) + sizeof(int));   // keys + sorted-space indices
    const TypeTab tt = make_typetab(m);
    // fp32 pre-filter margin: the fp32 copy is off by <= ulp(L)/2 per coordinate, the fp32 arithmetic by a few ulp of rc^2
    double Lmax = g.L[0] > g.L[1] ? g.L[0] : g.L[1];
    Lmax = Lmax > g.L[2] ? Lmax : g.L[2];
    // (and the fp32 minimum image d - L rint(d / L) by another ulp(L))
    NlistF32 gf;
    for (int d = 0; d < 3; ++d) { gf.L[d] = (float)g.L[d]; gf.invL[d] = (float)(1.0 / g.L[d]); }
    const double rl = m->rc + (m->list_mode ? m->md_skin : 0.0);      // search radius of pass 1
    gf.rc2_margin = (float)(rl * rl * (1.0 + 1e-5) + 12.0 * rl * Lmax * 1.2e-7 + 1e-6);
    gf.rc2_margin_rc = (float)(m->rc * m->rc * (1.0 + 1e-5) + 12.0 * m->rc * Lmax * 1.2e-7 + 1e-6);
    DP_SMEM_OPTIN(k_nlist2<0>, 4 * 4096 * 12);
    DP_SMEM_OPTIN(k_nlist2<1>, 4 * 4096 * 12);
    DP_SMEM_OPTIN(k_nlist2<2>, 4 * 4096 * 12);
    auto kern = m->list_mode == 1 ? k_nlist2<1> : (m->list_mode == 2 ? k_nlist2<2> : k_nlist2<0>);
    kern<<<(unsigned)((N + 3) / 4), 128, smem, st>>>(N, m->T, g, m->rc * m->rc, gf, cap, (int *)(ws + L.bin_start),
                                                    (double *)(ws + L.xs), (const float4 *)(ws + L.xsf), (int *)(ws + L.perm),
                                                    (int *)(ws + L.inv), m->Nm, tt, (int *)(ws + L.nlist),
                                                    (int *)(ws + L.nreal), !dp_uses_rows(m) ? nullptr : (int *)(ws + L.rowcnt),
                                                    (int *)(ws + L.status), m->md_cand, m->md_candcnt);
    if (dp_uses_rows(m))
        for (int b = 0; b < m->T; ++b)
            launch_scan((int)N, (int *)(ws + L.rowcnt) + (long)b * N, (int *)(ws + L.rowstart) + (long)b * (N + 1), (int *)(ws + L.scan_tmp), st);
    return cudaGetLastError();
}

cudaError_t launch_get_nlist(const dp_model *m, long N, char *ws, const WsLayout &L, int *out, cudaStream_t st) {
    long tot = N * m->Nm;
    k_get_nlist<<<(unsigned)((tot + 255) / 256), 256, 0, st>>>(N, m->Nm, (int *)(ws + L.nlist), (int *)(ws + L.perm), out);
    return cudaGetLastError();
}
