// S3 + S4 + S5 + S7 + S8 + S9 for WIDE embedding nets (W, 2 W, 4 W), W = 64 ... 512, in FP64 and MIX-32: the double and
// MIX-32 curves of the network-size study (Fig. 7: "the FLOPS curves of both double and MIX-32 versions
// flatten after the matrix size reaching 256 x 512"); the MIX-16 curve is wide.cu.
//
// The structure is the paper's own: one GEMM per layer with the bias / tanh / skip / tanh' work in its
// epilogue, the activations kept in HBM between the layers (row-major, in the precision of the nets) and reused by the
// backward pass, which overwrites them in place (dz3 over t3, dz2 over t2, dy2 over y2, dz1 over t1).  Rows are the compact
// rows of the mixed modes (the real rows of a (centre type, neighbour type) block, contiguous, plus one
// representative per atom and block for its padded slots, weighted by their number) and the row tiles are those of the
// tile table of wide.cu, so a tile never straddles two nets.
//   FP64   ("double"): k_wg_gemm_f64, the FP64 tensor pipe (DMMA m8n8k4), 64 x 64 x 16 tiles staged with cp.async, four CTAs per SM;
//   MIX-32 (nets in single precision): k_wg_gemm_tf32, tcgen05.mma kind::tf32 with TMEM accumulators; every operand
//          is split into a TF32 value and its TF32 remainder and each K step takes three products ("3xTF32": the product keeps
//          21+ mantissa bits; the accumulators are fp32); the activations arrive by TMA tensor copies, the weights' operand
//          images by bulk copies; exact tanhf.
//   Coordinates, environment rows, geometry derivative, force and virial accumulation stay fp64 in both modes.
// Forward:  k_wg_env -> k_wg_l1 (t1) -> gemm<0> (t2, y2 = (t1,t1) + t2) -> gemm<1> (t3) -> k_wg_contract (A_i = R^T G / Nm)
// Backward: k_wg_bwd_head (gG = R^ gA / Nm, dz3, skip share of dy2, dR^ = G gA^T / Nm) -> gemm<2> (dy2, dz2) -> gemm<3> (dz1)
//           -> k_wg_ds (ds^ = dz1 . w1, dE/dR~ = (dR^ + ds^ e0) / std) -> k_wg_force (N9 geometry derivative, ProdForce,
//           ProdViral).
#include <cstring>
#include <cuda.h>          // CUtensorMap (types only: the encoder is looked up through the runtime, no libcuda link)
#include <type_traits>
#include <vector>
#include "dp_internal.h"
#include "tanh64.cuh"
#include "tc_common.cuh"

namespace {

constexpr int GR = 128;                     // rows per tile (= the tile table's, wide.cu)
constexpr int GBM = 64, GBN = 64, GBK = 16;  // FP64 kernel: rows (half a tile of the table), columns, K step per CTA
constexpr int GNI = GBN / 16, GCTAS = 4;     // 8-column fragments per warp; CTAs per SM
constexpr int GTHREADS = 128;               // four warps as 2 (rows) x 2 (columns)
constexpr int GA_STRIDE = GBK + 4;          // A tile [64][20], B tile [16][68]: fragment loads hit distinct banks (per half warp)
struct GemmCfg {                             // the FP64 kernel's tiles
    static constexpr int BS = GBN + 4;                                  // B tile [32][BS]
    static constexpr int A_TILE = GBM * GA_STRIDE, B_TILE = GBK * BS;
    static constexpr int SMEM = 2 * (A_TILE + B_TILE) * 8;
    static constexpr int EPV = 2;                                       // doubles per 16-byte cp.async
};

__device__ __forceinline__ double wg_tanh(double x) { return dp_tanh64(x); }
__device__ __forceinline__ float wg_tanh(float x) { return tanhf(x); }

// 16 bytes of a row: 2 doubles / 4 floats (the element-wise kernels move whole vectors)
template <typename R> struct alignas(16) Vec {
    static constexpr int V = 16 / (int)sizeof(R);
    R v[V];
};
template <typename R> __device__ __forceinline__ Vec<R> vld(const R *p) { return *reinterpret_cast<const Vec<R> *>(p); }
template <typename R> __device__ __forceinline__ void vst(R *p, const Vec<R> &x) { *reinterpret_cast<Vec<R> *>(p) = x; }

__device__ __forceinline__ void dmma(double &c0, double &c1, double a, double b) {
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}
__device__ __forceinline__ void cp_async16(void *smem_dst, const void *gsrc, bool valid) {
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    const int sz = valid ? 16 : 0;
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(s), "l"(gsrc), "r"(sz));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N)); }

__device__ __forceinline__ double min_image(double t, double L, double halfL) {
    const double s = t > halfL ? -1.0 : (t < -halfL ? 1.0 : 0.0);
    return __dadd_rn(t, __dmul_rn(s, L));
}
struct EnvParams {
    double rc, rc_smth, inv_range;
    double L[3];
};
EnvParams make_env(const dp_model *m, const Grid3 &g) {
    EnvParams ep;
    ep.rc = m->rc; ep.rc_smth = m->rc_smth; ep.inv_range = 1.0 / (m->rc - m->rc_smth);
    ep.L[0] = g.L[0]; ep.L[1] = g.L[1]; ep.L[2] = g.L[2];
    return ep;
}
// N4 (+ N9 when sp_out): R~ = s (1, d / r), s = w(r) / r; sp = ds/dr
__device__ __forceinline__ void env_row(const EnvParams &p, double dx, double dy, double dz, double Rt[4], double *sp_out, double *r_out) {
    const double r2 = dx * dx + dy * dy + dz * dz;
    const double r = sqrt(r2);
    double w = 1.0, dw = 0.0;
    if (r >= p.rc_smth) {
        if (r < p.rc) {
            const double u = (r - p.rc_smth) * p.inv_range;
            w = u * u * u * (-6.0 * u * u + 15.0 * u - 10.0) + 1.0;
            dw = -30.0 * u * u * (u - 1.0) * (u - 1.0) * p.inv_range;
        } else {
            w = 0.0;
        }
    }
    const double s = w / r;
    Rt[0] = s; Rt[1] = s * dx / r; Rt[2] = s * dy / r; Rt[3] = s * dz / r;
    if (sp_out) { *sp_out = dw / r - w / r2; *r_out = r; }
}

// the block k = a T + b of a tile of the tile table (entry k = {first tile, first row, end row}; entry T T = {tiles})
__device__ __forceinline__ int wg_block(const int4 *tab, int nblk, int tile) {
    int k = 0;
    while (k + 1 < nblk && tile >= tab[k + 1].x) ++k;
    return k;
}

// per-net parameter block (elements of R): w1 | b1 | b2 | b3 | W2 [W][2W] | W3 [2W][4W] | W3^T [4W][2W] | W2^T [2W][W]
__host__ __device__ inline long wg_off_b2(int W) { return 2L * W; }
__host__ __device__ inline long wg_off_b3(int W) { return 4L * W; }
__host__ __device__ inline long wg_off_W2(int W) { return 8L * W; }
__host__ __device__ inline long wg_off_W3(int W) { return 8L * W + 2L * W * W; }
__host__ __device__ inline long wg_off_W3T(int W) { return 8L * W + 10L * W * W; }
__host__ __device__ inline long wg_off_W2T(int W) { return 8L * W + 18L * W * W; }

// S3: compact environment rows in the precision of the nets (computed in fp64), and their ids
template <typename R>
__global__ void __launch_bounds__(256)
k_wg_env(long N, int T, int ncell, int Nm, const __grid_constant__ TypeTab tt, EnvParams ep, const double *__restrict__ avg,
         const double *__restrict__ stdv, const int *__restrict__ bin_start, const double *__restrict__ xs,
         const int *__restrict__ nlist, const int *__restrict__ nreal, const int *__restrict__ rowstart, R *__restrict__ rh,
         int2 *__restrict__ rows_id) {
    const int lane = threadIdx.x & 31;
    const long i = blockIdx.x * 8L + (threadIdx.x >> 5);
    if (i >= N) return;
    int a = 0;
    for (int t = 1; t < T; ++t) a += i >= bin_start[t * ncell];
    double av[4], sd[4];
#pragma unroll
    for (int c = 0; c < 4; ++c) { av[c] = avg[4 * a + c]; sd[c] = stdv[4 * a + c]; }
    const double xi = xs[3 * i], yi = xs[3 * i + 1], zi = xs[3 * i + 2];
    const double hx = 0.5 * ep.L[0], hy = 0.5 * ep.L[1], hz = 0.5 * ep.L[2];
    for (int b = 0; b < T; ++b) {
        const int nr = nreal[i * T + b];
        const int tot = nr + (nr < tt.sel[b] ? 1 : 0);
        const long base = N * (long)tt.off[b] + rowstart[(long)b * (N + 1) + i];
        const int *nl = nlist + i * Nm + tt.off[b];
        for (int k = lane; k < tot; k += 32) {
            double Rt[4] = {0.0, 0.0, 0.0, 0.0};
            int j = -(tt.sel[b] - nr);
            if (k < nr) {
                j = nl[k];
                const double dx = min_image(xs[3 * (long)j] - xi, ep.L[0], hx);
                const double dy = min_image(xs[3 * (long)j + 1] - yi, ep.L[1], hy);
                const double dz = min_image(xs[3 * (long)j + 2] - zi, ep.L[2], hz);
                env_row(ep, dx, dy, dz, Rt, nullptr, nullptr);
            }
#pragma unroll
            for (int c = 0; c < 4; ++c) rh[4 * (base + k) + c] = (R)((Rt[c] - av[c]) / sd[c]);
            rows_id[base + k] = make_int2((int)i, j);
        }
    }
}

// Layer 1 (K = 1): t1 = tanh(s^ w1 + b1); one CTA per tile
template <typename R>
__global__ void __launch_bounds__(256)
k_wg_l1(long N, int T, int W, const __grid_constant__ TypeTab tt, const int4 *__restrict__ tab, const R *__restrict__ nets,
        long net_stride, const R *__restrict__ rh, R *__restrict__ T1) {
    const int nblk = T * T;
    const int tile = blockIdx.x;
    if (tile >= tab[nblk].x) return;
    const int k = wg_block(tab, nblk, tile);
    const int4 e = tab[k];
    const long rbase = N * (long)tt.off[k % T];
    const int row0 = e.y + (tile - e.x) * GR;
    const int nrows = min(GR, e.z - row0);
    const R *w1 = nets + k * net_stride, *b1 = w1 + W;
    constexpr int V = Vec<R>::V;
    const int vpr = W / V;                                   // vectors per row
    for (int idx = threadIdx.x; idx < nrows * vpr; idx += 256) {
        const int rr = idx / vpr, c = (idx % vpr) * V;
        const long Rg = rbase + row0 + rr;
        const R s = rh[4 * Rg];
        const Vec<R> w = vld(w1 + c), b = vld(b1 + c);
        Vec<R> o;
#pragma unroll
        for (int q = 0; q < V; ++q) o.v[q] = wg_tanh(s * w.v[q] + b.v[q]);
        vst(T1 + Rg * W + c, o);
    }
}

template <typename R>
struct GenArgs {
    long N;
    int T, W;
    int K, NTOT;                          // product shape: [rows x K] . [K x NTOT]
    const int4 *tab;
    const R *A;                           // [rows][K] row-major (one of the activation buffers)
    const R *nets;                        // parameter blocks, net k at nets + k * net_stride
    long net_stride, b_off;               // FP64: B [K][NTOT] row-major at offset b_off of the block; MIX-32: the operand images of B^T
    R *T1, *Y2, *T2, *T3;                 // activations [rows][W | 2 W | 2 W | 4 W]
    TypeTab tt;
};

// MODE 0: layer 2 forward   A = t1,  B = W2:    t2 = tanh(acc + b2) -> T2;  y2 = (t1,t1) + t2 -> Y2
// MODE 1: layer 3 forward   A = y2,  B = W3:    t3 = tanh(acc + b3) -> T3   (G = (y2,y2) + t3 is formed by its readers)
// MODE 2: layer 3 backward  A = dz3, B = W3^T:  dy2 = acc + (gG[f] + gG[f + 2 W], in Y2) -> Y2;  dz2 = dy2 (1 - t2^2) -> T2
// MODE 3: layer 2 backward  A = dz2, B = W2^T:  dy1 = acc + dy2[e] + dy2[e + W];  dz1 = dy1 (1 - t1^2) -> T1
// The FP64 epilogue of one pair of adjacent columns, in two steps so that the kernel can issue the loads of several pairs before
// the first store (the activation pointers may alias as far as the compiler knows: interleaved, every load would wait for the
// store before it).
struct EpiAux { double2 a, b, c; };

template <int MODE>
__device__ __forceinline__ EpiAux wg_epi_load(const GenArgs<double> &p, const double *__restrict__ net, long Rg, int col) {
    const int W = p.W;
    EpiAux x;
    if (MODE == 0) {
        x.a = *reinterpret_cast<const double2 *>(net + wg_off_b2(W) + col);
        x.b = *reinterpret_cast<const double2 *>(p.T1 + Rg * W + (col % W));
    } else if (MODE == 1) {
        x.a = *reinterpret_cast<const double2 *>(net + wg_off_b3(W) + col);
    } else if (MODE == 2) {
        x.a = *reinterpret_cast<const double2 *>(p.Y2 + Rg * 2 * W + col);
        x.b = *reinterpret_cast<const double2 *>(p.T2 + Rg * 2 * W + col);
    } else {
        x.a = *reinterpret_cast<const double2 *>(p.Y2 + Rg * 2 * W + col);
        x.b = *reinterpret_cast<const double2 *>(p.Y2 + Rg * 2 * W + W + col);
        x.c = *reinterpret_cast<const double2 *>(p.T1 + Rg * W + col);
    }
    return x;
}
template <int MODE>
__device__ __forceinline__ void wg_epi_store(const GenArgs<double> &p, long Rg, int col, double v0, double v1, const EpiAux &x) {
    const int W = p.W;
    double2 o;
    if (MODE == 0) {
        o.x = dp_tanh64(v0 + x.a.x); o.y = dp_tanh64(v1 + x.a.y);
        *reinterpret_cast<double2 *>(p.T2 + Rg * 2 * W + col) = o;
        o.x += x.b.x; o.y += x.b.y;
        *reinterpret_cast<double2 *>(p.Y2 + Rg * 2 * W + col) = o;
    } else if (MODE == 1) {
        o.x = dp_tanh64(v0 + x.a.x); o.y = dp_tanh64(v1 + x.a.y);
        *reinterpret_cast<double2 *>(p.T3 + Rg * 4 * W + col) = o;
    } else if (MODE == 2) {
        o.x = x.a.x + v0; o.y = x.a.y + v1;
        *reinterpret_cast<double2 *>(p.Y2 + Rg * 2 * W + col) = o;
        o.x *= 1.0 - x.b.x * x.b.x; o.y *= 1.0 - x.b.y * x.b.y;
        *reinterpret_cast<double2 *>(p.T2 + Rg * 2 * W + col) = o;
    } else {
        o.x = (v0 + x.a.x + x.b.x) * (1.0 - x.c.x * x.c.x);
        o.y = (v1 + x.a.y + x.b.y) * (1.0 - x.c.y * x.c.y);
        *reinterpret_cast<double2 *>(p.T1 + Rg * W + col) = o;
    }
}

// FP64: one 64 x 64 output tile per CTA (half a tile of the table), four warps as 2 (rows) x 2 (columns): warp tile 32 x 32 =
// 4 x 4 DMMA m8n8k4 fragments; FOUR CTAs per SM (128 registers x 128 threads, 37 KB of shared memory each), so that one CTA's
// barriers, prologue and epilogue run under the others' DMMAs.  A and B stages of K = 16 arrive by cp.async (two buffers); rows
// past the end of the tile's block and columns past NTOT are zero-filled and never stored.
template <int MODE>
__global__ void __launch_bounds__(GTHREADS, GCTAS) k_wg_gemm_f64(const __grid_constant__ GenArgs<double> p) {
    using C = GemmCfg;
    extern __shared__ __align__(16) unsigned char wg_smem[];
    double *sm = reinterpret_cast<double *>(wg_smem);
    const int nblk = p.T * p.T;
    const int ntn = (p.NTOT + GBN - 1) / GBN;
    constexpr int SUB = GR / GBM;                 // CTAs per tile of the table
    const int tile = blockIdx.x / (ntn * SUB), sub = (blockIdx.x / ntn) % SUB, n0 = (blockIdx.x % ntn) * GBN;
    if (tile >= p.tab[nblk].x) return;
    const int k = wg_block(p.tab, nblk, tile);
    const int4 e = p.tab[k];
    const long rbase = p.N * (long)p.tt.off[k % p.T];
    const int row0 = e.y + (tile - e.x) * GR + sub * GBM;
    const int nrows = min(GBM, e.z - row0);
    if (nrows <= 0) return;
    const double *net = p.nets + k * p.net_stride;
    const double *Ag = p.A + (rbase + row0) * (long)p.K;
    const double *Bg = net + p.b_off + n0;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wm = warp >> 1, wn = warp & 1, g = lane >> 2, t = lane & 3;

    auto load_stage = [&](int buf, int k0) {
        double *As = sm + buf * (C::A_TILE + C::B_TILE), *Bs = As + C::A_TILE;
        constexpr int AV = GBK / C::EPV, BV = GBN / C::EPV;       // 16-byte vectors per A row / per B row
#pragma unroll
        for (int q = 0; q < GBM * AV / GTHREADS; ++q) {
            const int idx = tid + q * GTHREADS, r = idx / AV, kv = (idx % AV) * C::EPV;
            const bool ok = r < nrows;
            cp_async16(As + r * GA_STRIDE + kv, Ag + (ok ? (long)r * p.K + k0 + kv : 0), ok);
        }
#pragma unroll
        for (int q = 0; q < GBK * BV / GTHREADS; ++q) {
            const int idx = tid + q * GTHREADS, kk = idx / BV, nv = (idx % BV) * C::EPV;
            const bool ok = n0 + nv < p.NTOT;
            cp_async16(Bs + kk * C::BS + nv, Bg + (ok ? (long)(k0 + kk) * p.NTOT + nv : 0), ok);
        }
        cp_async_commit();
    };

    double acc[8 * GNI];                         // 4 x GNI fragments of 2
#pragma unroll
    for (int q = 0; q < 8 * GNI; ++q) acc[q] = 0.0;

    const int nk = p.K / GBK;
    load_stage(0, 0);
    for (int ks = 0; ks < nk; ++ks) {
        if (ks + 1 < nk) { load_stage((ks + 1) & 1, (ks + 1) * GBK); cp_async_wait<1>(); } else { cp_async_wait<0>(); }
        __syncthreads();
        const double *As = sm + (ks & 1) * (C::A_TILE + C::B_TILE), *Bs = As + C::A_TILE;
#pragma unroll
        for (int kk = 0; kk < GBK / 4; ++kk) {
            double a[4], b[GNI];
#pragma unroll
            for (int mi = 0; mi < 4; ++mi) a[mi] = As[(32 * wm + 8 * mi + g) * GA_STRIDE + 4 * kk + t];
#pragma unroll
            for (int ni = 0; ni < GNI; ++ni) b[ni] = Bs[(4 * kk + t) * C::BS + 8 * GNI * wn + 8 * ni + g];
#pragma unroll
            for (int mi = 0; mi < 4; ++mi)
#pragma unroll
                for (int ni = 0; ni < GNI; ++ni) dmma(acc[2 * (mi * GNI + ni)], acc[2 * (mi * GNI + ni) + 1], a[mi], b[ni]);
        }
        __syncthreads();
    }

    // epilogue: pairs of adjacent columns, the eight pairs of one fragment row at a time (loads first)
#pragma unroll
    for (int mi = 0; mi < 4; ++mi) {
        const int r = 32 * wm + 8 * mi + g;
        if (r >= nrows) continue;
        const long Rg = rbase + row0 + r;
        EpiAux aux[GNI];
#pragma unroll
        for (int ni = 0; ni < GNI; ++ni) {
            const int col = n0 + 8 * GNI * wn + 8 * ni + 2 * t;
            if (col < p.NTOT) aux[ni] = wg_epi_load<MODE>(p, net, Rg, col);
        }
#pragma unroll
        for (int ni = 0; ni < GNI; ++ni) {
            const int col = n0 + 8 * GNI * wn + 8 * ni + 2 * t;
            if (col < p.NTOT) wg_epi_store<MODE>(p, Rg, col, acc[2 * (mi * GNI + ni)], acc[2 * (mi * GNI + ni) + 1], aux[ni]);
        }
    }
}

// ---- MIX-32 on the 5th-generation tensor cores: tcgen05.mma kind::tf32, three products per K step ("3xTF32") -------------------
// C = A B with A = the fp32 activations [rows][K] and B^T = a weight matrix [NTOT][K] (both K-major operands: dp_create keeps every
// matrix and its transpose).  Persistent, one CTA PAIR per two SMs (cluster of 2, tcgen05 cta_group::2): the pair computes
// two 128-row tiles of one net against one N tile; each CTA stages its own rows of A and HALF of the B tile, and the MMA of the
// leader (M = 256) reads both halves, so a CTA moves and reads half the weight bytes of a single-CTA tile.  Per CTA:
//   warp 13    loader (one thread): per K = 32 stage ONE TMA tensor copy of A (the row-major activations seen as a
//              (4, rows, K / 4) tensor, box {4, 128, 8}: it lands as the un-swizzled K-major operand image, per 16 bytes of K a
//              column [128 rows][16 B]) and ONE bulk copy of this CTA's half of the weights' operand images (TF32 values and TF32
//              remainders, laid out by dp_create), both counted by the stage's "landed" barrier;
//   warps 0-7  splitters: a_small = a - a_big (exact) into a second image, a_big = a with the 13 low mantissa bits cleared = what
//              the tensor core reads from the landed image itself; fence.proxy.async; arrive on the LEADER's "full" barrier
//              (the peer's threads through its cluster address);
//   warp 12    MMA issuer (leader only): per K = 8 step a_small b_big, a_big b_small, a_big b_big into one of two 256 x BN fp32
//              accumulators (128 TMEM lanes in each CTA); tcgen05.commit multicasts "stage free" and "accumulator ready" to both CTAs;
//   warps 8-11 epilogue: thread = row = TMEM lane, 32 columns per step, the layer's bias / tanh / skip / tanh' work on the
//              row-major fp32 activations; "accumulator drained" goes to the leader.
constexpr int TQ_KC = 32;                          // K per stage: 8 pieces of 16 bytes
constexpr int TQ_NST = 3;
constexpr int TQ_A_PIECE = 128 * 16;               // distance between the piece columns of an image (the descriptors' LBO)
constexpr int TQ_A_IMG = (TQ_KC / 4) * TQ_A_PIECE;   // 16 KB: [8 pieces][128 rows][16 B], written by one TMA tensor copy
constexpr int TQ_B_IMG = 128 * TQ_KC * 4;          // 16 KB: this CTA's half (<= 128 rows of B^T) of one weight image
constexpr int TQ_STAGE = 2 * TQ_A_IMG + 2 * TQ_B_IMG;      // a_big | a_small | b_big | b_small
constexpr int TQ_OFF_BAR = TQ_NST * TQ_STAGE;
constexpr int TQ_TOTAL = TQ_OFF_BAR + 256;
constexpr int TQ_THREADS = 448;                  // 8 splitter, 4 epilogue warps, the MMA warp, the loader warp
static_assert(TQ_TOTAL + 1024 <= 227 * 1024, "shared memory budget");
static_assert((3 * TQ_NST + 4) * 8 <= 256, "barriers");

__device__ __forceinline__ void mma_tf32_ss2(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t id, bool accumulate) {
    asm volatile("{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\ntcgen05.mma.cta_group::2.kind::tf32 [%0], %1, %2, %3, p;\n}"
                 ::"r"(tmem_d), "l"(da), "l"(db), "r"(id), "r"((uint32_t)accumulate) : "memory");
}
// kind::tf32 instruction descriptor: tf32 x tf32 -> fp32, M x N, both operands K-major
__host__ __device__ constexpr uint32_t idesc_tf32(int M, int N) {
    return (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}
// the MMAs issued so far by this thread arrive on the barrier at this shared-memory offset in BOTH CTAs of the pair
__device__ __forceinline__ void commit_pair(uint64_t *bar) {
    asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;"
                 ::"r"(tc::smem_u32(bar)), "h"((uint16_t)3) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx_cta(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(tc::smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s_cta(uint32_t sdst, const void *gsrc, uint32_t bytes, uint64_t *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(sdst), "l"(gsrc), "r"(bytes), "r"(tc::smem_u32(bar)) : "memory");
}
// arrive on the barrier at this shared-memory offset in the leader CTA (rank 0 of the pair), from either CTA.  Release at CTA
// scope (the default), as cluster barriers are commonly signalled: what the arrival publishes is shared memory of the arriving
// CTA that its own fence.proxy.async has handed to the asynchronous proxy.  A .release.cluster here compiles to a memory
// barrier per arrival and made the pairs 1.4x SLOWER than single CTAs (ncu: 9.9 membar stall cycles per issued instruction).
__device__ __forceinline__ void mbar_arrive_leader(uint64_t *bar) {
    asm volatile("{\n.reg .b32 ra;\nmapa.shared::cluster.u32 ra, %0, 0;\nmbarrier.arrive.shared::cluster.b64 _, [ra];\n}"
                 ::"r"(tc::smem_u32(bar)) : "memory");
}
// wait for a phase that CTAs of the cluster complete (acquire at cluster scope)
__device__ __forceinline__ void mbar_wait_cluster(uint64_t *bar, uint32_t parity) {
    asm volatile("{\n.reg .pred p;\nWAITC_%=:\nmbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%0], %1;\n@p bra DONEC_%=;\nbra WAITC_%=;\nDONEC_%=:\n}"
                 ::"r"(tc::smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;\nbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// box {4 elements, 128 rows, 8 pieces} of the activation tensor viewed as (4, rows, K / 4) -> the [8][128][16 B] operand image
__device__ __forceinline__ void tma_load_3d(uint32_t sdst, const CUtensorMap *tm, int c0, int c1, int c2, uint64_t *bar) {
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                 ::"r"(sdst), "l"((uint64_t)tm), "r"(c0), "r"(c1), "r"(c2), "r"(tc::smem_u32(bar)) : "memory");
}

// Work item w of the pairs: (pair of consecutive tiles of one block, N tile).  Returns the block; row0 / nrows of this CTA's tile
// (nrows <= 0: the block has an odd number of tiles and this CTA of its last pair has none: it stages operands, stores nothing).
__device__ __forceinline__ int pair_item(const GenArgs<float> &p, int nblk, int NT, long w, int rank, int &nt, long &row0, int &nrows) {
    const int pt = (int)(w / NT);
    nt = (int)(w % NT);
    int k = 0, base = 0;
    for (;; ++k) {
        const int ntk = k + 1 < nblk + 1 ? p.tab[k + 1].x - p.tab[k].x : 0;        // tiles of block k (entry nblk = {tiles})
        const int np = (ntk + 1) >> 1;
        if (pt < base + np || k == nblk - 1) break;
        base += np;
    }
    const int4 e = p.tab[k];
    const int t = 2 * (pt - base) + rank;
    const int r0 = e.y + t * GR;
    nrows = min(GR, e.z - r0);
    row0 = p.N * (long)p.tt.off[k % p.T] + r0;
    return k;
}
__device__ __forceinline__ long pair_count(const GenArgs<float> &p, int nblk) {
    long n = 0;
    for (int k = 0; k < nblk; ++k) n += (p.tab[k + 1].x - p.tab[k].x + 1) >> 1;
    return n;
}

template <int MODE>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(TQ_THREADS, 1)
k_wg_gemm_tf32(const __grid_constant__ GenArgs<float> p, const __grid_constant__ CUtensorMap tmA) {
    extern __shared__ __align__(1024) unsigned char tq_smem[];
    __shared__ uint32_t tmem_base_s;
    const int tid = threadIdx.x, lane = tid & 31;
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);
    uint32_t rank;
    asm("mov.u32 %0, %%cluster_ctarank;" : "=r"(rank));
    uint64_t *bars = reinterpret_cast<uint64_t *>(tq_smem + TQ_OFF_BAR);
    uint64_t *full = bars, *empty = bars + TQ_NST, *landed = bars + 2 * TQ_NST, *acc_full = bars + 3 * TQ_NST, *acc_empty = acc_full + 2;
    if (tid == 0) {
        for (int k = 0; k < TQ_NST; ++k) { tc::mbar_init(&full[k], 16); tc::mbar_init(&empty[k], 1); tc::mbar_init(&landed[k], 1); }
        for (int k = 0; k < 2; ++k) { tc::mbar_init(&acc_full[k], 1); tc::mbar_init(&acc_empty[k], 8); }
        asm volatile("fence.mbarrier_init.release.cluster;");
    }
    if (warp == 12) {      // the same warp of both CTAs, the same shared-memory word
        asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tc::smem_u32(&tmem_base_s)), "n"(512));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;");
    }
    tc::fence_before();
    cluster_sync_all();
    tc::fence_after();
    const uint32_t tmem = tmem_base_s;
    const uint32_t sbase = tc::smem_u32(tq_smem);
    const int nblk = p.T * p.T;
    const int W = p.W, K = p.K, BN = p.NTOT < 256 ? p.NTOT : 256, HB = BN / 2, NT = p.NTOT / BN, NKC = K / TQ_KC;
    const long nwork = pair_count(p, nblk) * NT;   // work item = (pair of row tiles, N tile), the N tiles of a pair adjacent
    const long pair0 = blockIdx.x >> 1, npair = gridDim.x >> 1;

    if (warp == 13) {
        // ------------------------------------------------------------------------------------------------ loader
        if (lane == 0) {
            const uint32_t b_half_bytes = 2u * HB * TQ_KC * 4;                  // TF32 values and remainders of HB rows of B^T
            uint32_t step = 0;
            for (long w = pair0; w < nwork; w += npair) {
                int nt, nrows;
                long row0;
                const int k = pair_item(p, nblk, NT, w, (int)rank, nt, row0, nrows);
                if (nrows <= 0) row0 -= GR;                                     // no tile of its own: any valid rows will do
                const float *Bg = p.nets + k * p.net_stride + p.b_off + ((long)nt * NKC * 2 + rank) * (2 * HB * TQ_KC);
                for (int kc = 0; kc < NKC; ++kc, ++step) {
                    const int st = step % TQ_NST;
                    tc::mbar_wait(&empty[st], ((step / TQ_NST) & 1) ^ 1);
                    mbar_expect_tx_cta(&landed[st], TQ_A_IMG + b_half_bytes);
                    tma_load_3d(sbase + st * TQ_STAGE, &tmA, 0, (int)row0, kc * (TQ_KC / 4), &landed[st]);
                    bulk_g2s_cta(sbase + st * TQ_STAGE + 2 * TQ_A_IMG, Bg + (long)kc * 2 * (2 * HB * TQ_KC), b_half_bytes, &landed[st]);
                }
            }
        }
    } else if (warp < 8) {
        // ------------------------------------------------------------------------------------------------ splitters
        // every thread splits four 16-byte pieces of the landed A image: a_small into the second image
        const uint32_t a_off = ((tid >> 3) & 3) * TQ_A_PIECE + (8 * (tid >> 5) + (tid & 7)) * 16;      // + 64 rows for the second piece
        const long nstage = nwork > pair0 ? ((nwork - pair0 + npair - 1) / npair) * NKC : 0;
        for (long it = 0; it < nstage; ++it) {
            const int st = (int)(it % TQ_NST);
            tc::mbar_wait(&landed[st], (uint32_t)((it / TQ_NST) & 1));
            unsigned char *stage = tq_smem + st * TQ_STAGE;
#pragma unroll
            for (int q = 0; q < TQ_KC / 8; ++q) {          // q & 1: + 64 rows; q >> 1: + 4 piece columns
                // (the landed image itself is a_big: the tensor core reads the top 19 bits of each fp32 word and ignores the 13
                // low mantissa bits; storing the masked words back changes no result bit and was measured, so it is not done)
                const uint4 *pb = reinterpret_cast<const uint4 *>(stage + a_off + (q & 1) * (64 * 16) + (q >> 1) * 4 * TQ_A_PIECE);
                uint4 *ps = reinterpret_cast<uint4 *>(stage + TQ_A_IMG + a_off + (q & 1) * (64 * 16) + (q >> 1) * 4 * TQ_A_PIECE);
                const uint4 x = *pb;
                uint4 b, sm;
                b.x = x.x & 0xffffe000u; b.y = x.y & 0xffffe000u; b.z = x.z & 0xffffe000u; b.w = x.w & 0xffffe000u;
                sm.x = __float_as_uint(__uint_as_float(x.x) - __uint_as_float(b.x));
                sm.y = __float_as_uint(__uint_as_float(x.y) - __uint_as_float(b.y));
                sm.z = __float_as_uint(__uint_as_float(x.z) - __uint_as_float(b.z));
                sm.w = __float_as_uint(__uint_as_float(x.w) - __uint_as_float(b.w));
                *ps = sm;
            }
            tc::proxy_fence();
            __syncwarp();
            if (lane == 0) mbar_arrive_leader(&full[st]);         // one arrival per warp: 8 local + 8 from the peer
        }
    } else if (warp == 12) {
        // ------------------------------------------------------------------------------------------------ MMA issuer (leader)
        if (rank == 0) {
            const uint32_t idesc = idesc_tf32(256, BN);
            const uint32_t B_PIECE = HB * 16;
            uint32_t step = 0, accn = 0;
            for (long w = pair0; w < nwork; w += npair, ++accn) {
                const int buf = accn & 1;
                mbar_wait_cluster(&acc_empty[buf], ((accn >> 1) & 1) ^ 1);
                tc::fence_after();
                for (int kc = 0; kc < NKC; ++kc, ++step) {
                    const int st = step % TQ_NST;
                    mbar_wait_cluster(&full[st], (step / TQ_NST) & 1);
                    tc::fence_after();
                    const uint32_t sa = sbase + st * TQ_STAGE;
                    const uint64_t dab = tc::desc(sa, TQ_A_PIECE, 128), das = tc::desc(sa + TQ_A_IMG, TQ_A_PIECE, 128);
                    const uint64_t dbb = tc::desc(sa + 2 * TQ_A_IMG, B_PIECE, 128), dbs = tc::desc(sa + 2 * TQ_A_IMG + HB * TQ_KC * 4, B_PIECE, 128);
                    if (tc::elect_one()) {
#pragma unroll
                        for (int ks = 0; ks < TQ_KC / 8; ++ks) {
                            const uint32_t oa = ks * 2 * TQ_A_PIECE, ob = ks * 2 * B_PIECE;
                            mma_tf32_ss2(tmem + buf * 256, tc::desc_at(das, oa), tc::desc_at(dbb, ob), idesc, (kc | ks) != 0);     // small terms first
                            mma_tf32_ss2(tmem + buf * 256, tc::desc_at(dab, oa), tc::desc_at(dbs, ob), idesc, true);
                            mma_tf32_ss2(tmem + buf * 256, tc::desc_at(dab, oa), tc::desc_at(dbb, ob), idesc, true);
                        }
                        commit_pair(&empty[st]);
                    }
                    __syncwarp();
                }
                if (tc::elect_one()) commit_pair(&acc_full[buf]);
                __syncwarp();
            }
        }
    } else {
        // ------------------------------------------------------------------------------------------------ epilogue
        const int q4 = warp & 3, r = q4 * 32 + lane;
        const uint32_t tm_lane = tmem + ((uint32_t)(q4 * 32) << 16);
        uint32_t accn = 0;
        for (long w = pair0; w < nwork; w += npair, ++accn) {
            int nt, nrows;
            long row0;
            const int k = pair_item(p, nblk, NT, w, (int)rank, nt, row0, nrows);
            const float *net = p.nets + k * p.net_stride;
            const long Rg = row0 + r;
            const bool ok = r < nrows;
            const int buf = accn & 1;
            tc::mbar_wait(&acc_full[buf], (accn >> 1) & 1);
            tc::fence_after();
            // 32 columns per step; the step's global loads are all issued before its first store (the activation pointers may
            // alias as far as the compiler knows: interleaved, every load would wait a full memory round trip behind a store)
            for (int c0 = 0; c0 < BN; c0 += 32) {
                const int col = nt * BN + c0;
                float4 xa[8], xb[8], xc[8];
                if (ok) {
#pragma unroll
                    for (int q = 0; q < 8; ++q) {
                        const int cq = col + 4 * q;
                        if (MODE == 0) {
                            xa[q] = *reinterpret_cast<const float4 *>(net + wg_off_b2(W) + cq);
                            xb[q] = *reinterpret_cast<const float4 *>(p.T1 + Rg * W + (cq % W));
                        } else if (MODE == 1) {
                            xa[q] = *reinterpret_cast<const float4 *>(net + wg_off_b3(W) + cq);
                        } else if (MODE == 2) {
                            xa[q] = *reinterpret_cast<const float4 *>(p.Y2 + Rg * 2 * W + cq);
                            xb[q] = *reinterpret_cast<const float4 *>(p.T2 + Rg * 2 * W + cq);
                        } else {
                            xa[q] = *reinterpret_cast<const float4 *>(p.Y2 + Rg * 2 * W + cq);
                            xb[q] = *reinterpret_cast<const float4 *>(p.Y2 + Rg * 2 * W + W + cq);
                            xc[q] = *reinterpret_cast<const float4 *>(p.T1 + Rg * W + cq);
                        }
                    }
                }
                uint32_t z[32];
                tc::ld16(tm_lane + buf * 256 + c0, *reinterpret_cast<uint32_t(*)[16]>(&z[0]));
                tc::ld16(tm_lane + buf * 256 + c0 + 16, *reinterpret_cast<uint32_t(*)[16]>(&z[16]));
                tc::wait_ld();
                if (!ok) continue;
#pragma unroll
                for (int q = 0; q < 8; ++q) {
                    const int cq = col + 4 * q;
                    float4 v = make_float4(__uint_as_float(z[4 * q]), __uint_as_float(z[4 * q + 1]), __uint_as_float(z[4 * q + 2]), __uint_as_float(z[4 * q + 3]));
                    if (MODE == 0) {
                        v.x = tanhf(v.x + xa[q].x); v.y = tanhf(v.y + xa[q].y); v.z = tanhf(v.z + xa[q].z); v.w = tanhf(v.w + xa[q].w);
                        *reinterpret_cast<float4 *>(p.T2 + Rg * 2 * W + cq) = v;
                        v.x += xb[q].x; v.y += xb[q].y; v.z += xb[q].z; v.w += xb[q].w;
                        *reinterpret_cast<float4 *>(p.Y2 + Rg * 2 * W + cq) = v;
                    } else if (MODE == 1) {
                        v.x = tanhf(v.x + xa[q].x); v.y = tanhf(v.y + xa[q].y); v.z = tanhf(v.z + xa[q].z); v.w = tanhf(v.w + xa[q].w);
                        *reinterpret_cast<float4 *>(p.T3 + Rg * 4 * W + cq) = v;
                    } else if (MODE == 2) {
                        const float4 t = xb[q];
                        v.x += xa[q].x; v.y += xa[q].y; v.z += xa[q].z; v.w += xa[q].w;
                        *reinterpret_cast<float4 *>(p.Y2 + Rg * 2 * W + cq) = v;
                        v.x *= 1.f - t.x * t.x; v.y *= 1.f - t.y * t.y; v.z *= 1.f - t.z * t.z; v.w *= 1.f - t.w * t.w;
                        *reinterpret_cast<float4 *>(p.T2 + Rg * 2 * W + cq) = v;
                    } else {
                        const float4 t = xc[q];
                        v.x = (v.x + xa[q].x + xb[q].x) * (1.f - t.x * t.x); v.y = (v.y + xa[q].y + xb[q].y) * (1.f - t.y * t.y);
                        v.z = (v.z + xa[q].z + xb[q].z) * (1.f - t.z * t.z); v.w = (v.w + xa[q].w + xb[q].w) * (1.f - t.w * t.w);
                        *reinterpret_cast<float4 *>(p.T1 + Rg * W + cq) = v;
                    }
                }
            }
            tc::fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive_leader(&acc_empty[buf]);
        }
    }
    tc::fence_before();
    cluster_sync_all();
    tc::fence_after();
    if (warp == 12) asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(512));
}

// S5: A_i[c][m] = (1 / Nm) sum over the atom's rows of wt R^[c] G[m], G[m] = y2[m mod 2 W] + t3[m]; wt = the number of padded
// slots a representative row stands for, 1 for a real row.  One thread per 16 bytes of columns.
template <typename R>
__global__ void __launch_bounds__(256)
k_wg_contract(long N, int T, int W, R inv_nm, const __grid_constant__ TypeTab tt, const int *__restrict__ rowstart,
              const R *__restrict__ rh, const int2 *__restrict__ rows_id, const R *__restrict__ Y2, const R *__restrict__ T3,
              R *__restrict__ Aout) {
    constexpr int V = Vec<R>::V;
    const long i = blockIdx.x;
    const int m = (blockIdx.y * blockDim.x + threadIdx.x) * V, f = m % (2 * W), M2 = 4 * W;
    R acc[4][V];
#pragma unroll
    for (int c = 0; c < 4; ++c)
#pragma unroll
        for (int q = 0; q < V; ++q) acc[c][q] = (R)0;
    for (int b = 0; b < T; ++b) {
        const int r0 = rowstart[(long)b * (N + 1) + i], r1 = rowstart[(long)b * (N + 1) + i + 1];
        const long base = N * (long)tt.off[b];
#pragma unroll 4
        for (int row = r0; row < r1; ++row) {
            const long Rg = base + row;
            const int jj = rows_id[Rg].y;
            const R wt = jj < 0 ? (R)(-jj) : (R)1;
            const Vec<R> y = vld(Y2 + Rg * 2 * W + f), t = vld(T3 + Rg * M2 + m);
            R r[4];
#pragma unroll
            for (int c = 0; c < 4; ++c) r[c] = rh[4 * Rg + c] * wt;
#pragma unroll
            for (int q = 0; q < V; ++q) {
                const R G = y.v[q] + t.v[q];
#pragma unroll
                for (int c = 0; c < 4; ++c) acc[c][q] += r[c] * G;
            }
        }
    }
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        Vec<R> o;
#pragma unroll
        for (int q = 0; q < V; ++q) o.v[q] = acc[c][q] * inv_nm;
        vst(Aout + (i * 4 + c) * M2 + m, o);
    }
}

// Head of the backward pass; one CTA per atom, one warp per row, a lane per pair of columns (f, f + 2 W):
//   gG[m]  = (1 / Nm) sum_c R^[c] gA[c][m]       gradient of E with respect to G of a real row
//   dz3    = gG (1 - t3^2)                       -> over t3 (A operand of gemm<2>)
//   gG[f] + gG[f + 2 W]                          -> over y2 (the skip connection's share of dy2, added in the epilogue of gemm<2>)
//   dR^[c] = (1 / Nm) sum_m G[m] gA[c][m]        -> dR
// The representative of the padded slots carries no gradient (R~ = 0 there is a constant): its rows are zeroed.
template <typename R>
__global__ void __launch_bounds__(256)
k_wg_bwd_head(long N, int T, int W, R inv_nm, const __grid_constant__ TypeTab tt, const int *__restrict__ rowstart,
              const R *__restrict__ rh, const int2 *__restrict__ rows_id, const R *__restrict__ gA, R *__restrict__ Y2,
              R *__restrict__ T3, R *__restrict__ dR) {
    const long i = blockIdx.x;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, M2 = 4 * W;
    const R *__restrict__ ga = gA + i * 4L * M2;
    for (int b = 0; b < T; ++b) {
        const int r0 = rowstart[(long)b * (N + 1) + i], r1 = rowstart[(long)b * (N + 1) + i + 1];
        const long base = N * (long)tt.off[b];
        for (int row = r0 + warp; row < r1; row += 8) {
            const long Rg = base + row;
            R *__restrict__ y2 = Y2 + Rg * 2 * W;
            R *__restrict__ t3 = T3 + Rg * M2;
            constexpr int V = Vec<R>::V;
            if (rows_id[Rg].y < 0) {
                Vec<R> zero;
#pragma unroll
                for (int q = 0; q < V; ++q) zero.v[q] = (R)0;
                for (int f = lane * V; f < 2 * W; f += 32 * V) { vst(y2 + f, zero); vst(t3 + f, zero); vst(t3 + f + 2 * W, zero); }
                if (lane < 4) dR[4 * Rg + lane] = (R)0;
                continue;
            }
            R r[4], acc[4] = {(R)0, (R)0, (R)0, (R)0};
#pragma unroll
            for (int c = 0; c < 4; ++c) r[c] = rh[4 * Rg + c] * inv_nm;
#pragma unroll 2
            for (int f = lane * V; f < 2 * W; f += 32 * V) {
                const Vec<R> y = vld(y2 + f), ta = vld(t3 + f), tb = vld(t3 + f + 2 * W);
                Vec<R> a[4], bq[4], oa, ob, oy;
#pragma unroll
                for (int c = 0; c < 4; ++c) { a[c] = vld(ga + c * M2 + f); bq[c] = vld(ga + c * M2 + 2 * W + f); }
#pragma unroll
                for (int q = 0; q < V; ++q) {
                    const R Ga = y.v[q] + ta.v[q], Gb = y.v[q] + tb.v[q];
                    R gGa = (R)0, gGb = (R)0;
#pragma unroll
                    for (int c = 0; c < 4; ++c) {
                        gGa += r[c] * a[c].v[q]; gGb += r[c] * bq[c].v[q];
                        acc[c] += Ga * a[c].v[q] + Gb * bq[c].v[q];
                    }
                    oa.v[q] = gGa * ((R)1 - ta.v[q] * ta.v[q]);
                    ob.v[q] = gGb * ((R)1 - tb.v[q] * tb.v[q]);
                    oy.v[q] = gGa + gGb;
                }
                vst(t3 + f, oa); vst(t3 + f + 2 * W, ob); vst(y2 + f, oy);
            }
#pragma unroll
            for (int c = 0; c < 4; ++c) {
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) acc[c] += __shfl_xor_sync(0xffffffffu, acc[c], o);
            }
            if (lane == 0) {
#pragma unroll
                for (int c = 0; c < 4; ++c) dR[4 * Rg + c] = acc[c] * inv_nm;
            }
        }
    }
}

// Layer 1 backward and the normalisation: ds^ = dz1 . w1 (dz1 in T1 after gemm<3>); dE/dR~[c] = (dR^[c] + [c = 0] ds^) / std[c],
// written over dR.  One CTA per tile, one warp per row.
template <typename R>
__global__ void __launch_bounds__(256)
k_wg_ds(long N, int T, int W, const __grid_constant__ TypeTab tt, const int4 *__restrict__ tab, const R *__restrict__ nets,
        long net_stride, const double *__restrict__ stdv, const R *__restrict__ T1, R *__restrict__ dR) {
    const int nblk = T * T;
    const int tile = blockIdx.x;
    if (tile >= tab[nblk].x) return;
    const int k = wg_block(tab, nblk, tile);
    const int4 e = tab[k];
    const long rbase = N * (long)tt.off[k % T];
    const int row0 = e.y + (tile - e.x) * GR;
    const int nrows = min(GR, e.z - row0);
    const R *w1 = nets + k * net_stride;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, a = k / T;
    for (int rr = warp; rr < nrows; rr += 8) {
        const long Rg = rbase + row0 + rr;
        R ds = (R)0;
        for (int c = lane; c < W; c += 32) ds += T1[Rg * W + c] * w1[c];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) ds += __shfl_xor_sync(0xffffffffu, ds, o);
        if (lane < 4) dR[4 * Rg + lane] = (R)(((double)dR[4 * Rg + lane] + (lane == 0 ? (double)ds : 0.0)) / stdv[4 * a + lane]);
    }
}

// S8 + S9: per real row, the geometry derivative N9 in fp64, F_i += g, F_j -= g, Xi_ab -= d_a g_b (Q18)
template <typename R>
__global__ void __launch_bounds__(256)
k_wg_force(long N, int b, long row_off, EnvParams ep, const int *__restrict__ rowstart, const int2 *__restrict__ rows_id,
           const R *__restrict__ gR, const double *__restrict__ xs, double *__restrict__ fsorted, double *__restrict__ virial) {
    const long row = blockIdx.x * 256L + threadIdx.x;
    const int nrow = rowstart[(long)b * (N + 1) + N];
    double vir[9];
#pragma unroll
    for (int k = 0; k < 9; ++k) vir[k] = 0.0;
    if (row < nrow) {
        const long Rg = row_off + row;
        const int2 id = rows_id[Rg];
        if (id.y >= 0) {
            const long i = id.x, j = id.y;
            const double dx = min_image(xs[3 * j] - xs[3 * i], ep.L[0], 0.5 * ep.L[0]);
            const double dy = min_image(xs[3 * j + 1] - xs[3 * i + 1], ep.L[1], 0.5 * ep.L[1]);
            const double dz = min_image(xs[3 * j + 2] - xs[3 * i + 2], ep.L[2], 0.5 * ep.L[2]);
            double Rt[4], sp, rl;
            env_row(ep, dx, dy, dz, Rt, &sp, &rl);
            const double s = Rt[0];
            const double g0 = (double)gR[4 * Rg], g1 = (double)gR[4 * Rg + 1], g2 = (double)gR[4 * Rg + 2], g3 = (double)gR[4 * Rg + 3];
            const double d[3] = {dx, dy, dz};
            const double gd = g1 * dx + g2 * dy + g3 * dz;
            const double coef = (sp / rl - s / (rl * rl)) / rl;
#pragma unroll
            for (int bb = 0; bb < 3; ++bb) {
                const double gk = g0 * sp * d[bb] / rl + coef * d[bb] * gd + (s / rl) * (bb == 0 ? g1 : (bb == 1 ? g2 : g3));
                atomicAdd(&fsorted[3 * i + bb], gk);
                atomicAdd(&fsorted[3 * j + bb], -gk);
#pragma unroll
                for (int aa = 0; aa < 3; ++aa) vir[3 * aa + bb] -= d[aa] * gk;
            }
        }
    }
#pragma unroll
    for (int k = 0; k < 9; ++k) {
        double v = vir[k];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if ((threadIdx.x & 31) == 0 && v != 0.0) atomicAdd(&virial[k], v);
    }
}

}  // namespace

// ---- host side -------------------------------------------------------------------------------------------------------------

// fp32 blocks carry the weight matrices twice: rounded to TF32, and the TF32 remainders (the 3xTF32 products of k_wg_gemm)
size_t wide_gen_net_elems(int W, bool f64) { return 8 * (size_t)W + (f64 ? 20 : 40) * (size_t)W * W; }

static float tf32_rna(float x) {          // cvt.rna.tf32.f32: nearest, ties away from zero, 13 low mantissa bits cleared
    uint32_t u;
    std::memcpy(&u, &x, 4);
    u = (u + 0x1000u) & 0xffffe000u;
    std::memcpy(&x, &u, 4);
    return x;
}

// net: w1[W] b1[W] W2[W][2W] b2[2W] W3[2W][4W] b3[4W] (dp_weights order) -> the parameter block of the kernels above
template <typename R>
static void build_net(int W, const double *net, R *out) {
    const double *w1 = net, *b1 = w1 + W, *W2 = b1 + W, *b2 = W2 + (size_t)W * 2 * W, *W3 = b2 + 2 * W, *b3 = W3 + (size_t)2 * W * 4 * W;
    for (int e = 0; e < W; ++e) { out[e] = (R)w1[e]; out[W + e] = (R)b1[e]; }
    for (int f = 0; f < 2 * W; ++f) out[wg_off_b2(W) + f] = (R)b2[f];
    for (int m = 0; m < 4 * W; ++m) out[wg_off_b3(W) + m] = (R)b3[m];
    for (int e = 0; e < W; ++e)
        for (int f = 0; f < 2 * W; ++f) {
            out[wg_off_W2(W) + (size_t)e * 2 * W + f] = (R)W2[(size_t)e * 2 * W + f];
            out[wg_off_W2T(W) + (size_t)f * W + e] = (R)W2[(size_t)e * 2 * W + f];
        }
    for (int f = 0; f < 2 * W; ++f)
        for (int m = 0; m < 4 * W; ++m) {
            out[wg_off_W3(W) + (size_t)f * 4 * W + m] = (R)W3[(size_t)f * 4 * W + m];
            out[wg_off_W3T(W) + (size_t)m * 2 * W + f] = (R)W3[(size_t)f * 4 * W + m];
        }
}
// MIX-32: the operand images of B^T [NTOT][K] of one product: per N tile (BN = min(256, NTOT) rows), per K = 32 stage and per half
// of the tile's rows (one half per CTA of a pair) the TF32 values [4 pieces][BN / 2][4] followed by the TF32 remainders in the
// same order, pieces of 16 bytes of K outermost (one contiguous bulk copy per stage and CTA)
static void tf32_image(const std::vector<float> &Bt, int NTOT, int K, float *out) {
    const int BN = NTOT < 256 ? NTOT : 256, HB = BN / 2, NKC = K / TQ_KC;
    for (int n = 0; n < NTOT; ++n)
        for (int k = 0; k < K; ++k) {
            const float x = Bt[(size_t)n * K + k], big = tf32_rna(x), small = tf32_rna(x - big);
            const size_t half = ((size_t)((n / BN) * NKC + k / TQ_KC) * 2 + (n % BN) / HB) * (2 * (size_t)HB * TQ_KC);
            const size_t in = (size_t)((k % TQ_KC) / 4) * (HB * 4) + (size_t)(n % HB) * 4 + (k % 4);
            out[half + in] = big;
            out[half + (size_t)HB * TQ_KC + in] = small;
        }
}
__host__ __device__ inline long wg_off_img(int W, int mode) {      // MODE 0: W2^T, 1: W3^T, 2: W3, 3: W2 as B^T [NTOT][K]
    return 8L * W + (mode == 0 ? 0L : mode == 1 ? 4L : mode == 2 ? 20L : 36L) * W * W;
}
void wide_gen_build_net(int W, bool f64, const double *net, void *out) {
    if (f64) { build_net<double>(W, net, (double *)out); return; }
    float *o = (float *)out;
    const double *w1 = net, *b1 = w1 + W, *W2 = b1 + W, *b2 = W2 + (size_t)W * 2 * W, *W3 = b2 + 2 * W, *b3 = W3 + (size_t)2 * W * 4 * W;
    for (int e = 0; e < W; ++e) { o[e] = (float)w1[e]; o[W + e] = (float)b1[e]; }
    for (int f = 0; f < 2 * W; ++f) o[wg_off_b2(W) + f] = (float)b2[f];
    for (int m = 0; m < 4 * W; ++m) o[wg_off_b3(W) + m] = (float)b3[m];
    std::vector<float> w2((size_t)W * 2 * W), w2t(w2.size()), w3((size_t)2 * W * 4 * W), w3t(w3.size());
    for (int e = 0; e < W; ++e)
        for (int f = 0; f < 2 * W; ++f) { w2[(size_t)e * 2 * W + f] = (float)W2[(size_t)e * 2 * W + f]; w2t[(size_t)f * W + e] = w2[(size_t)e * 2 * W + f]; }
    for (int f = 0; f < 2 * W; ++f)
        for (int m = 0; m < 4 * W; ++m) { w3[(size_t)f * 4 * W + m] = (float)W3[(size_t)f * 4 * W + m]; w3t[(size_t)m * 2 * W + f] = w3[(size_t)f * 4 * W + m]; }
    tf32_image(w2t, 2 * W, W, o + wg_off_img(W, 0));        // t1 . W2:     B^T[f][e]
    tf32_image(w3t, 4 * W, 2 * W, o + wg_off_img(W, 1));    // y2 . W3:     B^T[m][f]
    tf32_image(w3, 2 * W, 4 * W, o + wg_off_img(W, 2));     // dz3 . W3^T:  B^T[f][m]
    tf32_image(w2, W, 2 * W, o + wg_off_img(W, 3));         // dz2 . W2^T:  B^T[e][f]
}

template <typename R>
static GenArgs<R> gen_args(const dp_model *m, long N, char *ws, const WsLayout &L) {
    GenArgs<R> p{};
    p.N = N; p.T = m->T; p.W = m->m0;
    p.tab = (const int4 *)(ws + L.wide_tab);
    p.nets = (const R *)m->wide_vec_dev; p.net_stride = (long)wide_gen_net_elems(m->m0, sizeof(R) == 8);
    p.T1 = (R *)(ws + L.wide_t1); p.Y2 = (R *)(ws + L.wide_y2); p.T2 = (R *)(ws + L.wide_t2); p.T3 = (R *)(ws + L.wide_t3);
    p.tt = make_typetab(m);
    return p;
}

typedef CUresult (*tmap_encode_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                   const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                   CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static tmap_encode_fn tmap_encoder() {
    static const tmap_encode_fn fn = [] {
        void *q = nullptr;
        cudaDriverEntryPointQueryResult res;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &q, cudaEnableDefault, &res) != cudaSuccess || res != cudaDriverEntryPointSuccess)
            q = nullptr;
        return (tmap_encode_fn)q;
    }();
    return fn;
}

// MIX-32: the tcgen05 kernel; bt_off = offset of the product's B^T [Nn][K] (the transposed copy of the weight matrix)
template <int MODE>
static cudaError_t gen_gemm_tf32(const dp_model *m, GenArgs<float> p, int K, int Nn, const float *A, long bt_off, cudaStream_t st) {
    DP_SMEM_OPTIN((k_wg_gemm_tf32<MODE>), TQ_TOTAL);
    p.K = K; p.NTOT = Nn; p.A = A; p.b_off = bt_off;
    // the activations [rows][K] as a (4, rows, K / 4) tensor: strides K * 4 bytes (rows) and 16 bytes (pieces of a row)
    const tmap_encode_fn enc = tmap_encoder();
    if (!enc) return cudaErrorNotSupported;
    CUtensorMap tm;
    const cuuint64_t gdim[3] = {4, (cuuint64_t)p.N * (cuuint64_t)m->Nm, (cuuint64_t)(K / 4)};
    const cuuint64_t gstr[2] = {(cuuint64_t)K * 4, 16};
    const cuuint32_t box[3] = {4, 128, TQ_KC / 4}, estr[3] = {1, 1, 1};
    if (enc(&tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, (void *)A, gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
            CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return cudaErrorInvalidValue;
    k_wg_gemm_tf32<MODE><<<m->num_sms & ~1, TQ_THREADS, TQ_TOTAL, st>>>(p, tm);      // CTA pairs (__cluster_dims__(2, 1, 1))
    return cudaGetLastError();
}

// b_off: offset of the product's weight matrix in the FP64 parameter block (MIX-32: the product's images, by MODE)
template <typename R, int MODE>
static cudaError_t gen_gemm(const dp_model *m, long N, GenArgs<R> p, int K, int Nn, const R *A, long b_off, cudaStream_t st) {
    if constexpr (sizeof(R) == 4) {
        return gen_gemm_tf32<MODE>(m, p, K, Nn, A, wg_off_img(m->m0, MODE), st);
    } else {
        DP_SMEM_OPTIN((k_wg_gemm_f64<MODE>), GemmCfg::SMEM);
        p.K = K; p.NTOT = Nn; p.A = A; p.b_off = b_off;
        const long tiles = wide_tiles_cap(m, N) * (GR / GBM), ntn = (Nn + GBN - 1) / GBN;
        k_wg_gemm_f64<MODE><<<(unsigned)(tiles * ntn), GTHREADS, GemmCfg::SMEM, st>>>(p);
        return cudaGetLastError();
    }
}

template <typename R>
static cudaError_t fwd_gen(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st) {
    const int W = m->m0, T = m->T;
    const TypeTab tt = make_typetab(m);
    cudaError_t e = cudaSuccess;
    auto ok = [&](cudaError_t x) { if (e == cudaSuccess) e = x; };
    const GenArgs<R> p = gen_args<R>(m, N, ws, L);
    R *rh = (R *)(ws + L.wide_rh);
    int2 *rows_id = (int2 *)(ws + L.rows_id);
    const int *rowstart = (const int *)(ws + L.rowstart);
    k_wg_env<R><<<(unsigned)((N + 7) / 8), 256, 0, st>>>(N, T, g.ncell, m->Nm, tt, make_env(m, g), m->avg_dev, m->std_dev,
                                                         (const int *)(ws + L.bin_start), (const double *)(ws + L.xs),
                                                         (const int *)(ws + L.nlist), (const int *)(ws + L.nreal), rowstart, rh, rows_id);
    ok(cudaGetLastError());
    ok(launch_wide_tiles(m, N, g, ws, L, st));
    const unsigned tiles = (unsigned)wide_tiles_cap(m, N);
    k_wg_l1<R><<<tiles, 256, 0, st>>>(N, T, W, tt, p.tab, p.nets, p.net_stride, rh, p.T1);
    ok(cudaGetLastError());
    ok((gen_gemm<R, 0>(m, N, p, W, 2 * W, p.T1, wg_off_W2(W), st)));
    ok((gen_gemm<R, 1>(m, N, p, 2 * W, 4 * W, p.Y2, wg_off_W3(W), st)));
    const int cthreads = 4 * W / Vec<R>::V < 256 ? 4 * W / Vec<R>::V : 256;       // one thread per 16 bytes of the 4 W columns
    k_wg_contract<R><<<dim3((unsigned)N, (unsigned)(4 * W / Vec<R>::V / cthreads)), cthreads, 0, st>>>(N, T, W, (R)(1.0 / (double)m->Nm), tt, rowstart, rh, rows_id,
                                                                              p.Y2, p.T3, (R *)(ws + L.A));
    ok(cudaGetLastError());
    return e;
}

template <typename R>
static cudaError_t bwd_gen(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st) {
    const int W = m->m0, T = m->T;
    const TypeTab tt = make_typetab(m);
    cudaError_t e = cudaSuccess;
    auto ok = [&](cudaError_t x) { if (e == cudaSuccess) e = x; };
    const GenArgs<R> p = gen_args<R>(m, N, ws, L);
    const R *rh = (const R *)(ws + L.wide_rh);
    R *dR = (R *)(ws + L.wide_gr);
    const int2 *rows_id = (const int2 *)(ws + L.rows_id);
    const int *rowstart = (const int *)(ws + L.rowstart);
    // gA [N][4][m2]: FP64 from k_gA_wide (fit_f64.cu), MIX-32 left in the gD buffer by the last fitting product (fit_tc.cu MODE 6)
    const R *gA = sizeof(R) == 8 ? (const R *)(ws + L.gAf) : (const R *)(ws + L.gD);
    k_wg_bwd_head<R><<<(unsigned)N, 256, 0, st>>>(N, T, W, (R)(1.0 / (double)m->Nm), tt, rowstart, rh, rows_id, gA, p.Y2, p.T3, dR);
    ok(cudaGetLastError());
    if (m->profile) cudaEventRecord(m->ev[6], st);      // ev[6] .. ev[7]: the two backward GEMMs
    ok((gen_gemm<R, 2>(m, N, p, 4 * W, 2 * W, p.T3, wg_off_W3T(W), st)));
    ok((gen_gemm<R, 3>(m, N, p, 2 * W, W, p.T2, wg_off_W2T(W), st)));
    if (m->profile) cudaEventRecord(m->ev[7], st);
    const unsigned tiles = (unsigned)wide_tiles_cap(m, N);
    k_wg_ds<R><<<tiles, 256, 0, st>>>(N, T, W, tt, p.tab, p.nets, p.net_stride, m->std_dev, p.T1, dR);
    ok(cudaGetLastError());
    for (int b = 0; b < T; ++b) {
        const long cap = N * (long)m->sel[b];
        k_wg_force<R><<<(unsigned)((cap + 255) / 256), 256, 0, st>>>(N, b, N * (long)m->off[b], make_env(m, g), rowstart, rows_id, dR,
                                                                    (const double *)(ws + L.xs), (double *)(ws + L.fsorted),
                                                                    (double *)(ws + L.virial));
        ok(cudaGetLastError());
    }
    return e;
}

cudaError_t launch_embed_fwd_wide_gen(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st) {
    return m->prec == DP_FP64 ? fwd_gen<double>(m, N, g, ws, L, st) : fwd_gen<float>(m, N, g, ws, L, st);
}
cudaError_t launch_embed_bwd_wide_gen(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st) {
    return m->prec == DP_FP64 ? bwd_gen<double>(m, N, g, ws, L, st) : bwd_gen<float>(m, N, g, ws, L, st);
}
