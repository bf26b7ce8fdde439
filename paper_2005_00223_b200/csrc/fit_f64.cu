// S5 (descriptor) + S6 (fitting net forward and backward) of SURVEY.md section 8(a), FP64 mode.
//
// D_i = A_i^T A_i[:, :M2] ("the descriptor is the product of terms involving R~ and G"), fitting net
// 1600 -> 240 -> 240 -> 240 -> 1 with identity skips (Fig. 1(d),(f), 151), backward by hand with
// tanh' = 1 - tanh^2 fused into the GEMM epilogues.  The GEMMs are batched over the atoms of one
// centre type and run on the FP64 tensor pipe (DMMA m8n8k4); bias, tanh, skip and tanh' live in the epilogue
// (PAPER.md:133-134 merged them into cuBLAS GEMM calls; here they never reach memory as separate passes).
#include "dp_internal.h"
#include "tanh64.cuh"

namespace {

constexpr int BM = 64, BN = 80, BK = 16;
constexpr int AS_STRIDE = BK + 4;      // doubles; conflict-free A-fragment loads
constexpr int BS_STRIDE = BN + 4;      // doubles; conflict-free B-fragment loads (B stored [k][n])
constexpr int BT_STRIDE = BK + 4;      // B stored [n][k] for the transposed products
constexpr int AS_TILE = BM * AS_STRIDE;
constexpr int B_TILE = (BK * BS_STRIDE > BN * BT_STRIDE) ? BK * BS_STRIDE : BN * BT_STRIDE;

__device__ __forceinline__ void dmma(double &c0, double &c1, double a, double b) {
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
        : "+d"(c0), "+d"(c1)
        : "d"(a), "d"(b));
}

__device__ __forceinline__ void cp_async16(void *smem_dst, const void *gsrc, bool valid) {
    unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    int sz = valid ? 16 : 0;
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(s), "l"(gsrc), "r"(sz));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N)); }

struct FitArgs {
    int ncell;
    const int *bin_start;
    int K, N;                 // GEMM inner and output widths
    int ksplit;               // MODE 0 on small systems: K is split over ksplit CTAs per output tile (0 / 1: no split); the partial
                              // sums meet in out0 (zeroed by the launcher) through fp64 atomics and k_bias_tanh finishes the layer
    const double *A; int lda;             // [rows][K]
    const double *B; long b_type_stride; int ldb;   // weights of type a at B + a*b_type_stride
    const double *bias; int bias_type_stride;       // epilogue vector (c1/c2/c3 or v4)
    const double *v4; int v4_type_stride;
    const double *aux0; const double *aux1;         // epilogue inputs [rows][240]
    double *out0; double *out1; int ldo;
};

// MODE: 0 L1 fwd, 1 L2 fwd, 2 L3 fwd, 3 L3 bwd, 4 L2 bwd, 5 L1 bwd (see file header of DESIGN.md section "fitting")
template <int MODE>
__global__ void __launch_bounds__(256) k_fit_gemm(FitArgs p) {
    constexpr bool BT = MODE >= 3;
    __shared__ __align__(16) double sm[2 * (AS_TILE + B_TILE)];
    const int a = blockIdx.z;
    const int ts0 = p.bin_start[a * p.ncell], ts1 = p.bin_start[(a + 1) * p.ncell];
    const int row0 = ts0 + blockIdx.x * BM;
    if (row0 >= ts1) return;
    const int ntn = (p.N + BN - 1) / BN;
    const int n0 = (blockIdx.y % ntn) * BN, kpart = blockIdx.y / ntn;
    const bool split = MODE == 0 && p.ksplit > 1;
    const double *Bw = p.B + a * p.b_type_stride;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int wm = wid >> 1, wn = wid & 1;         // 4 x 2 warps, warp tile 16 x 40
    const int q4 = lane >> 2, r = lane & 3;

    auto load_tiles = [&](int stage, int k0) {
        double *As = sm + stage * (AS_TILE + B_TILE);
        double *Bs = As + AS_TILE;
#pragma unroll
        for (int c = tid; c < BM * (BK / 2); c += 256) {
            const int row = c >> 3, c8 = c & 7;
            const bool ok = row0 + row < ts1;
            const double *src = p.A + (long)(ok ? row0 + row : ts0) * p.lda + k0 + 2 * c8;
            cp_async16(As + row * AS_STRIDE + 2 * c8, src, ok);
        }
        if (!BT) {
            for (int c = tid; c < BK * (BN / 2); c += 256) {
                const int k = c / (BN / 2), cc = c % (BN / 2);
                const bool okn = n0 + 2 * cc < p.N;
                cp_async16(Bs + k * BS_STRIDE + 2 * cc, Bw + (long)(k0 + k) * p.ldb + (okn ? n0 + 2 * cc : 0), okn);
            }
        } else {
            for (int c = tid; c < BN * (BK / 2); c += 256) {
                const int n = c >> 3, c8 = c & 7;
                const bool okn = n0 + n < p.N;
                cp_async16(Bs + n * BT_STRIDE + 2 * c8, Bw + (long)(okn ? n0 + n : 0) * p.ldb + k0 + 2 * c8, okn);
            }
        }
        cp_async_commit();
    };

    double acc[2][5][2];
#pragma unroll
    for (int mt = 0; mt < 2; ++mt)
#pragma unroll
        for (int nt = 0; nt < 5; ++nt) acc[mt][nt][0] = acc[mt][nt][1] = 0.0;

    const int nk_all = p.K / BK;
    const int nk = split ? nk_all / p.ksplit : nk_all, kb = split ? kpart * nk : 0;      // k-steps of this CTA: [kb, kb + nk)
    load_tiles(0, kb * BK);
    for (int ks = 0; ks < nk; ++ks) {
        if (ks + 1 < nk) { load_tiles((ks + 1) & 1, (kb + ks + 1) * BK); cp_async_wait<1>(); }
        else cp_async_wait<0>();
        __syncthreads();
        const double *As = sm + (ks & 1) * (AS_TILE + B_TILE);
        const double *Bs = As + AS_TILE;
#pragma unroll
        for (int kc = 0; kc < BK / 4; ++kc) {
            double af[2], bf[5];
#pragma unroll
            for (int mt = 0; mt < 2; ++mt) af[mt] = As[(wm * 16 + mt * 8 + q4) * AS_STRIDE + kc * 4 + r];
#pragma unroll
            for (int nt = 0; nt < 5; ++nt)
                bf[nt] = BT ? Bs[(wn * 40 + nt * 8 + q4) * BT_STRIDE + kc * 4 + r]
                            : Bs[(kc * 4 + r) * BS_STRIDE + wn * 40 + nt * 8 + q4];
#pragma unroll
            for (int mt = 0; mt < 2; ++mt)
#pragma unroll
                for (int nt = 0; nt < 5; ++nt) dmma(acc[mt][nt][0], acc[mt][nt][1], af[mt], bf[nt]);
        }
        __syncthreads();
    }

    // epilogue: thread holds (row = wm*16 + mt*8 + q4, cols n0 + wn*40 + nt*8 + 2r + {0,1})
#pragma unroll
    for (int mt = 0; mt < 2; ++mt) {
        const int row = row0 + wm * 16 + mt * 8 + q4;
        if (row >= ts1) continue;
#pragma unroll
        for (int nt = 0; nt < 5; ++nt) {
            const int col = n0 + wn * 40 + nt * 8 + 2 * r;
            if (col >= p.N) continue;          // N = 16 m2 need not be a multiple of the tile width
            const long o = (long)row * p.ldo + col;
            double v0 = acc[mt][nt][0], v1 = acc[mt][nt][1];
            if (MODE == 0 && split) {
                atomicAdd(p.out0 + o, v0);
                atomicAdd(p.out0 + o + 1, v1);
            } else if (MODE == 0) {
                const double *b = p.bias + a * p.bias_type_stride + col;
                *reinterpret_cast<double2 *>(p.out0 + o) = make_double2(dp_tanh64(v0 + b[0]), dp_tanh64(v1 + b[1]));
            } else if (MODE == 1) {
                const double *b = p.bias + a * p.bias_type_stride + col;
                const double2 h = *reinterpret_cast<const double2 *>(p.aux0 + o);
                const double t0 = dp_tanh64(v0 + b[0]), t1 = dp_tanh64(v1 + b[1]);
                *reinterpret_cast<double2 *>(p.out0 + o) = make_double2(t0, t1);
                *reinterpret_cast<double2 *>(p.out1 + o) = make_double2(h.x + t0, h.y + t1);
            } else if (MODE == 2) {
                const double *b = p.bias + a * p.bias_type_stride + col;
                const double *v4 = p.v4 + a * p.v4_type_stride + col;
                const double2 h = *reinterpret_cast<const double2 *>(p.aux0 + o);
                const double t0 = dp_tanh64(v0 + b[0]), t1 = dp_tanh64(v1 + b[1]);
                *reinterpret_cast<double2 *>(p.out0 + o) = make_double2(v4[0] * (1.0 - t0 * t0), v4[1] * (1.0 - t1 * t1));
                *reinterpret_cast<double2 *>(p.out1 + o) = make_double2(h.x + t0, h.y + t1);
            } else if (MODE == 3) {
                const double *v4 = p.v4 + a * p.v4_type_stride + col;
                const double2 t = *reinterpret_cast<const double2 *>(p.aux0 + o);     // t2
                const double g0 = v4[0] + v0, g1 = v4[1] + v1;
                *reinterpret_cast<double2 *>(p.out0 + o) = make_double2(g0, g1);
                *reinterpret_cast<double2 *>(p.out1 + o) = make_double2(g0 * (1.0 - t.x * t.x), g1 * (1.0 - t.y * t.y));
            } else if (MODE == 4) {
                const double2 g = *reinterpret_cast<const double2 *>(p.aux0 + o);     // g2
                const double2 h = *reinterpret_cast<const double2 *>(p.aux1 + o);     // h1
                const double g0 = g.x + v0, g1 = g.y + v1;
                *reinterpret_cast<double2 *>(p.out0 + o) = make_double2(g0 * (1.0 - h.x * h.x), g1 * (1.0 - h.y * h.y));
            } else {
                *reinterpret_cast<double2 *>(p.out0 + o) = make_double2(v0, v1);
            }
        }
    }
}

// second half of the split-K first layer: h1 = tanh(h1 + c1[type]) in place
__global__ void __launch_bounds__(256) k_bias_tanh(long N, int T, int ncell, int F, const int *__restrict__ bin_start,
                                                   const double *__restrict__ bias, double *__restrict__ h) {
    const long k = blockIdx.x * 256L + threadIdx.x;
    if (k >= N * F) return;
    const long i = k / F;
    const int col = (int)(k % F);
    int a = 0;
    for (int t = 1; t < T; ++t) a += i >= bin_start[t * ncell];
    h[k] = dp_tanh64(h[k] + bias[a * F + col]);
}

// D[i][m*16 + a] = sum_c A[i][c][m] A[i][c][a]    (N6, Q6, Q7); one warp per atom
template <int W>
__global__ void __launch_bounds__(256) k_descr(long N, const double *__restrict__ Amat, double *__restrict__ D) {
    constexpr int M2E = EmbW<W>::M2E;
    __shared__ double sA[8][4 * M2E];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const long i = blockIdx.x * 8L + wid;
    if (i >= N) return;
    for (int k = lane; k < 4 * M2E; k += 32) sA[wid][k] = Amat[i * 4 * M2E + k];
    __syncwarp();
    for (int idx = lane; idx < M2E * 16; idx += 32) {
        const int m = idx >> 4, ax = idx & 15;
        double acc = 0.0;
#pragma unroll
        for (int c = 0; c < 4; ++c) acc += sA[wid][c * M2E + m] * sA[wid][c * M2E + ax];
        D[i * (M2E * 16) + idx] = acc;
    }
}

__device__ __forceinline__ int type_of_sorted(int i, int T, int ncell, const int *bin_start) {
    int a = 0;
    for (int t = 1; t < T; ++t) a += i >= bin_start[t * ncell];
    return a;
}

// E_i = h3 . v4 + c4 + ebias[type]   (N7, Q10); one warp per atom
__global__ void __launch_bounds__(256) k_energy(long N, int T, int ncell, const int *__restrict__ bin_start,
                                                const double *__restrict__ h3, const double *__restrict__ v4,
                                                const double *__restrict__ c4, const double *__restrict__ ebias,
                                                double *__restrict__ eatom) {
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const long i = blockIdx.x * 8L + wid;
    if (i >= N) return;
    const int a = type_of_sorted((int)i, T, ncell, bin_start);
    double acc = 0.0;
    for (int n = lane; n < 240; n += 32) acc += h3[i * 240 + n] * v4[a * 240 + n];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (lane == 0) eatom[i] = acc + c4[a] + ebias[a];
}

template <int W>
__device__ __forceinline__ int feature3(int nt3, int r, int j3) {
    const int e = 4 * (nt3 >> 1) + r;
    return e < W ? e + W * (nt3 & 1) + 2 * W * j3 : -1;
}

// gA[c][m] = sum_a gD[m][a] A[c][a] + [m < 16] sum_m' gD[m'][m] A[c][m']   (N8), written as the MMA fragments the
// embedding backward consumes (layout in embed_f64.cu), pre-scaled by 1/Nm.  One CTA of four warps works on one atom at a time
// (20 KB of shared memory per CTA: eleven CTAs per SM; one warp per atom with its own 20 KB left eight warps per SM).
template <int W>
__global__ void __launch_bounds__(128) k_gA(long N, double inv_nm, const double *__restrict__ Amat,
                                            const double *__restrict__ gD, double *__restrict__ gAf) {
    constexpr int M2E = EmbW<W>::M2E, NT3 = EmbW<W>::NT3;
    extern __shared__ double smg[];
    double *sA = smg;                       // [4][M2E]
    double *sG = sA + 4 * M2E;              // [M2E][17]: rows of gD padded (lanes walk consecutive rows m: stride 16 was a 16-way bank conflict)
    double *sO = sG + M2E * 17;             // [4][M2E]
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    for (long i = blockIdx.x; i < N; i += gridDim.x) {
        __syncthreads();
        for (int k = tid; k < 4 * M2E; k += 128) sA[k] = Amat[i * 4 * M2E + k];
        for (int k = tid; k < M2E * 16; k += 128) sG[(k >> 4) * 17 + (k & 15)] = gD[i * (M2E * 16) + k];
        __syncthreads();
        for (int idx = tid; idx < 4 * M2E; idx += 128) {
            const int c = idx / M2E, m = idx % M2E;
            double acc = 0.0;
#pragma unroll
            for (int ax = 0; ax < 16; ++ax) acc += sG[m * 17 + ax] * sA[c * M2E + ax];
            if (m < 16)
                for (int mp = 0; mp < M2E; ++mp) acc += sG[mp * 17 + m] * sA[c * M2E + mp];
            sO[idx] = acc * inv_nm;
        }
        __syncthreads();
        double *out = gAf + i * (3 * NT3 * 32);
        const int q4 = lane >> 2, r = lane & 3;
        for (int nt3 = wid; nt3 < NT3; nt3 += 4) {
            const int f = feature3<W>(nt3, q4 >> 1, q4 & 1);
            out[nt3 * 32 + lane] = f >= 0 ? sO[r * M2E + f] : 0.0;
        }
        for (int kc = wid; kc < 2 * NT3; kc += 4) {
            const int f = feature3<W>(kc >> 1, r, kc & 1);
            out[(NT3 + kc) * 32 + lane] = (f >= 0 && q4 < 4) ? sO[q4 * M2E + f] : 0.0;
        }
    }
}

// Wide nets (wide_gen.cu; m2 = 4 W up to 2,048, a run-time value).  The descriptor: one thread per entry.
__global__ void __launch_bounds__(256) k_descr_wide(int M2, const double *__restrict__ Amat, double *__restrict__ D) {
    const long i = blockIdx.x;
    const int idx = blockIdx.y * 256 + threadIdx.x;           // M2 * 16 is a multiple of 256
    const int mm = idx >> 4, ax = idx & 15;
    const double *A = Amat + i * 4L * M2;
    double acc = 0.0;
#pragma unroll
    for (int c = 0; c < 4; ++c) acc += A[c * M2 + mm] * A[c * M2 + ax];
    D[i * (M2 * 16L) + idx] = acc;
}
// gA[c][m] = sum_a gD[m][a] A[c][a] + [m < 16] sum_m' gD[m'][m] A[c][m']   (N8), row-major [N][4][M2], without the 1 / Nm that
// the backward head applies.  One CTA per atom.  Second sum (a 4 x M2 by M2 x 16 product): thread (m', quarter q of the 16
// columns) reads 32 contiguous bytes of gD[m'] and keeps 4 x 4 partial sums; lanes of equal q meet by shuffles, warps in
// shared memory.  First sum: a thread per (c, m) reads the 128 contiguous bytes of gD[m].
__global__ void __launch_bounds__(256) k_gA_wide(int M2, const double *__restrict__ Amat, const double *__restrict__ gD,
                                                 double *__restrict__ gA) {
    __shared__ double part[8][64];
    __shared__ double s2[64];
    const long i = blockIdx.x;
    const double *A = Amat + i * 4L * M2, *G = gD + i * (M2 * 16L);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, q = threadIdx.x & 3;
    double acc[4][4];
#pragma unroll
    for (int c = 0; c < 4; ++c)
#pragma unroll
        for (int k = 0; k < 4; ++k) acc[c][k] = 0.0;
    for (int mp = threadIdx.x >> 2; mp < M2; mp += 64) {
        const double2 g0 = *reinterpret_cast<const double2 *>(G + mp * 16 + 4 * q), g1 = *reinterpret_cast<const double2 *>(G + mp * 16 + 4 * q + 2);
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            const double a = A[c * M2 + mp];
            acc[c][0] += g0.x * a; acc[c][1] += g0.y * a; acc[c][2] += g1.x * a; acc[c][3] += g1.y * a;
        }
    }
#pragma unroll
    for (int c = 0; c < 4; ++c)
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            double v = acc[c][k];
            v += __shfl_xor_sync(0xffffffffu, v, 4);
            v += __shfl_xor_sync(0xffffffffu, v, 8);
            v += __shfl_xor_sync(0xffffffffu, v, 16);
            if (lane < 4) part[warp][c * 16 + 4 * q + k] = v;
        }
    __syncthreads();
    if (threadIdx.x < 64) {
        double v = 0.0;
#pragma unroll
        for (int w = 0; w < 8; ++w) v += part[w][threadIdx.x];
        s2[threadIdx.x] = v;
    }
    __syncthreads();
    for (int idx = threadIdx.x; idx < 4 * M2; idx += 256) {
        const int c = idx / M2, mm = idx % M2;
        double acc1 = mm < 16 ? s2[c * 16 + mm] : 0.0;
        const double2 *g = reinterpret_cast<const double2 *>(G + mm * 16);
#pragma unroll
        for (int ax = 0; ax < 8; ++ax) { const double2 v = g[ax]; acc1 += v.x * A[c * M2 + 2 * ax] + v.y * A[c * M2 + 2 * ax + 1]; }
        gA[i * 4L * M2 + idx] = acc1;
    }
}

}  // namespace

// W = 0: a wide net (m2 taken from the model; descriptor and gA by the run-time kernels above)
template <int W>
static cudaError_t launch_fit_w(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st) {
    const int M2E = W ? EmbW<(W ? W : 25)>::M2E : m->m2;
    const int F = 240, ND = M2E * 16;
    const int T = m->T;
    double *Amat = (double *)(ws + L.A);
    double *D = (double *)(ws + L.gD);          // D and gD share one [N][1600] buffer (D is dead after layer 1)
    double *act = (double *)(ws + L.fit_act);
    const size_t S = (size_t)N * F;
    double *h1 = act, *t2 = act + S, *h2 = act + 2 * S, *gz3 = act + 3 * S, *h3 = act + 4 * S, *g2 = act + 5 * S,
           *gz2 = act + 6 * S, *gz1 = h2;      // h2 is dead after the layer-3 forward
    const int *bin_start = (const int *)(ws + L.bin_start);
    const double *V1 = (const double *)m->fitV1_dev, *V2 = (const double *)m->fitV2_dev, *V3 = (const double *)m->fitV3_dev;
    const double *c1 = (const double *)m->fitc1_dev, *c2 = (const double *)m->fitc2_dev, *c3 = (const double *)m->fitc3_dev;
    const double *v4 = (const double *)m->fitv4_dev, *c4 = (const double *)m->fitc4_dev;
    const unsigned gx = (unsigned)((N + BM - 1) / BM);
    const unsigned nb8 = (unsigned)((N + 7) / 8);

    if constexpr (W == 0) k_descr_wide<<<dim3((unsigned)N, (unsigned)(ND / 256)), 256, 0, st>>>(M2E, Amat, D);
    else k_descr<W><<<nb8, 256, 0, st>>>(N, Amat, D);

    FitArgs p{};
    p.ncell = g.ncell; p.bin_start = bin_start; p.v4 = v4; p.v4_type_stride = F; p.bias_type_stride = F;
    // layer 1 forward: h1 = tanh(D V1 + c1)
    p.K = ND; p.N = F; p.A = D; p.lda = ND; p.B = V1; p.b_type_stride = (long)ND * F; p.ldb = F; p.bias = c1;
    p.out0 = h1; p.ldo = F;
    // few row tiles (configs 0, 1: 24 / 72 CTAs walking K = 1,600): split K four ways so that the GPU fills
    p.ksplit = fit_f64_splitk(m, N) ? 4 : 1;
    if (p.ksplit > 1) {
        cudaMemsetAsync(h1, 0, sizeof(double) * S, st);
        k_fit_gemm<0><<<dim3(gx, (F / BN) * p.ksplit, T), 256, 0, st>>>(p);
        k_bias_tanh<<<(unsigned)((S + 255) / 256), 256, 0, st>>>(N, T, g.ncell, F, bin_start, c1, h1);
    } else {
        k_fit_gemm<0><<<dim3(gx, F / BN, T), 256, 0, st>>>(p);
    }
    p.ksplit = 1;
    // layer 2 forward: t2 = tanh(h1 V2 + c2), h2 = h1 + t2
    p.K = F; p.A = h1; p.lda = F; p.B = V2; p.b_type_stride = (long)F * F; p.bias = c2; p.aux0 = h1; p.out0 = t2; p.out1 = h2;
    k_fit_gemm<1><<<dim3(gx, F / BN, T), 256, 0, st>>>(p);
    // layer 3 forward: t3 = tanh(h2 V3 + c3), h3 = h2 + t3, gz3 = v4 (1 - t3^2)
    p.A = h2; p.B = V3; p.bias = c3; p.aux0 = h2; p.out0 = gz3; p.out1 = h3;
    k_fit_gemm<2><<<dim3(gx, F / BN, T), 256, 0, st>>>(p);
    k_energy<<<nb8, 256, 0, st>>>(N, T, g.ncell, bin_start, h3, v4, c4, m->ebias_dev, (double *)(ws + L.eatom));
    // layer 3 backward: g2 = v4 + gz3 V3^T, gz2 = g2 (1 - t2^2)
    p.A = gz3; p.B = V3; p.aux0 = t2; p.out0 = g2; p.out1 = gz2;
    k_fit_gemm<3><<<dim3(gx, F / BN, T), 256, 0, st>>>(p);
    // layer 2 backward: g1 = g2 + gz2 V2^T, gz1 = g1 (1 - h1^2)
    p.A = gz2; p.B = V2; p.aux0 = g2; p.aux1 = h1; p.out0 = gz1; p.out1 = nullptr;
    k_fit_gemm<4><<<dim3(gx, F / BN, T), 256, 0, st>>>(p);
    // layer 1 backward: gD = gz1 V1^T
    p.A = gz1; p.N = ND; p.B = V1; p.b_type_stride = (long)ND * F; p.out0 = D; p.ldo = ND;
    k_fit_gemm<5><<<dim3(gx, (ND + BN - 1) / BN, T), 256, 0, st>>>(p);
    // gD, A -> gA fragments for the embedding backward
    if constexpr (W == 0) {
        k_gA_wide<<<(unsigned)N, 256, 0, st>>>(M2E, Amat, D, (double *)(ws + L.gAf));
    } else {
        const int smem = (4 * M2E + M2E * 17 + 4 * M2E) * 8;
        const long gmax = (long)m->num_sms * 11;
        k_gA<W><<<(unsigned)(N < gmax ? N : gmax), 128, smem, st>>>(N, 1.0 / (double)m->Nm, Amat, D, (double *)(ws + L.gAf));
    }
    return cudaGetLastError();
}

cudaError_t launch_fit_f64(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st) {
    if (m->wide) return launch_fit_w<0>(m, N, g, ws, L, st);
    return m->m0 == 32 ? launch_fit_w<32>(m, N, g, ws, L, st) : launch_fit_w<25>(m, N, g, ws, L, st);
}
