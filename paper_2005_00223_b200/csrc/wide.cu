// S4 + S5 + S7 for WIDE embedding nets (W, 2 W, 4 W), W = 64 ... 512: the network-size study of PAPER.md:273-279 (Fig. 7,
// last layer 128 x 256 ... 1024 x 2048), MIX-16.
//
// At these widths the layer products are GEMM-bound (tanh per flop falls as 1 / W), the weights no longer fit beside two
// tiles in one SM, and keeping a tile's activations on chip is impossible (128 rows x 7 W fp16 = 448 KB at W = 256).  So the
// path is the paper's own: one GEMM per layer with the bias / tanh / skip / tanh' work fused into its
// epilogue, activations kept in HBM between the layers (fp16) and reused by the backward pass.  What is B200-specific:
//   * activations live in HBM as ready-made tcgen05 operand images: per 128-row tile and per 8 columns one 2 KB block
//     [128 rows][8 fp16], so a K = 64 slice of the A operand is ONE contiguous 16 KB cp.async.bulk, and an epilogue thread
//     (= row) writes 16 bytes per 8 columns, a warp 512 contiguous bytes;
//   * k_wide_gemm: persistent, warp-specialised, CTA pairs (cluster of 2, tcgen05 cta_group::2: a pair takes two consecutive row
//     tiles of one net against one N tile, each CTA staging its own A tile and half of the B tile): warp 0 streams A and B
//     stages (mbarrier transactions), warp 1 of the leader issues tcgen05.mma 256 x BN x 16 (BN <= 256) into one of two TMEM
//     accumulators (warp 1 of the peer relays "stage landed"), eight epilogue warps drain the other one;
//   * the backward overwrites in place: dz3 over t3, dz2 over t2, (gG_lo + gG_hi) and then dy2 over y2.
// Forward:  k_wide_l1 (t1)  ->  gemm<0> (t2, y2 = (t1,t1) + t2)  ->  gemm<1> (t3)  ->  k_wide_contract (A_i = R^T G / Nm)
// Backward: k_wide_gscale  ->  k_wide_bwd_elem (gG = R^ gA, dz3, dR^ = G gA^T)  ->  gemm<2> (dy2, dz2)  ->  gemm<3> (dy1,
//           dz1, ds^, gradient of the environment row)  ->  k_prod_force_virial (embed_tc2_bwd.cu).
#include <cstdio>
#include <vector>
#include <cuda_fp16.h>
#include "dp_internal.h"
#include "tc_common.cuh"

namespace {

constexpr int WR = 128;                        // rows per tile
constexpr int WKC = 64;                        // K per pipeline stage: 8 chunks of 8 columns
constexpr int WNST = 6;                        // pipeline stages
constexpr int W_A_STAGE = WR * WKC * 2;        // 16 KB
constexpr int W_B_STAGE = 128 * WKC * 2;       // 16 KB: this CTA's half (<= 128 rows) of the B tile (BN <= 256)
constexpr int W_OFF_A = 0;
constexpr int W_OFF_B = WNST * W_A_STAGE;
constexpr int W_OFF_BAR = W_OFF_B + WNST * W_B_STAGE;
constexpr int W_OFF_RED = W_OFF_BAR + 256;     // float [2][2][128]: ds^ partial sums of the two column halves (double buffered)
constexpr int W_TOTAL = W_OFF_RED + 2 * 2 * 128 * 4;
constexpr int W_THREADS = 64 + 256;
static_assert(W_TOTAL + 1024 <= 227 * 1024, "shared memory budget");

__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(tc::smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(tc::smem_u32(bar)) : "memory");
}
// ---- CTA pairs (cluster of 2, tcgen05 cta_group::2): the leader (rank 0) issues M = 256 MMAs over both CTAs' operands
__device__ __forceinline__ void mma_ss2(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t id, bool accumulate) {
    asm volatile("{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\ntcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n}"
                 ::"r"(tmem_d), "l"(da), "l"(db), "r"(id), "r"((uint32_t)accumulate) : "memory");
}
// the MMAs issued so far by this thread arrive on the barrier at this shared-memory offset in BOTH CTAs of the pair
__device__ __forceinline__ void commit_pair(uint64_t *bar) {
    asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;"
                 ::"r"(tc::smem_u32(bar)), "h"((uint16_t)3) : "memory");
}
// arrive on the barrier at this shared-memory offset in the leader CTA, from either CTA (release at CTA scope, the default: a
// .release.cluster compiles to a memory barrier per arrival and made pairs slower than single CTAs)
__device__ __forceinline__ void mbar_arrive_leader(uint64_t *bar) {
    asm volatile("{\n.reg .b32 ra;\nmapa.shared::cluster.u32 ra, %0, 0;\nmbarrier.arrive.shared::cluster.b64 _, [ra];\n}"
                 ::"r"(tc::smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait_cluster(uint64_t *bar, uint32_t parity) {
    asm volatile("{\n.reg .pred p;\nWAITC_%=:\nmbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%0], %1;\n@p bra DONEC_%=;\nbra WAITC_%=;\nDONEC_%=:\n}"
                 ::"r"(tc::smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;\nbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// Pair pw of the tile table: two consecutive tiles of one block (one net).  Returns the block; tile = this CTA's tile, valid =
// false for the second CTA of the last pair of a block with an odd number of tiles (it stages operands and stores nothing).
__device__ __forceinline__ int wide_pair(const int4 *tab, int nblk, int pw, int rank, int &tile, bool &valid) {
    int k = 0, base = 0;
    for (;; ++k) {
        const int np = (tab[k + 1].x - tab[k].x + 1) >> 1;
        if (pw < base + np || k == nblk - 1) break;
        base += np;
    }
    tile = tab[k].x + 2 * (pw - base) + rank;
    valid = tile < tab[k + 1].x;
    return k;
}
__device__ __forceinline__ int wide_pair_count(const int4 *tab, int nblk) {
    int n = 0;
    for (int k = 0; k < nblk; ++k) n += (tab[k + 1].x - tab[k].x + 1) >> 1;
    return n;
}
__device__ __forceinline__ void bulk_g2s(uint32_t sdst, const void *gsrc, uint32_t bytes, uint64_t *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(sdst), "l"(gsrc), "r"(bytes), "r"(tc::smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void unpack8(const uint4 &u, float (&x)[8]) {
    const __half2 *h = reinterpret_cast<const __half2 *>(&u);
#pragma unroll
    for (int q = 0; q < 4; ++q) { const float2 f = __half22float2(h[q]); x[2 * q] = f.x; x[2 * q + 1] = f.y; }
}
__device__ __forceinline__ uint4 pack8(const float (&x)[8]) {
    return make_uint4(tc::pack_h2(x[0], x[1]), tc::pack_h2(x[2], x[3]), tc::pack_h2(x[4], x[5]), tc::pack_h2(x[6], x[7]));
}

// Tile table: entry k = a T + b = {first tile, first row, end row} of the (centre type a, neighbour type b) row block;
// entry T T = {number of tiles}.  Rows of a block are contiguous (sorted atoms of one type are contiguous).
__global__ void k_wide_tiles(long N, int T, int ncell, const int *__restrict__ bin_start, const int *__restrict__ rowstart,
                             int4 *__restrict__ tab) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    int base = 0;
    for (int a = 0; a < T; ++a) {
        const int ts0 = bin_start[a * ncell], ts1 = bin_start[(a + 1) * ncell];
        for (int b = 0; b < T; ++b) {
            const int rs = rowstart[(long)b * (N + 1) + ts0], re = rowstart[(long)b * (N + 1) + ts1];
            tab[a * T + b] = make_int4(base, rs, re, 0);
            base += (re - rs + WR - 1) / WR;
        }
    }
    tab[T * T] = make_int4(base, 0, 0, 0);
}
// the block of a tile; k = the block of an earlier tile of the same walk (tiles are visited in increasing order)
__device__ __forceinline__ int wide_block(const int4 *tab, int nblk, int tile, int k) {
    while (k + 1 < nblk && tile >= tab[k + 1].x) ++k;
    return k;
}

// Layer 1 (K = 1, ALUs): t1 = tanh(s^ w1 + b1) -> T1 image.  Rows past the end of a block are zero.
__global__ void __launch_bounds__(WR)
k_wide_l1(long N, int T, int W, const __grid_constant__ TypeTab tt, const int4 *__restrict__ tab, const float *__restrict__ vec,
          const float4 *__restrict__ rows_rh, uint8_t *__restrict__ T1) {
    const int nblk = T * T, ntiles = tab[nblk].x, r = threadIdx.x;
    int k = 0;
    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        k = wide_block(tab, nblk, tile, k);
        const int4 e = tab[k];
        const long rbase = N * (long)tt.off[k % T];
        const int row = e.y + (tile - e.x) * WR + r;
        const bool ok = row < e.z;
        const float s = ok ? __ldg(&rows_rh[rbase + row]).x : 0.f;
        const float *w1 = vec + (size_t)k * 8 * W, *b1 = w1 + W;
        uint4 *dst = reinterpret_cast<uint4 *>(T1 + (size_t)tile * (W / 8) * 2048) + r;
        for (int c = 0; c < W / 8; ++c) {
            float y[8];
#pragma unroll
            for (int q = 0; q < 8; ++q) y[q] = ok ? tc::tanh_approx(fmaf(s, __ldg(w1 + 8 * c + q), __ldg(b1 + 8 * c + q))) : 0.f;
            dst[c * WR] = pack8(y);
        }
    }
}

struct WideArgs {
    long N;
    int T, W, Nm;
    int K, NTOT, BN;                      // product shape: [rows x K] . [K x NTOT], N tile BN
    int G;                                // CTAs that share a row tile, each taking every G-th N tile (the A tile then comes
                                          // from HBM once and from L2 for the others: the working set is grid / G tiles)
    const int4 *tab;
    const uint8_t *Aimg;                  // A operand images: K / 8 chunks per tile
    const __half *Bimg;                   // B image of this product inside the first net's block, [NTOT / BN][K / 8][BN][8]
    long b_net_stride;                    // elements per net
    const float *vec;                     // [T T][8 W]: w1, b1, b2, b3
    uint8_t *T1, *Y2, *T2, *T3;           // activation images (W, 2 W, 2 W, 4 W columns)
    const int2 *rows_id;
    float4 *rows_g;
    const float *gscale;
    const double *stdv;
    TypeTab tt;
};

// MODE 0: layer 2 forward   A = t1 (K = W),    N = 2 W:  t2 = tanh(acc + b2) -> T2;  y2 = (t1,t1) + t2 -> Y2
// MODE 1: layer 3 forward   A = y2 (K = 2 W),  N = 4 W:  t3 = tanh(acc + b3) -> T3   (G = (y2,y2) + t3 is formed by its readers)
// MODE 2: layer 3 backward  A = dz3 (K = 4 W), N = 2 W:  dy2 = acc + (gG[f] + gG[f + 2 W], in Y2) -> Y2;  dz2 = dy2 (1 - t2^2) -> T2
// MODE 3: layer 2 backward  A = dz2 (K = 2 W), N = W:    dy1 = acc + dy2[e] + dy2[e + W];  dz1 = dy1 (1 - t1^2);  ds^ = dz1 . w1;
//                           rows_g = dE/dR~ of the row (dR^ from k_wide_bwd_elem + ds^ on component 0, unscaled, / std)
template <int MODE>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(W_THREADS, 1) k_wide_gemm(const __grid_constant__ WideArgs p) {
    extern __shared__ __align__(1024) uint8_t smem[];
    __shared__ uint32_t tmem_base_s;
    const int tid = threadIdx.x, lane = tid & 31;
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem + W_OFF_BAR);
    uint64_t *full = bars, *empty = bars + WNST, *pfull = bars + 2 * WNST, *acc_full = bars + 3 * WNST, *acc_empty = acc_full + 2;
    uint32_t rank;
    asm("mov.u32 %0, %%cluster_ctarank;" : "=r"(rank));
    if (tid == 0) {
        for (int k = 0; k < WNST; ++k) { tc::mbar_init(&full[k], 1); tc::mbar_init(&empty[k], 1); tc::mbar_init(&pfull[k], 1); }
        for (int k = 0; k < 2; ++k) { tc::mbar_init(&acc_full[k], 1); tc::mbar_init(&acc_empty[k], 16); }
        asm volatile("fence.mbarrier_init.release.cluster;");
    }
    if (warp == 0) {       // the same warp of both CTAs, the same shared-memory word
        asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tc::smem_u32(&tmem_base_s)), "n"(512));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;");
    }
    tc::fence_before();
    cluster_sync_all();
    tc::fence_after();
    const uint32_t tmem = __shfl_sync(0xffffffffu, tmem_base_s, 0);
    const uint32_t sbase = tc::smem_u32(smem);
    const int nblk = p.T * p.T;
    const int W = p.W, BN = p.BN, HB = BN / 2, NT = p.NTOT / BN, NKC = p.K / WKC;
    const uint32_t b_half_bytes = (uint32_t)HB * WKC * 2;
    // pairs of CTAs walk pairs of tiles; G pairs share one pair of tiles, each taking every G-th N tile
    const int G = p.G, npairs = wide_pair_count(p.tab, nblk);
    const int pw0 = (blockIdx.x >> 1) / G, pwstep = (gridDim.x >> 1) / G, nt0 = (blockIdx.x >> 1) % G;

    if (warp == 0) {
        // ---------------------------------------------------------------- loader: one A and one B (half) bulk copy per stage
        if (lane == 0) {
            uint32_t step = 0;
            for (int pw = pw0; pw < npairs; pw += pwstep) {
                int tile;
                bool valid;
                const int k = wide_pair(p.tab, nblk, pw, (int)rank, tile, valid);
                const __half *Bw = p.Bimg + (size_t)k * p.b_net_stride;
                const uint8_t *At = p.Aimg + (size_t)(valid ? tile : tile - 1) * (p.K / 8) * 2048;      // (no tile of its own: any tile will do)
                for (int nt = nt0; nt < NT; nt += G)
                    for (int kc = 0; kc < NKC; ++kc, ++step) {
                        const int st = step % WNST;
                        tc::mbar_wait(&empty[st], ((step / WNST) & 1) ^ 1);
                        mbar_expect_tx(&full[st], W_A_STAGE + b_half_bytes);
                        bulk_g2s(sbase + W_OFF_A + st * W_A_STAGE, At + (size_t)kc * W_A_STAGE, W_A_STAGE, &full[st]);
                        bulk_g2s(sbase + W_OFF_B + st * W_B_STAGE, Bw + (((size_t)nt * NKC + kc) * 2 + rank) * (WKC * HB), b_half_bytes, &full[st]);
                    }
            }
        }
    } else if (warp == 1) {
        if (rank == 0) {
            // ------------------------------------------------------------ MMA issuer (leader): M = 256 over both CTAs
            const uint32_t idesc = tc::idesc(256, BN, false, false);
            uint32_t step = 0, accn = 0;
            for (int pw = pw0; pw < npairs; pw += pwstep)
                for (int nt = nt0; nt < NT; nt += G, ++accn) {
                    const int buf = accn & 1;
                    mbar_wait_cluster(&acc_empty[buf], ((accn >> 1) & 1) ^ 1);
                    tc::fence_after();
                    for (int kc = 0; kc < NKC; ++kc, ++step) {
                        const int st = step % WNST;
                        tc::mbar_wait(&full[st], (step / WNST) & 1);
                        mbar_wait_cluster(&pfull[st], (step / WNST) & 1);
                        tc::fence_after();
                        const uint64_t da = tc::desc(sbase + W_OFF_A + st * W_A_STAGE, 2048, 128);
                        const uint64_t db = tc::desc(sbase + W_OFF_B + st * W_B_STAGE, HB * 16, 128);
                        if (tc::elect_one()) {
#pragma unroll
                            for (int ks = 0; ks < WKC / 16; ++ks)
                                mma_ss2(tmem + buf * 256, tc::desc_at(da, ks * 2 * 2048), tc::desc_at(db, ks * 2 * (HB * 16)), idesc, (kc | ks) != 0);
                            commit_pair(&empty[st]);
                        }
                        __syncwarp();
                    }
                    if (tc::elect_one()) commit_pair(&acc_full[buf]);
                    __syncwarp();
                }
        } else {
            // ------------------------------------------------------------ relay (peer): "my stage has landed" to the leader
            uint32_t step = 0;
            for (int pw = pw0; pw < npairs; pw += pwstep)
                for (int nt = nt0; nt < NT; nt += G)
                    for (int kc = 0; kc < NKC; ++kc, ++step) {
                        const int st = step % WNST;
                        tc::mbar_wait(&full[st], (step / WNST) & 1);
                        if (lane == 0) mbar_arrive_leader(&pfull[st]);
                        __syncwarp();
                    }
        }
    } else {
        // ---------------------------------------------------------------- epilogue: thread = (row, every other 16 columns)
        const int q4 = warp & 3, r = q4 * 32 + lane, hc = ((warp - 2) >> 2) & 1;
        const uint32_t tm_lane = tmem + ((uint32_t)(q4 * 32) << 16);
        float *red = reinterpret_cast<float *>(smem + W_OFF_RED);
        uint32_t accn = 0, it = 0;
        for (int pw = pw0; pw < npairs; pw += pwstep, ++it) {
            int tile;
            bool valid;
            const int k = wide_pair(p.tab, nblk, pw, (int)rank, tile, valid);
            if (!valid) {          // no tile of its own: keep the accumulator hand-shake of the pair going, store nothing
                for (int nt = nt0; nt < NT; nt += G, ++accn) {
                    const int buf = accn & 1;
                    tc::mbar_wait(&acc_full[buf], (accn >> 1) & 1);
                    tc::fence_before();
                    __syncwarp();
                    if (lane == 0) mbar_arrive_leader(&acc_empty[buf]);
                }
                continue;
            }
            const float *vec = p.vec + (size_t)k * 8 * W;
            // this row's 16-byte slot of chunk 0 of each image of the tile
            uint8_t *t1r = p.T1 + (size_t)tile * (W / 8) * 2048 + r * 16;
            uint8_t *y2r = p.Y2 + (size_t)tile * (2 * W / 8) * 2048 + r * 16;
            uint8_t *t2r = p.T2 + (size_t)tile * (2 * W / 8) * 2048 + r * 16;
            uint8_t *t3r = p.T3 + (size_t)tile * (4 * W / 8) * 2048 + r * 16;
            (void)t1r; (void)y2r; (void)t2r; (void)t3r;
            float ds = 0.f;
            // global operands of a group of 16 columns (two chunks), loaded one group ahead of their use
            struct Pre { uint4 a[2], b[2], c[2]; };
            const int ngrp = BN / 32;                       // groups of this thread per N tile (2, 4 or 8)
            auto fetch = [&](int nt, int g, Pre &P) {
                const int ch0 = (nt * BN + 16 * hc + 32 * g) / 8;
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const size_t ch = ch0 + h;
                    if (MODE == 0) P.a[h] = *reinterpret_cast<const uint4 *>(t1r + (ch % (W / 8)) * 2048);
                    if (MODE == 2) {
                        P.a[h] = *reinterpret_cast<const uint4 *>(y2r + ch * 2048);
                        P.b[h] = *reinterpret_cast<const uint4 *>(t2r + ch * 2048);
                    }
                    if (MODE == 3) {
                        P.a[h] = *reinterpret_cast<const uint4 *>(y2r + ch * 2048);
                        P.b[h] = *reinterpret_cast<const uint4 *>(y2r + (ch + W / 8) * 2048);
                        P.c[h] = *reinterpret_cast<const uint4 *>(t1r + ch * 2048);
                    }
                }
            };
            auto process = [&](int nt, int g, int buf, const Pre &P) {
                const int c0 = 16 * hc + 32 * g, n = nt * BN + c0;      // n: first of these 16 output columns
                uint32_t v[16];
                tc::ld16(tm_lane + buf * 256 + c0, v);
                tc::wait_ld();
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const size_t ch = n / 8 + h;
                    float x[8];
                    if (MODE == 0) {
                        const float4 b0 = __ldg(reinterpret_cast<const float4 *>(vec + 2 * W + n + 8 * h)), b1 = __ldg(reinterpret_cast<const float4 *>(vec + 2 * W + n + 8 * h + 4));
                        const float bb[8] = {b0.x, b0.y, b0.z, b0.w, b1.x, b1.y, b1.z, b1.w};
                        float t1[8];
                        unpack8(P.a[h], t1);
#pragma unroll
                        for (int q = 0; q < 8; ++q) x[q] = tc::tanh_approx(__uint_as_float(v[8 * h + q]) + bb[q]);
                        *reinterpret_cast<uint4 *>(t2r + ch * 2048) = pack8(x);
#pragma unroll
                        for (int q = 0; q < 8; ++q) x[q] += t1[q];
                        *reinterpret_cast<uint4 *>(y2r + ch * 2048) = pack8(x);
                    } else if (MODE == 1) {
                        const float4 b0 = __ldg(reinterpret_cast<const float4 *>(vec + 4 * W + n + 8 * h)), b1 = __ldg(reinterpret_cast<const float4 *>(vec + 4 * W + n + 8 * h + 4));
                        const float bb[8] = {b0.x, b0.y, b0.z, b0.w, b1.x, b1.y, b1.z, b1.w};
#pragma unroll
                        for (int q = 0; q < 8; ++q) x[q] = tc::tanh_approx(__uint_as_float(v[8 * h + q]) + bb[q]);
                        *reinterpret_cast<uint4 *>(t3r + ch * 2048) = pack8(x);
                    } else if (MODE == 2) {
                        float gs[8], t2[8];
                        unpack8(P.a[h], gs);
                        unpack8(P.b[h], t2);
#pragma unroll
                        for (int q = 0; q < 8; ++q) x[q] = __uint_as_float(v[8 * h + q]) + gs[q];
                        *reinterpret_cast<uint4 *>(y2r + ch * 2048) = pack8(x);
#pragma unroll
                        for (int q = 0; q < 8; ++q) x[q] *= fmaf(-t2[q], t2[q], 1.f);
                        *reinterpret_cast<uint4 *>(t2r + ch * 2048) = pack8(x);
                    } else {
                        float da[8], db[8], t1[8];
                        unpack8(P.a[h], da);
                        unpack8(P.b[h], db);
                        unpack8(P.c[h], t1);
                        const float4 w0 = __ldg(reinterpret_cast<const float4 *>(vec + n + 8 * h)), w1 = __ldg(reinterpret_cast<const float4 *>(vec + n + 8 * h + 4));
                        const float ww[8] = {w0.x, w0.y, w0.z, w0.w, w1.x, w1.y, w1.z, w1.w};
#pragma unroll
                        for (int q = 0; q < 8; ++q) {
                            const float dy1 = __uint_as_float(v[8 * h + q]) + da[q] + db[q];
                            ds = fmaf(dy1 * fmaf(-t1[q], t1[q], 1.f), ww[q], ds);
                        }
                    }
                }
            };
            Pre P0, P1;
            fetch(nt0, 0, P0);
            for (int nt = nt0; nt < NT; nt += G, ++accn) {
                const int buf = accn & 1;
                tc::mbar_wait(&acc_full[buf], (accn >> 1) & 1);
                tc::fence_after();
                for (int g = 0; g < ngrp; g += 2) {
                    fetch(nt, g + 1, P1);
                    process(nt, g, buf, P0);
                    if (g + 2 < ngrp) fetch(nt, g + 2, P0);
                    else if (nt + G < NT) fetch(nt + G, 0, P0);
                    process(nt, g + 1, buf, P1);
                }
                tc::fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive_leader(&acc_empty[buf]);
            }
            if (MODE == 3) {
                float *rd = red + (it & 1) * 256;
                rd[hc * 128 + r] = ds;
                tc::bar_sync(1, 256);
                const int4 e = p.tab[k];
                const int row = e.y + (tile - e.x) * WR + r;
                if (hc == 0 && row < e.z) {
                    const long rbase = p.N * (long)p.tt.off[k % p.T];
                    const int2 id = __ldg(&p.rows_id[rbase + row]);
                    if (id.y >= 0) {
                        const int a = k / p.T;
                        const float4 g = p.rows_g[rbase + row];          // gscale * dR^ (k_wide_bwd_elem)
                        const float osc = 1.0f / ((float)p.Nm * __ldg(&p.gscale[id.x]));
                        const float dsum = rd[r] + rd[128 + r];
                        p.rows_g[rbase + row] = make_float4((g.x + dsum) * osc / (float)p.stdv[4 * a], g.y * osc / (float)p.stdv[4 * a + 1],
                                                            g.z * osc / (float)p.stdv[4 * a + 2], g.w * osc / (float)p.stdv[4 * a + 3]);
                    }
                }
            }
        }
    }
    tc::fence_before();
    cluster_sync_all();
    tc::fence_after();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(512));
}

// S5: A_i[c][m] = (1 / Nm) sum_rows w R^[row][c] G[row][m],  G = (y2, y2) + t3.
// One CTA per atom, and per batch of up to 192 of its rows: S3 = R^T t3 [4][4 W] and S2 = R^T y2 [4][2 W] are accumulated
// separately (A_i[c][m] = S3[c][m] + S2[c][m mod 2 W]), so every activation is read from HBM once.  A group of 8 columns is
// one product [8 x rows] . [rows x 8] on the tensor cores (mma.sync m16n8k16, fp32 accumulate): M = the four components of the
// weighted row as fp16 hi parts (rows 0-3) and lo parts (rows 4-7), K = rows, N = the 8 columns; the B fragments come straight
// from the stored [row][8 fp16] blocks through ldmatrix.trans.  Every warp owns every 8th column group and stages it itself:
// bulk copies of the atom's rows of that group (contiguous inside a tile), three groups ahead, completion on its own mbarriers.
// With scalar fp32 FMAs (32 per 16 bytes loaded) the kernel was issue-bound at 4.3 TB/s.  No atomics, fixed summation order.
constexpr int WC_BATCH = 192;                   // rows per pass: 12 k-steps of 16
constexpr int WC_DEPTH = 3;                     // column groups in flight per warp
constexpr int WC_SLOT = WC_BATCH * 16;          // bytes of one staged column group
__global__ void __launch_bounds__(256)
k_wide_contract(long N, int T, int ncell, int W, int P, int Nm, const __grid_constant__ TypeTab tt, const int4 *__restrict__ tab,
                const int *__restrict__ bin_start, const int *__restrict__ rowstart, const float4 *__restrict__ rows_rh,
                const int2 *__restrict__ rows_id, const uint8_t *__restrict__ Y2, const uint8_t *__restrict__ T3,
                float *__restrict__ Aout) {
    extern __shared__ __align__(128) uint8_t csm[];
    __shared__ uint64_t cbar[8][WC_DEPTH];
    uint8_t *slots = csm;                                                    // [8 warps][WC_DEPTH][WC_SLOT]
    float4 *srw = reinterpret_cast<float4 *>(csm + 8 * WC_DEPTH * WC_SLOT);   // [WC_BATCH] weighted rows
    // P CTAs per atom (W = 512: two, so that two CTAs fit an SM): part h takes the y2 chunks [h ych / P, (h + 1) ych / P) and the
    // t3 chunks of the same columns f and of f + 2 W
    const int nch = 4 * W / 8, ych = 2 * W / 8, ychp = ych / P, WP = 8 * ychp;      // WP: y2 columns of one part
    float *sA = reinterpret_cast<float *>(srw + WC_BATCH);                   // S3 [2 (f, f + 2 W)][4][WP]
    float *sA2 = sA + 8 * WP;                                                // S2 [4][WP]
    const long i = blockIdx.x / P;
    const int part = blockIdx.x % P;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int g8 = lane >> 2, t4 = lane & 3;
    int a = 0;
    for (int t = 1; t < T; ++t) a += i >= bin_start[t * ncell];
    for (int k = tid; k < 12 * WP; k += 256) sA[k] = 0.f;
    // staged rows beyond a batch's count keep older (finite) activations: they meet zero rows of R.  Start from zeros.
    for (int k = tid; k < 8 * WC_DEPTH * WC_SLOT / 16; k += 256) reinterpret_cast<uint4 *>(slots)[k] = make_uint4(0u, 0u, 0u, 0u);
    if (lane == 0)
        for (int d = 0; d < WC_DEPTH; ++d) tc::mbar_init(&cbar[wid][d], 1);
    asm volatile("fence.mbarrier_init.release.cluster;");
    const int ngroups = 3 * ychp;               // group q: q < 2 ychp: t3 chunk (lower then upper columns), else y2 chunk
    uint32_t issued = 0, consumed = 0;          // per warp: column groups handed to / taken from the staging ring (all batches)
    uint8_t *myslots = slots + wid * WC_DEPTH * WC_SLOT;
    for (int b = 0; b < T; ++b) {
        const int4 e = tab[a * T + b];
        const long rbase = N * (long)tt.off[b];
        const int r0 = rowstart[(long)b * (N + 1) + i], r1 = rowstart[(long)b * (N + 1) + i + 1];
        for (int rb = r0; rb < r1; rb += WC_BATCH) {
            const int nb = min(WC_BATCH, r1 - rb), nks = (nb + 15) / 16;
            __syncthreads();
            for (int j = tid; j < WC_BATCH; j += 256) {
                float4 rh = make_float4(0.f, 0.f, 0.f, 0.f);
                if (j < nb) {
                    rh = __ldg(&rows_rh[rbase + rb + j]);
                    const int2 id = __ldg(&rows_id[rbase + rb + j]);
                    if (id.y < 0) { const float w = (float)(-id.y); rh.x *= w; rh.y *= w; rh.z *= w; rh.w *= w; }
                }
                srw[j] = rh;
            }
            __syncthreads();
            // A fragments of all k-steps: lane (g8, t4) holds rows 2 t4, 2 t4 + 1 (a0) and 2 t4 + 8, 2 t4 + 9 (a2) of the step, M row g8:
            // component g8 & 3, hi part for g8 < 4, lo part otherwise
            uint32_t afr[WC_BATCH / 16][2];
            {
                const float *sr = reinterpret_cast<const float *>(srw);
                const int c = g8 & 3;
#pragma unroll
                for (int ks = 0; ks < WC_BATCH / 16; ++ks) {
                    const int rr = 16 * ks + 2 * t4;
                    uint32_t h0, l0, h1, l1;
                    tc::split_h2(sr[rr * 4 + c], sr[(rr + 1) * 4 + c], h0, l0);
                    tc::split_h2(sr[(rr + 8) * 4 + c], sr[(rr + 9) * 4 + c], h1, l1);
                    afr[ks][0] = g8 < 4 ? h0 : l0;
                    afr[ks][1] = g8 < 4 ? h1 : l1;
                }
            }
            // this warp's column groups of the batch: vc = wid, wid + 8, ...
            const int rel0 = rb - e.y;
            auto issue = [&](int vc) {
                if (lane == 0) {
                    const bool isy = vc >= 2 * ychp;
                    const uint8_t *img = isy ? Y2 : T3;
                    const int cpt = isy ? ych : nch;
                    const int ch = isy ? part * ychp + (vc - 2 * ychp) : (vc < ychp ? part * ychp + vc : ych + part * ychp + (vc - ychp));
                    uint64_t *bar = &cbar[wid][issued % WC_DEPTH];
                    uint8_t *dst = myslots + (issued % WC_DEPTH) * WC_SLOT;
                    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                    mbar_expect_tx(bar, (uint32_t)nb * 16u);
                    for (int done = 0; done < nb;) {          // the rows are contiguous inside a tile: one copy per tile touched
                        const int rel = rel0 + done, tl = rel / WR, rr = rel % WR;
                        const int cnt = min(nb - done, WR - rr);
                        bulk_g2s(tc::smem_u32(dst + done * 16), img + (((size_t)e.x + tl) * cpt + ch) * 2048 + rr * 16, (uint32_t)cnt * 16u, bar);
                        done += cnt;
                    }
                }
                ++issued;
            };
            const int nmine = (ngroups - wid + 7) / 8;
            __syncwarp();
            for (int q = 0; q < WC_DEPTH && q < nmine; ++q) issue(wid + 8 * q);
            for (int q = 0; q < nmine; ++q) {
                const int vc = wid + 8 * q;
                const uint32_t sl = consumed % WC_DEPTH;
                tc::mbar_wait(&cbar[wid][sl], (consumed / WC_DEPTH) & 1);
                ++consumed;
                const uint32_t sbase = tc::smem_u32(myslots + sl * WC_SLOT) + lane * 16;
                float c0 = 0.f, c1 = 0.f, c2 = 0.f, c3 = 0.f;
#pragma unroll
                for (int kp = 0; kp < WC_BATCH / 32; ++kp) {
                    if (2 * kp < nks) {
                        uint32_t b0, b1, b2, b3;
                        asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0, %1, %2, %3}, [%4];"
                                     : "=r"(b0), "=r"(b1), "=r"(b2), "=r"(b3) : "r"(sbase + kp * 512));
                        asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, {%8, %9}, {%0, %1, %2, %3};"
                                     : "+f"(c0), "+f"(c1), "+f"(c2), "+f"(c3) : "r"(afr[2 * kp][0]), "r"(0u), "r"(afr[2 * kp][1]), "r"(0u), "r"(b0), "r"(b1));
                        if (2 * kp + 1 < nks)
                            asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, {%8, %9}, {%0, %1, %2, %3};"
                                         : "+f"(c0), "+f"(c1), "+f"(c2), "+f"(c3) : "r"(afr[2 * kp + 1][0]), "r"(0u), "r"(afr[2 * kp + 1][1]), "r"(0u), "r"(b2), "r"(b3));
                    }
                }
                (void)c2; (void)c3;
                __syncwarp();                                   // every lane has read the slot: it may be refilled
                if (q + WC_DEPTH < nmine) issue(vc + 8 * WC_DEPTH);
                // hi rows (g8 < 4) + lo rows (g8 >= 4): lanes 16 apart
                c0 += __shfl_xor_sync(0xffffffffu, c0, 16);
                c1 += __shfl_xor_sync(0xffffffffu, c1, 16);
                if (g8 < 4) {
                    // vc < ychp: S3 lower columns, < 2 ychp: S3 upper columns, else S2; each [4][WP]
                    const int sec = vc >= 2 * ychp ? 2 : (vc >= ychp ? 1 : 0);
                    float *dst = sA + sec * 4 * WP + g8 * WP + 8 * (vc - sec * ychp);
                    dst[2 * t4] += c0;
                    dst[2 * t4 + 1] += c1;
                }
            }
        }
    }
    __syncthreads();
    const float inv_nm = 1.0f / (float)Nm;
    for (int k = tid; k < 8 * WP; k += 256) {           // (upper / lower, component, column of the part)
        const int u = k / (4 * WP), c = (k / WP) & 3, f = k % WP;
        Aout[i * 16L * W + c * 4 * W + u * 2 * W + part * WP + f] = (sA[k] + sA2[c * WP + f]) * inv_nm;
    }
}

// per-atom power-of-two scale of the gradient images: max |gA_i| in [0.5, 1) (fp16 range; undone in gemm<3>)
__global__ void __launch_bounds__(256) k_wide_gscale(long N, int n, const float *__restrict__ gA, float *__restrict__ gscale) {
    const int lane = threadIdx.x & 31;
    const long i = blockIdx.x * 8L + (threadIdx.x >> 5);
    if (i >= N) return;
    const float4 *g = reinterpret_cast<const float4 *>(gA + i * (long)n);
    float mx = 0.f;
    for (int k = lane; k < n / 4; k += 32) {
        const float4 v = __ldg(g + k);
        mx = fmaxf(fmaxf(mx, fmaxf(fabsf(v.x), fabsf(v.y))), fmaxf(fabsf(v.z), fabsf(v.w)));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    int ex = 0;
    if (mx > 0.f) frexpf(mx, &ex);
    if (lane == 0) gscale[i] = ldexpf(1.f, -ex);
}

// Head of the backward pass, thread = row, per pair of column groups (f, f + 2 W):
//   gG[m] = sc sum_c R^[c] gA[c][m]          (gradient of E with respect to G, scaled by the atom's sc, without 1 / Nm)
//   dz3   = gG (1 - t3^2)                     -> over t3 (A operand of gemm<2>)
//   gG[f] + gG[f + 2 W]                       -> over y2 (the skip connection's share of dy2, added in the epilogue of gemm<2>)
//   dR^[c] = sc sum_m G[m] gA[c][m]           -> rows_g (finished by gemm<3>)
// Padded-row representatives carry no gradient (R~ = 0 there is a constant): skipped.
// The three 2 KB activation chunks of a step (per column half) are staged in shared memory by a producer warp with bulk copies, four
// steps (48 KB per CTA, 96 KB per SM) ahead of the arithmetic: with per-thread loads one step ahead the kernel reached 4.5 TB/s.
constexpr int BE_STAGES = 4;
constexpr int BE_STAGE_BYTES = 2 * 3 * 2048;          // [column half][y2, t3 lower, t3 upper][128 rows x 16 B]
constexpr int BE_THREADS = 2 * WR + 32;               // 256 consumers (row, column half) + the producer warp
__global__ void __launch_bounds__(BE_THREADS, 2)
k_wide_bwd_elem(long N, int T, int W, const __grid_constant__ TypeTab tt, const int4 *__restrict__ tab,
                const float4 *__restrict__ rows_rh, const int2 *__restrict__ rows_id, const float *__restrict__ gA,
                const float *__restrict__ gscale, uint8_t *__restrict__ Y2, uint8_t *__restrict__ T3, float4 *__restrict__ rows_g) {
    extern __shared__ __align__(128) uint8_t bsm[];
    __shared__ float4 sdr[WR];
    __shared__ uint64_t full[BE_STAGES], empty[BE_STAGES];
    const int nblk = T * T, ntiles = tab[nblk].x;
    const int ych = 2 * W / 8, M2 = 4 * W, nstep = ych / 2;
    if (threadIdx.x == 0) {
        for (int k = 0; k < BE_STAGES; ++k) { tc::mbar_init(&full[k], 1); tc::mbar_init(&empty[k], 8); }
        asm volatile("fence.mbarrier_init.release.cluster;");
    }
    __syncthreads();
    if (threadIdx.x >= 2 * WR) {
        // ---------------------------------------------------------------- producer warp
        if (threadIdx.x == 2 * WR) {
            uint32_t step = 0;
            for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
                const uint8_t *y2t = Y2 + (size_t)tile * ych * 2048, *t3t = T3 + (size_t)tile * (2 * ych) * 2048;
                for (int sidx = 0; sidx < nstep; ++sidx, ++step) {
                    const int st = step % BE_STAGES;
                    tc::mbar_wait(&empty[st], ((step / BE_STAGES) & 1) ^ 1);
                    mbar_expect_tx(&full[st], BE_STAGE_BYTES);
                    const uint32_t dst = tc::smem_u32(bsm + st * BE_STAGE_BYTES);
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        const size_t f = (size_t)sidx + h * nstep;
                        bulk_g2s(dst + h * 6144, y2t + f * 2048, 2048, &full[st]);
                        bulk_g2s(dst + h * 6144 + 2048, t3t + f * 2048, 2048, &full[st]);
                        bulk_g2s(dst + h * 6144 + 4096, t3t + (f + ych) * 2048, 2048, &full[st]);
                    }
                }
            }
        }
        return;
    }
    // -------------------------------------------------------------------- consumers: thread = (row, column half)
    const int r = threadIdx.x & (WR - 1), hf = threadIdx.x >> 7, lane = threadIdx.x & 31;
    uint32_t step = 0;
    int k = 0;
    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        k = wide_block(tab, nblk, tile, k);
        const int4 e = tab[k];
        const long rbase = N * (long)tt.off[k % T];
        const int row = e.y + (tile - e.x) * WR + r;
        int2 id = make_int2(-1, -1);
        if (row < e.z) id = __ldg(&rows_id[rbase + row]);
        const bool real = id.y >= 0;
        float dR[4] = {0.f, 0.f, 0.f, 0.f};
        float sc = 0.f;
        float R[4] = {0.f, 0.f, 0.f, 0.f};
        const float *g = gA;
        if (real) {
            const float4 rh = __ldg(&rows_rh[rbase + row]);
            sc = __ldg(&gscale[id.x]);
            R[0] = rh.x * sc; R[1] = rh.y * sc; R[2] = rh.z * sc; R[3] = rh.w * sc;
            g = gA + (long)id.x * 4 * M2;
        }
        uint8_t *y2r = Y2 + (size_t)tile * ych * 2048 + r * 16;
        uint8_t *t3r = T3 + (size_t)tile * (2 * ych) * 2048 + r * 16;
        for (int sidx = 0; sidx < nstep; ++sidx, ++step) {
            const int st = step % BE_STAGES;
            const int f = sidx + hf * nstep;
            tc::mbar_wait(&full[st], (step / BE_STAGES) & 1);
            if (real) {
                const uint8_t *src = bsm + st * BE_STAGE_BYTES + hf * 6144 + r * 16;
                float y2[8], ta[8], tb[8], oa[8], ob[8], os[8];
                unpack8(*reinterpret_cast<const uint4 *>(src), y2);
                unpack8(*reinterpret_cast<const uint4 *>(src + 2048), ta);
                unpack8(*reinterpret_cast<const uint4 *>(src + 4096), tb);
#pragma unroll
                for (int q = 0; q < 8; ++q) { oa[q] = 0.f; ob[q] = 0.f; }
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    const float4 a0 = __ldg(reinterpret_cast<const float4 *>(g + c * M2 + 8 * f)), a1 = __ldg(reinterpret_cast<const float4 *>(g + c * M2 + 8 * f + 4));
                    const float4 b0 = __ldg(reinterpret_cast<const float4 *>(g + c * M2 + 2 * W + 8 * f)), b1 = __ldg(reinterpret_cast<const float4 *>(g + c * M2 + 2 * W + 8 * f + 4));
                    const float ga[8] = {a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w};
                    const float gb[8] = {b0.x, b0.y, b0.z, b0.w, b1.x, b1.y, b1.z, b1.w};
                    float acc = 0.f;
#pragma unroll
                    for (int q = 0; q < 8; ++q) {
                        oa[q] = fmaf(R[c], ga[q], oa[q]);
                        ob[q] = fmaf(R[c], gb[q], ob[q]);
                        acc = fmaf(ta[q] + y2[q], ga[q], acc);
                        acc = fmaf(tb[q] + y2[q], gb[q], acc);
                    }
                    dR[c] += acc;
                }
#pragma unroll
                for (int q = 0; q < 8; ++q) {
                    os[q] = oa[q] + ob[q];
                    oa[q] *= fmaf(-ta[q], ta[q], 1.f);
                    ob[q] *= fmaf(-tb[q], tb[q], 1.f);
                }
                *reinterpret_cast<uint4 *>(y2r + (size_t)f * 2048) = pack8(os);
                *reinterpret_cast<uint4 *>(t3r + (size_t)f * 2048) = pack8(oa);
                *reinterpret_cast<uint4 *>(t3r + (size_t)(f + ych) * 2048) = pack8(ob);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[st]);
        }
        if (hf == 1) sdr[r] = make_float4(dR[0], dR[1], dR[2], dR[3]);
        tc::bar_sync(1, 2 * WR);
        if (hf == 0 && real) {
            const float4 o = sdr[r];
            rows_g[rbase + row] = make_float4((dR[0] + o.x) * sc, (dR[1] + o.y) * sc, (dR[2] + o.z) * sc, (dR[3] + o.w) * sc);
        }
        tc::bar_sync(1, 2 * WR);
    }
}

}  // namespace

// ---------------------------------------------------------------------------------------------------------------------
// Host side.  Weight images of one net, in this order: W2 (K = W, N = 2 W), W3 (K = 2 W, N = 4 W), W3^T (K = 4 W, N = 2 W),
// W2^T (K = 2 W, N = W); each [N / BN][K / 8][BN][8] fp16 with BN = min(N, 256): a (N tile, K = 64) stage is contiguous.
static int wide_bn(int n) { return n < 256 ? n : 256; }
static size_t wide_img_off(int W, int g) {
    const size_t w2 = (size_t)W * W;
    const size_t off[5] = {0, 2 * w2, 10 * w2, 18 * w2, 20 * w2};
    return off[g];
}
size_t wide_net_img_elems(int W) { return wide_img_off(W, 4); }

// B image of one product: per N tile (BN columns), per K = 64 stage and per half of the tile's columns (one half per CTA of a
// pair) the block [8 chunks][BN / 2][8 fp16]: one contiguous bulk copy per stage and CTA
static void wide_image(const double *Wt, int ldw, bool transpose, int K, int Nn, __half *out) {
    const int BN = wide_bn(Nn), HB = BN / 2, nkc = K / WKC;
    for (int nn = 0; nn < Nn; ++nn)
        for (int k = 0; k < K; ++k) {
            const double v = transpose ? Wt[(size_t)nn * ldw + k] : Wt[(size_t)k * ldw + nn];
            const int nt = nn / BN, n = nn % BN, kc = k / WKC, k8 = (k % WKC) / 8, kk = k % 8;
            out[((((size_t)nt * nkc + kc) * 2 + n / HB) * 8 + k8) * ((size_t)HB * 8) + (size_t)(n % HB) * 8 + kk] = __float2half_rn((float)v);
        }
}

// net: w1[W], b1[W], W2[W][2 W], b2[2 W], W3[2 W][4 W], b3[4 W] (dp.h weight order); vec: w1, b1, b2, b3
void wide_build_net(int W, const double *net, float *vec, __half *img) {
    const double *w1 = net, *b1 = w1 + W, *W2 = b1 + W, *b2 = W2 + (size_t)W * 2 * W, *W3 = b2 + 2 * W, *b3 = W3 + (size_t)2 * W * 4 * W;
    for (int e = 0; e < W; ++e) { vec[e] = (float)w1[e]; vec[W + e] = (float)b1[e]; }
    for (int f = 0; f < 2 * W; ++f) vec[2 * W + f] = (float)b2[f];
    for (int m = 0; m < 4 * W; ++m) vec[4 * W + m] = (float)b3[m];
    wide_image(W2, 2 * W, false, W, 2 * W, img + wide_img_off(W, 0));
    wide_image(W3, 4 * W, false, 2 * W, 4 * W, img + wide_img_off(W, 1));
    wide_image(W3, 4 * W, true, 4 * W, 2 * W, img + wide_img_off(W, 2));      // B[k = m][n = f] = W3[f][m]
    wide_image(W2, 2 * W, true, 2 * W, W, img + wide_img_off(W, 3));          // B[k = f][n = e] = W2[e][f]
}

// capacity of the tile table: every (type, type) block may end in a partial tile
long wide_tiles_cap(const dp_model *m, long N) {
    long t = (long)m->T * m->T + 1;
    for (int b = 0; b < m->T; ++b) t += (N * (long)m->sel[b] + WR - 1) / WR;
    return t;
}

static WideArgs wide_args(const dp_model *m, long N, char *ws, const WsLayout &L) {
    WideArgs p{};
    p.N = N; p.T = m->T; p.W = m->m0; p.Nm = m->Nm;
    p.tab = (const int4 *)(ws + L.wide_tab);
    p.b_net_stride = (long)wide_net_img_elems(m->m0);
    p.vec = (const float *)m->wide_vec_dev;
    p.T1 = (uint8_t *)(ws + L.wide_t1); p.Y2 = (uint8_t *)(ws + L.wide_y2);
    p.T2 = (uint8_t *)(ws + L.wide_t2); p.T3 = (uint8_t *)(ws + L.wide_t3);
    p.rows_id = (const int2 *)(ws + L.rows_id);
    p.rows_g = (float4 *)(ws + L.rows_g);
    p.gscale = (const float *)(ws + L.gscale);
    p.stdv = m->std_dev;
    p.tt = make_typetab(m);
    return p;
}

template <int MODE>
static cudaError_t wide_gemm(const dp_model *m, WideArgs p, int K, int Nn, const uint8_t *Aimg, int img, cudaStream_t st) {
    DP_SMEM_OPTIN(k_wide_gemm<MODE>, W_TOTAL);
    p.K = K; p.NTOT = Nn; p.BN = wide_bn(Nn);
    p.Aimg = Aimg;
    p.Bimg = (const __half *)m->wide_img_dev + wide_img_off(m->m0, img);
    // MODE 3 sums ds^ over all the N tiles of a row in one thread: no sharing there
    const int nt = Nn / p.BN;
    // (worth it when the A tiles of all CTAs, grid x 128 x K fp16, overflow the L2: K = 2048, the layer-3 backward at W = 512)
    p.G = (MODE != 3 && K >= 2048 && nt >= 4) ? 4 : 1;
    k_wide_gemm<MODE><<<m->num_sms - m->num_sms % (2 * p.G), W_THREADS, W_TOTAL, st>>>(p);      // CTA pairs
    return cudaGetLastError();
}

cudaError_t launch_env_rows(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st);

// the tile table alone (the FP64 / MIX-32 wide path of wide_gen.cu walks the same 128-row tiles)
cudaError_t launch_wide_tiles(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st) {
    k_wide_tiles<<<1, 32, 0, st>>>(N, m->T, g.ncell, (const int *)(ws + L.bin_start), (const int *)(ws + L.rowstart), (int4 *)(ws + L.wide_tab));
    return cudaGetLastError();
}

cudaError_t launch_embed_fwd_wide(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st) {
    const int W = m->m0;
    const TypeTab tt = make_typetab(m);
    cudaError_t e = launch_env_rows(m, N, g, ws, L, st);
    auto ok = [&](cudaError_t x) { if (e == cudaSuccess) e = x; };
    int4 *tab = (int4 *)(ws + L.wide_tab);
    k_wide_tiles<<<1, 32, 0, st>>>(N, m->T, g.ncell, (const int *)(ws + L.bin_start), (const int *)(ws + L.rowstart), tab);
    k_wide_l1<<<m->num_sms * 8, WR, 0, st>>>(N, m->T, W, tt, tab, (const float *)m->wide_vec_dev, (const float4 *)(ws + L.rows_rh),
                                           (uint8_t *)(ws + L.wide_t1));
    ok(cudaGetLastError());
    const WideArgs p = wide_args(m, N, ws, L);
    ok(wide_gemm<0>(m, p, W, 2 * W, p.T1, 0, st));
    ok(wide_gemm<1>(m, p, 2 * W, 4 * W, p.Y2, 1, st));
    const int P = W >= 512 ? 2 : 1;             // CTAs per atom: two CTAs (100 KB each) must fit an SM
    const int csm = 8 * WC_DEPTH * WC_SLOT + WC_BATCH * 16 + 24 * W * 4 / P;
    DP_SMEM_OPTIN(k_wide_contract, 8 * WC_DEPTH * WC_SLOT + WC_BATCH * 16 + 24 * 256 * 4);
    k_wide_contract<<<(unsigned)(N * P), 256, csm, st>>>(N, m->T, g.ncell, W, P, m->Nm, tt, tab, (const int *)(ws + L.bin_start),
                                                   (const int *)(ws + L.rowstart), (const float4 *)(ws + L.rows_rh),
                                                   (const int2 *)(ws + L.rows_id), p.Y2, p.T3, (float *)(ws + L.A));
    ok(cudaGetLastError());
    return e;
}

cudaError_t launch_embed_bwd_wide(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st) {
    const int W = m->m0;
    const TypeTab tt = make_typetab(m);
    cudaError_t e = cudaSuccess;
    auto ok = [&](cudaError_t x) { if (e == cudaSuccess) e = x; };
    const WideArgs p = wide_args(m, N, ws, L);
    // the last fitting GEMM left gA itself in the gD buffer (fit_tc.cu MODE 6)
    const float *gA = (const float *)(ws + L.gD);
    k_wide_gscale<<<(unsigned)((N + 7) / 8), 256, 0, st>>>(N, 16 * W, gA, (float *)(ws + L.gscale));
    DP_SMEM_OPTIN(k_wide_bwd_elem, BE_STAGES * BE_STAGE_BYTES);
    k_wide_bwd_elem<<<m->num_sms * 2, BE_THREADS, BE_STAGES * BE_STAGE_BYTES, st>>>(N, m->T, W, tt, p.tab, (const float4 *)(ws + L.rows_rh), p.rows_id, gA, p.gscale,
                                                 p.Y2, p.T3, p.rows_g);
    ok(cudaGetLastError());
    if (m->profile) cudaEventRecord(m->ev[6], st);      // ev[6] .. ev[7]: the two backward GEMMs
    ok(wide_gemm<2>(m, p, 4 * W, 2 * W, p.T3, 2, st));
    ok(wide_gemm<3>(m, p, 2 * W, W, p.T2, 3, st));
    if (m->profile) cudaEventRecord(m->ev[7], st);
    ok(launch_prod_force_virial(m, N, g, ws, L, st));
    return e;
}
