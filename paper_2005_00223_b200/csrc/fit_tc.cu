// S6 (fitting net forward + backward GEMMs) on tcgen05 tensor cores, mixed-precision modes.
//
// One persistent, warp-specialised GEMM kernel C[rows x N] = A[rows x K] . B[K x N] per layer product, batched over the
// atoms of each centre type (row ranges from the device-side type boundaries, no host sync):
//   warp 0      : streams the weight images B (fp16, pre-tiled at dp_create) with cp.async.bulk + mbarrier transactions
//   warp 1      : issues tcgen05.mma (one thread); accumulators in TMEM, double buffered (2 x BN columns)
//   warps 2-9   : A producers: fp32 activations from global memory -> fp16 hi + lo operand images in shared memory
//                 (activations are carried as hi + lo pairs: single-precision activations on fp16 tensor cores)
//   warps 10-13 : epilogue: tcgen05.ld, bias / tanh / residual / tanh' per MODE, fp32 results to global memory
// K = 1600 (first layer) streams A and B chunk by chunk; K = 240 keeps the A tile resident and streams B over the N tiles.
#include <cstdio>
#include <cuda_fp16.h>
#include "dp_internal.h"
#include "tc_common.cuh"

namespace {

constexpr int BM = 128;
constexpr int KC = 80;                    // K chunk: 5 k-steps of 16
constexpr int SUB = KC / 8;               // 16-byte sub-chunks per K chunk
constexpr int A_SUB_STRIDE = BM * 16 + 16;   // bytes between sub-chunks of the A image (+16: conflict-free producer stores)
constexpr int A_PART = SUB * A_SUB_STRIDE;   // one part (hi or lo) of one K chunk
// gz1 as the tcgen05 A operand of the last product, written by k_fit_chain tile by tile in the shared-memory layout of
// k_fit_tc<6>: [K chunk 3][hi, lo][sub-chunk 10][row 128 (+ pad)][16 B]; one cp.async.bulk per K chunk brings it in
constexpr int GZ_TILE_BYTES = 3 * 2 * A_PART;
static_assert((size_t)GZ_TILE_BYTES == FIT_GZ_TILE_BYTES, "workspace layout (dp_api.cu) sizes the gz1 images");
// producer threads (MODE 6 produces its resident A tile once per row tile: fewer producers leave registers to its epilogue)
__host__ __device__ constexpr int nprod(int mode) { return mode == 6 ? 32 : 256; }
// epilogue threads.  MODE 6 (gA in the epilogue): four per row, one per component c; other modes: two per row, each owns
// every other group of 16 columns (the epilogues are bound by the latency of their loads: more of them in flight)
__host__ __device__ constexpr int nepi(int mode) { return mode == 6 ? 512 : 256; }
__host__ __device__ constexpr int nthreads(int mode) { return 64 + nprod(mode) + nepi(mode); }

// WS (MIX-32: weights as hi + lo fp16 parts, "single precision"): a B stage holds the hi image followed by the lo
// image and every k-step issues three products (A hi B hi, A lo B hi, A hi B lo; lo lo is below fp32 rounding)
template <int KTOT, int NTOT, bool WS = false>
struct Cfg {
    static constexpr bool RESIDENT = KTOT == 240;            // the A tile stays in shared memory for all N tiles
    // K chunk.  K = 1600 (the descriptor producer): 64 = 4 values of m, so that A_i[c][4 kc .. 4 kc + 3] is one aligned float4
    static constexpr bool DESCR_K = KTOT != 240;             // K = 16 m2 (1600 / 2048): the first layer, A = the descriptor
    static constexpr bool GA_N = NTOT != 240;                // N = 16 m2: the last backward product, gA in the epilogue
    static constexpr int M2 = (DESCR_K ? KTOT : (GA_N ? NTOT : 1600)) / 16;     // embedding output width m2 (100 / 128)
    static constexpr int KCH = DESCR_K ? 64 : KC;
    static constexpr int SUBS = KCH / 8;
    // bytes between sub-chunks of the A image.  K = 1600: the two threads of a row are neighbouring lanes and write
    // sub-chunks 2 mm and 2 mm + 1: 64 bytes of padding put them on disjoint banks
    static constexpr int ASS = DESCR_K ? BM * 16 + 64 : A_SUB_STRIDE;
    static constexpr int A_PARTC = SUBS * ASS;               // one part (hi or lo) of one K chunk
    static constexpr int BN = NTOT == 240 ? 240 : (NTOT == 1600 ? 160 : 128);
    static constexpr int NTILES = NTOT / BN;
    static constexpr int NKC = KTOT / KCH;
    static constexpr int NA = RESIDENT ? NKC : 3;            // A buffers
    static constexpr int B_PART = KCH * BN * 2;                       // one weight image (hi or lo) of a stage
    static constexpr int B_STAGE = (WS ? 2 : 1) * B_PART;
    static constexpr int NSTAGE = WS ? 2 : (GA_N ? 4 : (DESCR_K ? 3 : 2));   // B pipeline depth (short stages need more copies in flight)
    static constexpr int A_BUF = 2 * A_PARTC;                // hi + lo
    static constexpr int OFF_A = 0;
    static constexpr int OFF_B = ((NA * A_BUF + 1023) / 1024) * 1024;
    static constexpr int OFF_BAR = OFF_B + NSTAGE * B_STAGE;
    static constexpr int TOTAL = OFF_BAR + 256;
    static constexpr int TM_BUF = 256;                       // TMEM columns per accumulator buffer
    static_assert(KTOT % KCH == 0 && NTOT % BN == 0 && BN % 16 == 0, "tile shapes");
    static_assert(TOTAL + 1024 + 64 <= 227 * 1024, "shared memory budget (1 KB: alignment of the dynamic array behind the static word)");
};

struct FitTcArgs {
    int T, ncell;
    const int *bin_start;
    const float *A; int lda;
    const uint8_t *Aimg;                         // MODE 6: the A operand as pre-built hi + lo fp16 tile images (k_fit_chain), or null
    const __half *Bimg; long b_type_stride;      // elements per type
    const float *bias;                           // [T][240]
    const float *aux0;                           // MODE 6: A [rows][4][100]
    float *out0; int ldo;
};

__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(tc::smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(tc::smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t sdst, const void *gsrc, uint32_t bytes, uint64_t *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(sdst), "l"(gsrc), "r"(bytes), "r"(tc::smem_u32(bar)) : "memory");
}

// row tile -> (type, first row, end of the type's rows)
__device__ __forceinline__ bool tile_rows(const FitTcArgs &p, int tile, int &a, int &row0, int &rend) {
    for (a = 0; a < p.T; ++a) {
        const int ts0 = p.bin_start[a * p.ncell], ts1 = p.bin_start[(a + 1) * p.ncell];
        const int nt = (ts1 - ts0 + BM - 1) / BM;
        if (tile < nt) { row0 = ts0 + tile * BM; rend = ts1; return true; }
        tile -= nt;
    }
    return false;
}

// MODE (epilogue):
//   0: out0 = tanh(acc + bias)                                   (h1; the A operand is the descriptor, formed by the producers)
//   6: gD is consumed in registers: out0[row][c][m] = gA[c][m] = sum_a gD[m][a] A[c][a] + [m < 16] sum_m' gD[m'][m] A[c][m']
//      (aux0 = A [rows][4][100]); the gD tensor never reaches memory
#ifdef DP_FIT_TIMING
__device__ long long fit_dbg[8];
#define FT(i) do { long long n_ = clock64(); if (blockIdx.x == 0) ft[i] += n_ - ftl; ftl = n_; } while (0)
#else
#define FT(i) do { } while (0)
#endif
template <int MODE, int KTOT, int NTOT, bool WS>
__global__ void __launch_bounds__(nthreads(MODE), 1) k_fit_tc(FitTcArgs p) {
    static_assert(MODE == 0 || MODE == 6, "the 240 x 240 products run in k_fit_chain");
    constexpr int NEPI = nepi(MODE), NPROD = nprod(MODE);
    using C = Cfg<KTOT, NTOT, WS>;
    extern __shared__ __align__(1024) uint8_t smem[];
    __shared__ uint32_t tmem_base_s;
    const int tid = threadIdx.x, lane = tid & 31;
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);       // warp-uniform role index
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem + C::OFF_BAR);
    uint64_t *b_full = bars, *b_empty = bars + C::NSTAGE, *a_full = bars + 2 * C::NSTAGE, *a_empty = a_full + C::NA;
    uint64_t *acc_full = a_empty + C::NA, *acc_empty = acc_full + 2;
    if (tid == 0) {
        for (int k = 0; k < C::NSTAGE; ++k) { tc::mbar_init(&b_full[k], 1); tc::mbar_init(&b_empty[k], 1); }
        for (int k = 0; k < C::NA; ++k) { tc::mbar_init(&a_full[k], NPROD / 32); tc::mbar_init(&a_empty[k], 1); }
        for (int k = 0; k < 2; ++k) { tc::mbar_init(&acc_full[k], 1); tc::mbar_init(&acc_empty[k], NEPI / 32); }
        asm volatile("fence.mbarrier_init.release.cluster;");
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tc::smem_u32(&tmem_base_s)), "n"(512));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    tc::fence_before();
    __syncthreads();
    tc::fence_after();
    const uint32_t tmem = __shfl_sync(0xffffffffu, tmem_base_s, 0);
    const uint32_t sbase = tc::smem_u32(smem);
    int ntiles_total = 0;
    for (int a = 0; a < p.T; ++a) ntiles_total += (p.bin_start[(a + 1) * p.ncell] - p.bin_start[a * p.ncell] + BM - 1) / BM;

    if (warp == 0) {
        // ---------------------------------------------------------------- B loader
        if (lane == 0) {
            uint32_t step = 0;
            for (int tile = blockIdx.x; tile < ntiles_total; tile += gridDim.x) {
                int a, row0, rend;
                tile_rows(p, tile, a, row0, rend);
                const __half *Bw = p.Bimg + a * p.b_type_stride;
                for (int nt = 0; nt < C::NTILES; ++nt)
                    for (int kc = 0; kc < C::NKC; ++kc, ++step) {
                        const int st = step % C::NSTAGE;
                        tc::mbar_wait(&b_empty[st], ((step / C::NSTAGE) & 1) ^ 1);
                        mbar_expect_tx(&b_full[st], C::B_STAGE);
                        bulk_g2s(sbase + C::OFF_B + st * C::B_STAGE, Bw + ((long)nt * C::NKC + kc) * (C::B_STAGE / 2), C::B_STAGE, &b_full[st]);
                    }
            }
        }
    } else if (warp == 1) {
        // ---------------------------------------------------------------- MMA issuer (whole warp walks the loop, one lane issues)
        {
            constexpr uint32_t idesc = tc::idesc(128, C::BN, false, false);
            uint32_t step = 0, astep = 0, accn = 0, it = 0;
#ifdef DP_FIT_TIMING
            long long ft[8] = {0, 0, 0, 0, 0, 0, 0, 0}, ftl = clock64();
#endif
            for (int tile = blockIdx.x; tile < ntiles_total; tile += gridDim.x, ++it) {
                for (int nt = 0; nt < C::NTILES; ++nt, ++accn) {
                    const int buf = accn & 1;
                    FT(0);
                    tc::mbar_wait(&acc_empty[buf], ((accn >> 1) & 1) ^ 1);
                    tc::fence_after();
                    FT(1);
                    for (int kc = 0; kc < C::NKC; ++kc, ++step) {
                        const int st = step % C::NSTAGE;
                        int ab;
                        if (C::RESIDENT) { ab = kc; tc::mbar_wait(&a_full[ab], it & 1); }
                        else { ab = astep % C::NA; tc::mbar_wait(&a_full[ab], (astep / C::NA) & 1); }
                        FT(2);
                        tc::mbar_wait(&b_full[st], (step / C::NSTAGE) & 1);
                        tc::fence_after();
                        FT(3);
                        const uint64_t da = tc::desc(sbase + C::OFF_A + ab * C::A_BUF, C::ASS, 128);
                        const uint64_t db = tc::desc(sbase + C::OFF_B + st * C::B_STAGE, C::BN * 16, 128);
                        if (tc::elect_one()) {
#pragma unroll
                            for (int part = 0; part < 2; ++part)
#pragma unroll
                                for (int ks = 0; ks < C::KCH / 16; ++ks)
                                    tc::mma_ss(tmem + buf * C::TM_BUF, tc::desc_at(da, part * C::A_PARTC + ks * 2 * C::ASS),
                                               tc::desc_at(db, ks * 2 * (C::BN * 16)), idesc, (kc | part | ks) != 0);
                            if (WS) {       // A hi . B lo
#pragma unroll
                                for (int ks = 0; ks < C::KCH / 16; ++ks)
                                    tc::mma_ss(tmem + buf * C::TM_BUF, tc::desc_at(da, ks * 2 * C::ASS),
                                               tc::desc_at(db, C::B_PART + ks * 2 * (C::BN * 16)), idesc, true);
                            }
                            tc::commit(&b_empty[st]);
                            if (!C::RESIDENT || nt == C::NTILES - 1) tc::commit(&a_empty[ab]);
                        }
                        __syncwarp();
                        FT(4);
                        if (!C::RESIDENT) ++astep;
                    }
                    if (tc::elect_one()) tc::commit(&acc_full[buf]);
                    __syncwarp();
                }
            }
#ifdef DP_FIT_TIMING
            if (blockIdx.x == 0 && lane == 0) for (int k = 0; k < 5; ++k) fit_dbg[k] = ft[k];
#endif
        }
    } else if (warp < 2 + NPROD / 32) {
        // ---------------------------------------------------------------- A producers
        const int pt = tid - 64;
        uint32_t astep = 0, it = 0;
#ifdef DP_FIT_TIMING
        long long ft[8] = {0, 0, 0, 0, 0, 0, 0, 0}, ftl = clock64();
#endif
        for (int tile = blockIdx.x; tile < ntiles_total; tile += gridDim.x, ++it) {
            int a, row0, rend;
            tile_rows(p, tile, a, row0, rend);
            if (MODE == 6 && p.Aimg) {      // the operand image exists already: one bulk copy per K chunk
                if (lane == 0)
                    for (int kc = 0; kc < C::NKC; ++kc) {
                        tc::mbar_wait(&a_empty[kc], (it & 1) ^ 1);
                        mbar_expect_tx(&a_full[kc], C::A_BUF);
                        bulk_g2s(sbase + C::OFF_A + kc * C::A_BUF, p.Aimg + (size_t)tile * GZ_TILE_BYTES + kc * C::A_BUF, C::A_BUF, &a_full[kc]);
                    }
                __syncwarp();
                continue;
            }
            // MODE 0: the A operand is the descriptor D[m*16 + a] = sum_c A[c][m] A[c][a] (S5), formed here from the
            // 4 x 100 matrix A_i (p.A, lda = 400): D never reaches memory.  Thread = (row, half of the axis range a).
            constexpr bool DESCR = MODE == 0;
            const int dr = pt >> 1, dah = pt & 1;       // neighbouring lanes share a row: their loads coalesce in L1
            const bool drow_ok = row0 + dr < rend;
            constexpr int M2 = C::M2;
            const float *Ai = p.A + (long)(drow_ok ? row0 + dr : row0) * (4 * M2);
            tc::f32x2 axp[4][4];                        // A_i[c][8 dah + 2 jp, + 1] as packed pairs
            float4 nx[4];                               // A_i[c][4 kc .. 4 kc + 3] of the next chunk (prefetched)
            if (DESCR) {
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    const float4 u0 = __ldg(reinterpret_cast<const float4 *>(Ai + c * M2 + 8 * dah));
                    const float4 u1 = __ldg(reinterpret_cast<const float4 *>(Ai + c * M2 + 8 * dah + 4));
                    axp[c][0] = tc::pk2(u0.x, u0.y); axp[c][1] = tc::pk2(u0.z, u0.w);
                    axp[c][2] = tc::pk2(u1.x, u1.y); axp[c][3] = tc::pk2(u1.z, u1.w);
                    nx[c] = u0;
                }
                if (dah) {
#pragma unroll
                    for (int c = 0; c < 4; ++c) nx[c] = __ldg(reinterpret_cast<const float4 *>(Ai + c * M2));
                }
            }
            for (int kc = 0; kc < C::NKC; ++kc, ++astep) {
                float4 cur[4];
                if (DESCR) {
#pragma unroll
                    for (int c = 0; c < 4; ++c) {
                        cur[c] = nx[c];
                        if (kc + 1 < C::NKC) nx[c] = __ldg(reinterpret_cast<const float4 *>(Ai + c * M2 + 4 * (kc + 1)));
                    }
                }
                int ab;
                FT(5);
                if (C::RESIDENT) { ab = kc; tc::mbar_wait(&a_empty[ab], (it & 1) ^ 1); }
                else { ab = astep % C::NA; tc::mbar_wait(&a_empty[ab], ((astep / C::NA) & 1) ^ 1); }
                FT(6);
                uint8_t *img = smem + C::OFF_A + ab * C::A_BUF;
                if (DESCR) {
                    // chunk kc covers m = 4 kc .. 4 kc + 3 (KCH / 16 = 4 values of m, 16 axis columns each)
#pragma unroll
                    for (int mm = 0; mm < C::KCH / 16; ++mm) {
                        const float a0 = reinterpret_cast<const float *>(&cur[0])[mm], a1 = reinterpret_cast<const float *>(&cur[1])[mm];
                        const float a2 = reinterpret_cast<const float *>(&cur[2])[mm], a3 = reinterpret_cast<const float *>(&cur[3])[mm];
                        const tc::f32x2 s0 = tc::pk2(a0, a0), s1 = tc::pk2(a1, a1), s2 = tc::pk2(a2, a2), s3 = tc::pk2(a3, a3);
                        float d[8];
#pragma unroll
                        for (int jp = 0; jp < 4; ++jp) {
                            const tc::f32x2 dp = tc::fma2(s3, axp[3][jp], tc::fma2(s2, axp[2][jp], tc::fma2(s1, axp[1][jp], tc::mul2(s0, axp[0][jp]))));
                            tc::upk2(dp, d[2 * jp], d[2 * jp + 1]);
                            if (!drow_ok) d[2 * jp] = d[2 * jp + 1] = 0.f;
                        }
                        uint4 hi, lo;
                        tc::split_h2(d[0], d[1], hi.x, lo.x); tc::split_h2(d[2], d[3], hi.y, lo.y);
                        tc::split_h2(d[4], d[5], hi.z, lo.z); tc::split_h2(d[6], d[7], hi.w, lo.w);
                        const int sub = 2 * mm + dah;
                        *reinterpret_cast<uint4 *>(img + sub * C::ASS + dr * 16) = hi;
                        *reinterpret_cast<uint4 *>(img + C::A_PARTC + sub * C::ASS + dr * 16) = lo;
                    }
                }
                // item = (row, sub-chunk): 8 consecutive fp32 -> one 16-byte hi chunk and one lo chunk
#pragma unroll
                for (int j = 0; j < (DESCR ? 0 : BM * C::SUBS / NPROD); ++j) {
                    const int idx = pt + j * NPROD;
                    const int r = idx / C::SUBS, sub = idx % C::SUBS;
                    float4 x0 = make_float4(0.f, 0.f, 0.f, 0.f), x1 = x0;
                    if (row0 + r < rend) {
                        const float4 *src = reinterpret_cast<const float4 *>(p.A + (long)(row0 + r) * p.lda + kc * C::KCH + sub * 8);
                        x0 = __ldg(src); x1 = __ldg(src + 1);
                    }
                    uint4 hi, lo;
                    tc::split_h2(x0.x, x0.y, hi.x, lo.x); tc::split_h2(x0.z, x0.w, hi.y, lo.y);
                    tc::split_h2(x1.x, x1.y, hi.z, lo.z); tc::split_h2(x1.z, x1.w, hi.w, lo.w);
                    *reinterpret_cast<uint4 *>(img + sub * C::ASS + r * 16) = hi;
                    *reinterpret_cast<uint4 *>(img + C::A_PARTC + sub * C::ASS + r * 16) = lo;
                }
                tc::proxy_fence();
                __syncwarp();
                if (lane == 0) mbar_arrive(&a_full[ab]);
            }
        }
#ifdef DP_FIT_TIMING
        FT(5);
        if (blockIdx.x == 0 && tid == 64) { fit_dbg[5] = ft[5]; fit_dbg[6] = ft[6]; }
#endif
    } else {
        // ---------------------------------------------------------------- epilogue (thread = row)
        const int q = warp & 3, r = q * 32 + lane;
        const uint32_t tm_lane = tmem + ((uint32_t)(q * 32) << 16);
        uint32_t accn = 0;
        for (int tile = blockIdx.x; tile < ntiles_total; tile += gridDim.x) {
            int a, row0, rend;
            tile_rows(p, tile, a, row0, rend);
            const bool ok = row0 + r < rend;
            const float *bias = p.bias ? p.bias + a * 240 : nullptr;
            if (MODE == 6) {
                // thread (row, c): one of the four components.  Per 16 accumulator columns = gD[m][0..16) of one m.
                // (four threads per row: the epilogue is bound by its load-to-use latencies, not by the FMA pipe)
                const int c = ((warp - 2 - NPROD / 32) >> 2) & 3;
                constexpr int M2 = C::M2;
                const float *Arow = p.aux0 + (long)(ok ? row0 + r : row0) * (4 * M2) + c * M2;
                float *Grow = p.out0 + (long)(row0 + r) * (4 * M2) + c * M2;
                float a16[16], acc2[16];
#pragma unroll
                for (int k4 = 0; k4 < 4; ++k4) {
                    const float4 v = __ldg(reinterpret_cast<const float4 *>(Arow) + k4);
                    a16[4 * k4] = v.x; a16[4 * k4 + 1] = v.y; a16[4 * k4 + 2] = v.z; a16[4 * k4 + 3] = v.w;
                    acc2[4 * k4] = acc2[4 * k4 + 1] = acc2[4 * k4 + 2] = acc2[4 * k4 + 3] = 0.f;
                }
                // A_i[c][m .. m + 3] is loaded one group of four m ahead of its use, the accumulator columns one group of 16 ahead
                float4 am0, an0, go0 = make_float4(0.f, 0.f, 0.f, 0.f);
                an0 = __ldg(reinterpret_cast<const float4 *>(Arow));
                am0 = an0;
                for (int nt = 0; nt < C::NTILES; ++nt, ++accn) {
                    const int buf = accn & 1;
                    tc::mbar_wait(&acc_full[buf], (accn >> 1) & 1);
                    tc::fence_after();
                    uint32_t v[2][16];
                    tc::ld16(tm_lane + buf * C::TM_BUF, v[0]);
#pragma unroll
                    for (int mm = 0; mm < C::BN / 16; ++mm) {
                        const int m = nt * (C::BN / 16) + mm;            // BN / 16 = 10: the unrolled mm gives m & 3 statically per nt parity
                        if ((m & 3) == 0) {
                            am0 = an0;
                            if (m + 4 < M2) an0 = __ldg(reinterpret_cast<const float4 *>(Arow + m + 4));
                        }
                        tc::wait_ld();
                        if (mm + 1 < C::BN / 16) tc::ld16(tm_lane + buf * C::TM_BUF + 16 * (mm + 1), v[(mm + 1) & 1]);
                        const float a0 = (m & 3) == 0 ? am0.x : (m & 3) == 1 ? am0.y : (m & 3) == 2 ? am0.z : am0.w;
                        float g0 = 0.f, g1 = 0.f;      // two partial sums: half the dependent-FMA chain
#pragma unroll
                        for (int ax = 0; ax < 16; ax += 2) {
                            const float gd0 = __uint_as_float(v[mm & 1][ax]), gd1 = __uint_as_float(v[mm & 1][ax + 1]);
                            g0 = fmaf(gd0, a16[ax], g0);
                            g1 = fmaf(gd1, a16[ax + 1], g1);
                            acc2[ax] = fmaf(gd0, a0, acc2[ax]);
                            acc2[ax + 1] = fmaf(gd1, a0, acc2[ax + 1]);
                        }
                        g0 += g1;
                        // m < 16: the first term joins the second one in registers (written once, after the last N tile)
                        if (nt == 0) acc2[mm] += g0;
                        else if (nt == 1 && mm < 16 - C::BN / 16) acc2[(C::BN / 16 + mm) & 15] += g0;
                        if ((m & 3) == 0) go0.x = g0;
                        else if ((m & 3) == 1) go0.y = g0;
                        else if ((m & 3) == 2) go0.z = g0;
                        else {
                            go0.w = g0;
                            if (ok && m >= 16) *reinterpret_cast<float4 *>(Grow + m - 3) = go0;
                        }
                    }
                    tc::fence_before();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&acc_empty[buf]);
                }
                if (ok) {
#pragma unroll
                    for (int k4 = 0; k4 < 4; ++k4)
                        *reinterpret_cast<float4 *>(Grow + 4 * k4) = make_float4(acc2[4 * k4], acc2[4 * k4 + 1], acc2[4 * k4 + 2], acc2[4 * k4 + 3]);
                }
                continue;
            }
            // MODE 0: h1 = tanh(acc + c1); two threads per row, each owns every other group of 16 columns
            for (int nt = 0; nt < C::NTILES; ++nt, ++accn) {
                const int buf = accn & 1;
                tc::mbar_wait(&acc_full[buf], (accn >> 1) & 1);
                tc::fence_after();
                const long o = (long)(row0 + r) * p.ldo + nt * C::BN;
                const int half = ((warp - 2 - NPROD / 32) >> 2) & 1;
#pragma unroll 1
                for (int c0 = 16 * half; c0 < C::BN; c0 += 32) {
                    uint32_t v[16];
                    tc::ld16(tm_lane + buf * C::TM_BUF + c0, v);
                    tc::wait_ld();
                    if (ok) {
#pragma unroll
                        for (int g4 = 0; g4 < 4; ++g4) {
                            const int c = c0 + 4 * g4;
                            const float4 b = *reinterpret_cast<const float4 *>(bias + c);
                            const float bb[4] = {b.x, b.y, b.z, b.w};
                            float r0[4];
#pragma unroll
                            for (int k = 0; k < 4; ++k) {
                                const float z = __uint_as_float(v[4 * g4 + k]) + bb[k];
                                r0[k] = WS ? tanhf(z) : tc::tanh_approx(z);        // MIX-32: exact single-precision tanh
                            }
                            *reinterpret_cast<float4 *>(p.out0 + o + c) = make_float4(r0[0], r0[1], r0[2], r0[3]);
                        }
                    }
                }
                tc::fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(&acc_empty[buf]);
            }
        }
    }
    tc::fence_before();
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(512));
}

// ---------------------------------------------------------------------------------------------------------------------
// The four 240 x 240 products of the fitting net in ONE kernel (layers 2, 3 forward, their backward):
//   S1: t2 = tanh(h1 V2 + c2), h2 = h1 + t2         S2: t3 = tanh(h2 V3 + c3), h3 = h2 + t3, E_i = h3.v4 + c4 + ebias,
//   S3: gh2 = v4 + gz3 V3^T, gz2 = gh2 (1 - t2^2)        gz3 = v4 (1 - t3^2)
//   S4: gh1 = gh2 + gz2 V2^T, gz1 = gh1 (1 - h1^2)  -> global (A operand of the last product, MODE 6)
// One 128-row tile per CTA at a time; the operand of every stage is written by the previous epilogue straight into the
// shared-memory operand image (hi + lo fp16), 1 - t2^2 waits in TMEM (fp32), gh2 stays in the accumulator and the S4
// product accumulates on top of it.  h1 is read from global memory twice (S1 operand, S4 epilogue), prefetched into
// registers under the preceding MMAs; nothing else of the chain touches HBM.
// Warps: 0 weight loader (cp.async.bulk), 1 MMA issuer, 2-9 epilogue / operand producers: thread (row, half of the columns).
struct FitChainArgs {
    int T, ncell;
    const int *bin_start;
    const float *h1;                      // [rows][240]
    const __half *Bimg; long b_type_stride;
    const float *c2, *c3, *v4, *c4;       // [T][240], c4 [T]
    const double *ebias;                  // [T]
    long nd240;                           // elements of the V1 image (16 m2 x 240): the 240 x 240 images follow it
    uint8_t *gz1img;                      // per 128-row tile the hi + lo fp16 operand image of the last product (GZ_TILE_BYTES)
    double *eatom;                        // [rows]
};
constexpr int CH_THREADS = 64 + 256;
constexpr int CH_BN = 240, CH_NKC = 3, CH_BSTAGE = KC * CH_BN * 2;
constexpr int CH_OFF_B = ((CH_NKC * 2 * A_PART + 1023) / 1024) * 1024;
constexpr int CH_OFF_BAR = CH_OFF_B + 2 * CH_BSTAGE;
constexpr int CH_OFF_RED = CH_OFF_BAR + 128;                 // float [2][128] energy partial sums
constexpr int CH_TOTAL = CH_OFF_RED + 2 * 128 * 4;
constexpr int CH_TM_ACC = 0, CH_TM_D2 = 256;                 // TMEM: accumulator [0,240), 1 - t2^2 (fp32) [256,496)
static_assert(CH_TOTAL <= 227 * 1024, "shared memory budget");

__global__ void __launch_bounds__(CH_THREADS, 1) k_fit_chain(FitChainArgs p) {
    extern __shared__ __align__(1024) uint8_t smem[];
    __shared__ uint32_t tmem_base_s;
    const int tid = threadIdx.x, lane = tid & 31;
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem + CH_OFF_BAR);
    uint64_t *b_full = bars, *b_empty = bars + 2, *a_ready = bars + 4, *acc_ready = bars + 5;
    float *red = reinterpret_cast<float *>(smem + CH_OFF_RED);
    if (tid == 0) {
        for (int k = 0; k < 2; ++k) { tc::mbar_init(&b_full[k], 1); tc::mbar_init(&b_empty[k], 1); }
        tc::mbar_init(a_ready, 8);
        tc::mbar_init(acc_ready, 1);
        asm volatile("fence.mbarrier_init.release.cluster;");
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tc::smem_u32(&tmem_base_s)), "n"(512));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    tc::fence_before();
    __syncthreads();
    tc::fence_after();
    const uint32_t tmem = __shfl_sync(0xffffffffu, tmem_base_s, 0);
    const uint32_t sbase = tc::smem_u32(smem);
    int ntiles_total = 0;
    for (int a = 0; a < p.T; ++a) ntiles_total += (p.bin_start[(a + 1) * p.ncell] - p.bin_start[a * p.ncell] + BM - 1) / BM;
    auto tile_of = [&](int tile, int &a, int &row0, int &rend) {
        for (a = 0; a < p.T; ++a) {
            const int ts0 = p.bin_start[a * p.ncell], ts1 = p.bin_start[(a + 1) * p.ncell];
            const int nt = (ts1 - ts0 + BM - 1) / BM;
            if (tile < nt) { row0 = ts0 + tile * BM; rend = ts1; return; }
            tile -= nt;
        }
    };
    // weight images of the four stages inside one type's block (FIT_TC_OFF[1..4]): V2, V3, V3^T, V2^T
    const long img_off[4] = {p.nd240, p.nd240 + 240L * 240, p.nd240 + 2L * 240 * 240, p.nd240 + 3L * 240 * 240};

    if (warp == 0) {
        // ---------------------------------------------------------------- weight loader
        if (lane == 0) {
            uint32_t step = 0;
            for (int tile = blockIdx.x; tile < ntiles_total; tile += gridDim.x) {
                int a, row0, rend;
                tile_of(tile, a, row0, rend);
                const __half *Bw = p.Bimg + a * p.b_type_stride;
                for (int sidx = 0; sidx < 4; ++sidx)
                    for (int kc = 0; kc < CH_NKC; ++kc, ++step) {
                        const int st = step & 1;
                        tc::mbar_wait(&b_empty[st], ((step >> 1) & 1) ^ 1);
                        mbar_expect_tx(&b_full[st], CH_BSTAGE);
                        bulk_g2s(sbase + CH_OFF_B + st * CH_BSTAGE, Bw + img_off[sidx] + (long)kc * (KC * CH_BN), CH_BSTAGE, &b_full[st]);
                    }
            }
        }
    } else if (warp == 1) {
        // ---------------------------------------------------------------- MMA issuer
        constexpr uint32_t idesc = tc::idesc(128, CH_BN, false, false);
        uint32_t step = 0, stage = 0;
        for (int tile = blockIdx.x; tile < ntiles_total; tile += gridDim.x)
            for (int sidx = 0; sidx < 4; ++sidx, ++stage) {
                tc::mbar_wait(a_ready, stage & 1);
                tc::fence_after();
                for (int kc = 0; kc < CH_NKC; ++kc, ++step) {
                    const int st = step & 1;
                    tc::mbar_wait(&b_full[st], (step >> 1) & 1);
                    tc::fence_after();
                    const uint64_t da = tc::desc(sbase + kc * 2 * A_PART, A_SUB_STRIDE, 128);
                    const uint64_t db = tc::desc(sbase + CH_OFF_B + st * CH_BSTAGE, CH_BN * 16, 128);
                    if (tc::elect_one()) {
#pragma unroll
                        for (int part = 0; part < 2; ++part)
#pragma unroll
                            for (int ks = 0; ks < KC / 16; ++ks)       // S4 accumulates on gh2, left in TMEM by the S3 epilogue
                                tc::mma_ss(tmem + CH_TM_ACC, tc::desc_at(da, part * A_PART + ks * 2 * A_SUB_STRIDE),
                                           tc::desc_at(db, ks * 2 * (CH_BN * 16)), idesc, sidx == 3 || (kc | part | ks) != 0);
                        tc::commit(&b_empty[st]);
                    }
                    __syncwarp();
                }
                if (tc::elect_one()) tc::commit(acc_ready);
                __syncwarp();
            }
    } else {
        // ---------------------------------------------------------------- epilogue / operand producers: thread = (row, column half)
        const int q4 = warp & 3, r = q4 * 32 + lane, hc = ((warp - 2) >> 2) & 1;
        const uint32_t tm_lane = tmem + ((uint32_t)(q4 * 32) << 16);
        uint32_t stage = 0;
        // 8 consecutive values of this row -> the hi and lo 16-byte chunks of column group j (columns 120 hc + 8 j ..)
        auto put_group = [&](int j, const float (&x)[8]) {
            const int g = 15 * hc + j, kc = g / SUB, sub = g % SUB;
            uint8_t *dst = smem + kc * 2 * A_PART + sub * A_SUB_STRIDE + r * 16;
            uint4 hi, lo;
            tc::split_h2(x[0], x[1], hi.x, lo.x); tc::split_h2(x[2], x[3], hi.y, lo.y);
            tc::split_h2(x[4], x[5], hi.z, lo.z); tc::split_h2(x[6], x[7], hi.w, lo.w);
            *reinterpret_cast<uint4 *>(dst) = hi;
            *reinterpret_cast<uint4 *>(dst + A_PART) = lo;
        };
        auto publish = [&]() {        // operand image (and TMEM stores) of this warp are complete: one arrival per warp
            tc::wait_st();
            tc::proxy_fence();
            tc::fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(a_ready);
        };
        auto wait_acc = [&]() {
            tc::mbar_wait(acc_ready, stage & 1);
            ++stage;
            tc::fence_after();
        };
        for (int tile = blockIdx.x; tile < ntiles_total; tile += gridDim.x) {
            int a, row0, rend;
            tile_of(tile, a, row0, rend);
            const bool ok = row0 + r < rend;
            const float *h1row = p.h1 + (long)(ok ? row0 + r : row0) * 240 + 120 * hc;
            const float *c2 = p.c2 + a * 240 + 120 * hc, *c3 = p.c3 + a * 240 + 120 * hc, *v4 = p.v4 + a * 240 + 120 * hc;
            float H[120];
            // ---- operand of S1: h1 ----
#pragma unroll
            for (int k4 = 0; k4 < 30; ++k4) {
                float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
                if (ok) v = __ldg(reinterpret_cast<const float4 *>(h1row) + k4);
                H[4 * k4] = v.x; H[4 * k4 + 1] = v.y; H[4 * k4 + 2] = v.z; H[4 * k4 + 3] = v.w;
            }
#pragma unroll
            for (int j = 0; j < 15; ++j) {
                const float x[8] = {H[8 * j], H[8 * j + 1], H[8 * j + 2], H[8 * j + 3], H[8 * j + 4], H[8 * j + 5], H[8 * j + 6], H[8 * j + 7]};
                put_group(j, x);
            }
            publish();
            // ---- S1: t2 = tanh(acc + c2); 1 - t2^2 -> TMEM; h2 = h1 + t2 -> operand of S2 ----
            wait_acc();
#pragma unroll
            for (int j = 0; j < 15; ++j) {
                uint32_t v[8], d[8];
                tc::ld8(tm_lane + CH_TM_ACC + 120 * hc + 8 * j, v);
                tc::wait_ld();
                float x[8];
#pragma unroll
                for (int q = 0; q < 8; ++q) {
                    const float z = __uint_as_float(v[q]) + __ldg(c2 + 8 * j + q);
                    const float t = tc::tanh_approx(z);
                    d[q] = __float_as_uint(fmaf(-t, t, 1.f));
                    H[8 * j + q] += t;
                    x[q] = H[8 * j + q];
                }
                tc::st8(tm_lane + CH_TM_D2 + 120 * hc + 8 * j, d);
                put_group(j, x);
            }
            publish();
            // ---- S2: t3 = tanh(acc + c3); h3 = h2 + t3 -> E_i; gz3 = v4 (1 - t3^2) -> operand of S3 ----
            wait_acc();
            float esum = 0.f;
#pragma unroll
            for (int j = 0; j < 15; ++j) {
                uint32_t v[8];
                tc::ld8(tm_lane + CH_TM_ACC + 120 * hc + 8 * j, v);
                tc::wait_ld();
                float x[8];
#pragma unroll
                for (int q = 0; q < 8; ++q) {
                    const float w = __ldg(v4 + 8 * j + q);
                    const float t = tanhf(__uint_as_float(v[q]) + __ldg(c3 + 8 * j + q));
                    esum = fmaf(H[8 * j + q] + t, w, esum);
                    x[q] = w * fmaf(-t, t, 1.f);
                }
                put_group(j, x);
            }
            red[hc * 128 + r] = esum;
            tc::bar_sync(1, 256);
            if (hc == 0 && ok) p.eatom[row0 + r] = (double)(red[r] + red[128 + r] + __ldg(p.c4 + a)) + p.ebias[a];
            publish();
            // ---- S3: gh2 = v4 + acc (left in the accumulator); gz2 = gh2 (1 - t2^2) -> operand of S4 ----
            wait_acc();
#pragma unroll
            for (int j = 0; j < 15; ++j) {
                uint32_t v[8], d[8], o[8];
                tc::ld8(tm_lane + CH_TM_ACC + 120 * hc + 8 * j, v);
                tc::ld8(tm_lane + CH_TM_D2 + 120 * hc + 8 * j, d);
                tc::wait_ld();
                float x[8];
#pragma unroll
                for (int q = 0; q < 8; ++q) {
                    const float gh = __ldg(v4 + 8 * j + q) + __uint_as_float(v[q]);
                    o[q] = __float_as_uint(gh);
                    x[q] = gh * __uint_as_float(d[q]);
                }
                tc::st8(tm_lane + CH_TM_ACC + 120 * hc + 8 * j, o);
                put_group(j, x);
            }
            publish();
            // h1 again (for 1 - h1^2), in flight under the S4 products
#pragma unroll
            for (int k4 = 0; k4 < 30; ++k4) {
                float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
                if (ok) v = __ldg(reinterpret_cast<const float4 *>(h1row) + k4);
                H[4 * k4] = v.x; H[4 * k4 + 1] = v.y; H[4 * k4 + 2] = v.z; H[4 * k4 + 3] = v.w;
            }
            // ---- S4: gh1 = acc (= gh2 + gz2 V2^T); gz1 = gh1 (1 - h1^2) -> global ----
            wait_acc();
            uint8_t *gzimg = p.gz1img + (size_t)tile * GZ_TILE_BYTES + r * 16;
#pragma unroll
            for (int j = 0; j < 15; ++j) {
                uint32_t v[8];
                tc::ld8(tm_lane + CH_TM_ACC + 120 * hc + 8 * j, v);
                tc::wait_ld();
                float x[8];
#pragma unroll
                for (int q = 0; q < 8; ++q) x[q] = ok ? __uint_as_float(v[q]) * fmaf(-H[8 * j + q], H[8 * j + q], 1.f) : 0.f;
                const int g = 15 * hc + j, kc = g / SUB, sub = g % SUB;
                uint4 hi, lo;
                tc::split_h2(x[0], x[1], hi.x, lo.x); tc::split_h2(x[2], x[3], hi.y, lo.y);
                tc::split_h2(x[4], x[5], hi.z, lo.z); tc::split_h2(x[6], x[7], hi.w, lo.w);
                uint8_t *dst = gzimg + kc * 2 * A_PART + sub * A_SUB_STRIDE;
                *reinterpret_cast<uint4 *>(dst) = hi;
                *reinterpret_cast<uint4 *>(dst + A_PART) = lo;
            }
            tc::fence_before();      // the accumulator reads above precede the next tile's products (ordered by its first publish)
        }
    }
    tc::fence_before();
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(512));
}

template <int MODE, int KTOT, int NTOT, bool WS = false>
cudaError_t launch(const FitTcArgs &p, int grid, cudaStream_t st) {
    using C = Cfg<KTOT, NTOT, WS>;
    DP_SMEM_OPTIN((k_fit_tc<MODE, KTOT, NTOT, WS>), C::TOTAL);
    k_fit_tc<MODE, KTOT, NTOT, WS><<<grid, nthreads(MODE), C::TOTAL, st>>>(p);
#ifdef DP_FIT_TIMING
    {
        cudaStreamSynchronize(st);
        long long h[8];
        cudaMemcpyFromSymbol(h, fit_dbg, sizeof(h));
        long long tot = 0;
        for (int k = 0; k < 5; ++k) tot += h[k];
        fprintf(stderr, "fit_tc mode %d MMA warp cycles %lld: other %.1f%% acc_empty %.1f%% a_full %.1f%% b_full %.1f%% issue %.1f%%; producer: work %.1f%% wait a_empty %.1f%%\n", MODE, tot,
                100.0 * h[0] / tot, 100.0 * h[1] / tot, 100.0 * h[2] / tot, 100.0 * h[3] / tot, 100.0 * h[4] / tot, 100.0 * h[5] / tot, 100.0 * h[6] / tot);
    }
#endif
    return cudaGetLastError();
}

}  // namespace

// Host side: weight images.  For product g the image of type a is [NTILES][K/8][BN][8] fp16 with
// element (nt, k8, n, kk) = B[k = k8*8 + kk][nt*BN + n]  (any K chunking of the kernels reads it contiguously).
void fit_tc_build_image(const double *W, int ldw, bool transpose, int K, int Nn, __half *out) {
    const int BN = Nn == 240 ? 240 : (Nn == 1600 ? 160 : 128);
    const int ntl = Nn / BN, nk8 = K / 8;
    for (int nt = 0; nt < ntl; ++nt)
        for (int k8 = 0; k8 < nk8; ++k8)
            for (int n = 0; n < BN; ++n)
                for (int kk = 0; kk < 8; ++kk) {
                    const int k = k8 * 8 + kk, nn = nt * BN + n;
                    const double v = transpose ? W[(size_t)nn * ldw + k] : W[(size_t)k * ldw + nn];
                    out[(((size_t)nt * nk8 + k8) * BN + n) * 8 + kk] = __float2half_rn((float)v);
                }
}

// offsets (elements) of the six product images inside one type's block: g0 V1, g1 V2, g2 V3, g3 V3^T, g4 V2^T, g5 V1^T
static size_t fit_tc_off(int nd, int g) {
    const size_t a = (size_t)nd * 240, b = 240 * 240;
    const size_t off[7] = {0, a, a + b, a + 2 * b, a + 3 * b, a + 4 * b, 2 * a + 4 * b};
    return off[g];
}
size_t fit_tc_type_elems(int nd) { return fit_tc_off(nd, 6); }
void fit_tc_build_type(int nd, const double *V1, const double *V2, const double *V3, __half *out) {
    fit_tc_build_image(V1, 240, false, nd, 240, out + fit_tc_off(nd, 0));
    fit_tc_build_image(V2, 240, false, 240, 240, out + fit_tc_off(nd, 1));
    fit_tc_build_image(V3, 240, false, 240, 240, out + fit_tc_off(nd, 2));
    fit_tc_build_image(V3, 240, true, 240, 240, out + fit_tc_off(nd, 3));
    fit_tc_build_image(V2, 240, true, 240, 240, out + fit_tc_off(nd, 4));
    fit_tc_build_image(V1, 240, true, 240, nd, out + fit_tc_off(nd, 5));
}

// S5 + S6 in MIX-16: first layer (descriptor formed in the operand producer), the fused 240 x 240 chain with the energy,
// and the last backward product with gA in its epilogue (the gD buffer receives gA [N][4][100]; gD is never written).
// gz1 travels from the chain to the last product as ready-made hi + lo fp16 tile images in the activation buffers 2 S .. 4 S.
template <int ND>
static cudaError_t launch_fit_tc_nd(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st) {
    const int F = 240;
    constexpr int M2E = ND / 16;
    float *Amat = (float *)(ws + L.A);
    float *act = (float *)(ws + L.fit_act);
    float *h1 = act;
    uint8_t *gzimg = reinterpret_cast<uint8_t *>(act + 2 * (size_t)N * F);
    const int *bin_start = (const int *)(ws + L.bin_start);
    const int grid = m->num_sms;
    cudaError_t e = cudaSuccess;
    auto ok = [&](cudaError_t x) { if (e == cudaSuccess) e = x; };
    FitTcArgs p{};
    p.T = m->T; p.ncell = g.ncell; p.bin_start = bin_start; p.b_type_stride = (long)fit_tc_off(ND, 6);
    p.A = Amat; p.lda = 4 * M2E; p.Bimg = (const __half *)m->fit_tc_img_dev + fit_tc_off(ND, 0);
    p.bias = (const float *)m->fitc1_dev; p.out0 = h1; p.ldo = F;
    ok(launch<0, ND, 240>(p, grid, st));
    FitChainArgs c{};
    c.T = m->T; c.ncell = g.ncell; c.bin_start = bin_start; c.h1 = h1;
    c.Bimg = (const __half *)m->fit_tc_img_dev; c.b_type_stride = (long)fit_tc_off(ND, 6);
    c.c2 = (const float *)m->fitc2_dev; c.c3 = (const float *)m->fitc3_dev; c.v4 = (const float *)m->fitv4_dev;
    c.c4 = (const float *)m->fitc4_dev; c.nd240 = (long)ND * 240; c.ebias = m->ebias_dev; c.gz1img = gzimg; c.eatom = (double *)(ws + L.eatom);
    DP_SMEM_OPTIN(k_fit_chain, CH_TOTAL);
    k_fit_chain<<<grid, CH_THREADS, CH_TOTAL, st>>>(c);
    ok(cudaGetLastError());
    FitTcArgs q{};
    q.T = m->T; q.ncell = g.ncell; q.bin_start = bin_start; q.b_type_stride = (long)fit_tc_off(ND, 6);
    q.Aimg = gzimg; q.lda = F; q.Bimg = (const __half *)m->fit_tc_img_dev + fit_tc_off(ND, 5);
    q.aux0 = Amat; q.out0 = (float *)(ws + L.gD); q.ldo = ND;
    ok(launch<6, 240, ND>(q, grid, st));
    return e;
}

// ---- MIX-32: the two large products of the fitting net (first layer forward, K = 16 m2; last product backward, N = 16 m2)
// on the same kernels with the weights as hi + lo fp16 parts (WS) and the exact tanhf; the four 240 x 240 products stay in
// fit_mix.cu.  Images of one type: V1 for MODE 0 (K chunks of 64), then V1^T for MODE 6 (K chunks of 80); per stage (N tile, K
// chunk) the hi image [KCH / 8][BN][8] followed by the lo image.
static void fit_tc32_build_image(const double *W, int ldw, bool transpose, int K, int Nn, int KCH, __half *out) {
    const int BN = Nn == 240 ? 240 : (Nn == 1600 ? 160 : 128);
    const int ntl = Nn / BN, nkc = K / KCH, sub = KCH / 8;
    for (int nt = 0; nt < ntl; ++nt)
        for (int kc = 0; kc < nkc; ++kc)
            for (int k8 = 0; k8 < sub; ++k8)
                for (int n = 0; n < BN; ++n)
                    for (int kk = 0; kk < 8; ++kk) {
                        const int k = kc * KCH + k8 * 8 + kk, nn = nt * BN + n;
                        const double v = transpose ? W[(size_t)nn * ldw + k] : W[(size_t)k * ldw + nn];
                        const float vf = (float)v;                  // "cast to single", then hi + lo fp16 parts
                        const __half hi = __float2half_rn(vf);
                        const __half lo = __float2half_rn(vf - __half2float(hi));
                        const size_t stage = ((size_t)nt * nkc + kc) * 2 * ((size_t)KCH * BN);
                        const size_t e = ((size_t)k8 * BN + n) * 8 + kk;
                        out[stage + e] = hi;
                        out[stage + (size_t)KCH * BN + e] = lo;
                    }
}
size_t fit_tc32_type_elems(int nd) { return 4 * (size_t)nd * 240; }
void fit_tc32_build_type(int nd, const double *V1, __half *out) {
    fit_tc32_build_image(V1, 240, false, nd, 240, 64, out);
    fit_tc32_build_image(V1, 240, true, 240, nd, 80, out + 2 * (size_t)nd * 240);
}

template <int ND>
static cudaError_t launch_fit_tc32_first_nd(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st) {
    constexpr int M2E = ND / 16;
    FitTcArgs p{};
    p.T = m->T; p.ncell = g.ncell; p.bin_start = (const int *)(ws + L.bin_start); p.b_type_stride = (long)fit_tc32_type_elems(ND);
    p.A = (const float *)(ws + L.A); p.lda = 4 * M2E; p.Bimg = (const __half *)m->fit_tc_img_dev;
    p.bias = (const float *)m->fitc1_dev; p.out0 = (float *)(ws + L.fit_act); p.ldo = 240;
    return launch<0, ND, 240, true>(p, m->num_sms, st);
}
template <int ND>
static cudaError_t launch_fit_tc32_last_nd(const dp_model *m, long N, const float *gz1, const Grid3 &g, char *ws, const WsLayout &L,
                                           cudaStream_t st) {
    FitTcArgs q{};
    q.T = m->T; q.ncell = g.ncell; q.bin_start = (const int *)(ws + L.bin_start); q.b_type_stride = (long)fit_tc32_type_elems(ND);
    q.A = gz1; q.lda = 240; q.Aimg = nullptr; q.Bimg = (const __half *)m->fit_tc_img_dev + 2 * (size_t)ND * 240;
    q.aux0 = (const float *)(ws + L.A); q.out0 = (float *)(ws + L.gD); q.ldo = ND;
    return launch<6, 240, ND, true>(q, m->num_sms, st);
}
// h1 [N][240] (first activation buffer) = tanh(D V1 + c1), the descriptor D formed in the operand producer from A_i
cudaError_t launch_fit_tc32_first(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st) {
    switch (m->m2) {
        case 128: return launch_fit_tc32_first_nd<2048>(m, N, g, ws, L, st);
        case 256: return launch_fit_tc32_first_nd<4096>(m, N, g, ws, L, st);       // wide nets (wide_gen.cu)
        case 512: return launch_fit_tc32_first_nd<8192>(m, N, g, ws, L, st);
        case 1024: return launch_fit_tc32_first_nd<16384>(m, N, g, ws, L, st);
        case 2048: return launch_fit_tc32_first_nd<32768>(m, N, g, ws, L, st);
        default: return launch_fit_tc32_first_nd<1600>(m, N, g, ws, L, st);
    }
}
// gA [N][4][m2] (in the gD buffer) from gz1 [N][240]: the last backward product with gD consumed in its epilogue
cudaError_t launch_fit_tc32_last(const dp_model *m, long N, const float *gz1, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st) {
    switch (m->m2) {
        case 128: return launch_fit_tc32_last_nd<2048>(m, N, gz1, g, ws, L, st);
        case 256: return launch_fit_tc32_last_nd<4096>(m, N, gz1, g, ws, L, st);
        case 512: return launch_fit_tc32_last_nd<8192>(m, N, gz1, g, ws, L, st);
        case 1024: return launch_fit_tc32_last_nd<16384>(m, N, gz1, g, ws, L, st);
        case 2048: return launch_fit_tc32_last_nd<32768>(m, N, gz1, g, ws, L, st);
        default: return launch_fit_tc32_last_nd<1600>(m, N, gz1, g, ws, L, st);
    }
}

cudaError_t launch_fit_tc(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st) {
    switch (m->m2) {
        case 128: return launch_fit_tc_nd<2048>(m, N, g, ws, L, st);
        case 256: return launch_fit_tc_nd<4096>(m, N, g, ws, L, st);       // wide nets (wide.cu)
        case 512: return launch_fit_tc_nd<8192>(m, N, g, ws, L, st);
        case 1024: return launch_fit_tc_nd<16384>(m, N, g, ws, L, st);
        case 2048: return launch_fit_tc_nd<32768>(m, N, g, ws, L, st);
        default: return launch_fit_tc_nd<1600>(m, N, g, ws, L, st);
    }
}
