// S7 + S8 + S9 (embedding backward, ProdForce, ProdViral) on tcgen05 tensor cores, MIX-16.
//
// One warpgroup = one 128-row tile (thread = neighbour row = TMEM lane), two warpgroups per CTA, one CTA per SM.
// The forward is recomputed (storing the tanh outputs would cost 94 GB at config 4) with the
// activations carried as fp16 hi + lo pairs: the hi parts live in TMEM and feed tcgen05.mma as the A operand, the lo
// parts in shared memory.  With t_l = tanh(z_l) and T = [t1 | t2 | t3] (embed_tc2.cuh) the residual folds are linear, so
//   dR^[k][c]  = sum_col T[k][col] g~[c][col]                      (g~ = gA folded onto the T columns, per atom)
//   dT[k][col] = sum_c R^[k][c] g~[c][col]                         (direct part of every layer's gradient)
//   dz3 = dT3 (1 - t3^2);   dy2 = dT2 + dz3 W3^T;   dz2 = dy2 (1 - t2^2)
//   dy1 = dT1 + dz3 (W3^T folded) + dz2 W2^T;   dz1 = dy1 (1 - t1^2);   ds^ = dz1 . w1
// followed, per row, by the fp64 geometry derivative, the force scatter and the virial (S8, S9).
// Per-atom operand images g~ (hi, lo) come from k_gA_img (the tail of the fitting backward), scaled by a power of two.
#include <cstdio>
#include <cstdlib>
#include "embed_tc2.cuh"
#include "tc_common.cuh"

namespace {

#ifdef DP_BWD_TIMING
#define DP_TICK(i) do { if (dbg_t) { long long now_ = clock64(); tacc[i] += now_ - tlast; tlast = now_; } } while (0)
#else
#define DP_TICK(i) do { } while (0)
#endif

constexpr int NWG = 2;
// TMEM columns per warpgroup
constexpr int TM_T = 0;                        // T hi parts, packed fp16 pairs: t1 [0,16) t2 [16,48) t3 [48,48 + K3/2)
constexpr int TM_Z = 112;                      // accumulator: z2 -> z3 -> dT3 -> [dy2 | dy1]      (K3 columns)
constexpr int TM_WG = 256;

template <int W>
struct BwdSmem {
    using L = T2<W>;
    static constexpr int TM_DR = TM_Z + L::K3;                     // dR^: 2 slots x 8 columns (TMEM columns 224 / 240)
    static_assert(TM_DR + 16 <= TM_WG && 48 + L::K3 / 2 <= TM_Z, "TMEM budget");
    static constexpr int W2 = 0;                                   // [4][64][16 B]
    static constexpr int W3 = W2 + 4 * 64 * 16;                    // [12][K3][16 B]
    static constexpr int W3T = W3 + 12 * L::K3 * 16;               // [K3/8][96][16 B]
    static constexpr int W2T = W3T + (L::K3 / 8) * 96 * 16;        // [8][32][16 B]
    static constexpr int BB2 = W2T + 8 * 32 * 16;                  // ONES_STEP: bias chunks and the ones image (embed_tc2.cuh)
    static constexpr int BB3 = BB2 + (L::ONES_STEP ? 64 * 16 : 0);
    static constexpr int ONES = BB3 + (L::ONES_STEP ? L::K3 * 16 : 0);
    static constexpr int VEC = ONES + (L::ONES_STEP ? 256 : 0);    // w1[32] b1[32]
    static constexpr int BARS = VEC + 256;
    static constexpr int WG0 = ((BARS + 64 + 127) / 128) * 128;
    // per warpgroup
    static constexpr int TLO = 0;                                  // T lo parts / dz2 / dz3: CHUNKS x 2 KB
    static constexpr int RIMG = TLO + L::CHUNKS * 2048;            // A of the direct products: [4][128][16 B]
    // per slot the atom's gradient image C [COLS][16 B]: K-major B of the direct products (K = 16 per slot: both K chunks
    // read the same image; W = 25 keeps two copies, W = 32 aliases them through a zero leading stride) and, viewed MN-major,
    // B of the dR^ product (N = 16)
    static constexpr int QCOPIES = W == 25 ? 2 : 1;
    static constexpr int QIMG = RIMG + 4 * 2048;
    static constexpr int META = QIMG + 2 * QCOPIES * L::COLS * 16;
    static constexpr int WG_BYTES = ((META + 2 * 3072 + 127) / 128) * 128;   // META: two stages of prefetched row data
    static constexpr int TOTAL = WG0 + NWG * WG_BYTES;
    static_assert(TOTAL + 1024 <= 227 * 1024, "shared memory budget (1 KB: alignment of the dynamic array behind the static word)");
};

__device__ __forceinline__ double min_image(double t, double L, double halfL) {
    double s = t > halfL ? -1.0 : (t < -halfL ? 1.0 : 0.0);
    return __dadd_rn(t, __dmul_rn(s, L));
}
struct EnvParams {
    double rc, rc_smth, inv_range;
    double L[3];
};

__device__ __forceinline__ void cp_async16(uint32_t sdst, const void *gsrc) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sdst), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async8(uint32_t sdst, const void *gsrc) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(sdst), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

__device__ __forceinline__ float2 unpack_h2(uint32_t v) {
    return __half22float2(*reinterpret_cast<const __half2 *>(&v));
}

// 16 accumulator columns: t = tanh(z); hi parts -> 8 TMEM columns, lo parts -> two 16-byte chunks, 1 - t^2 -> dpk (fp16 pairs)
__device__ __forceinline__ void act16(const uint32_t (&z)[16], uint32_t tm_dst, uint8_t *lo_row, int chunk, uint32_t *dpk) {
    uint32_t hi[8], lo[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        const float x = tc::tanh_approx(__uint_as_float(z[2 * q])), y = tc::tanh_approx(__uint_as_float(z[2 * q + 1]));
        tc::split_h2(x, y, hi[q], lo[q]);
        dpk[q] = tc::pack_h2(fmaf(-x, x, 1.f), fmaf(-y, y, 1.f));
    }
    tc::st8(tm_dst, hi);
    *reinterpret_cast<uint4 *>(lo_row + chunk * 2048) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
    *reinterpret_cast<uint4 *>(lo_row + (chunk + 1) * 2048) = make_uint4(lo[4], lo[5], lo[6], lo[7]);
}
// Per-atom operand image of the folded gradient g~[c][col] = fold(gA)[c][col] * 2^e, split in hi + lo fp16 parts:
//   C [COLS][8] : per T column {hi[0..3], lo[0..3]} (16 bytes); 3,328 / 3,584 bytes per atom
// Built from gA (fp32 [N][4][100], written by the epilogue of the last fitting-backward GEMM, fit_tc.cu MODE 6).
template <int W>
__global__ void __launch_bounds__(256) k_gA_fold(long N, const float *__restrict__ gA, uint8_t *__restrict__ img,
                                                  float *__restrict__ gscale) {
    constexpr int M0 = T2<W>::M0, M1 = T2<W>::M1, M2E = T2<W>::M2E, COLS = T2<W>::COLS, GA_IMG_BYTES = COLS * 16;
    __shared__ __align__(16) float sO_all[8][4 * M2E];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const long i = blockIdx.x * 8L + wid;
    if (i >= N) return;
    float *sO = sO_all[wid];
    const float4 *g4 = reinterpret_cast<const float4 *>(gA + i * 4 * M2E);
    for (int k = lane; k < M2E; k += 32) reinterpret_cast<float4 *>(sO)[k] = __ldg(g4 + k);
    __syncwarp();
    float v[7][4];
    float mx = 0.f;
#pragma unroll
    for (int j = 0; j < 7; ++j) {
        const int col = lane + 32 * j;
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            const float *o = sO + c * M2E;
            float x = 0.f;
            if (col < T2_O2) { if (col < M0) x = (o[col] + o[col + M0]) + (o[col + 2 * M0] + o[col + 3 * M0]); }
            else if (col < T2_O3) { const int f = col - T2_O2; if (f < M1) x = o[f] + o[f + M1]; }
            else if (col < COLS) { const int m = col - T2_O3; if (m < M2E) x = o[m]; }
            v[j][c] = x;
            mx = fmaxf(mx, fabsf(x));
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    int ex = 0;
    if (mx > 0.f) frexpf(mx, &ex);
    const float sc = ldexpf(1.f, -ex);          // max |g~| in [0.5, 1)
    if (lane == 0) gscale[i] = sc;
    uint4 *C = reinterpret_cast<uint4 *>(img + i * (long)GA_IMG_BYTES);
#pragma unroll
    for (int j = 0; j < 7; ++j) {
        const int col = lane + 32 * j;
        if (col < COLS) {
            uint32_t h01, l01, h23, l23;
            tc::split_h2(v[j][0] * sc, v[j][1] * sc, h01, l01);
            tc::split_h2(v[j][2] * sc, v[j][3] * sc, h23, l23);
            C[col] = make_uint4(h01, h23, l01, l23);
        }
    }
}

// hi parts -> 8 TMEM columns, lo parts -> two 16-byte chunks, 1 - t^2 -> dpk (fp16 pairs); t given in fp32
__device__ __forceinline__ void emit16(const float (&y)[16], uint32_t tm_dst, uint8_t *lo_row, int chunk, uint32_t *dpk) {
    uint32_t hi[8], lo[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        tc::split_h2(y[2 * q], y[2 * q + 1], hi[q], lo[q]);
        dpk[q] = tc::pack_h2(fmaf(-y[2 * q], y[2 * q], 1.f), fmaf(-y[2 * q + 1], y[2 * q + 1], 1.f));
    }
    tc::st8(tm_dst, hi);
    *reinterpret_cast<uint4 *>(lo_row + chunk * 2048) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
    *reinterpret_cast<uint4 *>(lo_row + (chunk + 1) * 2048) = make_uint4(lo[4], lo[5], lo[6], lo[7]);
}
__device__ __forceinline__ uint32_t hmul2(uint32_t a, uint32_t b) {
    __half2 r = __hmul2(*reinterpret_cast<const __half2 *>(&a), *reinterpret_cast<const __half2 *>(&b));
    return *reinterpret_cast<uint32_t *>(&r);
}
// 16 gradient columns (fp32 accumulators) times 1 - t^2 (fp16 pairs) -> fp16 pairs -> 8 TMEM columns (A operand of the
// next product: dz3 / dz2 overwrite the hi parts of t3 / t2, which are dead once dR^ = T g~ has been formed)
__device__ __forceinline__ void gradh16(const uint32_t (&g)[16], const uint32_t *dpk, uint32_t tm_dst) {
    uint32_t o[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        const float2 d = unpack_h2(dpk[q]);
        o[q] = tc::pack_h2(__uint_as_float(g[2 * q]) * d.x, __uint_as_float(g[2 * q + 1]) * d.y);
    }
    tc::st8(tm_dst, o);
}

constexpr int WGT = 128;       // threads per warpgroup: thread = row; every stage walks its two column halves h = 0, 1

// flag[a * T + b] = 1 if some 128-row tile of the (centre type a, neighbour type b) block spans more than T2_NSLOT atoms
__global__ void __launch_bounds__(256) k_bwd_classify(long N, int T, int ncell, const __grid_constant__ TypeTab tt,
                                                      const int *__restrict__ bin_start, const int *__restrict__ rowstart,
                                                      const int2 *__restrict__ rows_id, int *__restrict__ flag) {
    const int a = blockIdx.y / T, b = blockIdx.y % T;
    const int ts0 = bin_start[a * ncell], ts1 = bin_start[(a + 1) * ncell];
    if (ts0 == ts1) return;
    const int rs = rowstart[(long)b * (N + 1) + ts0], re = rowstart[(long)b * (N + 1) + ts1];
    const long rbase = N * (long)tt.off[b];
    const long tile = blockIdx.x * 256L + threadIdx.x;
    const long r0 = rs + tile * T2_ROWS;
    if (r0 >= re) return;
    const long rl = r0 + T2_ROWS - 1 < re ? r0 + T2_ROWS - 1 : re - 1;
    if ((__ldg(&rows_id[rbase + rl]).x - __ldg(&rows_id[rbase + r0]).x) / T2_NSLOT > 0) flag[blockIdx.y] = 1;
}

// The products with the per-atom gradient images take T2_NSLOT atoms per pass.  MULTI = false serves the (centre, neighbour)
// type blocks in which no 128-row tile spans more atoms than that (copper: >= 128 rows per atom): one pass, straight-line code.
// MULTI = true serves the other blocks (short neighbour blocks: water) with pass loops.  k_bwd_classify sets the per-block
// flag; each launch skips the blocks of the other kind.  Two kernels, not one with both paths: with both in one kernel
// the single-pass path loses 3.4 % at config 4 (register allocation), and a per-tile branch in its loop head 1.3 %.
template <int W, bool MULTI>
__global__ void __launch_bounds__(NWG * WGT, 1)
k_embed_bwd_tc2(long N, int T, int ncell, int Nm, const __grid_constant__ TypeTab tt, const EmbedNetTC2<W> *__restrict__ nets,
                const double *__restrict__ stdv, const int *__restrict__ bin_start, const int *__restrict__ rowstart,
                const float4 *__restrict__ rows_rh, const int2 *__restrict__ rows_id, const uint8_t *__restrict__ gimg,
                const float *__restrict__ gscale, float4 *__restrict__ rows_g, unsigned long long *__restrict__ row_counter,
                const int *__restrict__ multi_flag, long long *__restrict__ tdbg) {
    using SL = BwdSmem<W>;
    using LY = T2<W>;
    constexpr int M0 = LY::M0, K3 = LY::K3, COLS = LY::COLS, GA_IMG_BYTES = COLS * 16, TM_DR = SL::TM_DR, QC = SL::QCOPIES;
    constexpr int HW3 = K3 / 2 - (W == 25 ? 8 : 0);     // t3 columns handled per column half by full 16-column groups: 48 / 64
    constexpr int NU3 = HW3 / 16;                      // 16-column groups per half: 3 / 4
    constexpr bool PF3 = W == 25;                      // E3: software-pipelined TMEM loads (the same in E4 was measured 4 % slower)
    extern __shared__ __align__(1024) uint8_t smem[];
    __shared__ uint32_t tmem_base_s;
    const int tid = threadIdx.x;
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);      // warp-uniform: keeps the MMA operands in uniform registers
    const int wg = warp >> 2, t = tid & (WGT - 1), tw = t;
    const bool issuer_warp = (warp & 3) == 0;
    float *sw1 = reinterpret_cast<float *>(smem + SL::VEC), *sb1 = sw1 + 32;
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem + SL::BARS);
    uint8_t *wgs = smem + SL::WG0 + wg * SL::WG_BYTES;
    uint8_t *lo_row = wgs + SL::TLO + t * 16;
    const int *off = tt.off;

    if (tid == 0) {
        for (int k = 0; k < NWG; ++k) tc::mbar_init(&bars[k], 1);
        asm volatile("fence.mbarrier_init.release.cluster;");
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tc::smem_u32(&tmem_base_s)), "n"(512));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    for (int k = tw; k < SL::WG_BYTES / 16; k += WGT) reinterpret_cast<uint4 *>(wgs)[k] = make_uint4(0u, 0u, 0u, 0u);
    tc::fence_before();
    __syncthreads();
    tc::fence_after();
    const uint32_t tmem = __shfl_sync(0xffffffffu, tmem_base_s, 0) + wg * TM_WG;
    const uint32_t tm_lane = tmem + ((uint32_t)((warp & 3) * 32) << 16);
    const uint32_t sbase = tc::smem_u32(smem);
    const uint32_t s_tlo = tc::smem_u32(wgs + SL::TLO), s_rimg = tc::smem_u32(wgs + SL::RIMG);
    const uint32_t s_qimg = tc::smem_u32(wgs + SL::QIMG);
    // operand descriptors are built once; every MMA adds a compile-time offset
    const uint64_t d_tlo = tc::desc(s_tlo, 2048, 128), d_rimg = tc::desc(s_rimg, 2048, 128);
    const uint64_t d_qk = tc::desc(s_qimg, QC == 2 ? COLS * 16 : 0, 128), d_qmn = tc::desc(s_qimg, 128, QC * COLS * 16);
    const uint64_t d_w2 = tc::desc(sbase + SL::W2, 64 * 16, 128), d_w3 = tc::desc(sbase + SL::W3, K3 * 16, 128);
    const uint64_t d_ones = tc::desc(sbase + SL::ONES, 128, 0), d_bb2 = tc::desc(sbase + SL::BB2, 0, 128), d_bb3 = tc::desc(sbase + SL::BB3, 0, 128);
    (void)d_ones; (void)d_bb2; (void)d_bb3;
    const uint64_t d_w3t = tc::desc(sbase + SL::W3T, 96 * 16, 128), d_w2t = tc::desc(sbase + SL::W2T, 32 * 16, 128);
    uint64_t *bar = &bars[wg];
    uint32_t ph = 0;
    unsigned long long my_rows = 0;
#ifdef DP_BWD_TIMING
    const bool dbg_t = tdbg && blockIdx.x == 0 && tid == 0;
    long long tacc[20], tlast = clock64();
    for (int k = 0; k < 20; ++k) tacc[k] = 0;
#endif
    // zero the T hi region once: its padding columns are read as K of the products and must stay finite (zero)
    {
        uint32_t z8[8] = {0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u};
#pragma unroll
        for (int c = 0; c < 48 + K3 / 2; c += 8) tc::st8(tm_lane + TM_T + c, z8);
    }
    tc::wait_st();

    auto sync_issue = [&]() {          // make this warpgroup's operand writes visible to the tensor core, then meet
        tc::proxy_fence();
        tc::fence_before();
        tc::bar_sync(1 + wg, WGT);
    };
    auto sync_issue_tmem = [&]() {     // the same after an epilogue that wrote TMEM only: no shared-memory operand to publish, no proxy fence
        tc::fence_before();
        tc::bar_sync(1 + wg, WGT);
    };
    auto wait_mma = [&]() {
        tc::mbar_wait(bar, ph); ph ^= 1;
        tc::fence_after();
    };

    for (int a = 0; a < T; ++a) {
        const int ts0 = bin_start[a * ncell], ts1 = bin_start[(a + 1) * ncell];
        if (ts0 == ts1) continue;
        const float isd[4] = {(float)(1.0 / stdv[4 * a]), (float)(1.0 / stdv[4 * a + 1]), (float)(1.0 / stdv[4 * a + 2]),
                              (float)(1.0 / stdv[4 * a + 3])};
        for (int b = 0; b < T; ++b) {
            const long rbase = N * (long)off[b];
            const int rs = rowstart[(long)b * (N + 1) + ts0], re = rowstart[(long)b * (N + 1) + ts1];
            const int ntiles = (re - rs + T2_ROWS - 1) / T2_ROWS;
            if (ntiles == 0 || (multi_flag[a * T + b] != 0) != MULTI) continue;      // CTA-uniform
            __syncthreads();
            {   // stage the (a, b) net
                const EmbedNetTC2<W> *net = nets + (a * T + b);
                const uint4 *src = reinterpret_cast<const uint4 *>(&net->W2[0][0][0]);
                // W2, W3, W3T, W2T (and, with the ones step, the bias chunks) are contiguous in the struct and in shared memory
                constexpr int NW = (4 * 64 + 12 * K3 + (K3 / 8) * 96 + 8 * 32) + (LY::ONES_STEP ? 64 + K3 : 0);
                for (int k = tid; k < NW; k += NWG * WGT) reinterpret_cast<uint4 *>(smem + SL::W2)[k] = src[k];
                if (LY::ONES_STEP && tid < 16)
                    reinterpret_cast<uint4 *>(smem + SL::ONES)[tid] = tid < 8 ? make_uint4(0x3c003c00u, 0u, 0u, 0u) : make_uint4(0u, 0u, 0u, 0u);
                if (tid < 64) sw1[tid] = reinterpret_cast<const float *>(net)[tid];
            }
            tc::proxy_fence();
            __syncthreads();
            const int G = gridDim.x * NWG, gw = blockIdx.x * NWG + wg;
            const int tile0 = (int)((long)ntiles * gw / G), tile1 = (int)((long)ntiles * (gw + 1) / G);
            // Row data (R^, {atom, j}) is prefetched one tile ahead with cp.async into a two-stage buffer: stage = tile parity.
            auto prefetch_rows = [&](int first_row, int stage) {
                uint8_t *pf = wgs + SL::META + stage * 3072;
                if (first_row + t < re) {
                    cp_async16(tc::smem_u32(pf + t * 16), &rows_rh[rbase + first_row + t]);
                    cp_async8(tc::smem_u32(pf + 2048 + t * 8), &rows_id[rbase + first_row + t]);
                } else {
                    *reinterpret_cast<float4 *>(pf + t * 16) = make_float4(0.f, 0.f, 0.f, 0.f);
                    *reinterpret_cast<int2 *>(pf + 2048 + t * 8) = make_int2(-1, -1);
                }
            };
            if (tile0 < tile1) {
                prefetch_rows(rs + tile0 * T2_ROWS, tile0 & 1);
                cp_async_wait_all();
            }
            tc::bar_sync(1 + wg, WGT);
            for (int tile = tile0; tile < tile1; ++tile) {
                const int r0 = rs + tile * T2_ROWS;
                const int nrows = min(T2_ROWS, re - r0);
                const uint8_t *pf = wgs + SL::META + (tile & 1) * 3072;
                const float4 rh = *reinterpret_cast<const float4 *>(pf + t * 16);
                const int2 id = *reinterpret_cast<const int2 *>(pf + 2048 + t * 8);
                const int atom0 = reinterpret_cast<const int2 *>(pf + 2048)[0].x;
                const int atomL = reinterpret_cast<const int2 *>(pf + 2048)[nrows - 1].x;
                // next tile: lands before this tile's backward stage (cp.async.wait_all + warpgroup barrier there)
                if (tile + 1 < tile1) prefetch_rows(r0 + T2_ROWS, (tile + 1) & 1);
                const int atom = id.x;
                DP_TICK(17);
                // A tile that spans more than T2_NSLOT atoms runs several passes over the SAME recomputed tile: a row is masked
                // out of the passes of other atoms (its R image rows are zero), so the direct products dT = R^ g~ ACCUMULATE
                // over the passes, and dR^ = T g~ is read out per pass by the rows of that pass.
                const int npass = MULTI ? (atomL - atom0) / T2_NSLOT + 1 : 1;
                const int slot = atom & (T2_NSLOT - 1);
                                // operand images of one pass: R (A of the direct products) and the per-atom gradient images (async copies)
                auto setup_images = [&](int p0) {
                    const bool in = atom >= p0 && atom - p0 < T2_NSLOT;
                    uint32_t rh01, rl01, rh23, rl23;
                    tc::split_h2(rh.x, rh.y, rh01, rl01);
                    tc::split_h2(rh.z, rh.w, rh23, rl23);
                    const uint4 c0 = make_uint4(rh01, rh23, rh01, rh23), c1 = make_uint4(rl01, rl23, 0u, 0u), z4 = make_uint4(0u, 0u, 0u, 0u);
#pragma unroll
                    for (int s_ = 0; s_ < T2_NSLOT; ++s_) {
                        const bool mine = in && slot == s_;
                        *reinterpret_cast<uint4 *>(wgs + SL::RIMG + (2 * s_) * 2048 + t * 16) = mine ? c0 : z4;
                        *reinterpret_cast<uint4 *>(wgs + SL::RIMG + (2 * s_ + 1) * 2048 + t * 16) = mine ? c1 : z4;
                    }
                    for (int q = p0; q < p0 + T2_NSLOT && q <= atomL; ++q) {
                        const int s_ = q & (T2_NSLOT - 1);
                        const uint4 *C = reinterpret_cast<const uint4 *>(gimg + (long)q * GA_IMG_BYTES);
                        for (int k = tw; k < COLS; k += WGT) {
                            cp_async16(s_qimg + (QC * s_) * (COLS * 16) + k * 16, C + k);
                            if (QC == 2) cp_async16(s_qimg + (2 * s_ + 1) * (COLS * 16) + k * 16, C + k);
                        }
                    }
                };
                {
                    setup_images(atom0);          // first pass: the copies land under the recomputed forward
                    DP_TICK(18);
                    uint32_t d1p[2][8], d2p[2][16], d3p[2][HW3 / 2 + 2];   // 1 - t^2 per column half (fp16 pairs; only layer 3's are read back)
                    float d2f[2][32], d1f[2][16];     // layers 1-2 keep 1 - t^2 in fp32: fp16 here costs 2x in force error
                    DP_TICK(0);
                    // ---- E1: layer 1 on the ALUs; h = 0: t1[0..16), h = 1: t1[16..25), ones, padding ----
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        const float s = rh.x;
                        float y[16];
#pragma unroll
                        for (int e = 0; e < 16; ++e) {
                            const int ee = 16 * h + e;
                            if (ee < M0) y[e] = tc::tanh_approx(fmaf(s, sw1[ee], sb1[ee]));
                            else y[e] = (!LY::ONES_STEP && ee <= T2_ONE_LO) ? 1.f : 0.f;
                        }
                        emit16(y, tm_lane + TM_T + 8 * h, lo_row, 2 * h, d1p[h]);
#pragma unroll
                        for (int q = 0; q < 16; ++q) d1f[h][q] = fmaf(-y[q], y[q], 1.f);
                    }
                    tc::wait_st();
                    DP_TICK(1);
                    sync_issue();
                    if (issuer_warp && tc::elect_one()) {
                        tc::fence_after();
                        constexpr uint32_t id2 = tc::idesc(128, 64, false, false);
#pragma unroll
                        for (int ks = 0; ks < 2; ++ks) {
                            const uint64_t db = tc::desc_at(d_w2, ks * 2 * (64 * 16));
                            tc::mma_ts(tmem + TM_Z, tmem + TM_T + 8 * ks, db, id2, ks > 0);
                            tc::mma_ss(tmem + TM_Z, tc::desc_at(d_tlo, ks * 2 * 2048), db, id2, true);
                        }
                        if (LY::ONES_STEP) tc::mma_ss(tmem + TM_Z, d_ones, d_bb2, id2, true);
                        tc::commit(bar);
                    }
                    DP_TICK(2);
                    wait_mma();
                    DP_TICK(3);
                    // ---- E2: h = 0: t2[0..32), h = 1: t2[32..50)  (pipelining these TMEM loads as in E3 was measured 4 % slower) ----
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        uint8_t *img = lo_row + (T2_O2 / 8) * 2048;
                        uint32_t z0[16], z1[16];
                        const bool full = h == 0 || W != 25;        // this half has 32 real columns (W = 25, h = 1: 18)
                        tc::ld16(tm_lane + TM_Z + 32 * h, z0);
                        if (full) tc::ld16(tm_lane + TM_Z + 32 * h + 16, z1);
                        else tc::ld2(tm_lane + TM_Z + 48, reinterpret_cast<uint32_t (&)[2]>(z1));
                        tc::wait_ld();
                        act16(z0, tm_lane + TM_T + 16 + 16 * h, img, 4 * h, d2p[h]);
#pragma unroll
                        for (int q = 0; q < 16; ++q) { const float tt = tc::tanh_approx(__uint_as_float(z0[q])); d2f[h][q] = fmaf(-tt, tt, 1.f); }
#pragma unroll
                        for (int q = 0; q < 16; ++q) { const float tt = tc::tanh_approx(__uint_as_float(z1[q & (full ? 15 : 1)])); d2f[h][16 + q] = fmaf(-tt, tt, 1.f); }
                        if (full) {
                            act16(z1, tm_lane + TM_T + 24 + 16 * h, img, 4 * h + 2, d2p[h] + 8);
                        } else {
                            const float x = tc::tanh_approx(__uint_as_float(z1[0])), y = tc::tanh_approx(__uint_as_float(z1[1]));
                            uint32_t hi, lo;
                            tc::split_h2(x, y, hi, lo);
                            d2p[h][8] = tc::pack_h2(fmaf(-x, x, 1.f), fmaf(-y, y, 1.f));
                            tc::st4(tm_lane + TM_T + 40, hi, 0u, 0u, 0u);
                            *reinterpret_cast<uint4 *>(img + 6 * 2048) = make_uint4(lo, 0u, 0u, 0u);
                        }
                    }
                    tc::wait_st();
                    DP_TICK(4);
                    sync_issue();
                    if (issuer_warp && tc::elect_one()) {
                        tc::fence_after();
                        constexpr uint32_t id3 = tc::idesc(128, K3, false, false);
#pragma unroll
                        for (int ks = 0; ks < 6; ++ks) {
                            const int acol = ks < 4 ? 16 + 8 * ks : 8 * (ks - 4);              // TMEM column of the hi part
                            const int achunk = ks < 4 ? T2_O2 / 8 + 2 * ks : 2 * (ks - 4);     // chunk of the lo part
                            const uint64_t db = tc::desc_at(d_w3, ks * 2 * (K3 * 16));
                            tc::mma_ts(tmem + TM_Z, tmem + TM_T + acol, db, id3, ks > 0);
                            tc::mma_ss(tmem + TM_Z, tc::desc_at(d_tlo, achunk * 2048), db, id3, true);
                        }
                        if (LY::ONES_STEP) tc::mma_ss(tmem + TM_Z, d_ones, d_bb3, id3, true);
                        tc::commit(bar);
                    }
                    DP_TICK(5);
                    wait_mma();
                    DP_TICK(6);
                    // ---- E3: h = 0: t3[0..48), h = 1: t3[48..100) ----
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        uint8_t *img = lo_row + (T2_O3 / 8 + (HW3 / 8) * h) * 2048;
                        if (PF3) {   // TMEM loads one group ahead of the tanh / split work (measured: -3.8 % at W = 25, +1 % at W = 32)
                            uint32_t zb[2][16];
                            tc::ld16(tm_lane + TM_Z + HW3 * h, zb[0]);
#pragma unroll
                            for (int u = 0; u < NU3; ++u) {
                                tc::wait_ld();
                                if (u + 1 < NU3) tc::ld16(tm_lane + TM_Z + HW3 * h + 16 * (u + 1), zb[(u + 1) & 1]);
                                act16(zb[u & 1], tm_lane + TM_T + 48 + (HW3 / 2) * h + 8 * u, img, 2 * u, d3p[h] + 8 * u);
                            }
                        } else {
#pragma unroll
                        for (int u = 0; u < NU3; ++u) {
                            uint32_t z0[16];
                            tc::ld16(tm_lane + TM_Z + HW3 * h + 16 * u, z0);
                            tc::wait_ld();
                            act16(z0, tm_lane + TM_T + 48 + (HW3 / 2) * h + 8 * u, img, 2 * u, d3p[h] + 8 * u);
                        }
                        }
                        if (W == 25 && h == 1) {
                            uint32_t z3[4];
                            tc::ld4(tm_lane + TM_Z + 96, z3);
                            tc::wait_ld();
                            const float x0 = tc::tanh_approx(__uint_as_float(z3[0])), x1 = tc::tanh_approx(__uint_as_float(z3[1]));
                            const float x2 = tc::tanh_approx(__uint_as_float(z3[2])), x3 = tc::tanh_approx(__uint_as_float(z3[3]));
                            uint32_t h0, l0, h1, l1;
                            tc::split_h2(x0, x1, h0, l0); tc::split_h2(x2, x3, h1, l1);
                            d3p[h][24] = tc::pack_h2(fmaf(-x0, x0, 1.f), fmaf(-x1, x1, 1.f));
                            d3p[h][25] = tc::pack_h2(fmaf(-x2, x2, 1.f), fmaf(-x3, x3, 1.f));
                            tc::st4(tm_lane + TM_T + 96, h0, h1, 0u, 0u);
                            *reinterpret_cast<uint4 *>(img + 6 * 2048) = make_uint4(l0, l1, 0u, 0u);
                        }
                    }
                    tc::wait_st();
                    // ---- backward ----
                    {
                    const int NP = MULTI ? npass : 1;
                    float gsc = 1.f;
                    float dR[4] = {0.f, 0.f, 0.f, 0.f};
                    for (int pi = 0; pi < NP; ++pi) {
                        const int p0 = atom0 + pi * T2_NSLOT;
                        const bool in = atom >= p0 && atom - p0 < T2_NSLOT;
                        if (pi > 0) setup_images(p0);        // the products of the previous pass are complete (wait_mma below)
                        cp_async_wait_all();
                        DP_TICK(7);
                        sync_issue();
                        if (issuer_warp && tc::elect_one()) {
                            tc::fence_after();
                            constexpr uint32_t idr = tc::idesc(128, 8 * T2_NSLOT, false, true);
                            // dR^ = T g~.  Single pass: only the t3 columns of T must be read before E4 overwrites them with dz3;
                            // the t1 / t2 part (12 small MMAs) is issued behind the commit, off the E3 -> E4 critical path, and is
                            // covered by the next commit (E5 is the first stage that overwrites t2); dR^ is read in E6
                            constexpr int KS_A = MULTI ? 0 : T2_O3 / 16;
#pragma unroll
                            for (int ks = KS_A; ks < COLS / 16; ++ks) {
                                const uint64_t db = tc::desc_at(d_qmn, ks * 256);
                                tc::mma_ts(tmem + TM_DR, tmem + TM_T + 8 * ks, db, idr, ks > KS_A);
                                tc::mma_ss(tmem + TM_DR, tc::desc_at(d_tlo, ks * 2 * 2048), db, idr, true);
                            }
                            constexpr uint32_t idg = tc::idesc(128, K3, false, false);
#pragma unroll
                            for (int ks = 0; ks < T2_NSLOT; ++ks)      // dT3 accumulates over the passes
                                tc::mma_ss(tmem + TM_Z, tc::desc_at(d_rimg, ks * 2 * 2048), tc::desc_at(d_qk, T2_O3 * 16 + ks * QC * (COLS * 16)), idg, pi > 0 || ks > 0);
                            tc::commit(bar);
#pragma unroll
                            for (int ks = 0; ks < KS_A; ++ks) {
                                const uint64_t db = tc::desc_at(d_qmn, ks * 256);
                                tc::mma_ts(tmem + TM_DR, tmem + TM_T + 8 * ks, db, idr, true);
                                tc::mma_ss(tmem + TM_DR, tc::desc_at(d_tlo, ks * 2 * 2048), db, idr, true);
                            }
                        }
                        if (in) gsc = __ldg(&gscale[atom]);
                        DP_TICK(8);
                        wait_mma();
                        if (MULTI) {      // dR^ of the rows of this pass (a single pass reads it in E6)
                            uint32_t v[16];
                            tc::ld16(tm_lane + TM_DR, v);
                            tc::wait_ld();
                            if (in) {
#pragma unroll
                                for (int c = 0; c < 4; ++c)
                                    dR[c] = slot ? __uint_as_float(v[8 + c]) + __uint_as_float(v[12 + c]) : __uint_as_float(v[c]) + __uint_as_float(v[4 + c]);
                            }
                        }
                    }
                    DP_TICK(9);
                    // ---- E4: dz3 = dT3 (1 - t3^2) -> TMEM, over the hi parts of t3 ----
                    {
#pragma unroll
                        for (int h = 0; h < 2; ++h) {
#pragma unroll
                            for (int u = 0; u < NU3; ++u) {
                                uint32_t g0[16];
                                tc::ld16(tm_lane + TM_Z + HW3 * h + 16 * u, g0);
                                tc::wait_ld();
                                gradh16(g0, d3p[h] + 8 * u, tm_lane + TM_T + 48 + (HW3 / 2) * h + 8 * u);
                            }
                            if (W == 25 && h == 1) {
                                uint32_t g3[4];
                                tc::ld4(tm_lane + TM_Z + 96, g3);
                                tc::wait_ld();
                                const float2 da = unpack_h2(d3p[h][24]), db = unpack_h2(d3p[h][25]);
                                tc::st4(tm_lane + TM_T + 96, tc::pack_h2(__uint_as_float(g3[0]) * da.x, __uint_as_float(g3[1]) * da.y),
                                        tc::pack_h2(__uint_as_float(g3[2]) * db.x, __uint_as_float(g3[3]) * db.y), 0u, 0u);
                            }
                        }
                        tc::wait_st();
                    }
                    DP_TICK(10);
                    // direct parts dT2, dT1 of the other passes first (their images are reloaded; the last pass's are still
                    // resident and go last, together with the products of dz3)
                    for (int pi = 0; pi < NP; ++pi) {
                        const bool last = pi == NP - 1;
                        if (!last) { setup_images(atom0 + pi * T2_NSLOT); cp_async_wait_all(); }
                        else if (MULTI) { setup_images(atom0 + pi * T2_NSLOT); cp_async_wait_all(); }
                        if (MULTI) sync_issue(); else sync_issue_tmem();
                        if (issuer_warp && tc::elect_one()) {
                            tc::fence_after();
                            constexpr uint32_t idy2 = tc::idesc(128, 64, false, false);
                            constexpr uint32_t idy1 = tc::idesc(128, 32, false, false);
#pragma unroll
                            for (int ks = 0; ks < T2_NSLOT; ++ks)      // direct part dT2 -> accumulator columns [32,96)
                                tc::mma_ss(tmem + TM_Z + 32, tc::desc_at(d_rimg, ks * 2 * 2048), tc::desc_at(d_qk, T2_O2 * 16 + ks * QC * (COLS * 16)), idy2, pi > 0 || ks > 0);
                            if (!last) {
#pragma unroll
                                for (int ks = 0; ks < T2_NSLOT; ++ks)  // direct part dT1 -> accumulator columns [0,32)
                                    tc::mma_ss(tmem + TM_Z, tc::desc_at(d_rimg, ks * 2 * 2048), tc::desc_at(d_qk, ks * QC * (COLS * 16)), idy1, pi > 0 || ks > 0);
                                tc::commit(bar);
                            } else {
                                // dy2 first (the next stage needs it) ...
#pragma unroll
                                for (int ks = 0; ks < K3 / 16; ++ks)
                                    tc::mma_ts(tmem + TM_Z + 32, tmem + TM_T + 48 + 8 * ks, tc::desc_at(d_w3t, 32 * 16 + ks * 2 * (96 * 16)), idy2, true);
                                tc::commit(bar);
                                // ... then the part of dy1 that does not depend on dz2 (waited for with the last stage)
#pragma unroll
                                for (int ks = 0; ks < T2_NSLOT; ++ks)
                                    tc::mma_ss(tmem + TM_Z, tc::desc_at(d_rimg, ks * 2 * 2048), tc::desc_at(d_qk, ks * QC * (COLS * 16)), idy1, pi > 0 || ks > 0);
#pragma unroll
                                for (int ks = 0; ks < K3 / 16; ++ks)
                                    tc::mma_ts(tmem + TM_Z, tmem + TM_T + 48 + 8 * ks, tc::desc_at(d_w3t, ks * 2 * (96 * 16)), idy1, true);
                            }
                        }
                        DP_TICK(11);
                        wait_mma();
                    }
                    DP_TICK(12);
                    // ---- E5: dz2 = dy2 (1 - t2^2) -> TMEM, over the hi parts of t2 ----
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        uint32_t g0[16], g1[16];
                        const bool full = h == 0 || W != 25;
                        tc::ld16(tm_lane + TM_Z + 32 + 32 * h, g0);
                        if (full) tc::ld16(tm_lane + TM_Z + 48 + 32 * h, g1);
                        else tc::ld2(tm_lane + TM_Z + 80, reinterpret_cast<uint32_t (&)[2]>(g1));
                        tc::wait_ld();
                        uint32_t o[8];
#pragma unroll
                        for (int q = 0; q < 8; ++q) o[q] = tc::pack_h2(__uint_as_float(g0[2 * q]) * d2f[h][2 * q], __uint_as_float(g0[2 * q + 1]) * d2f[h][2 * q + 1]);
                        tc::st8(tm_lane + TM_T + 16 + 16 * h, o);
                        if (full) {
#pragma unroll
                            for (int q = 0; q < 8; ++q) o[q] = tc::pack_h2(__uint_as_float(g1[2 * q]) * d2f[h][16 + 2 * q], __uint_as_float(g1[2 * q + 1]) * d2f[h][16 + 2 * q + 1]);
                            tc::st8(tm_lane + TM_T + 24 + 16 * h, o);
                        } else {
                            tc::st4(tm_lane + TM_T + 40, tc::pack_h2(__uint_as_float(g1[0]) * d2f[h][16], __uint_as_float(g1[1]) * d2f[h][17]), 0u, 0u, 0u);
                        }
                    }
                    tc::wait_st();
                    DP_TICK(13);
                    sync_issue_tmem();
                    if (issuer_warp && tc::elect_one()) {
                        tc::fence_after();
                        constexpr uint32_t id1 = tc::idesc(128, 32, false, false);
#pragma unroll
                        for (int ks = 0; ks < T2_K2 / 16; ++ks)
                            tc::mma_ts(tmem + TM_Z, tmem + TM_T + 16 + 8 * ks, tc::desc_at(d_w2t, ks * 2 * (32 * 16)), id1, true);
                        tc::commit(bar);
                    }
                    DP_TICK(14);
                    wait_mma();
                    DP_TICK(15);
                    // ---- E6: ds^ = sum_e dy1 (1 - t1^2) w1; gradient of the environment row; S8 + S9 in fp64 ----
                    {
                        float ds = 0.f;
                        if (!MULTI) {      // dR^ is complete only now (its t1 / t2 part was issued behind the dT3 commit)
                            uint32_t v[16];
                            tc::ld16(tm_lane + TM_DR, v);
                            tc::wait_ld();
#pragma unroll
                            for (int c = 0; c < 4; ++c)
                                dR[c] = slot ? __uint_as_float(v[8 + c]) + __uint_as_float(v[12 + c]) : __uint_as_float(v[c]) + __uint_as_float(v[4 + c]);
                        }
#pragma unroll
                        for (int h = 0; h < 2; ++h) {
                            uint32_t g0[16];
                            tc::ld16(tm_lane + TM_Z + 16 * h, g0);
                            tc::wait_ld();
#pragma unroll
                            for (int q = 0; q < 8; ++q) {
                                const float2 d = make_float2(d1f[h][2 * q], d1f[h][2 * q + 1]);
                                if (16 * h + 2 * q < M0) ds = fmaf(__uint_as_float(g0[2 * q]) * d.x, sw1[16 * h + 2 * q], ds);
                                if (16 * h + 2 * q + 1 < M0) ds = fmaf(__uint_as_float(g0[2 * q + 1]) * d.y, sw1[16 * h + 2 * q + 1], ds);
                            }
                        }
                        // gradient of E with respect to this row of the environment matrix R~ (S8 + S9 run in k_prod_force_virial)
                        if (atom >= 0) {
                            const float osc = 1.0f / ((float)Nm * gsc);
                            rows_g[rbase + r0 + t] = make_float4((dR[0] + ds) * osc * isd[0], dR[1] * osc * isd[1], dR[2] * osc * isd[2],
                                                                 dR[3] * osc * isd[3]);
                        }
                    }
                    }
                    DP_TICK(16);
                }
                if (tw == 0) my_rows += (unsigned long long)nrows;
            }
        }
    }
    tc::fence_before();
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base_s), "n"(512));
    if (tw == 0 && my_rows) atomicAdd(row_counter, my_rows);
#ifdef DP_BWD_TIMING
    if (dbg_t) for (int k = 0; k < 20; ++k) tdbg[k] = tacc[k];
#endif
}


// S8 + S9 (ProdForce, ProdViral): one thread per compact neighbour row.  g = dE/dR~ of the row (fp32, from
// the backward kernel); the geometry derivative, the force scatter and the virial are fp64 (configs 3-4).
__global__ void __launch_bounds__(256)
k_prod_force_virial(long N, int T, const __grid_constant__ TypeTab tt, EnvParams ep, const int *__restrict__ rowstart,
                    const int2 *__restrict__ rows_id, const float4 *__restrict__ rows_g, const double *__restrict__ xs,
                    double *__restrict__ fsorted, float4 *__restrict__ fj32, double *__restrict__ virial) {
    const int lane = threadIdx.x & 31;
    const int *sel = tt.sel, *off = tt.off;
    const double hx = 0.5 * ep.L[0], hy = 0.5 * ep.L[1], hz = 0.5 * ep.L[2];
    double vir[9];
#pragma unroll
    for (int k = 0; k < 9; ++k) vir[k] = 0.0;
    for (int b = 0; b < T; ++b) {
        const long rbase = N * (long)off[b];
        const long nrows = rowstart[(long)b * (N + 1) + N];
        (void)sel;
        // whole warps walk the rows so that the warp-level reduction below is always convergent
        for (long r0 = (blockIdx.x * (long)blockDim.x + threadIdx.x) - lane; r0 < nrows; r0 += (long)gridDim.x * blockDim.x) {
            const long row = r0 + lane;
            int2 id = make_int2(-1, -1);
            if (row < nrows) id = __ldg(&rows_id[rbase + row]);
            const bool real = id.y >= 0;
            const int atom = id.x;
            double gk[3] = {0.0, 0.0, 0.0};
            if (real) {
                const float4 g = __ldg(&rows_g[rbase + row]);
                const int j = id.y;
                const double dx = min_image(xs[3 * (long)j] - xs[3 * (long)atom], ep.L[0], hx);
                const double dy = min_image(xs[3 * (long)j + 1] - xs[3 * (long)atom + 1], ep.L[1], hy);
                const double dz = min_image(xs[3 * (long)j + 2] - xs[3 * (long)atom + 2], ep.L[2], hz);
                const double r2 = dx * dx + dy * dy + dz * dz;
                const double ir = rsqrt(r2), r = r2 * ir;
                double w = 1.0, dw = 0.0;
                if (r >= ep.rc_smth) {
                    if (r < ep.rc) {
                        const double u = (r - ep.rc_smth) * ep.inv_range;
                        w = u * u * u * (-6.0 * u * u + 15.0 * u - 10.0) + 1.0;
                        dw = -30.0 * u * u * (u - 1.0) * (u - 1.0) * ep.inv_range;
                    } else {
                        w = 0.0;
                    }
                }
                const double s = w * ir;
                const double sp = dw * ir - w * ir * ir;          // ds/dr
                const double g0_ = g.x, g1_ = g.y, g2_ = g.z, g3_ = g.w;
                const double gd = g1_ * dx + g2_ * dy + g3_ * dz;
                const double coef = (sp * ir - s * ir * ir) * ir;
                const double c0 = g0_ * sp * ir + coef * gd, c1 = s * ir;
                gk[0] = c0 * dx + c1 * g1_;
                gk[1] = c0 * dy + c1 * g2_;
                gk[2] = c0 * dz + c1 * g3_;
#pragma unroll
                for (int bb = 0; bb < 3 && !fj32; ++bb) atomicAdd(&fsorted[3 * (long)j + bb], -gk[bb]);
                // the neighbour's share: ONE 16-byte fp32 vector reduction per row instead of three fp64 ones (the L2 reduction
                // rate bounds this kernel); k_force_add32 adds the fp32 sums to the fp64 forces afterwards
                if (fj32)
                    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(fj32 + j), "f"((float)-gk[0]), "f"((float)-gk[1]),
                                 "f"((float)-gk[2]), "f"(0.f) : "memory");
                vir[0] -= dx * gk[0]; vir[1] -= dx * gk[1]; vir[2] -= dx * gk[2];
                vir[3] -= dy * gk[0]; vir[4] -= dy * gk[1]; vir[5] -= dy * gk[2];
                vir[6] -= dz * gk[0]; vir[7] -= dz * gk[1]; vir[8] -= dz * gk[2];
            }
            // centre atom: one atomic per warp when all its real rows belong to the same atom
            const unsigned rm = __ballot_sync(0xffffffffu, real);
            if (rm) {
                const int a0 = __shfl_sync(0xffffffffu, atom, __ffs(rm) - 1);
                if (__all_sync(0xffffffffu, !real || atom == a0)) {
#pragma unroll
                    for (int bb = 0; bb < 3; ++bb) {
                        double v = gk[bb];
#pragma unroll
                        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
                        if (lane == 0) atomicAdd(&fsorted[3 * (long)a0 + bb], v);
                    }
                } else if (real) {
#pragma unroll
                    for (int bb = 0; bb < 3; ++bb) atomicAdd(&fsorted[3 * (long)atom + bb], gk[bb]);
                }
            }
        }
    }
    __shared__ double red[8][9];
#pragma unroll
    for (int k = 0; k < 9; ++k) {
        double v = vir[k];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) red[threadIdx.x >> 5][k] = v;
    }
    __syncthreads();
    if (threadIdx.x < 9) {
        double v = 0.0;
        for (int w = 0; w < 8; ++w) v += red[w][threadIdx.x];
        if (v != 0.0) atomicAdd(&virial[threadIdx.x], v);
    }
}

// fsorted[k] += fj32[k] (the neighbour shares accumulated in fp32 by k_prod_force_virial)
__global__ void __launch_bounds__(256) k_force_add32(long n, const float4 *__restrict__ fj32, double *__restrict__ fsorted) {
    const long k = blockIdx.x * 256L + threadIdx.x;
    if (k >= n) return;
    const float4 v = fj32[k];
    fsorted[3 * k] += (double)v.x;
    fsorted[3 * k + 1] += (double)v.y;
    fsorted[3 * k + 2] += (double)v.z;
}

}  // namespace

// S8 + S9 from the per-row gradients in rows_g (the tail of the MIX-16 backward and of the wide-network backward, wide.cu)
cudaError_t launch_prod_force_virial(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st) {
    const TypeTab tt = make_typetab(m);
    EnvParams ep;
    ep.rc = m->rc; ep.rc_smth = m->rc_smth; ep.inv_range = 1.0 / (m->rc - m->rc_smth);
    ep.L[0] = g.L[0]; ep.L[1] = g.L[1]; ep.L[2] = g.L[2];
    float4 *fj32 = (float4 *)(ws + L.fj32);
    cudaMemsetAsync(fj32, 0, sizeof(float4) * (size_t)g.cap_ext, st);
    k_prod_force_virial<<<m->num_sms * 8, 256, 0, st>>>(N, m->T, tt, ep, (int *)(ws + L.rowstart),
                                                        (const int2 *)(ws + L.rows_id), (const float4 *)(ws + L.rows_g),
                                                        (double *)(ws + L.xs), (double *)(ws + L.fsorted), fj32, (double *)(ws + L.virial));
    k_force_add32<<<(unsigned)((g.cap_ext + 255) / 256), 256, 0, st>>>(g.cap_ext, fj32, (double *)(ws + L.fsorted));
    return cudaGetLastError();
}

template <int W>
static cudaError_t launch_bwd_w(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st) {
    DP_SMEM_OPTIN((k_embed_bwd_tc2<W, false>), BwdSmem<W>::TOTAL);
    DP_SMEM_OPTIN((k_embed_bwd_tc2<W, true>), BwdSmem<W>::TOTAL);
    const TypeTab tt = make_typetab(m);
    EnvParams ep;
    ep.rc = m->rc; ep.rc_smth = m->rc_smth; ep.inv_range = 1.0 / (m->rc - m->rc_smth);
    ep.L[0] = g.L[0]; ep.L[1] = g.L[1]; ep.L[2] = g.L[2];
    // the last fitting GEMM left gA itself in the gD buffer (fit_tc.cu MODE 6)
    k_gA_fold<W><<<(unsigned)((N + 7) / 8), 256, 0, st>>>(N, (const float *)(ws + L.gD), (uint8_t *)(ws + L.gAf), (float *)(ws + L.gscale));
    long long *tdbg = nullptr;
#ifdef DP_BWD_TIMING
    static long long *tbuf = nullptr;
    if (!tbuf) cudaMalloc(&tbuf, 20 * sizeof(long long));
    tdbg = tbuf;
#endif
    if (m->profile) cudaEventRecord(m->ev[6], st);
    int *multi_flag = (int *)(ws + L.multi_cnt);
    cudaMemsetAsync(multi_flag, 0, sizeof(int) * DP_MAX_TYPES * DP_MAX_TYPES, st);
    {
        int maxsel = 0;
        for (int b = 0; b < m->T; ++b) maxsel = m->sel[b] > maxsel ? m->sel[b] : maxsel;
        const long maxtiles = (N * (long)maxsel + T2_ROWS - 1) / T2_ROWS + 1;
        k_bwd_classify<<<dim3((unsigned)((maxtiles + 255) / 256), (unsigned)(m->T * m->T)), 256, 0, st>>>(
            N, m->T, g.ncell, tt, (int *)(ws + L.bin_start), (int *)(ws + L.rowstart), (const int2 *)(ws + L.rows_id), multi_flag);
    }
    k_embed_bwd_tc2<W, false><<<m->num_sms, NWG * WGT, BwdSmem<W>::TOTAL, st>>>(
        N, m->T, g.ncell, m->Nm, tt, (const EmbedNetTC2<W> *)m->embed_tc2_dev, m->std_dev, (int *)(ws + L.bin_start),
        (int *)(ws + L.rowstart), (const float4 *)(ws + L.rows_rh), (const int2 *)(ws + L.rows_id),
        (const uint8_t *)(ws + L.gAf), (const float *)(ws + L.gscale), (float4 *)(ws + L.rows_g),
        (unsigned long long *)(ws + L.status + 16), multi_flag, tdbg);
    // the blocks with tiles that span more than T2_NSLOT atoms (none for copper: the launch finds no block of its kind)
    k_embed_bwd_tc2<W, true><<<m->num_sms, NWG * WGT, BwdSmem<W>::TOTAL, st>>>(
        N, m->T, g.ncell, m->Nm, tt, (const EmbedNetTC2<W> *)m->embed_tc2_dev, m->std_dev, (int *)(ws + L.bin_start),
        (int *)(ws + L.rowstart), (const float4 *)(ws + L.rows_rh), (const int2 *)(ws + L.rows_id),
        (const uint8_t *)(ws + L.gAf), (const float *)(ws + L.gscale), (float4 *)(ws + L.rows_g),
        (unsigned long long *)(ws + L.status + 16), multi_flag, nullptr);
    if (m->profile) cudaEventRecord(m->ev[7], st);
    {
        const cudaError_t e2 = launch_prod_force_virial(m, N, g, ws, L, st);
        if (e2 != cudaSuccess) return e2;
    }
#ifdef DP_BWD_TIMING
    if (tdbg) {
        cudaStreamSynchronize(st);
        long long h[20];
        cudaMemcpy(h, tdbg, sizeof(h), cudaMemcpyDeviceToHost);
        long long tot = 0;
        for (int k = 0; k < 20; ++k) tot += h[k];
        fprintf(stderr, "bwd phase cycles (WG0 of CTA 0), total %lld:", tot);
        for (int k = 0; k < 20; ++k) fprintf(stderr, " %d:%.1f%%", k, 100.0 * h[k] / (double)tot);
        fprintf(stderr, "\n");
    }
#endif
    return cudaGetLastError();
}

cudaError_t launch_embed_bwd_tc2(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st) {
    return m->m0 == 32 ? launch_bwd_w<32>(m, N, g, ws, L, st) : launch_bwd_w<25>(m, N, g, ws, L, st);
}
