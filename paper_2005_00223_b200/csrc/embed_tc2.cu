// S3 + S4 + S5 (forward) on tcgen05 tensor cores, MIX-16, second generation (see embed_tc2.cuh for the layout).
//
// One warpgroup = one 128-row tile in flight (thread = row = TMEM lane); three warpgroups per CTA, one CTA per SM.
// Per tile:  E1  t1 = tanh(s^ w1 + b1)            (ALUs, K = 1 as in PAPER.md:125)        -> T image (fp16)
//            L2  z2 = [t1 | 1] . [W2 ; b2]         tcgen05.mma 128 x 64 x 32             -> TMEM
//            E2  t2 = tanh(z2)                                                            -> T image
//            L3  z3 = [t2 | t1 | 1] . [W3 ; W3fold ; b3]   tcgen05.mma 128 x 112 x 96    -> TMEM
//            E3  t3 = tanh(z3)                                                            -> T image
//            C   DA[feature][slot, c] += T^T . R^w   two tcgen05.mma 128 x 16 x 128, accumulated in TMEM ACROSS tiles
//            flush (once per atom): fold the t1 / t2 / t3 lanes into A_i[c][m] and add to global memory.
// The embedding matrix G and the environment matrix never reach HBM.
#include "embed_tc2.cuh"
#include "tc_common.cuh"

namespace {

constexpr int NWG = 3;                         // warpgroups (tiles in flight) per CTA
constexpr int TM_Z = 0;

// TMEM columns per warpgroup: Z [0,K3) D1 [K3,K3+16) D2 [K3+16,K3+32)
template <int W>
struct FwdSmem {
    using L = T2<W>;
    static constexpr int W2 = 0;                                   // 4 chunks x 64 x 16 B
    static constexpr int W3 = W2 + 4 * 64 * 16;                    // 12 chunks x K3 x 16 B
    static constexpr int BB2 = W3 + 12 * L::K3 * 16;               // ONES_STEP: bias images (one K chunk each) and the ones image
    static constexpr int BB3 = BB2 + (L::ONES_STEP ? 64 * 16 : 0);
    static constexpr int ONES = BB3 + (L::ONES_STEP ? L::K3 * 16 : 0);   // two 128-byte core matrices: {1,1,0..} rows, zeros
    static constexpr int VEC = ONES + (L::ONES_STEP ? 256 : 0);    // w1[32] b1[32]
    static constexpr int BARS = VEC + 256;
    static constexpr int WG0 = ((BARS + 64 + 1023) / 1024) * 1024;
    // per warpgroup
    static constexpr int TIMG = 0;                                 // CHUNKS x 2 KB
    static constexpr int RIMG = TIMG + L::CHUNKS * 2048;           // T2_NSLOT chunks x 2 KB
    static constexpr int SCR = RIMG + T2_NSLOT * 2048;             // float [4][COLS]
    static constexpr int META = SCR + (W == 25 ? 8 : 4) * L::COLS * 4;
    static constexpr int WG_BYTES = ((META + 64 + 127) / 128) * 128;
    // the second contraction MMA reads T-image chunks 16..31 (lanes >= COLS - 128 of its result are never used): keep that
    // window inside the allocation
    static constexpr int SLACK = W == 25 ? 2048 : 1024;
    static constexpr int TOTAL = WG0 + NWG * WG_BYTES + SLACK;
    static_assert(32 * 2048 <= WG_BYTES + SLACK, "contraction over-read must stay inside the allocation");
    // (the 1024-byte alignment of the dynamic array behind the static tmem_base_s costs up to 1 KB of the 227 KB)
    static_assert(TOTAL + 1024 <= 227 * 1024, "shared memory budget");
    static constexpr int TM_D1 = L::K3, TM_D2 = L::K3 + 16, TM_WG = L::K3 + 32;
    static_assert(NWG * TM_WG <= 512, "TMEM budget");
};

// tanh of 16 accumulator columns -> two 16-byte chunks of the T image
__device__ __forceinline__ void tanh16_store(const uint32_t (&z)[16], uint8_t *img_row, int chunk) {
    uint4 a, b;
    a.x = tc::pack_h2(tc::tanh_approx(__uint_as_float(z[0])), tc::tanh_approx(__uint_as_float(z[1])));
    a.y = tc::pack_h2(tc::tanh_approx(__uint_as_float(z[2])), tc::tanh_approx(__uint_as_float(z[3])));
    a.z = tc::pack_h2(tc::tanh_approx(__uint_as_float(z[4])), tc::tanh_approx(__uint_as_float(z[5])));
    a.w = tc::pack_h2(tc::tanh_approx(__uint_as_float(z[6])), tc::tanh_approx(__uint_as_float(z[7])));
    b.x = tc::pack_h2(tc::tanh_approx(__uint_as_float(z[8])), tc::tanh_approx(__uint_as_float(z[9])));
    b.y = tc::pack_h2(tc::tanh_approx(__uint_as_float(z[10])), tc::tanh_approx(__uint_as_float(z[11])));
    b.z = tc::pack_h2(tc::tanh_approx(__uint_as_float(z[12])), tc::tanh_approx(__uint_as_float(z[13])));
    b.w = tc::pack_h2(tc::tanh_approx(__uint_as_float(z[14])), tc::tanh_approx(__uint_as_float(z[15])));
    *reinterpret_cast<uint4 *>(img_row + chunk * 2048) = a;
    *reinterpret_cast<uint4 *>(img_row + (chunk + 1) * 2048) = b;
}

template <int W>
__global__ void __launch_bounds__(NWG * 128, 1)
k_embed_fwd_tc2(long N, int T, int ncell, int Nm, const __grid_constant__ TypeTab tt, const EmbedNetTC2<W> *__restrict__ nets,
                const int *__restrict__ bin_start, const int *__restrict__ rowstart, const float4 *__restrict__ rows_rh,
                const int2 *__restrict__ rows_id, float *__restrict__ Aout, unsigned long long *__restrict__ row_counter) {
    using SL = FwdSmem<W>;
    using LY = T2<W>;
    constexpr int M0 = LY::M0, M1 = LY::M1, M2E = LY::M2E, K3 = LY::K3, COLS = LY::COLS;
    constexpr int TM_D1 = SL::TM_D1, TM_D2 = SL::TM_D2, TM_WG = SL::TM_WG;
    extern __shared__ __align__(1024) uint8_t smem[];
    __shared__ uint32_t tmem_base_s;
    const int tid = threadIdx.x, t = tid & 127;
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0), wg = warp >> 2;     // warp-uniform (MMA operands in uniform registers)
    const bool issuer_warp = (warp & 3) == 0;
    float *sw1 = reinterpret_cast<float *>(smem + SL::VEC), *sb1 = sw1 + 32;
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem + SL::BARS);
    uint8_t *wgs = smem + SL::WG0 + wg * SL::WG_BYTES;
    uint8_t *timg_row = wgs + SL::TIMG + t * 16;            // this row's 16-byte slot of chunk 0
    float *scr = reinterpret_cast<float *>(wgs + SL::SCR);
    int *meta = reinterpret_cast<int *>(wgs + SL::META);
    const int *off = tt.off;
    const float inv_nm = 1.0f / (float)Nm;

    if (tid == 0) {
        for (int k = 0; k < NWG; ++k) tc::mbar_init(&bars[k], 1);
        asm volatile("fence.mbarrier_init.release.cluster;");
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tc::smem_u32(&tmem_base_s)), "n"(512));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    // zero this warpgroup's T image (padding columns stay zero for the whole kernel), R image and scratch
    for (int k = t; k < SL::WG_BYTES / 16; k += 128) reinterpret_cast<uint4 *>(wgs)[k] = make_uint4(0u, 0u, 0u, 0u);
    if (wg == NWG - 1)
        for (int k = t; k < SL::SLACK / 16; k += 128) reinterpret_cast<uint4 *>(wgs + SL::WG_BYTES)[k] = make_uint4(0u, 0u, 0u, 0u);
    tc::fence_before();
    __syncthreads();
    tc::fence_after();
    const uint32_t tmem = __shfl_sync(0xffffffffu, tmem_base_s, 0) + wg * TM_WG;
    const uint32_t tm_lane = tmem + ((uint32_t)((warp & 3) * 32) << 16);
    const uint32_t sbase = tc::smem_u32(smem);
    const uint32_t s_timg = tc::smem_u32(wgs + SL::TIMG), s_rimg = tc::smem_u32(wgs + SL::RIMG);
    const uint64_t d_timg = tc::desc(s_timg, 2048, 128), d_timg_mn = tc::desc(s_timg, 128, 2048), d_rimg_mn = tc::desc(s_rimg, 128, 2048);
    const uint64_t d_w2 = tc::desc(sbase + SL::W2, 64 * 16, 128), d_w3 = tc::desc(sbase + SL::W3, K3 * 16, 128);
    // ONES_STEP: A = the ones image (every 8-row group reads the same core matrix: stride 0), B = one bias chunk read twice
    // (leading stride 0; the second K chunk of the ones image is zero)
    const uint64_t d_ones = tc::desc(sbase + SL::ONES, 128, 0), d_bb2 = tc::desc(sbase + SL::BB2, 0, 128), d_bb3 = tc::desc(sbase + SL::BB3, 0, 128);
    (void)d_ones; (void)d_bb2; (void)d_bb3;
    uint64_t *bar = &bars[wg];
    uint32_t ph = 0;
    unsigned long long my_rows = 0;
    // the contraction accumulators start at zero
#pragma unroll
    for (int c = 0; c < 32; c += 4) tc::st4(tm_lane + TM_D1 + c, 0u, 0u, 0u, 0u);
    tc::wait_st();

    // fold the lanes of one finished atom into A_i and clear its accumulator block
    auto flush = [&](int atom) {
        const int slot = atom & (T2_NSLOT - 1);
        uint32_t v1[8], v2[8];
        const uint32_t z8[8] = {0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u};
        tc::ld8(tm_lane + TM_D1 + 8 * slot, v1);
        tc::ld8(tm_lane + TM_D2 + 8 * slot, v2);
        tc::wait_ld();
        tc::st8(tm_lane + TM_D1 + 8 * slot, z8);
        tc::st8(tm_lane + TM_D2 + 8 * slot, z8);
#pragma unroll
        for (int c = 0; c < 4; ++c) {      // columns c: T . R^w(hi), columns 4 + c: T . R^w(lo)
            scr[c * COLS + t] = __uint_as_float(v1[c]) + __uint_as_float(v1[4 + c]);
            if (t < COLS - 128) scr[c * COLS + 128 + t] = __uint_as_float(v2[c]) + __uint_as_float(v2[4 + c]);
        }
        tc::bar_sync(1 + wg, 128);
        if (t < M2E) {
            float *dst = Aout + (long)atom * 4 * M2E + t;
            const int f2 = T2_O2 + (t >= M1 ? t - M1 : t);
            const int f1 = T2_O1 + (t % M0);
#pragma unroll
            for (int c = 0; c < 4; ++c)
                atomicAdd(dst + c * M2E, (scr[c * COLS + T2_O3 + t] + scr[c * COLS + f2] + scr[c * COLS + f1]) * inv_nm);
        }
        tc::wait_st();
        tc::fence_before();
        tc::bar_sync(1 + wg, 128);
    };

    for (int a = 0; a < T; ++a) {
        const int ts0 = bin_start[a * ncell], ts1 = bin_start[(a + 1) * ncell];
        if (ts0 == ts1) continue;
        for (int b = 0; b < T; ++b) {
            const long rbase = N * (long)off[b];
            const int rs = rowstart[(long)b * (N + 1) + ts0], re = rowstart[(long)b * (N + 1) + ts1];
            const int ntiles = (re - rs + T2_ROWS - 1) / T2_ROWS;
            __syncthreads();
            {   // stage the (a, b) net: forward operand images and the layer-1 vectors
                const EmbedNetTC2<W> *net = nets + (a * T + b);
                const uint4 *s2 = reinterpret_cast<const uint4 *>(&net->W2[0][0][0]);
                const uint4 *s3 = reinterpret_cast<const uint4 *>(&net->W3[0][0][0]);
                for (int k = tid; k < 4 * 64; k += NWG * 128) reinterpret_cast<uint4 *>(smem + SL::W2)[k] = s2[k];
                for (int k = tid; k < 12 * K3; k += NWG * 128) reinterpret_cast<uint4 *>(smem + SL::W3)[k] = s3[k];
                if (LY::ONES_STEP) {
                    const uint4 *sb2 = reinterpret_cast<const uint4 *>(&net->Bb2[0][0]), *sb3 = reinterpret_cast<const uint4 *>(&net->Bb3[0][0]);
                    for (int k = tid; k < 64; k += NWG * 128) reinterpret_cast<uint4 *>(smem + SL::BB2)[k] = sb2[k];
                    for (int k = tid; k < K3; k += NWG * 128) reinterpret_cast<uint4 *>(smem + SL::BB3)[k] = sb3[k];
                    if (tid < 16) reinterpret_cast<uint4 *>(smem + SL::ONES)[tid] = tid < 8 ? make_uint4(0x3c003c00u, 0u, 0u, 0u) : make_uint4(0u, 0u, 0u, 0u);
                }
                if (tid < 64) sw1[tid] = reinterpret_cast<const float *>(net)[tid];
            }
            tc::proxy_fence();
            __syncthreads();
            const int G = gridDim.x * NWG, gw = blockIdx.x * NWG + wg;
            const int tile0 = (int)((long)ntiles * gw / G), tile1 = (int)((long)ntiles * (gw + 1) / G);
            int pending = -1;
            float4 nrh = make_float4(0.f, 0.f, 0.f, 0.f);
            int2 nid = make_int2(-1, 1);
            if (tile0 < tile1) {
                const int r0 = rs + tile0 * T2_ROWS;
                if (r0 + t < re) { nrh = __ldg(&rows_rh[rbase + r0 + t]); nid = __ldg(&rows_id[rbase + r0 + t]); }
            }
            for (int tile = tile0; tile < tile1; ++tile) {
                const int r0 = rs + tile * T2_ROWS;
                const int nrows = min(T2_ROWS, re - r0);
                const float4 rh = nrh;
                const int2 id = nid;
                nrh = make_float4(0.f, 0.f, 0.f, 0.f);
                nid = make_int2(-1, 1);
                if (tile + 1 < tile1 && r0 + T2_ROWS + t < re) {
                    nrh = __ldg(&rows_rh[rbase + r0 + T2_ROWS + t]);
                    nid = __ldg(&rows_id[rbase + r0 + T2_ROWS + t]);
                }
                const int atom = id.x;
                const float wgt = id.y < 0 ? (float)(-id.y) : 1.f;
                if (t == 0) meta[0] = atom;
                if (t == nrows - 1) meta[1] = atom;
                // ---- E1: layer 1 on the ALUs ----
                {
                    const float s = rh.x;
                    float y[32];
#pragma unroll
                    for (int e = 0; e < 32; ++e) y[e] = e < M0 ? tc::tanh_approx(fmaf(s, sw1[e], sb1[e])) : 0.f;
                    if (!LY::ONES_STEP) { y[T2_ONE_HI] = 1.0f; y[T2_ONE_LO] = 1.0f; }     // W = 25: the constant-one columns
#pragma unroll
                    for (int c = 0; c < 4; ++c)
                        *reinterpret_cast<uint4 *>(timg_row + c * 2048) =
                            make_uint4(tc::pack_h2(y[8 * c], y[8 * c + 1]), tc::pack_h2(y[8 * c + 2], y[8 * c + 3]),
                                       tc::pack_h2(y[8 * c + 4], y[8 * c + 5]), tc::pack_h2(y[8 * c + 6], y[8 * c + 7]));
                }
                tc::proxy_fence();
                tc::fence_before();
                tc::bar_sync(1 + wg, 128);
                const int atom0 = meta[0], atomL = meta[1];
                if (issuer_warp && tc::elect_one()) {
                    tc::fence_after();
                    constexpr uint32_t id2 = tc::idesc(128, 64, false, false);
#pragma unroll
                    for (int ks = 0; ks < 2; ++ks)
                        tc::mma_ss(tmem + TM_Z, tc::desc_at(d_timg, ks * 2 * 2048), tc::desc_at(d_w2, ks * 2 * (64 * 16)), id2, ks > 0);
                    if (LY::ONES_STEP) tc::mma_ss(tmem + TM_Z, d_ones, d_bb2, id2, true);
                    tc::commit(bar);
                }
                // while layer 2 runs: retire the previous tile's last atom if this tile starts a new one
                if (pending >= 0 && pending != atom0) flush(pending);
                // ... and write the contraction operand of the first pass
                {
                    const bool in = atom >= 0 && atom - atom0 < T2_NSLOT;
                    uint4 rw;          // {hi[0..3], lo[0..3]} of the weighted row: the lo parts ride in the four spare columns of the slot
                    tc::split_h2(wgt * rh.x, wgt * rh.y, rw.x, rw.z);
                    tc::split_h2(wgt * rh.z, wgt * rh.w, rw.y, rw.w);
                    const uint4 z4 = make_uint4(0u, 0u, 0u, 0u);
#pragma unroll
                    for (int s_ = 0; s_ < T2_NSLOT; ++s_)
                        *reinterpret_cast<uint4 *>(wgs + SL::RIMG + s_ * 2048 + t * 16) = (in && (atom & (T2_NSLOT - 1)) == s_) ? rw : z4;
                }
                tc::mbar_wait(bar, ph); ph ^= 1;
                tc::fence_after();
                // ---- E2 ----
                {
                    uint8_t *img = timg_row + (T2_O2 / 8) * 2048;
                    if (W == 25) {
                        uint32_t z0[16], z1[16], z2[16], z3[2];
                        tc::ld16(tm_lane + TM_Z, z0); tc::ld16(tm_lane + TM_Z + 16, z1); tc::ld16(tm_lane + TM_Z + 32, z2);
                        tc::ld2(tm_lane + TM_Z + 48, z3);
                        tc::wait_ld();
                        tanh16_store(z0, img, 0); tanh16_store(z1, img, 2); tanh16_store(z2, img, 4);
                        *reinterpret_cast<uint4 *>(img + 6 * 2048) =
                            make_uint4(tc::pack_h2(tc::tanh_approx(__uint_as_float(z3[0])), tc::tanh_approx(__uint_as_float(z3[1]))), 0u, 0u, 0u);
                    } else {
                        uint32_t z0[16], z1[16], z2[16], z3[16];
                        tc::ld16(tm_lane + TM_Z, z0); tc::ld16(tm_lane + TM_Z + 16, z1); tc::ld16(tm_lane + TM_Z + 32, z2);
                        tc::ld16(tm_lane + TM_Z + 48, z3);
                        tc::wait_ld();
                        tanh16_store(z0, img, 0); tanh16_store(z1, img, 2); tanh16_store(z2, img, 4); tanh16_store(z3, img, 6);
                    }
                }
                tc::proxy_fence();
                tc::fence_before();
                tc::bar_sync(1 + wg, 128);
                if (issuer_warp && tc::elect_one()) {
                    tc::fence_after();
                    constexpr uint32_t id3 = tc::idesc(128, K3, false, false);
#pragma unroll
                    for (int ks = 0; ks < 6; ++ks) {
                        const int achunk = ks < 4 ? T2_O2 / 8 + 2 * ks : 2 * (ks - 4);
                        tc::mma_ss(tmem + TM_Z, tc::desc_at(d_timg, achunk * 2048), tc::desc_at(d_w3, ks * 2 * (K3 * 16)), id3, ks > 0);
                    }
                    if (LY::ONES_STEP) tc::mma_ss(tmem + TM_Z, d_ones, d_bb3, id3, true);
                    tc::commit(bar);
                }
                tc::mbar_wait(bar, ph); ph ^= 1;
                tc::fence_after();
                // ---- E3 ----
                {
                    uint8_t *img = timg_row + (T2_O3 / 8) * 2048;
                    {   // the first 96 columns in six groups of 16, each TMEM load one group ahead of its tanh work
                        uint32_t zb[2][16];
                        tc::ld16(tm_lane + TM_Z, zb[0]);
#pragma unroll
                        for (int u = 0; u < 6; ++u) {
                            tc::wait_ld();
                            if (u + 1 < 6) tc::ld16(tm_lane + TM_Z + 16 * (u + 1), zb[(u + 1) & 1]);
                            tanh16_store(zb[u & 1], img, 2 * u);
                        }
                    }
                    if (W == 25) {
                        uint32_t z3[4];
                        tc::ld4(tm_lane + TM_Z + 96, z3);
                        tc::wait_ld();
                        *reinterpret_cast<uint4 *>(img + 12 * 2048) =
                            make_uint4(tc::pack_h2(tc::tanh_approx(__uint_as_float(z3[0])), tc::tanh_approx(__uint_as_float(z3[1]))),
                                       tc::pack_h2(tc::tanh_approx(__uint_as_float(z3[2])), tc::tanh_approx(__uint_as_float(z3[3]))), 0u, 0u);
                    } else {
                        uint32_t z0[16], z1[16];
                        tc::ld16(tm_lane + TM_Z + 96, z0); tc::ld16(tm_lane + TM_Z + 112, z1);
                        tc::wait_ld();
                        tanh16_store(z0, img, 12); tanh16_store(z1, img, 14);
                    }
                }
                // ---- contraction, T2_NSLOT atoms per pass, accumulated in TMEM across tiles ----
                for (int p0 = atom0; p0 <= atomL; p0 += T2_NSLOT) {
                    if (p0 != atom0) {
                        const bool in = atom >= p0 && atom - p0 < T2_NSLOT;
                        uint4 rw;          // {hi[0..3], lo[0..3]} of the weighted row: the lo parts ride in the four spare columns of the slot
                    tc::split_h2(wgt * rh.x, wgt * rh.y, rw.x, rw.z);
                    tc::split_h2(wgt * rh.z, wgt * rh.w, rw.y, rw.w);
                        const uint4 z4 = make_uint4(0u, 0u, 0u, 0u);
#pragma unroll
                        for (int s_ = 0; s_ < T2_NSLOT; ++s_)
                            *reinterpret_cast<uint4 *>(wgs + SL::RIMG + s_ * 2048 + t * 16) = (in && (atom & (T2_NSLOT - 1)) == s_) ? rw : z4;
                    }
                    tc::proxy_fence();
                    tc::fence_before();
                    tc::bar_sync(1 + wg, 128);
                    if (issuer_warp && tc::elect_one()) {
                        tc::fence_after();
                        constexpr uint32_t idc = tc::idesc(128, 8 * T2_NSLOT, true, true);
#pragma unroll
                        for (int half = 0; half < 2; ++half)
#pragma unroll
                            for (int ks = 0; ks < T2_ROWS / 16; ++ks)
                                tc::mma_ss(tmem + (half ? TM_D2 : TM_D1), tc::desc_at(d_timg_mn, half * 16 * 2048 + ks * 256), tc::desc_at(d_rimg_mn, ks * 256), idc, true);
                        tc::commit(bar);
                    }
                    tc::mbar_wait(bar, ph); ph ^= 1;
                    tc::fence_after();
                    for (int q = p0; q < p0 + T2_NSLOT && q < atomL; ++q) flush(q);
                }
                pending = atomL;
                if (t == 0) my_rows += (unsigned long long)nrows;
            }
            if (pending >= 0) flush(pending);
        }
    }
    tc::fence_before();
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base_s), "n"(512));
    if (t == 0 && my_rows) atomicAdd(row_counter, my_rows);
}

}  // namespace

// declared in embed_tc.cu
cudaError_t launch_env_rows(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st);

template <int W>
static cudaError_t launch_fwd_w(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st) {
    DP_SMEM_OPTIN(k_embed_fwd_tc2<W>, FwdSmem<W>::TOTAL);
    const TypeTab tt = make_typetab(m);
    cudaError_t e = launch_env_rows(m, N, g, ws, L, st);
    if (e != cudaSuccess) return e;
    cudaMemsetAsync(ws + L.A, 0, sizeof(float) * (size_t)N * 4 * T2<W>::M2E, st);
    k_embed_fwd_tc2<W><<<m->num_sms, NWG * 128, FwdSmem<W>::TOTAL, st>>>(
        N, m->T, g.ncell, m->Nm, tt, (const EmbedNetTC2<W> *)m->embed_tc2_dev, (int *)(ws + L.bin_start),
        (int *)(ws + L.rowstart), (const float4 *)(ws + L.rows_rh), (const int2 *)(ws + L.rows_id), (float *)(ws + L.A),
        (unsigned long long *)(ws + L.status + 8));
    return cudaGetLastError();
}

cudaError_t launch_embed_fwd_tc2(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st) {
    return m->m0 == 32 ? launch_fwd_w<32>(m, N, g, ws, L, st) : launch_fwd_w<25>(m, N, g, ws, L, st);
}
