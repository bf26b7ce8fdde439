// S3 + S4 + S5 on the 5th-generation tensor cores (tcgen05.mma, accumulators in TMEM), mixed-precision modes.
//
// Pipeline of one 128-row tile (layouts in embed_tc.cuh):
//   rows:   compact env rows (k_env_rows: fp64 env matrix -> fp32 R^, 24 B per row) -> s^ and weighted R^ operand image
//   E1:     layer 1 (K = 1) on the ALUs, y1 -> fp16 hi/lo A-operand image
//   MMA L2: D2[128 x 64]  = y1 . W2    (tcgen05.mma kind::f16, one issuing thread, hi and lo activation parts)
//   E2:     tcgen05.ld D2, + bias, tanh, + (y1,y1) -> y2 -> A-operand image
//   MMA L3: D3[128 x 128] = y2 . W3
//   E3:     tcgen05.ld D3, + bias, tanh, + (y2,y2) -> G  -> operand image (MN-major use)
//   MMA C:  DA[128 features x 8*slots] = G^T . R^w   (K = 128 rows; per-atom slots mask the rows of other atoms)
//   E4:     tcgen05.ld DA -> A_i (fp32, global), scaled by 1/Nm
// G never leaves the SM.  This kernel serves MIX-32 (NS = 3: hi + lo activations and weights) and MIX-16 models with
// Nm < 128 (NS = 2: hi + lo activations); MIX-16 otherwise runs embed_tc2.cu.
// k_env_rows (S3, the compact fp32 environment rows) serves both mixed modes.
#include "embed_tc.cuh"

namespace {

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
    uint64_t d = 0;
    d |= (uint64_t)((saddr & 0x3FFFF) >> 4);
    d |= (uint64_t)((lbo_bytes >> 4) & 0x3FFF) << 16;
    d |= (uint64_t)((sbo_bytes >> 4) & 0x3FFF) << 32;
    d |= (uint64_t)1 << 46;                     // sm_100 descriptor version; no swizzle, base offset 0
    return d;
}
// kind::f16 instruction descriptor: fp16 x fp16 -> fp32, M x N, optional MN-major operands
__device__ __forceinline__ uint32_t umma_idesc(int M, int N, bool a_mn, bool b_mn) {
    uint32_t d = 1u << 4;                        // D format F32
    d |= (a_mn ? 1u : 0u) << 15;
    d |= (b_mn ? 1u : 0u) << 16;
    d |= (uint32_t)(N >> 3) << 17;
    d |= (uint32_t)(M >> 4) << 24;
    return d;
}
__device__ __forceinline__ void umma_f16(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, bool accumulate) {
    asm volatile("{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\ntcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n}"
                 ::"r"(tmem_d), "l"(da), "l"(db), "r"(idesc), "r"((uint32_t)accumulate));
}
__device__ __forceinline__ void umma_commit(uint64_t *bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)));
}
__device__ __forceinline__ void mbar_init(uint64_t *bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
    asm volatile("{\n.reg .pred p;\nWAIT_%=:\nmbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n@p bra DONE_%=;\nbra WAIT_%=;\nDONE_%=:\n}"
                 ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void proxy_fence() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, float (&v)[16]) {
    uint32_t r[16];
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
                   "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
                 : "r"(taddr));
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
    for (int k = 0; k < 16; ++k) v[k] = __uint_as_float(r[k]);
}

__device__ __forceinline__ void tmem_ld8(uint32_t taddr, float (&v)[8]) {
    uint32_t r[8];
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
                 : "r"(taddr));
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
    for (int k = 0; k < 8; ++k) v[k] = __uint_as_float(r[k]);
}

__device__ __forceinline__ uint32_t pack_h2(float x, float y) {
    __half2 h = __floats2half2_rn(x, y);
    return *reinterpret_cast<uint32_t *>(&h);
}
__device__ __forceinline__ void split_h2(float x, float y, uint32_t &hi, uint32_t &lo) {
    const float xh = __int_as_float(__float_as_int(x) & 0xFFFFE000), yh = __int_as_float(__float_as_int(y) & 0xFFFFE000);
    hi = pack_h2(xh, yh);
    lo = pack_h2(x - xh, y - yh);
}
// 8 consecutive fp32 values -> one 16-byte chunk of the hi image and one of the lo image
__device__ __forceinline__ void store_chunk(uint8_t *hi_img, uint8_t *lo_img, int chunk, int row, const float *v) {
    uint4 h, l;
    split_h2(v[0], v[1], h.x, l.x); split_h2(v[2], v[3], h.y, l.y);
    split_h2(v[4], v[5], h.z, l.z); split_h2(v[6], v[7], h.w, l.w);
    const int o = chunk * (TC_ROWS * 16) + row * 16;
    *reinterpret_cast<uint4 *>(hi_img + o) = h;
    *reinterpret_cast<uint4 *>(lo_img + o) = l;
}
template <bool APPROX>
__device__ __forceinline__ float act_tanh(float x) {
    if (APPROX) {
        float y;
        asm("tanh.approx.f32 %0, %1;" : "=f"(y) : "f"(x));
        return y;
    } else {
        return tanhf(x);
    }
}

__device__ __forceinline__ double min_image(double t, double L, double halfL) {
    double s = t > halfL ? -1.0 : (t < -halfL ? 1.0 : 0.0);
    return __dadd_rn(t, __dmul_rn(s, L));
}
struct EnvParams {
    double rc, rc_smth, inv_range;
    double L[3];
};
__device__ __forceinline__ void env_row(const EnvParams &p, double dx, double dy, double dz, double Rt[4]) {
    const double r2 = dx * dx + dy * dy + dz * dz;
    const double r = sqrt(r2);
    double w = 1.0;
    if (r >= p.rc_smth) {
        if (r < p.rc) {
            const double u = (r - p.rc_smth) * p.inv_range;
            w = u * u * u * (-6.0 * u * u + 15.0 * u - 10.0) + 1.0;
        } else {
            w = 0.0;
        }
    }
    const double s = w / r;
    Rt[0] = s; Rt[1] = s * dx / r; Rt[2] = s * dy / r; Rt[3] = s * dz / r;
}

// shared-memory carve-up (bytes)
template <int NSW>
struct SmemLayout {
    static constexpr int W2 = 0;
    static constexpr int W3 = W2 + NSW * 4096;
    static constexpr int VEC = W3 + NSW * 16384;               // w1[32] b1[32] b2[64] b3[128] floats
    static constexpr int BUF = ((VEC + 256 * 4 + 1023) / 1024) * 1024;   // 64 KB operand images
    static constexpr int A1H = BUF, A1L = BUF + 8192, A2H = BUF + 16384, A2L = BUF + 32768;
    static constexpr int GH = BUF, GL = BUF + 32768;          // G aliases A1/A2 (dead once the layer-3 MMAs are done)
    static constexpr int RH = BUF + 65536, RL = RH + TC_NSLOT * 2048;
    static constexpr int S = RL + TC_NSLOT * 2048;               // s^ [128] floats
    static constexpr int META = S + 512;                       // ints
    static constexpr int BARS = META + 128;
    static constexpr int TOTAL = BARS + 64;
};

struct TileMeta {
    int atom0, atom_last;
};

// Compact env rows (S3): one record per processed row, block b at row offset N*off[b]:
//   rh = R^ (fp32, unweighted), id = {sorted atom, neighbour j (sorted index)} for a real row and {sorted atom, -npad}
//   for the representative of the npad padded slots; rows of atom i start at rowstart[b][i].
__global__ void __launch_bounds__(256)
k_env_rows(long N, int T, int ncell, int Nm, const __grid_constant__ TypeTab tt, EnvParams ep, const double *__restrict__ avg,
           const double *__restrict__ stdv, const int *__restrict__ bin_start, const double *__restrict__ xs,
           const int *__restrict__ nlist, const int *__restrict__ nreal, const int *__restrict__ rowstart,
           float4 *__restrict__ rows_rh, int2 *__restrict__ rows_id) {
    const int lane = threadIdx.x & 31;
    const long i = blockIdx.x * 8L + (threadIdx.x >> 5);
    if (i >= N) return;
    const int *sel = tt.sel, *off = tt.off;
    int a = 0;
    for (int t = 1; t < T; ++t) a += i >= bin_start[t * ncell];
    double av[4], isd[4];
#pragma unroll
    for (int c = 0; c < 4; ++c) { av[c] = avg[4 * a + c]; isd[c] = 1.0 / stdv[4 * a + c]; }
    const double xi = xs[3 * i], yi = xs[3 * i + 1], zi = xs[3 * i + 2];
    const double hx = 0.5 * ep.L[0], hy = 0.5 * ep.L[1], hz = 0.5 * ep.L[2];
    for (int b = 0; b < T; ++b) {
        const int nr = nreal[i * T + b];
        const int tot = nr + (nr < sel[b] ? 1 : 0);
        const long base = N * (long)off[b] + rowstart[(long)b * (N + 1) + i];
        // software pipeline over the lane's rows: list entries two rows ahead, coordinates one row ahead of the arithmetic
        const int *nl = nlist + i * Nm + off[b];
        int jn0 = lane < nr ? nl[lane] : -1, jn1 = lane + 32 < nr ? nl[lane + 32] : -1;
        double xn = 0.0, yn = 0.0, zn = 0.0;
        if (jn0 >= 0) { xn = xs[3 * (long)jn0]; yn = xs[3 * (long)jn0 + 1]; zn = xs[3 * (long)jn0 + 2]; }
        for (int k = lane; k < tot; k += 32) {
            const int j = jn0;
            const double xj = xn, yj = yn, zj = zn;
            jn0 = jn1;
            jn1 = k + 64 < nr ? nl[k + 64] : -1;
            if (jn0 >= 0) { xn = xs[3 * (long)jn0]; yn = xs[3 * (long)jn0 + 1]; zn = xs[3 * (long)jn0 + 2]; }
            double Rt[4] = {0.0, 0.0, 0.0, 0.0};
            if (k < nr) {
                const double dx = min_image(xj - xi, ep.L[0], hx);
                const double dy = min_image(yj - yi, ep.L[1], hy);
                const double dz = min_image(zj - zi, ep.L[2], hz);
                // fp64 environment row with one reciprocal square root instead of a square root and four divisions
                // (the result is rounded to fp32 below; PAPER.md:125 keeps the environment matrix in double)
                const double r2 = dx * dx + dy * dy + dz * dz;
                const double ir = rsqrt(r2), r = r2 * ir;
                double w = 1.0;
                if (r >= ep.rc_smth) {
                    if (r < ep.rc) {
                        const double u = (r - ep.rc_smth) * ep.inv_range;
                        w = u * u * u * (-6.0 * u * u + 15.0 * u - 10.0) + 1.0;
                    } else {
                        w = 0.0;
                    }
                }
                const double sr = w * ir, q = sr * ir;
                Rt[0] = sr; Rt[1] = q * dx; Rt[2] = q * dy; Rt[3] = q * dz;
            }
            rows_rh[base + k] = make_float4((float)((Rt[0] - av[0]) * isd[0]), (float)((Rt[1] - av[1]) * isd[1]),
                                            (float)((Rt[2] - av[2]) * isd[2]), (float)((Rt[3] - av[3]) * isd[3]));
            rows_id[base + k] = make_int2((int)i, k < nr ? j : -(sel[b] - nr));
        }
    }
}

template <int NS, bool APPROX, int W>
__global__ void __launch_bounds__(256, (NS == 2 ? 2 : 1))
k_embed_fwd_tc(long N, int T, int ncell, int Nm, const __grid_constant__ TypeTab tt, const EmbedNetTC<(NS == 3 ? 2 : 1)> *__restrict__ nets,
               const int *__restrict__ bin_start, const int *__restrict__ rowstart, const float4 *__restrict__ rows_rh,
               const int2 *__restrict__ rows_id, float *__restrict__ Aout, unsigned long long *__restrict__ row_counter) {
    constexpr int NSW = NS == 3 ? 2 : 1;
    constexpr int M2E = 4 * W;
    using SL = SmemLayout<NSW>;
    extern __shared__ __align__(1024) uint8_t smem[];
    __shared__ uint32_t tmem_base_s;
    float *sw1 = reinterpret_cast<float *>(smem + SL::VEC), *sb1 = sw1 + 32, *sb2 = sb1 + 32, *sb3 = sb2 + 64;
    float *sS = reinterpret_cast<float *>(smem + SL::S);
    TileMeta *meta = reinterpret_cast<TileMeta *>(smem + SL::META);
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem + SL::BARS);
    const int tid = threadIdx.x, warp = tid >> 5;
    const int row = tid & 127, h = tid >> 7;
    const int *sel = tt.sel, *off = tt.off;
    const float inv_nm = 1.0f / (float)Nm;

    if (tid == 0) {
        mbar_init(&bars[0], 1); mbar_init(&bars[1], 1); mbar_init(&bars[2], 1);
        asm volatile("fence.mbarrier_init.release.cluster;");
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)), "n"(256));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = tmem_base_s;
    const uint32_t tm_lane = tmem + ((uint32_t)((warp & 3) * 32) << 16);
    const uint32_t TM_D2 = 0, TM_D3 = 64, TM_DA = 192;
    const uint32_t sbase = smem_u32(smem);
    uint32_t ph0 = 0, ph1 = 0, ph2 = 0;          // parities of the three MMA barriers
    unsigned long long my_rows = 0;

    for (int a = 0; a < T; ++a) {
        const int ts0 = bin_start[a * ncell], ts1 = bin_start[(a + 1) * ncell];
        if (ts0 == ts1) continue;
        for (int b = 0; b < T; ++b) {
            const long rbase = N * (long)off[b];
            const int rs = rowstart[(long)b * (N + 1) + ts0], re = rowstart[(long)b * (N + 1) + ts1];
            const int ntiles = (re - rs + TC_ROWS - 1) / TC_ROWS;
            if ((int)blockIdx.x >= ntiles) continue;
            __syncthreads();
            {   // stage the (a, b) net: forward weight images and the bias vectors
                const EmbedNetTC<NSW> *net = nets + (a * T + b);
                const uint4 *s2 = reinterpret_cast<const uint4 *>(&net->W2[0][0][0][0]);
                const uint4 *s3 = reinterpret_cast<const uint4 *>(&net->W3[0][0][0][0]);
                for (int k = tid; k < NSW * 256; k += 256) reinterpret_cast<uint4 *>(smem + SL::W2)[k] = s2[k];
                for (int k = tid; k < NSW * 1024; k += 256) reinterpret_cast<uint4 *>(smem + SL::W3)[k] = s3[k];
                sw1[tid] = reinterpret_cast<const float *>(net)[tid];    // w1 b1 b2 b3 are contiguous (256 floats)
            }
            proxy_fence();
            __syncthreads();
            for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
                const int r0 = rs + tile * TC_ROWS;
                const int nrows = min(TC_ROWS, re - r0);
                // ---- rows: compact env rows -> s^, weights, slot bookkeeping ----
                float4 rh = make_float4(0.f, 0.f, 0.f, 0.f);
                int atom = -1;
                float wgt = 0.f;
                if (h == 0) {
                    if (row < nrows) {
                        rh = rows_rh[rbase + r0 + row];
                        const int2 id = rows_id[rbase + r0 + row];
                        atom = id.x;
                        wgt = id.y < 0 ? (float)(-id.y) : 1.f;
                    }
                    sS[row] = rh.x;
                    if (row == 0) meta->atom0 = atom;
                    if (row == nrows - 1) meta->atom_last = atom;
                }
                __syncthreads();
                const int atom0 = meta->atom0, na = meta->atom_last - atom0 + 1;
                const int slot = atom - atom0;
                // ---- E1: layer 1 on the ALUs ----
                float y1[16];
                {
                    const float s = sS[row];
#pragma unroll
                    for (int t = 0; t < 16; ++t) {
                        const int p1 = 16 * h + t;
                        y1[t] = t < tc_ce<W>(h) ? act_tanh<APPROX>(fmaf(s, sw1[p1], sb1[p1])) : 0.f;
                    }
                    store_chunk(smem + SL::A1H, smem + SL::A1L, 2 * h, row, y1);
                    store_chunk(smem + SL::A1H, smem + SL::A1L, 2 * h + 1, row, y1 + 8);
                }
                proxy_fence();
                tc_fence_before();
                __syncthreads();
                if (tid == 0) {
                    tc_fence_after();
                    const uint32_t idesc = umma_idesc(128, TC_N2, false, false);
                    bool acc = false;
#pragma unroll
                    for (int part = 0; part < 2; ++part)           // activation hi, lo
#pragma unroll
                        for (int wp = 0; wp < NSW; ++wp) {
                            if (part == 1 && wp == 1) continue;    // lo * lo dropped
                            for (int ks = 0; ks < TC_K1 / 16; ++ks) {
                                const uint64_t da = umma_desc(sbase + (part ? SL::A1L : SL::A1H) + ks * 2 * 2048, 2048, 128);
                                const uint64_t db = umma_desc(sbase + SL::W2 + wp * 4096 + ks * 2 * (TC_N2 * 16), TC_N2 * 16, 128);
                                umma_f16(tmem + TM_D2, da, db, idesc, acc);
                                acc = true;
                            }
                        }
                    umma_commit(&bars[0]);
                }
                // ---- E2: layer-2 epilogue ----
                float y2[32];
                mbar_wait(&bars[0], ph0); ph0 ^= 1;
                tc_fence_after();
#pragma unroll
                for (int j = 0; j < 2; ++j) {
                    float z[16];
                    tmem_ld16(tm_lane + TM_D2 + 32 * h + 16 * j, z);
#pragma unroll
                    for (int t = 0; t < 16; ++t) {
                        const int n = 32 * h + 16 * j + t;
                        y2[16 * j + t] = t < tc_ce<W>(h) ? y1[t] + act_tanh<APPROX>(z[t] + sb2[n]) : 0.f;
                    }
                    store_chunk(smem + SL::A2H, smem + SL::A2L, 4 * h + 2 * j, row, y2 + 16 * j);
                    store_chunk(smem + SL::A2H, smem + SL::A2L, 4 * h + 2 * j + 1, row, y2 + 16 * j + 8);
                }
                proxy_fence();
                tc_fence_before();
                __syncthreads();
                if (tid == 0) {
                    tc_fence_after();
                    const uint32_t idesc = umma_idesc(128, TC_N3, false, false);
                    bool acc = false;
#pragma unroll
                    for (int part = 0; part < 2; ++part)
#pragma unroll
                        for (int wp = 0; wp < NSW; ++wp) {
                            if (part == 1 && wp == 1) continue;
                            for (int ks = 0; ks < TC_N2 / 16; ++ks) {
                                const uint64_t da = umma_desc(sbase + (part ? SL::A2L : SL::A2H) + ks * 2 * 2048, 2048, 128);
                                const uint64_t db = umma_desc(sbase + SL::W3 + wp * 16384 + ks * 2 * (TC_N3 * 16), TC_N3 * 16, 128);
                                umma_f16(tmem + TM_D3, da, db, idesc, acc);
                                acc = true;
                            }
                        }
                    umma_commit(&bars[1]);
                }
                // ---- E3: layer-3 epilogue -> G image ----
                mbar_wait(&bars[1], ph1); ph1 ^= 1;
                tc_fence_after();
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    float z[16], gv[16];
                    tmem_ld16(tm_lane + TM_D3 + 64 * h + 16 * q, z);
#pragma unroll
                    for (int t = 0; t < 16; ++t) {
                        const int c3 = 64 * h + 16 * q + t;
                        const int u = 16 * (q & 1) + t;
                        gv[t] = t < tc_ce<W>(h) ? y2[u] + act_tanh<APPROX>(z[t] + sb3[c3]) : 0.f;
                    }
                    store_chunk(smem + SL::GH, smem + SL::GL, 8 * h + 2 * q, row, gv);
                    store_chunk(smem + SL::GH, smem + SL::GL, 8 * h + 2 * q + 1, row, gv + 8);
                }
                // ---- contraction, TC_NSLOT atoms per pass ----
                for (int g0 = 0; g0 < na; g0 += TC_NSLOT) {
                    if (h == 0) {
                        float rw[8] = {wgt * rh.x, wgt * rh.y, wgt * rh.z, wgt * rh.w, 0.f, 0.f, 0.f, 0.f};
                        const float zero8[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
#pragma unroll
                        for (int s = 0; s < TC_NSLOT; ++s)
                            store_chunk(smem + SL::RH, smem + SL::RL, s, row, (atom >= 0 && s == slot - g0) ? rw : zero8);
                    }
                    proxy_fence();
                    tc_fence_before();
                    __syncthreads();
                    if (tid == 0) {
                        tc_fence_after();
                        const uint32_t idesc = umma_idesc(128, 8 * TC_NSLOT, true, true);
                        bool acc = false;
#pragma unroll
                        for (int combo = 0; combo < 3; ++combo) {       // Gh Rh, Gl Rh, Gh Rl
                            const uint32_t ga = sbase + (combo == 1 ? SL::GL : SL::GH), ra = sbase + (combo == 2 ? SL::RL : SL::RH);
                            for (int ks = 0; ks < TC_ROWS / 16; ++ks) {
                                const uint64_t da = umma_desc(ga + ks * 256, 128, 2048);
                                const uint64_t db = umma_desc(ra + ks * 256, 128, 2048);
                                umma_f16(tmem + TM_DA, da, db, idesc, acc);
                                acc = true;
                            }
                        }
                        umma_commit(&bars[2]);
                    }
                    // ---- E4: read-out: lane = layer-3 column c3, columns = 8*slot + c; h selects slots 3h..3h+2 ----
                    mbar_wait(&bars[2], ph2); ph2 ^= 1;
                    tc_fence_after();
                    const int m = tc_m_of_c3<W>(row);
#pragma unroll
                    for (int sl = 0; sl < TC_NSLOT / 2; ++sl) {
                        float v[8];
                        const int s_ = (TC_NSLOT / 2) * h + sl;
                        tmem_ld8(tm_lane + TM_DA + 8 * s_, v);
                        if (m >= 0 && g0 + s_ < na) {
                            float *dst = Aout + (long)(atom0 + g0 + s_) * 4 * M2E + m;
#pragma unroll
                            for (int c = 0; c < 4; ++c) atomicAdd(dst + c * M2E, v[c] * inv_nm);
                        }
                    }
                    tc_fence_before();
                    __syncthreads();
                }
                if (tid == 0) my_rows += (unsigned long long)nrows;
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(256));
    if (tid == 0 && my_rows) atomicAdd(row_counter, my_rows);
}

EnvParams make_env(const dp_model *m, const Grid3 &g) {
    EnvParams ep;
    ep.rc = m->rc; ep.rc_smth = m->rc_smth; ep.inv_range = 1.0 / (m->rc - m->rc_smth);
    ep.L[0] = g.L[0]; ep.L[1] = g.L[1]; ep.L[2] = g.L[2];
    return ep;
}

}  // namespace

// S3: compact fp32 environment rows for the tcgen05 embedding kernels
cudaError_t launch_env_rows(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st) {
    const TypeTab tt = make_typetab(m);
    k_env_rows<<<(unsigned)((N + 7) / 8), 256, 0, st>>>(N, m->T, g.ncell, m->Nm, tt, make_env(m, g), m->avg_dev, m->std_dev,
                                                         (int *)(ws + L.bin_start), (double *)(ws + L.xs), (int *)(ws + L.nlist),
                                                         (int *)(ws + L.nreal), (int *)(ws + L.rowstart),
                                                         (float4 *)(ws + L.rows_rh), (int2 *)(ws + L.rows_id));
    return cudaGetLastError();
}

namespace {

template <int NS, bool APPROX, int W>
cudaError_t launch_fwd(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st) {
    constexpr int M2E = 4 * W;
    constexpr int NSW = NS == 3 ? 2 : 1;
    const int smem = SmemLayout<NSW>::TOTAL;
    DP_SMEM_OPTIN((k_embed_fwd_tc<NS, APPROX, W>), smem);
    const TypeTab tt = make_typetab(m);
    launch_env_rows(m, N, g, ws, L, st);
    cudaMemsetAsync(ws + L.A, 0, sizeof(float) * (size_t)N * 4 * M2E, st);
    const int grid = m->num_sms * (NS == 2 ? 2 : 1);
    k_embed_fwd_tc<NS, APPROX, W><<<grid, 256, smem, st>>>(
        N, m->T, g.ncell, m->Nm, tt, (const EmbedNetTC<NSW> *)m->embed_tc_dev, (int *)(ws + L.bin_start),
        (int *)(ws + L.rowstart), (const float4 *)(ws + L.rows_rh), (const int2 *)(ws + L.rows_id), (float *)(ws + L.A),
        (unsigned long long *)(ws + L.status + 8));
    return cudaGetLastError();
}

}  // namespace

// MIX-32: activations and weights as hi + lo fp16 pairs (three products per MMA step), exact tanhf.
// MIX-16 models with a short neighbour row (Nm < 128, dp_model::fwd_split): activations as hi + lo pairs, fp16 weights,
// tanh.approx; the single-fp16 activations of embed_tc2.cu average over too few rows there.
cudaError_t launch_embed_fwd_tc(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st) {
    if (m->prec == DP_MIX32) return m->m0 == 32 ? launch_fwd<3, false, 32>(m, N, g, ws, L, st) : launch_fwd<3, false, 25>(m, N, g, ws, L, st);
    return launch_fwd<2, true, 25>(m, N, g, ws, L, st);
}
