// S6 (fitting net forward and backward) in MIX-32 (MIX-16 runs fit_tc.cu): the four 240 x 240 products, the
// energy and the gA fragments; the two large products (first layer with the descriptor S5 formed in its operand producer, and
// the last backward product) run on the tcgen05 kernels of fit_tc.cu with hi + lo weight images.
// GEMMs batched over the atoms of one centre type on fp16 tensor-core MMAs (m16n8k16) with fp32 accumulation; every
// operand is split hi + lo (NS = 3: hi hi + hi lo + lo hi), i.e. single-precision products on the tensor pipe, exact
// tanhf, activations stored in fp32 ("all the arithmetic operations ... performed in single precision").
#include "embed_mix.cuh"

namespace {

constexpr int BM = 128, BN = 80, BK = 16;      // K = 240 and 1600 are multiples of 16, not of 32
constexpr int AS_STRIDE = BK + 8;       // floats: conflict-free float2 fragment loads
constexpr int BS_STRIDE = BN + 4;       // B stored [k][n]
constexpr int BT_STRIDE = BK + 8;       // B stored [n][k]
constexpr int AS_TILE = BM * AS_STRIDE;
constexpr int B_TILE = (BK * BS_STRIDE > BN * BT_STRIDE) ? BK * BS_STRIDE : BN * BT_STRIDE;
constexpr int FIT_SMEM_BYTES = 2 * (AS_TILE + B_TILE) * 4;

__device__ __forceinline__ void cp_async16(void *smem_dst, const void *gsrc, bool valid) {
    unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    int sz = valid ? 16 : 0;
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(s), "l"(gsrc), "r"(sz));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N)); }

struct FitArgsF {
    int ncell;
    const int *bin_start;
    int K, N;
    const float *A; int lda;
    const float *B; long b_type_stride; int ldb;
    const float *bias; int bias_type_stride;
    const float *v4; int v4_type_stride;
    const float *aux0; const float *aux1;
    float *out0; float *out1; int ldo;
};

template <bool SPLIT>
__device__ __forceinline__ void cvt_pair(float x, float y, uint32_t &hi, uint32_t &lo) {
    if (!SPLIT) { hi = pack_h2(x, y); lo = 0; }
    else split_h2(x, y, hi, lo);
}

template <int MODE, int NS, bool APPROX>
__global__ void __launch_bounds__(256) k_fitm_gemm(FitArgsF p) {
    constexpr bool BT = MODE >= 3;
    extern __shared__ __align__(16) float smf[];
    const int a = blockIdx.z;
    const int ts0 = p.bin_start[a * p.ncell], ts1 = p.bin_start[(a + 1) * p.ncell];
    const int row0 = ts0 + blockIdx.y * BM;
    if (row0 >= ts1) return;
    const int n0 = blockIdx.x * BN;
    const float *Bw = p.B + a * p.b_type_stride;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int wm = wid >> 1, wn = wid & 1;          // 4 x 2 warps, warp tile 32 x 40
    const int g = lane >> 2, r = lane & 3;

    auto load_tiles = [&](int stage, int k0) {
        float *As = smf + stage * (AS_TILE + B_TILE);
        float *Bs = As + AS_TILE;
        for (int c = tid; c < BM * (BK / 4); c += 256) {
            const int row = c / (BK / 4), c4 = c % (BK / 4);
            const bool ok = row0 + row < ts1;
            cp_async16(As + row * AS_STRIDE + 4 * c4, p.A + (long)(ok ? row0 + row : ts0) * p.lda + k0 + 4 * c4, ok);
        }
        if (!BT) {
            for (int c = tid; c < BK * (BN / 4); c += 256) {
                const int k = c / (BN / 4), cc = c % (BN / 4);
                const bool okn = n0 + 4 * cc < p.N;
                cp_async16(Bs + k * BS_STRIDE + 4 * cc, Bw + (long)(k0 + k) * p.ldb + (okn ? n0 + 4 * cc : 0), okn);
            }
        } else {
            for (int c = tid; c < BN * (BK / 4); c += 256) {
                const int n = c / (BK / 4), c4 = c % (BK / 4);
                const bool okn = n0 + n < p.N;
                cp_async16(Bs + n * BT_STRIDE + 4 * c4, Bw + (long)(okn ? n0 + n : 0) * p.ldb + k0 + 4 * c4, okn);
            }
        }
        cp_async_commit();
    };

    float acc[2][5][4];
#pragma unroll
    for (int mt = 0; mt < 2; ++mt)
#pragma unroll
        for (int nt = 0; nt < 5; ++nt)
#pragma unroll
            for (int k = 0; k < 4; ++k) acc[mt][nt][k] = 0.f;

    const int nk = p.K / BK;
    load_tiles(0, 0);
    for (int ks = 0; ks < nk; ++ks) {
        if (ks + 1 < nk) { load_tiles((ks + 1) & 1, (ks + 1) * BK); cp_async_wait<1>(); }
        else cp_async_wait<0>();
        __syncthreads();
        const float *As = smf + (ks & 1) * (AS_TILE + B_TILE);
        const float *Bs = As + AS_TILE;
#pragma unroll
        for (int kk = 0; kk < BK / 16; ++kk) {
            uint32_t ah[2][4], al[2][4], bh[5][2], bl[5][2];
#pragma unroll
            for (int mt = 0; mt < 2; ++mt) {
                const float *ap = As + (wm * 32 + mt * 16 + g) * AS_STRIDE + kk * 16 + 2 * r;
                const float2 x0 = *reinterpret_cast<const float2 *>(ap);
                const float2 x1 = *reinterpret_cast<const float2 *>(ap + 8 * AS_STRIDE);
                const float2 x2 = *reinterpret_cast<const float2 *>(ap + 8);
                const float2 x3 = *reinterpret_cast<const float2 *>(ap + 8 * AS_STRIDE + 8);
                cvt_pair<ns_asplit(NS)>(x0.x, x0.y, ah[mt][0], al[mt][0]); cvt_pair<ns_asplit(NS)>(x1.x, x1.y, ah[mt][1], al[mt][1]);
                cvt_pair<ns_asplit(NS)>(x2.x, x2.y, ah[mt][2], al[mt][2]); cvt_pair<ns_asplit(NS)>(x3.x, x3.y, ah[mt][3], al[mt][3]);
            }
#pragma unroll
            for (int nt = 0; nt < 5; ++nt) {
                const int n = wn * 40 + nt * 8 + g;
                if (BT) {
                    const float *bp = Bs + n * BT_STRIDE + kk * 16 + 2 * r;
                    const float2 y0 = *reinterpret_cast<const float2 *>(bp);
                    const float2 y1 = *reinterpret_cast<const float2 *>(bp + 8);
                    cvt_pair<ns_wsplit(NS)>(y0.x, y0.y, bh[nt][0], bl[nt][0]); cvt_pair<ns_wsplit(NS)>(y1.x, y1.y, bh[nt][1], bl[nt][1]);
                } else {
                    const float *bp = Bs + (kk * 16 + 2 * r) * BS_STRIDE + n;
                    cvt_pair<ns_wsplit(NS)>(bp[0], bp[BS_STRIDE], bh[nt][0], bl[nt][0]);
                    cvt_pair<ns_wsplit(NS)>(bp[8 * BS_STRIDE], bp[9 * BS_STRIDE], bh[nt][1], bl[nt][1]);
                }
            }
#pragma unroll
            for (int mt = 0; mt < 2; ++mt)
#pragma unroll
                for (int nt = 0; nt < 5; ++nt) {
                    mma16816(acc[mt][nt], ah[mt][0], ah[mt][1], ah[mt][2], ah[mt][3], bh[nt][0], bh[nt][1]);
                    if (ns_wsplit(NS)) mma16816(acc[mt][nt], ah[mt][0], ah[mt][1], ah[mt][2], ah[mt][3], bl[nt][0], bl[nt][1]);
                    if (ns_asplit(NS)) mma16816(acc[mt][nt], al[mt][0], al[mt][1], al[mt][2], al[mt][3], bh[nt][0], bh[nt][1]);
                }
        }
        __syncthreads();
    }

#pragma unroll
    for (int mt = 0; mt < 2; ++mt)
#pragma unroll
        for (int hrow = 0; hrow < 2; ++hrow) {
            const int row = row0 + wm * 32 + mt * 16 + g + 8 * hrow;
            if (row >= ts1) continue;
#pragma unroll
            for (int nt = 0; nt < 5; ++nt) {
                const int col = n0 + wn * 40 + nt * 8 + 2 * r;
                if (col >= p.N) continue;          // N = 16 m2 need not be a multiple of the tile width
                const long o = (long)row * p.ldo + col;
                const float v0 = acc[mt][nt][2 * hrow], v1 = acc[mt][nt][2 * hrow + 1];
                if (MODE == 0) {
                    const float *b = p.bias + a * p.bias_type_stride + col;
                    *reinterpret_cast<float2 *>(p.out0 + o) = make_float2(act_tanh<APPROX>(v0 + b[0]), act_tanh<APPROX>(v1 + b[1]));
                } else if (MODE == 1) {
                    const float *b = p.bias + a * p.bias_type_stride + col;
                    const float2 h = *reinterpret_cast<const float2 *>(p.aux0 + o);
                    const float t0 = act_tanh<APPROX>(v0 + b[0]), t1 = act_tanh<APPROX>(v1 + b[1]);
                    *reinterpret_cast<float2 *>(p.out0 + o) = make_float2(t0, t1);
                    *reinterpret_cast<float2 *>(p.out1 + o) = make_float2(h.x + t0, h.y + t1);
                } else if (MODE == 2) {
                    const float *b = p.bias + a * p.bias_type_stride + col;
                    const float *v4 = p.v4 + a * p.v4_type_stride + col;
                    const float2 h = *reinterpret_cast<const float2 *>(p.aux0 + o);
                    const float t0 = tanhf(v0 + b[0]), t1 = tanhf(v1 + b[1]);
                    *reinterpret_cast<float2 *>(p.out0 + o) = make_float2(v4[0] * (1.f - t0 * t0), v4[1] * (1.f - t1 * t1));
                    *reinterpret_cast<float2 *>(p.out1 + o) = make_float2(h.x + t0, h.y + t1);
                } else if (MODE == 3) {
                    const float *v4 = p.v4 + a * p.v4_type_stride + col;
                    const float2 t = *reinterpret_cast<const float2 *>(p.aux0 + o);
                    const float g0 = v4[0] + v0, g1 = v4[1] + v1;
                    *reinterpret_cast<float2 *>(p.out0 + o) = make_float2(g0, g1);
                    *reinterpret_cast<float2 *>(p.out1 + o) = make_float2(g0 * (1.f - t.x * t.x), g1 * (1.f - t.y * t.y));
                } else if (MODE == 4) {
                    const float2 gg = *reinterpret_cast<const float2 *>(p.aux0 + o);
                    const float2 h = *reinterpret_cast<const float2 *>(p.aux1 + o);
                    const float g0 = gg.x + v0, g1 = gg.y + v1;
                    *reinterpret_cast<float2 *>(p.out0 + o) = make_float2(g0 * (1.f - h.x * h.x), g1 * (1.f - h.y * h.y));
                } else {
                    *reinterpret_cast<float2 *>(p.out0 + o) = make_float2(v0, v1);
                }
            }
        }
}


__device__ __forceinline__ int type_of_sorted(int i, int T, int ncell, const int *bin_start) {
    int a = 0;
    for (int t = 1; t < T; ++t) a += i >= bin_start[t * ncell];
    return a;
}

// E_i: last layer in fp32, result converted to fp64 and the fp64 energy bias added
__global__ void __launch_bounds__(256) k_energy_f(long N, int T, int ncell, const int *__restrict__ bin_start,
                                                  const float *__restrict__ h3, const float *__restrict__ v4,
                                                  const float *__restrict__ c4, const double *__restrict__ ebias,
                                                  double *__restrict__ eatom) {
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const long i = blockIdx.x * 8L + wid;
    if (i >= N) return;
    const int a = type_of_sorted((int)i, T, ncell, bin_start);
    float acc = 0.f;
    for (int n = lane; n < 240; n += 32) acc = fmaf(h3[i * 240 + n], v4[a * 240 + n], acc);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (lane == 0) eatom[i] = (double)(acc + c4[a]) + ebias[a];
}


// gA (fp32 [N][4][m2], written by the epilogue of the tcgen05 last product, fit_tc.cu) -> scaled fp16 MMA fragments
// for the embedding backward (layout in embed_mix.cu)
template <int NSW, int W>
__global__ void __launch_bounds__(128) k_gA_frag(long N, const float *__restrict__ gA, uint32_t *__restrict__ gAf,
                                                 float *__restrict__ gscale) {
    constexpr int M2E = HW<W>::M2E, HNT3 = HW<W>::HNT3, GP = 2 * HNT3;
    __shared__ float sO_all[4][4 * M2E];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const long i = blockIdx.x * 4L + wid;
    if (i >= N) return;
    float *sO = sO_all[wid];
    float mx = 0.f;
    for (int k = lane; k < 4 * M2E; k += 32) {
        const float v = gA[i * 4 * M2E + k];
        sO[k] = v;
        mx = fmaxf(mx, fabsf(v));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    int ex = 0;
    if (mx > 0.f) frexpf(mx, &ex);
    const float sc = ldexpf(1.f, -ex);          // power-of-two scale bringing max|gA| into [0.5, 1)
    if (lane == 0) gscale[i] = sc;
    __syncwarp();
    uint32_t *out = gAf + i * (2 * GP * 32);
    const int g = lane >> 2, r = lane & 3;
    for (int nt3 = 0; nt3 < HNT3; ++nt3) {
        const int f = h_f3<W>(nt3, g >> 1, g & 1);
        float x = 0.f, y = 0.f;
        if (f >= 0 && r < 2) { x = sO[(2 * r) * M2E + f] * sc; y = sO[(2 * r + 1) * M2E + f] * sc; }
        uint32_t hi, lo;
        split_h2(x, y, hi, lo);
        out[nt3 * 32 + lane] = hi;
        if (NSW == 2) out[(GP + nt3) * 32 + lane] = lo;
    }
    for (int t = 0; t < HNT3; ++t) {
        const int f0 = h_f3<W>(t, r, 0), f1 = h_f3<W>(t, r, 1);
        float x = 0.f, y = 0.f;
        if (f0 >= 0 && g < 4) { x = sO[g * M2E + f0] * sc; y = sO[g * M2E + f1] * sc; }
        uint32_t hi, lo;
        split_h2(x, y, hi, lo);
        out[(HNT3 + t) * 32 + lane] = hi;
        if (NSW == 2) out[(GP + HNT3 + t) * 32 + lane] = lo;
    }
}

// MIX-32: every operand split hi + lo (NS = 3), exact tanhf
template <int MODE>
cudaError_t launch_gemm(const FitArgsF &p, dim3 grid, cudaStream_t st) {
    DP_SMEM_OPTIN((k_fitm_gemm<MODE, 3, false>), FIT_SMEM_BYTES);
    k_fitm_gemm<MODE, 3, false><<<grid, 256, FIT_SMEM_BYTES, st>>>(p);
    return cudaGetLastError();
}

}  // namespace

template <int W>
static cudaError_t launch_fit_mix_w(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st) {
    const int F = 240;
    const int T = m->T;
    float *D = (float *)(ws + L.gD);
    float *act = (float *)(ws + L.fit_act);
    const size_t S = (size_t)N * F;
    float *h1 = act, *t2 = act + S, *h2 = act + 2 * S, *gz3 = act + 3 * S, *h3 = act + 4 * S, *g2 = act + 5 * S,
          *gz2 = act + 6 * S, *gz1 = h2;
    const int *bin_start = (const int *)(ws + L.bin_start);
    const float *V2 = (const float *)m->fitV2_dev, *V3 = (const float *)m->fitV3_dev;
    const float *c2 = (const float *)m->fitc2_dev, *c3 = (const float *)m->fitc3_dev;
    const float *v4 = (const float *)m->fitv4_dev, *c4 = (const float *)m->fitc4_dev;
    const unsigned gy = (unsigned)((N + BM - 1) / BM);
    const unsigned nb8 = (unsigned)((N + 7) / 8);
    cudaError_t e = cudaSuccess;
    auto ok = [&](cudaError_t x) { if (e == cudaSuccess) e = x; };

    // first layer (K = 16 m2) on the tcgen05 kernel with hi + lo weights: h1 = tanh(D V1 + c1), D formed in its operand producer
    ok(launch_fit_tc32_first(m, N, g, ws, L, st));
    FitArgsF p{};
    p.ncell = g.ncell; p.bin_start = bin_start; p.v4 = v4; p.v4_type_stride = F; p.bias_type_stride = F;
    p.N = F; p.ldb = F; p.ldo = F;
    const dim3 g240(F / BN, gy, T);
    p.K = F; p.A = h1; p.lda = F; p.B = V2; p.b_type_stride = (long)F * F; p.bias = c2; p.aux0 = h1; p.out0 = t2; p.out1 = h2;
    ok(launch_gemm<1>(p, g240, st));
    p.A = h2; p.B = V3; p.bias = c3; p.aux0 = h2; p.out0 = gz3; p.out1 = h3;
    ok(launch_gemm<2>(p, g240, st));
    k_energy_f<<<nb8, 256, 0, st>>>(N, T, g.ncell, bin_start, h3, v4, c4, m->ebias_dev, (double *)(ws + L.eatom));
    p.A = gz3; p.B = V3; p.aux0 = t2; p.out0 = g2; p.out1 = gz2;
    ok(launch_gemm<3>(p, g240, st));
    p.A = gz2; p.B = V2; p.aux0 = g2; p.aux1 = h1; p.out0 = gz1; p.out1 = nullptr;
    ok(launch_gemm<4>(p, g240, st));
    // last product (N = 16 m2) on the tcgen05 kernel: gD is consumed in its epilogue, gA [N][4][m2] lands in the gD buffer
    ok(launch_fit_tc32_last(m, N, gz1, g, ws, L, st));
    if (!m->wide) {     // (the wide path of wide_gen.cu reads gA itself)
        k_gA_frag<2, W><<<(unsigned)((N + 3) / 4), 128, 0, st>>>(N, D, (uint32_t *)(ws + L.gAf), (float *)(ws + L.gscale));
        ok(cudaGetLastError());
    }
    return e;
}

cudaError_t launch_fit_mix(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st) {
    return m->m0 == 32 ? launch_fit_mix_w<32>(m, N, g, ws, L, st) : launch_fit_mix_w<25>(m, N, g, ws, L, st);
}
