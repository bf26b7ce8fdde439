// S3 + S4 + S7 + S8 + S9 (embedding backward, ProdForce, ProdViral) of SURVEY.md section 8(a), MIX-32 mode
// (PAPER.md:125): coordinates, environment matrix, switching function, its derivative, force and virial
// accumulation in fp64; the embedding net on fp16 tensor-core MMAs with fp32 accumulation (operand splitting gives
// single-precision products in MIX-32); tanh and tanh' in fp32; first embedding layer (K = 1) on the ALUs as in
// the paper ("do not meet the size requirements for using Tensor Cores").  See embed_mix.cuh for the layouts.
#include "embed_mix.cuh"

namespace {

__device__ __forceinline__ double min_image(double t, double L, double halfL) {
    double s = t > halfL ? -1.0 : (t < -halfL ? 1.0 : 0.0);
    return __dadd_rn(t, __dmul_rn(s, L));
}

struct EnvParams {
    double rc, rc_smth, inv_range;
    double L[3];
};

__device__ __forceinline__ void env_row(const EnvParams &p, double dx, double dy, double dz, double Rt[4],
                                        double *sp_out, double *r_out) {
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
    Rt[0] = s;
    Rt[1] = s * dx / r;
    Rt[2] = s * dy / r;
    Rt[3] = s * dz / r;
    if (sp_out) { *sp_out = dw / r - w / r2; *r_out = r; }
}

// Forward of one 16-row tile.  All C-layout arrays are X[tile][4] with index 2*row + j (row 0 = lane/4, row 1 = +8).
//   y1c[t][2row+j] : layer-1 slot q = 2t + j              t2c[nt] : tanh of layer-2 pre-activation
//   y2 = y1c[nt/2][2row + nt%2] + t2c[nt][.]              t3c[nt3]: tanh of layer-3 pre-activation
//   G  = y2(nt3/2)[2row + nt3%2] + t3c[nt3][.]
template <int NS, bool APPROX, int W>
__device__ __forceinline__ void forward_tile(const EmbedNetFragH<ns_wparts(NS), W> *__restrict__ net, int lane,
                                             float s0, float s1, float (&y1c)[4][4], float (&t2c)[HW<W>::HNT2][4],
                                             float (&t3c)[HW<W>::HNT3][4]) {
    constexpr int M2E = HW<W>::M2E, HNT2 = HW<W>::HNT2, HNT3 = HW<W>::HNT3;
    constexpr bool ODD2 = (HNT2 & 1) != 0;      // the K of HNT2 tiles ends with a k8 step
    (void)M2E; (void)ODD2;
    constexpr int NSW = ns_wparts(NS);
    const int r = lane & 3;
#pragma unroll
    for (int t = 0; t < 4; ++t)
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            const int e = 8 * t + 2 * r + j;
            const float w = net->w1[e], b = net->b1[e];
            y1c[t][j] = act_tanh<APPROX>(fmaf(s0, w, b));
            y1c[t][2 + j] = act_tanh<APPROX>(fmaf(s1, w, b));
        }
    // layer 2: K = 32 slots (2 k16 steps), N = 7 tiles
    {
        float acc[HNT2][4];
#pragma unroll
        for (int nt = 0; nt < HNT2; ++nt) {
            acc[nt][0] = acc[nt][2] = net->b2[nt * 8 + 2 * r];
            acc[nt][1] = acc[nt][3] = net->b2[nt * 8 + 2 * r + 1];
        }
#pragma unroll
        for (int s = 0; s < 2; ++s) {
            AFrag<NS> a;
            make_afrag<NS>(a, y1c[2 * s][0], y1c[2 * s][1], y1c[2 * s][2], y1c[2 * s][3], y1c[2 * s + 1][0],
                           y1c[2 * s + 1][1], y1c[2 * s + 1][2], y1c[2 * s + 1][3]);
#pragma unroll
            for (int nt = 0; nt < HNT2; ++nt)
                mma_k16<NS>(acc[nt], a, net->W2f[0][s][nt][lane], net->W2f[NSW - 1][s][nt][lane]);
        }
#pragma unroll
        for (int nt = 0; nt < HNT2; ++nt)
#pragma unroll
            for (int k = 0; k < 4; ++k) t2c[nt][k] = act_tanh<APPROX>(acc[nt][k]);
    }
    // layer 3: K = 56 positions (3 k16 + 1 k8), N = 14 tiles, two halves of 7 tiles
#pragma unroll
    for (int half = 0; half < 2; ++half) {
        float acc[HNT3 / 2][4];
#pragma unroll
        for (int t = 0; t < HNT3 / 2; ++t) {
            const int nt3 = half * (HNT3 / 2) + t;
            acc[t][0] = acc[t][2] = net->b3[nt3 * 8 + 2 * r];
            acc[t][1] = acc[t][3] = net->b3[nt3 * 8 + 2 * r + 1];
        }
#pragma unroll
        for (int s = 0; s < 4; ++s) {
            AFrag<NS> a;
            float v[2][4];
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int nt = 2 * s + h;
                if (nt < HNT2) {
#pragma unroll
                    for (int row = 0; row < 2; ++row)
#pragma unroll
                        for (int j = 0; j < 2; ++j)
                            v[h][2 * row + j] = y1c[nt >> 1][2 * row + (nt & 1)] + t2c[nt][2 * row + j];
                }
            }
            if (s < 3 || !ODD2) {
                make_afrag<NS>(a, v[0][0], v[0][1], v[0][2], v[0][3], v[1][0], v[1][1], v[1][2], v[1][3]);
#pragma unroll
                for (int t = 0; t < HNT3 / 2; ++t) {
                    const int nt3 = half * (HNT3 / 2) + t;
                    mma_k16<NS>(acc[t], a, net->W3f[0][s][nt3][lane], net->W3f[NSW - 1][s][nt3][lane]);
                }
            } else {
                make_afrag8<NS>(a, v[0][0], v[0][1], v[0][2], v[0][3]);
#pragma unroll
                for (int t = 0; t < HNT3 / 2; ++t) {
                    const int nt3 = half * (HNT3 / 2) + t;
                    mma_k8<NS>(acc[t], a, net->W3f[0][s][nt3][lane], net->W3f[NSW - 1][s][nt3][lane]);
                }
            }
        }
#pragma unroll
        for (int t = 0; t < HNT3 / 2; ++t) {
            const int nt3 = half * (HNT3 / 2) + t;
#pragma unroll
            for (int k = 0; k < 4; ++k) t3c[nt3][k] = act_tanh<APPROX>(acc[t][k]);
        }
    }
}

// G value of layer-3 tile nt3, element k = 2*row + j3
#define GVAL(nt3, k) ((y1c[(nt3) >> 2][((k) & 2) + (((nt3) >> 1) & 1)] + t2c[(nt3) >> 1][((k) & 2) + ((nt3) & 1)]) + t3c[nt3][k])

template <int NSW, int W>
__device__ __forceinline__ void copy_net_to_smem(EmbedNetFragH<NSW, W> *dst, const EmbedNetFragH<NSW, W> *__restrict__ src,
                                                 int nwords) {
    const uint32_t *s = reinterpret_cast<const uint32_t *>(src);
    uint32_t *d = reinterpret_cast<uint32_t *>(dst);
    for (int k = threadIdx.x; k < nwords; k += blockDim.x) d[k] = s[k];
}

constexpr int MIX_ROWCHUNK = 64;
constexpr int MIX_WARP_BUF_FLOATS = MIX_ROWCHUNK * 5;    // rbuf[64][4] + sbuf[64]

// ------------------------------------------------------------------------------------------------ backward
// gAf per atom (written by the mixed fitting backward, fit_mix.cu), per weight part p < NSW, 28*32 words:
//   [p][0..14)[lane]     dG  MMA (k8) B fragment of tile nt3:  (r < 2) ? half2(gA[2r][f], gA[2r+1][f]) : 0, f = f3(nt3, g/2, g%2)
//   [p][14 + 2s + h][lane] dR^ MMA (k16 step s) B registers h = 0,1: (g < 4) ? half2(gA[g][f3(2s+h, r, 0)], gA[g][f3(2s+h, r, 1)]) : 0
// all scaled by gscale[i] (a power of two that brings max|gA| near 1); results are multiplied by 1/(Nm*gscale).
template <int NS, int NSC, bool APPROX, int NSB, int W>
__global__ void __launch_bounds__(DP_WARPS_PER_CTA * 32, 1)
k_embed_bwd_mix(int T, int ncell, int Nm, const __grid_constant__ TypeTab tt, EnvParams ep, const EmbedNetFragH<ns_wparts(NS), W> *__restrict__ nets,
                const double *__restrict__ avg, const double *__restrict__ stdv, const int *__restrict__ bin_start,
                const double *__restrict__ xs, const int *__restrict__ nlist, const int *__restrict__ nreal,
                const uint32_t *__restrict__ gAf, const float *__restrict__ gscale, double *__restrict__ fsorted,
                double *__restrict__ virial, unsigned long long *__restrict__ row_counter) {
    constexpr int M2E = HW<W>::M2E, HNT2 = HW<W>::HNT2, HNT3 = HW<W>::HNT3;
    constexpr bool ODD2 = (HNT2 & 1) != 0;      // the K of HNT2 tiles ends with a k8 step
    (void)M2E; (void)ODD2;
    constexpr int NSW = ns_wparts(NS);
    constexpr int GP = 2 * HNT3;              // gA fragment words per weight part and lane: HNT3 dG tiles + HNT3 dR^ registers
    extern __shared__ __align__(16) uint32_t smem_u[];
    EmbedNetFragH<NSW, W> *net = reinterpret_cast<EmbedNetFragH<NSW, W> *>(smem_u);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    float *rbuf = reinterpret_cast<float *>(smem_u) + sizeof(EmbedNetFragH<NSW, W>) / 4 + wid * MIX_WARP_BUF_FLOATS;
    float *sbuf = rbuf + MIX_ROWCHUNK * 4;
    const int *sel = tt.sel;
    const int r = lane & 3, g = lane >> 2;
    const double hx = 0.5 * ep.L[0], hy = 0.5 * ep.L[1], hz = 0.5 * ep.L[2];
    unsigned long long my_rows = 0;
    double vir[9];
#pragma unroll
    for (int k = 0; k < 9; ++k) vir[k] = 0.0;

    for (int a = 0; a < T; ++a) {
        const int ts0 = bin_start[a * ncell], ts1 = bin_start[(a + 1) * ncell];
        if (ts0 == ts1) continue;
        double av[4], sd[4];
#pragma unroll
        for (int c = 0; c < 4; ++c) { av[c] = avg[4 * a + c]; sd[c] = stdv[4 * a + c]; }
        const float isd0 = (float)(1.0 / sd[2 * (r & 1)]), isd1 = (float)(1.0 / sd[2 * (r & 1) + 1]);
        int off = 0;
        for (int b = 0; b < T; ++b) {
            __syncthreads();
            copy_net_to_smem<NSW, W>(net, nets + (a * T + b), (int)(sizeof(EmbedNetFragH<NSW, W>) / 4));
            __syncthreads();
            // The eight warps of a CTA walk their atoms in lockstep, one barrier per 16-row tile: the unrolled tile body (95 KB of
            // code) then streams through the instruction cache once per tile for all eight warps instead of once per warp
            // (ncu: 2.5 no_instruction stalls per issue without it).  Loop bounds are CTA-uniform: sel[b] bounds the rows.
            for (int ibase = ts0 + blockIdx.x * DP_WARPS_PER_CTA; ibase < ts1; ibase += gridDim.x * DP_WARPS_PER_CTA) {
                const bool active = ibase + wid < ts1;
                const int i = active ? ibase + wid : ts0;
                const int nr = active ? nreal[i * T + b] : 0;
                const double xi = xs[3 * (long)i], yi = xs[3 * (long)i + 1], zi = xs[3 * (long)i + 2];
                const uint32_t *gf = gAf + (long)i * (2 * GP * 32);
                const float oscale = 1.0f / ((float)Nm * gscale[i]);
                double fi[3] = {0.0, 0.0, 0.0};
                for (int r0 = 0; r0 < sel[b]; r0 += MIX_ROWCHUNK) {
                    const int nrow_c = max(0, min(MIX_ROWCHUNK, nr - r0));
                    const int ntile = (nrow_c + HROWS - 1) / HROWS;
                    const int ntile_u = (min(MIX_ROWCHUNK, sel[b] - r0) + HROWS - 1) / HROWS;      // CTA-uniform
                    for (int rr = lane; rr < ntile * HROWS; rr += 32) {
                        const int row = r0 + rr;
                        double Rt[4] = {0.0, 0.0, 0.0, 0.0};
                        if (row < nr) {
                            const int j = nlist[(long)i * Nm + off + row];
                            const double dx = min_image(xs[3 * (long)j] - xi, ep.L[0], hx);
                            const double dy = min_image(xs[3 * (long)j + 1] - yi, ep.L[1], hy);
                            const double dz = min_image(xs[3 * (long)j + 2] - zi, ep.L[2], hz);
                            env_row(ep, dx, dy, dz, Rt, nullptr, nullptr);
                        }
#pragma unroll
                        for (int c = 0; c < 4; ++c) rbuf[rr * 4 + c] = (float)((Rt[c] - av[c]) / sd[c]);
                        sbuf[rr] = rbuf[rr * 4];
                    }
                    __syncwarp();
                    for (int t = 0; t < ntile_u; ++t) {
                        __syncthreads();
                        if (t >= ntile) continue;
                        float y1c[4][4], t2c[HNT2][4], t3c[HNT3][4];
                        forward_tile<NS, APPROX, W>(net, lane, sbuf[t * HROWS + g], sbuf[t * HROWS + g + 8], y1c, t2c, t3c);
                        // dR^[row][c] = sum_m G[row][m] gA[c][m]     (C: c0,c1 row g c=2r,2r+1 ; c2,c3 row g+8)
                        float dR[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
                        for (int s = 0; s < HNT3 / 2; ++s) {
                            AFrag<NSC> a_;
                            const int ta = 2 * s, tb = 2 * s + 1;
                            make_afrag<NSC>(a_, GVAL(ta, 0), GVAL(ta, 1), GVAL(ta, 2), GVAL(ta, 3), GVAL(tb, 0), GVAL(tb, 1),
                                           GVAL(tb, 2), GVAL(tb, 3));
                            uint32_t bh[2], bl[2];
                            bh[0] = gf[(HNT3 + 2 * s) * 32 + lane]; bh[1] = gf[(HNT3 + 1 + 2 * s) * 32 + lane];
                            if (NSC == 3) { bl[0] = gf[(GP + HNT3 + 2 * s) * 32 + lane]; bl[1] = gf[(GP + HNT3 + 1 + 2 * s) * 32 + lane]; }
                            else { bl[0] = bl[1] = 0; }
                            mma_k16<NSC>(dR, a_, bh, bl);
                        }
                        // dG = R^ gA ; dz3 = dG (1 - t3^2) (stored over t3c) ; residual dy2[nt3] = dG[.,0] + dG[.,1]
                        float dy2[HNT2][4];
                        {
                            AFrag<NSC> ar;
                            const float *rb = rbuf + t * HROWS * 4;
                            const float v0 = r < 2 ? rb[g * 4 + 2 * r] : 0.f, v1 = r < 2 ? rb[g * 4 + 2 * r + 1] : 0.f;
                            const float v2 = r < 2 ? rb[(g + 8) * 4 + 2 * r] : 0.f, v3 = r < 2 ? rb[(g + 8) * 4 + 2 * r + 1] : 0.f;
                            make_afrag8<NSC>(ar, v0, v1, v2, v3);
#pragma unroll
                            for (int nt3 = 0; nt3 < HNT3; ++nt3) {
                                float d[4] = {0.f, 0.f, 0.f, 0.f};
                                uint32_t bh[1], bl[1];
                                bh[0] = gf[nt3 * 32 + lane];
                                bl[0] = NSC == 3 ? gf[(GP + nt3) * 32 + lane] : 0u;
                                mma_k8<NSC>(d, ar, bh, bl);
#pragma unroll
                                for (int k = 0; k < 4; ++k) d[k] *= oscale;
                                dy2[nt3 >> 1][(nt3 & 1)] = d[0] + d[1];
                                dy2[nt3 >> 1][2 + (nt3 & 1)] = d[2] + d[3];
#pragma unroll
                                for (int k = 0; k < 4; ++k) t3c[nt3][k] = d[k] * (1.f - t3c[nt3][k] * t3c[nt3][k]);
                            }
                        }
                        // dy2 += dz3 W3^T   (K = 14 tiles = 7 k16 steps, N = 7 tiles)
#pragma unroll
                        for (int s = 0; s < HNT3 / 2; ++s) {
                            AFrag<NSB> a_;
                            make_afrag<NSB>(a_, t3c[2 * s][0], t3c[2 * s][1], t3c[2 * s][2], t3c[2 * s][3], t3c[2 * s + 1][0],
                                           t3c[2 * s + 1][1], t3c[2 * s + 1][2], t3c[2 * s + 1][3]);
#pragma unroll
                            for (int nt2 = 0; nt2 < HNT2; ++nt2)
                                mma_k16<NSB>(dy2[nt2], a_, net->W3Tf[0][s][nt2][lane], net->W3Tf[NSW - 1][s][nt2][lane]);
                        }
                        // residual dy1 (slot q = 2t + j1 <- dy2 tile q, both j2) ; dz2 = dy2 (1 - t2^2)
                        float dy1[4][4];
#pragma unroll
                        for (int q = 0; q < 8; ++q) {
                            dy1[q >> 1][(q & 1)] = q < HNT2 ? dy2[q][0] + dy2[q][1] : 0.f;
                            dy1[q >> 1][2 + (q & 1)] = q < HNT2 ? dy2[q][2] + dy2[q][3] : 0.f;
                        }
#pragma unroll
                        for (int nt2 = 0; nt2 < HNT2; ++nt2)
#pragma unroll
                            for (int k = 0; k < 4; ++k) dy2[nt2][k] *= (1.f - t2c[nt2][k] * t2c[nt2][k]);
                        // dy1 += dz2 W2^T   (K = 7 tiles = 3 k16 + 1 k8, N = 4 tiles of y1 slots)
#pragma unroll
                        for (int s = 0; s < 4; ++s) {
                            AFrag<NSB> a_;
                            if (s < 3 || !ODD2) {
                                constexpr int LAST = HNT2 - 1;
                                const int ta_ = 2 * s, tb_ = 2 * s + 1 <= LAST ? 2 * s + 1 : LAST;
                                make_afrag<NSB>(a_, dy2[ta_][0], dy2[ta_][1], dy2[ta_][2], dy2[ta_][3], dy2[tb_][0],
                                               dy2[tb_][1], dy2[tb_][2], dy2[tb_][3]);
#pragma unroll
                                for (int t1 = 0; t1 < 4; ++t1)
                                    mma_k16<NSB>(dy1[t1], a_, net->W2Tf[0][s][t1][lane], net->W2Tf[NSW - 1][s][t1][lane]);
                            } else {
                                make_afrag8<NSB>(a_, dy2[HNT2 - 1][0], dy2[HNT2 - 1][1], dy2[HNT2 - 1][2], dy2[HNT2 - 1][3]);
#pragma unroll
                                for (int t1 = 0; t1 < 4; ++t1)
                                    mma_k8<NSB>(dy1[t1], a_, net->W2Tf[0][s][t1][lane], net->W2Tf[NSW - 1][s][t1][lane]);
                            }
                        }
                        // layer 1: ds[row] = sum_e dy1 (1 - y1^2) W1[e]
                        float ds0 = 0.f, ds1 = 0.f;
#pragma unroll
                        for (int t1 = 0; t1 < 4; ++t1)
#pragma unroll
                            for (int j = 0; j < 2; ++j) {
                                const float w = net->w1[8 * t1 + 2 * r + j];
                                ds0 = fmaf(dy1[t1][j] * (1.f - y1c[t1][j] * y1c[t1][j]), w, ds0);
                                ds1 = fmaf(dy1[t1][2 + j] * (1.f - y1c[t1][2 + j] * y1c[t1][2 + j]), w, ds1);
                            }
                        ds0 += __shfl_xor_sync(0xffffffffu, ds0, 1); ds0 += __shfl_xor_sync(0xffffffffu, ds0, 2);
                        ds1 += __shfl_xor_sync(0xffffffffu, ds1, 1); ds1 += __shfl_xor_sync(0xffffffffu, ds1, 2);
#pragma unroll
                        for (int k = 0; k < 4; ++k) dR[k] *= oscale;
                        if (r == 0) { dR[0] += ds0; dR[2] += ds1; }
                        __syncwarp();
                        if (r < 2) {
                            float *rb = rbuf + t * HROWS * 4;
                            rb[g * 4 + 2 * r] = dR[0] * isd0; rb[g * 4 + 2 * r + 1] = dR[1] * isd1;
                            rb[(g + 8) * 4 + 2 * r] = dR[2] * isd0; rb[(g + 8) * 4 + 2 * r + 1] = dR[3] * isd1;
                        }
                    }
                    my_rows += (unsigned long long)ntile * HROWS;
                    __syncwarp();
                    for (int rr = lane; rr < nrow_c; rr += 32) {
                        const int j = nlist[(long)i * Nm + off + r0 + rr];
                        const double dx = min_image(xs[3 * (long)j] - xi, ep.L[0], hx);
                        const double dy = min_image(xs[3 * (long)j + 1] - yi, ep.L[1], hy);
                        const double dz = min_image(xs[3 * (long)j + 2] - zi, ep.L[2], hz);
                        double Rt[4], sp, rl;
                        env_row(ep, dx, dy, dz, Rt, &sp, &rl);
                        const double s = Rt[0];
                        const double g0 = rbuf[rr * 4], g1 = rbuf[rr * 4 + 1], g2 = rbuf[rr * 4 + 2], g3 = rbuf[rr * 4 + 3];
                        const double d[3] = {dx, dy, dz};
                        const double gd = g1 * dx + g2 * dy + g3 * dz;
                        const double coef = (sp / rl - s / (rl * rl)) / rl;
                        double gk[3];
#pragma unroll
                        for (int bb = 0; bb < 3; ++bb)
                            gk[bb] = g0 * sp * d[bb] / rl + coef * d[bb] * gd + (s / rl) * (bb == 0 ? g1 : (bb == 1 ? g2 : g3));
#pragma unroll
                        for (int bb = 0; bb < 3; ++bb) {
                            fi[bb] += gk[bb];
                            atomicAdd(&fsorted[3 * (long)j + bb], -gk[bb]);
                        }
#pragma unroll
                        for (int aa = 0; aa < 3; ++aa)
#pragma unroll
                            for (int bb = 0; bb < 3; ++bb) vir[3 * aa + bb] -= d[aa] * gk[bb];
                    }
                    __syncwarp();
                }
#pragma unroll
                for (int bb = 0; bb < 3; ++bb) {
                    double v = fi[bb];
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
                    if (lane == 0 && nr > 0) atomicAdd(&fsorted[3 * (long)i + bb], v);
                }
            }
            off += sel[b];
        }
    }
#pragma unroll
    for (int k = 0; k < 9; ++k) {
        double v = vir[k];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0 && v != 0.0) atomicAdd(&virial[k], v);
    }
    if (lane == 0 && my_rows) atomicAdd(row_counter, my_rows);
}

EnvParams make_env(const dp_model *m, const Grid3 &g) {
    EnvParams ep;
    ep.rc = m->rc; ep.rc_smth = m->rc_smth; ep.inv_range = 1.0 / (m->rc - m->rc_smth);
    ep.L[0] = g.L[0]; ep.L[1] = g.L[1]; ep.L[2] = g.L[2];
    return ep;
}

template <int NS, int W>
int smem_bytes() {
    return (int)sizeof(EmbedNetFragH<ns_wparts(NS), W>) + DP_WARPS_PER_CTA * MIX_WARP_BUF_FLOATS * 4;
}

int embed_grid(const dp_model *m, long N) {
    long grid = (N + DP_WARPS_PER_CTA - 1) / DP_WARPS_PER_CTA;
    return (int)(grid > m->num_sms ? m->num_sms : grid);
}

template <int NS, int NSC, bool APPROX, int NSB, int W>
cudaError_t launch_bwd(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st) {
    DP_SMEM_OPTIN((k_embed_bwd_mix<NS, NSC, APPROX, NSB, W>), (smem_bytes<NS, W>()));
    const TypeTab tt = make_typetab(m);
    k_embed_bwd_mix<NS, NSC, APPROX, NSB, W><<<embed_grid(m, N), DP_WARPS_PER_CTA * 32, smem_bytes<NS, W>(), st>>>(
        m->T, g.ncell, m->Nm, tt, make_env(m, g), (const EmbedNetFragH<ns_wparts(NS), W> *)m->embed_frag_dev, m->avg_dev,
        m->std_dev, (int *)(ws + L.bin_start), (double *)(ws + L.xs), (int *)(ws + L.nlist), (int *)(ws + L.nreal),
        (const uint32_t *)(ws + L.gAf), (const float *)(ws + L.gscale), (double *)(ws + L.fsorted),
        (double *)(ws + L.virial), (unsigned long long *)(ws + L.status + 16));
    return cudaGetLastError();
}

}  // namespace

// MIX-32 ("all the arithmetic operations ... in single precision"): every operand split hi + lo, exact tanhf
cudaError_t launch_embed_bwd_mix(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st) {
    return m->m0 == 32 ? launch_bwd<3, 3, false, 3, 32>(m, N, g, ws, L, st) : launch_bwd<3, 3, false, 3, 25>(m, N, g, ws, L, st);
}
