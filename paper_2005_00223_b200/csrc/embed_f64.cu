// S3 + S4 + S5 (forward) and S3 + S4 + S7 + S8 + S9 (backward) of SURVEY.md section 8(a), FP64 mode.
//
// Environment matrix rows are recomputed from the neighbour list and coordinates (never stored in HBM,
// PAPER.md:125 keeps them fp64), pushed through the embedding net 1->25->50->100
// with FP64 tensor-core MMAs (DMMA m8n8k4) whose accumulator fragments are chained in registers from layer to
// layer, and contracted with R^ into A_i = R^T G / Nm, so G never leaves the SM (BASELINE north_star).
// The backward kernel recomputes the forward (trading flops for memory, the opposite choice to PAPER.md:137,
// see DESIGN.md), applies tanh' = 1 - tanh^2, and finishes with ProdForce / ProdViral
// (PAPER.md:121).
//
// Register chaining: an m8n8k4 C fragment holds (row = lane/4, cols 2*(lane%4)+{0,1}); an A fragment holds
// (row = lane/4, k = lane%4).  Because the k index of a product can be permuted freely as long as both
// operands agree, the two C registers of an 8-wide output tile are used directly as two A fragments of the
// next layer; the weights are stored pre-permuted in "fragment order" by dp_create (dp_internal.h).
#include "dp_internal.h"
#include "tanh64.cuh"

namespace {

__device__ __forceinline__ void dmma(double &c0, double &c1, double a, double b) {
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
        : "+d"(c0), "+d"(c1)
        : "d"(a), "d"(b));
}

// tanh64.cuh: branch-free, 24 fp64-pipe operations, |error| <= 2.3e-16 (inlined: the lockstep tile loops below keep the
// instruction cache fed; a called copy was faster only before them)
__device__ __forceinline__ double dp_tanh(double x) { return dp_tanh64(x); }

__device__ __forceinline__ double min_image(double t, double L, double halfL) {
    double s = t > halfL ? -1.0 : (t < -halfL ? 1.0 : 0.0);
    return __dadd_rn(t, __dmul_rn(s, L));
}

struct EnvParams {
    double rc, rc_smth, inv_range;   // 1/(rc - rc_smth)
    double L[3];
};

// N4 (+ N9 when DERIV): R~ = s (1, d/r), s = w(r)/r; optional derivative pieces.
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

// Forward of one 8-row tile.  s = s^ of row lane/4.  Outputs (registers):
//   y1[kc]  layer-1 output, slot (kc, r=lane%4)
//   t2[p]   tanh of layer-2 pre-activation at position p = 2*nt2 + j2 ;  y2[p] = y1[p>>1] + t2[p]
//   t3[q]   tanh of layer-3 pre-activation at position q = 2*nt3 + j3 ;  G[q]  = y2[q>>1] + t3[q]
template <int W>
__device__ __forceinline__ void embed_forward_tile(const EmbedNetFrag<double, W> *__restrict__ net, int lane, double s,
                                                   double (&y1)[EmbW<W>::KC1], double (&t2)[2 * EmbW<W>::NT2], double (&t3)[2 * EmbW<W>::NT3]) {
    constexpr int M0 = EmbW<W>::M0, M1 = EmbW<W>::M1, M2E = EmbW<W>::M2E, KC1 = EmbW<W>::KC1, NT2 = EmbW<W>::NT2, NT3 = EmbW<W>::NT3, NT1 = EmbW<W>::NT1;
    (void)M0; (void)M1; (void)M2E; (void)KC1; (void)NT2; (void)NT3; (void)NT1;
    const int r = lane & 3;
#pragma unroll
    for (int kc = 0; kc < KC1; ++kc) y1[kc] = dp_tanh(fma(s, net->w1[4 * kc + r], net->b1[4 * kc + r]));
    {
        double acc[NT2][2];
#pragma unroll
        for (int nt = 0; nt < NT2; ++nt) {
            acc[nt][0] = net->b2[nt * 8 + 2 * r];
            acc[nt][1] = net->b2[nt * 8 + 2 * r + 1];
        }
#pragma unroll
        for (int kc = 0; kc < KC1; ++kc) {
#pragma unroll
            for (int nt = 0; nt < NT2; ++nt) dmma(acc[nt][0], acc[nt][1], y1[kc], net->W2f[(kc * NT2 + nt) * 32 + lane]);
        }
#pragma unroll
        for (int nt = 0; nt < NT2; ++nt) {
            t2[2 * nt] = dp_tanh(acc[nt][0]);
            t2[2 * nt + 1] = dp_tanh(acc[nt][1]);
        }
    }
#pragma unroll
    for (int half = 0; half < 2; ++half) {
        double acc[NT3 / 2][2];
#pragma unroll
        for (int t = 0; t < NT3 / 2; ++t) {
            const int nt3 = half * (NT3 / 2) + t;
            acc[t][0] = net->b3[nt3 * 8 + 2 * r];
            acc[t][1] = net->b3[nt3 * 8 + 2 * r + 1];
        }
#pragma unroll
        for (int kc = 0; kc < 2 * NT2; ++kc) {
            const double a = y1[kc >> 1] + t2[kc];
#pragma unroll
            for (int t = 0; t < NT3 / 2; ++t) {
                const int nt3 = half * (NT3 / 2) + t;
                dmma(acc[t][0], acc[t][1], a, net->W3f[(kc * NT3 + nt3) * 32 + lane]);
            }
        }
#pragma unroll
        for (int t = 0; t < NT3 / 2; ++t) {
            const int nt3 = half * (NT3 / 2) + t;
            t3[2 * nt3] = dp_tanh(acc[t][0]);
            t3[2 * nt3 + 1] = dp_tanh(acc[t][1]);
        }
    }
}

// logical layer-3 feature of internal position (nt3, r, j3); -1 for padding
template <int W>
__device__ __forceinline__ int feature3(int nt3, int r, int j3) {
    const int e = 4 * (nt3 >> 1) + r;
    return e < W ? e + W * (nt3 & 1) + 2 * W * j3 : -1;
}

// Stage one (centre type, neighbour type) net in shared memory: ONE bulk copy (cp.async.bulk, completion on an mbarrier) issued
// by thread 0; every thread waits on the barrier.  (A loop of per-thread loads took 20-50 us per net: a third of the forward
// at 500 atoms.)  Callers bracket it with __syncthreads(); phase = parity of the number of copies this CTA has made.
__device__ __forceinline__ void stage_net(double *dst, const double *__restrict__ src, int n, uint64_t *bar, uint32_t &phase) {
    const uint32_t b = (uint32_t)__cvta_generic_to_shared(bar);
    if (threadIdx.x == 0) {
        const uint32_t bytes = (uint32_t)n * 8u;
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(b), "r"(bytes) : "memory");
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                     ::"r"((uint32_t)__cvta_generic_to_shared(dst)), "l"(src), "r"(bytes), "r"(b) : "memory");
    }
    asm volatile("{\n.reg .pred p;\nSW_%=:\nmbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n@p bra SD_%=;\nbra SW_%=;\nSD_%=:\n}"
                 ::"r"(b), "r"(phase) : "memory");
    phase ^= 1u;
}
__device__ __forceinline__ void stage_init(uint64_t *bar) {
    if (threadIdx.x == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"((uint32_t)__cvta_generic_to_shared(bar)));
        asm volatile("fence.mbarrier_init.release.cluster;");
    }
    __syncthreads();
}

template <int W> __host__ __device__ constexpr int fwd_net_doubles() {
    using E = EmbW<W>;
    return E::KC1 * 4 * 2 + E::NT2 * 8 + E::NT3 * 8 + E::KC1 * E::NT2 * 32 + E::NT3 * E::NT3 * 32;
}
template <int W> __host__ __device__ constexpr int bwd_net_doubles() { return (int)(sizeof(EmbedNetFrag<double, W>) / sizeof(double)); }
constexpr int WARP_BUF_DOUBLES = ROWCHUNK * 5;   // rbuf[ROWCHUNK][4] + sbuf[ROWCHUNK]

// ------------------------------------------------------------------------------------------------ forward
template <int W>
__global__ void __launch_bounds__(DP_WARPS_PER_CTA * 32, 1)
k_embed_fwd_f64(int T, int ncell, int Nm, int CH, const __grid_constant__ TypeTab tt, EnvParams ep, const EmbedNetFrag<double, W> *__restrict__ nets,
                const double *__restrict__ avg, const double *__restrict__ stdv, const int *__restrict__ bin_start,
                const double *__restrict__ xs, const int *__restrict__ nlist, const int *__restrict__ nreal,
                double *__restrict__ Aout, unsigned long long *__restrict__ row_counter) {
    constexpr int M0 = EmbW<W>::M0, M1 = EmbW<W>::M1, M2E = EmbW<W>::M2E, KC1 = EmbW<W>::KC1, NT2 = EmbW<W>::NT2, NT3 = EmbW<W>::NT3, NT1 = EmbW<W>::NT1;
    (void)M0; (void)M1; (void)M2E; (void)KC1; (void)NT2; (void)NT3; (void)NT1;
    constexpr int FWD_NET_DOUBLES = fwd_net_doubles<W>();
    static_assert(FWD_NET_DOUBLES % 2 == 0 && sizeof(EmbedNetFrag<double, W>) % 16 == 0, "bulk copies move multiples of 16 bytes");
    extern __shared__ __align__(16) double smem[];
    __shared__ uint64_t stage_bar;
    uint32_t stage_phase = 0;
    stage_init(&stage_bar);
    EmbedNetFrag<double, W> *net = reinterpret_cast<EmbedNetFrag<double, W> *>(smem);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    double *rbuf = smem + FWD_NET_DOUBLES + wid * WARP_BUF_DOUBLES;
    double *sbuf = rbuf + ROWCHUNK * 4;
    const int *sel = tt.sel;
    const int NW = gridDim.x * DP_WARPS_PER_CTA;
    const int r = lane & 3, q4 = lane >> 2;
    const double inv_nm = 1.0 / (double)Nm;
    const double hx = 0.5 * ep.L[0], hy = 0.5 * ep.L[1], hz = 0.5 * ep.L[2];
    unsigned long long my_rows = 0;

    for (int a = 0; a < T; ++a) {
        const int ts0 = bin_start[a * ncell], ts1 = bin_start[(a + 1) * ncell];
        if (ts0 == ts1) continue;
        double av[4], sd[4];
#pragma unroll
        for (int c = 0; c < 4; ++c) { av[c] = avg[4 * a + c]; sd[c] = stdv[4 * a + c]; }
        int off = 0;
        for (int b = 0; b < T; ++b) {
            __syncthreads();
            stage_net(smem, reinterpret_cast<const double *>(nets + (a * T + b)), FWD_NET_DOUBLES, &stage_bar, stage_phase);
            __syncthreads();
            // work item = (atom, row chunk).  CH == ROWCHUNK (large systems): one item per atom walks all its chunks and writes
            // A_i itself.  CH < ROWCHUNK (systems with fewer atoms than warps): S items per atom, one chunk of CH rows each, so
            // that every warp has work; their partial sums meet in A_i (zeroed by the launcher) through fp64 atomics.
            // The items are walked in LOCKSTEP: the eight warps of a CTA meet at a barrier before every 8-row tile, so that the
            // unrolled tile body (90 KB of code) streams through the instruction cache once per tile for all of them instead of
            // once per warp (ncu: 2.2 no_instruction stalls per issue without it).  All loop bounds are CTA-uniform: sel[b] + 1
            // bounds the rows.
            // (Split items, S > 1, run free: measured slower in lockstep, their empty items would idle at the barriers.)
            const int S = CH == ROWCHUNK ? 1 : (sel[b] + CH) / CH;
            const bool LS = S == 1;
            const long nitems = (long)(ts1 - ts0) * S;
            for (long itb = LS ? (long)blockIdx.x * DP_WARPS_PER_CTA : (long)blockIdx.x * DP_WARPS_PER_CTA + wid; itb < nitems; itb += NW) {
                const long it = LS ? itb + wid : itb;
                const bool active = it < nitems;
                const int i = active ? ts0 + (int)(it / S) : ts0, part = active ? (int)(it % S) : 0;
                const int nr = active ? nreal[i * T + b] : 0;
                const int npad = sel[b] - nr;
                const int rows = active ? nr + (npad > 0 ? 1 : 0) : 0;
                if (!LS && part * CH >= rows) continue;
                const int rows_u = LS ? sel[b] + 1 : rows;          // bound of the chunk loop (CTA-uniform in lockstep)
                const double xi = xs[3 * (long)i], yi = xs[3 * (long)i + 1], zi = xs[3 * (long)i + 2];
                double accA[NT3][2];
#pragma unroll
                for (int t = 0; t < NT3; ++t) accA[t][0] = accA[t][1] = 0.0;
                for (int r0 = part * CH; r0 < rows_u; r0 += S * CH) {
                    const int nrow_c = max(0, min(CH, rows - r0));
                    const int ntile = (nrow_c + 7) >> 3;
                    const int ntile_u = LS ? (min(CH, rows_u - r0) + 7) >> 3 : ntile;
                    // pre-pass: weighted R^ rows and s^ of this chunk
                    for (int rr = lane; rr < ntile * 8; rr += 32) {
                        const int row = r0 + rr;
                        double Rt[4] = {0.0, 0.0, 0.0, 0.0};
                        double wgt = 0.0;
                        if (row < nr) {
                            const int j = nlist[(long)i * Nm + off + row];
                            const double dx = min_image(xs[3 * (long)j] - xi, ep.L[0], hx);
                            const double dy = min_image(xs[3 * (long)j + 1] - yi, ep.L[1], hy);
                            const double dz = min_image(xs[3 * (long)j + 2] - zi, ep.L[2], hz);
                            env_row(ep, dx, dy, dz, Rt, nullptr, nullptr);
                            wgt = 1.0;
                        } else if (row == nr && npad > 0) {
                            wgt = (double)npad;      // all padded slots of the block share this row (R~ = 0)
                        }
                        double Rh0 = (Rt[0] - av[0]) / sd[0];
                        sbuf[rr] = Rh0;
                        rbuf[rr * 4 + 0] = wgt * Rh0;
#pragma unroll
                        for (int c = 1; c < 4; ++c) rbuf[rr * 4 + c] = wgt * ((Rt[c] - av[c]) / sd[c]);
                    }
                    __syncwarp();
                    for (int t = 0; t < ntile_u; ++t) {
                        if (LS) __syncthreads();
                        if (t >= ntile) continue;
                        double y1[KC1], t2[2 * NT2], t3[2 * NT3];
                        embed_forward_tile<W>(net, lane, sbuf[t * 8 + q4], y1, t2, t3);
                        // G in C-fragment layout -> B fragments of the contraction A^T[c][m] += R^[k][c] G[k][m]
#pragma unroll
                        for (int g = 0; g < 2; ++g) {
                            const double ahat = q4 < 4 ? rbuf[(t * 8 + 4 * g + r) * 4 + q4] : 0.0;
                            const int src = 16 * g + 4 * r + (q4 >> 1);
#pragma unroll
                            for (int nt3 = 0; nt3 < NT3; ++nt3) {
                                const double y2 = y1[nt3 >> 1] + t2[nt3];
                                const double g0 = y2 + t3[2 * nt3], g1 = y2 + t3[2 * nt3 + 1];
                                const double v0 = __shfl_sync(0xffffffffu, g0, src);
                                const double v1 = __shfl_sync(0xffffffffu, g1, src);
                                dmma(accA[nt3][0], accA[nt3][1], ahat, (q4 & 1) ? v1 : v0);
                            }
                        }
                    }
                    my_rows += (unsigned long long)ntile * 8;
                    __syncwarp();
                }
                // accA: (c = lane/4, feature of (nt3, r, j)); lanes with c >= 4 hold zeros
                if (q4 < 4 && active) {
                    double *Ai = Aout + ((long)i * 4 + q4) * M2E;
#pragma unroll
                    for (int nt3 = 0; nt3 < NT3; ++nt3) {
#pragma unroll
                        for (int j = 0; j < 2; ++j) {
                            const int f = feature3<W>(nt3, r, j);
                            if (f >= 0) {
                                const double v = accA[nt3][j] * inv_nm;
                                if (S > 1) atomicAdd(&Ai[f], v);
                                else Ai[f] = (b == 0) ? v : Ai[f] + v;
                            }
                        }
                    }
                }
            }
            off += sel[b];
        }
    }
    if (lane == 0 && my_rows) atomicAdd(row_counter, my_rows);
}

// ------------------------------------------------------------------------------------------------ backward
// gAf: per atom 42 fragments of 32 doubles, already scaled by 1/Nm (written by the fitting backward):
//   [0..14)  : dG MMA   B fragment of tile nt3: lane -> gA[c = lane%4][feature3(nt3, (lane/4)/2, (lane/4)%2)]
//   [14..42) : dR^ MMA  B fragment of chunk kc = 2*nt3 + j3: lane -> (lane/4 < 4) ? gA[c = lane/4][feature3(nt3, lane%4, j3)] : 0
template <int W>
__global__ void __launch_bounds__(DP_WARPS_PER_CTA * 32, 1)
k_embed_bwd_f64(int T, int ncell, int Nm, int CH, const __grid_constant__ TypeTab tt, EnvParams ep, const EmbedNetFrag<double, W> *__restrict__ nets,
                const double *__restrict__ avg, const double *__restrict__ stdv, const int *__restrict__ bin_start,
                const double *__restrict__ xs, const int *__restrict__ nlist, const int *__restrict__ nreal,
                const double *__restrict__ gAf, double *__restrict__ fsorted, double *__restrict__ virial,
                unsigned long long *__restrict__ row_counter) {
    constexpr int M0 = EmbW<W>::M0, M1 = EmbW<W>::M1, M2E = EmbW<W>::M2E, KC1 = EmbW<W>::KC1, NT2 = EmbW<W>::NT2, NT3 = EmbW<W>::NT3, NT1 = EmbW<W>::NT1;
    (void)M0; (void)M1; (void)M2E; (void)KC1; (void)NT2; (void)NT3; (void)NT1;
    constexpr int BWD_NET_DOUBLES = bwd_net_doubles<W>();
    extern __shared__ __align__(16) double smem[];
    __shared__ uint64_t stage_bar;
    uint32_t stage_phase = 0;
    stage_init(&stage_bar);
    EmbedNetFrag<double, W> *net = reinterpret_cast<EmbedNetFrag<double, W> *>(smem);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    double *rbuf = smem + BWD_NET_DOUBLES + wid * WARP_BUF_DOUBLES;
    double *sbuf = rbuf + ROWCHUNK * 4;
    const int *sel = tt.sel;
    const int NW = gridDim.x * DP_WARPS_PER_CTA;
    const int r = lane & 3, q4 = lane >> 2;
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
        int off = 0;
        for (int b = 0; b < T; ++b) {
            __syncthreads();
            stage_net(smem, reinterpret_cast<const double *>(nets + (a * T + b)), BWD_NET_DOUBLES, &stage_bar, stage_phase);
            __syncthreads();
            const int S = CH == ROWCHUNK ? 1 : (sel[b] + CH) / CH;       // work items per atom; lockstep when S == 1 (see the forward kernel)
            const bool LS = S == 1;
            const long nitems = (long)(ts1 - ts0) * S;
            for (long itb = LS ? (long)blockIdx.x * DP_WARPS_PER_CTA : (long)blockIdx.x * DP_WARPS_PER_CTA + wid; itb < nitems; itb += NW) {
                const long it = LS ? itb + wid : itb;
                const bool active = it < nitems;
                const int i = active ? ts0 + (int)(it / S) : ts0, part = active ? (int)(it % S) : 0;
                const int nr = active ? nreal[i * T + b] : 0;
                if (!LS && part * CH >= nr) continue;
                const int rows_u = LS ? sel[b] : nr;
                const double xi = xs[3 * (long)i], yi = xs[3 * (long)i + 1], zi = xs[3 * (long)i + 2];
                const double *gf = gAf + (long)i * (3 * NT3 * 32);
                double fi[3] = {0.0, 0.0, 0.0};
                for (int r0 = part * CH; r0 < rows_u; r0 += S * CH) {
                    const int nrow_c = max(0, min(CH, nr - r0));
                    const int ntile = (nrow_c + 7) >> 3;
                    const int ntile_u = LS ? (min(CH, rows_u - r0) + 7) >> 3 : ntile;
                    for (int rr = lane; rr < ntile * 8; rr += 32) {
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
                        for (int c = 0; c < 4; ++c) rbuf[rr * 4 + c] = (Rt[c] - av[c]) / sd[c];
                        sbuf[rr] = rbuf[rr * 4];
                    }
                    __syncwarp();
                    for (int t = 0; t < ntile_u; ++t) {
                        if (LS) __syncthreads();
                        if (t >= ntile) continue;
                        double y1[KC1], t2[2 * NT2], t3[2 * NT3];
                        embed_forward_tile<W>(net, lane, sbuf[t * 8 + q4], y1, t2, t3);
                        const double rfrag = rbuf[(t * 8 + q4) * 4 + r];
                        // dR^[row][c] = sum_m gA[c][m] G[row][m]      (C frag: c = 2r + {0,1}, valid for r < 2)
                        double dR0 = 0.0, dR1 = 0.0;
#pragma unroll
                        for (int kc = 0; kc < 2 * NT3; ++kc) {
                            const double gval = (y1[kc >> 2] + t2[kc >> 1]) + t3[kc];
                            dmma(dR0, dR1, gval, gf[(NT3 + kc) * 32 + lane]);
                        }
                        // dG[row][m] = sum_c R^[row][c] gA[c][m] ; dz3 = dG (1 - t3^2) ; residual dy2 = dG[f] + dG[f+50]
                        double dy2[2 * NT2];
#pragma unroll
                        for (int nt3 = 0; nt3 < NT3; ++nt3) {
                            double d0 = 0.0, d1 = 0.0;
                            dmma(d0, d1, rfrag, gf[nt3 * 32 + lane]);
                            dy2[nt3] = d0 + d1;
                            t3[2 * nt3] = d0 * (1.0 - t3[2 * nt3] * t3[2 * nt3]);
                            t3[2 * nt3 + 1] = d1 * (1.0 - t3[2 * nt3 + 1] * t3[2 * nt3 + 1]);
                        }
                        // dy2 += dz3 W3^T
#pragma unroll
                        for (int kc = 0; kc < 2 * NT3; ++kc) {
#pragma unroll
                            for (int nt2 = 0; nt2 < NT2; ++nt2)
                                dmma(dy2[2 * nt2], dy2[2 * nt2 + 1], t3[kc], net->W3Tf[(kc * NT2 + nt2) * 32 + lane]);
                        }
                        // dz2 = dy2 (1 - t2^2) ; residual dy1[kc1] = dy2[2 kc1] + dy2[2 kc1 + 1]
                        double dy1[2 * NT1];
#pragma unroll
                        for (int kc1 = 0; kc1 < 2 * NT1; ++kc1) dy1[kc1] = kc1 < KC1 ? dy2[2 * kc1] + dy2[2 * kc1 + 1] : 0.0;
#pragma unroll
                        for (int p = 0; p < 2 * NT2; ++p) dy2[p] *= (1.0 - t2[p] * t2[p]);
#pragma unroll
                        for (int kc = 0; kc < 2 * NT2; ++kc) {
#pragma unroll
                            for (int nt1 = 0; nt1 < NT1; ++nt1)
                                dmma(dy1[2 * nt1], dy1[2 * nt1 + 1], dy2[kc], net->W2Tf[(kc * NT1 + nt1) * 32 + lane]);
                        }
                        // layer 1: ds = sum_e dy1[e] (1 - y1[e]^2) W1[e]
                        double ds = 0.0;
#pragma unroll
                        for (int kc1 = 0; kc1 < KC1; ++kc1)
                            ds = fma(dy1[kc1] * (1.0 - y1[kc1] * y1[kc1]), net->w1[4 * kc1 + r], ds);
                        ds += __shfl_xor_sync(0xffffffffu, ds, 1);
                        ds += __shfl_xor_sync(0xffffffffu, ds, 2);
                        if (r == 0) dR0 += ds;
                        __syncwarp();
                        if (r < 2) {     // gR~[c] = dR^[c] / std[c], overwrite this row's R^ in the buffer
                            rbuf[(t * 8 + q4) * 4 + 2 * r] = dR0 / sd[2 * r];
                            rbuf[(t * 8 + q4) * 4 + 2 * r + 1] = dR1 / sd[2 * r + 1];
                        }
                    }
                    my_rows += (unsigned long long)ntile * 8;
                    __syncwarp();
                    // post-pass: N9 geometry derivative, ProdForce scatter, ProdViral partial sums
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

}  // namespace

template <int W> constexpr int smem_fwd() { return (fwd_net_doubles<W>() + DP_WARPS_PER_CTA * WARP_BUF_DOUBLES) * 8; }
template <int W> constexpr int smem_bwd() { return (bwd_net_doubles<W>() + DP_WARPS_PER_CTA * WARP_BUF_DOUBLES) * 8; }

// rows per work item: a whole atom in chunks of ROWCHUNK when there are several atoms' worth of chunks per warp, else chunks of
// 16 rows (two 8-row tiles) as items of their own (config 0: 500 atoms for 1,184 warps, 18 tiles per atom)
static int embed_chunk(const dp_model *m, long N) {
    return N * (long)m->Nm / ROWCHUNK >= 4L * m->num_sms * DP_WARPS_PER_CTA ? ROWCHUNK : 16;
}
static int embed_grid(const dp_model *m, long N) {
    const int CH = embed_chunk(m, N);
    long items = CH == ROWCHUNK ? N : N * ((m->Nm + CH) / CH);
    long grid = (items + DP_WARPS_PER_CTA - 1) / DP_WARPS_PER_CTA;
    return (int)(grid > m->num_sms ? m->num_sms : grid);
}

template <int W>
static cudaError_t launch_fwd_w(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st) {
    DP_SMEM_OPTIN(k_embed_fwd_f64<W>, smem_fwd<W>());
    const TypeTab tt = make_typetab(m);
    const int CH = embed_chunk(m, N);
    if (CH != ROWCHUNK) cudaMemsetAsync(ws + L.A, 0, sizeof(double) * (size_t)N * 4 * m->m2, st);      // partial sums meet by atomics
    k_embed_fwd_f64<W><<<embed_grid(m, N), DP_WARPS_PER_CTA * 32, smem_fwd<W>(), st>>>(
        m->T, g.ncell, m->Nm, CH, tt, make_env(m, g), (const EmbedNetFrag<double, W> *)m->embed_frag_dev, m->avg_dev,
        m->std_dev, (int *)(ws + L.bin_start), (double *)(ws + L.xs), (int *)(ws + L.nlist), (int *)(ws + L.nreal),
        (double *)(ws + L.A), (unsigned long long *)(ws + L.status + 8));
    return cudaGetLastError();
}

template <int W>
static cudaError_t launch_bwd_w(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st) {
    DP_SMEM_OPTIN(k_embed_bwd_f64<W>, smem_bwd<W>());
    const TypeTab tt = make_typetab(m);
    k_embed_bwd_f64<W><<<embed_grid(m, N), DP_WARPS_PER_CTA * 32, smem_bwd<W>(), st>>>(
        m->T, g.ncell, m->Nm, embed_chunk(m, N), tt, make_env(m, g), (const EmbedNetFrag<double, W> *)m->embed_frag_dev, m->avg_dev,
        m->std_dev, (int *)(ws + L.bin_start), (double *)(ws + L.xs), (int *)(ws + L.nlist), (int *)(ws + L.nreal),
        (double *)(ws + L.gAf), (double *)(ws + L.fsorted), (double *)(ws + L.virial),
        (unsigned long long *)(ws + L.status + 16));
    return cudaGetLastError();
}

cudaError_t launch_embed_fwd_f64(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st) {
    return m->m0 == 32 ? launch_fwd_w<32>(m, N, g, ws, L, st) : launch_fwd_w<25>(m, N, g, ws, L, st);
}

cudaError_t launch_embed_bwd_f64(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st) {
    return m->m0 == 32 ? launch_bwd_w<32>(m, N, g, ws, L, st) : launch_bwd_w<25>(m, N, g, ws, L, st);
}
