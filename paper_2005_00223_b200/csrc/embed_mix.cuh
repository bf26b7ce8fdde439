// Shared pieces of the mixed-precision embedding kernels (MIX-32 and MIX-16).
//
// Tensor-core shape: mma.sync m16n8k16 / m16n8k8, fp16 operands, fp32 accumulation.  A 16-row tile of
// neighbour rows is pushed through the three embedding layers with the accumulator fragments chained in
// registers (C fragment of layer l -> A fragment of layer l+1, same thread, no shared memory).
//   NS = 1 : operands rounded to fp16 once (MIX-16: "parameters ... stored in half precision ... GEMM on Tensor
//            Cores with accumulations in single precision").
//   NS = 3 : every operand is split x = hi + lo (two fp16), products hi*hi + hi*lo + lo*hi are accumulated in
//            fp32: ~2^-21 relative product error, i.e. single-precision nets executed on the tensor pipe
//            (MIX-32: "all the arithmetic operations of the embedding net and the fitting net are performed in
//            single precision").
// Logical feature <-> internal position maps (in-thread residuals):
//   layer-1 slot (q, r)         : e  = 8*(q/2) + 2*r + (q%2)            (valid if < 25), q = 0..7
//   layer-2 position (nt, r, j) : f2 = e(nt, r) + 25*j                  (valid if e < 25), nt = 0..6
//   layer-3 position (nt3,r,j3) : f3 = f2(nt3/2, r, nt3%2) + 50*j3      (valid if f2 valid), nt3 = 0..13
#pragma once
#include <cuda_fp16.h>
#include "dp_internal.h"

constexpr int HQ1 = 8;        // layer-1 slots per thread per row
constexpr int HROWS = 16;     // rows per MMA tile

// widths (W, 2 W, 4 W): W = 25 (BASELINE) or 32 (the paper's networks)
template <int W>
struct HW {
    static constexpr int M0 = W, M1 = 2 * W, M2E = 4 * W;
    static constexpr int HNT2 = (W + 3) / 4;     // layer-2 8-wide tiles (7 / 8)
    static constexpr int HNT3 = 2 * HNT2;        // layer-3 8-wide tiles (14 / 16)
};

__host__ __device__ inline int h_e1(int q, int r) { return 8 * (q >> 1) + 2 * r + (q & 1); }
template <int W> __host__ __device__ inline int h_f2(int nt, int r, int j) { int e = h_e1(nt, r); return e < W ? e + W * j : -1; }
template <int W> __host__ __device__ inline int h_f3(int nt3, int r, int j3) { int f = h_f2<W>(nt3 >> 1, r, nt3 & 1); return f < 0 ? -1 : f + 2 * W * j3; }

// Fragment-ordered embedding net for the fp16 tensor path.  NSW = 1 (hi only) or 2 (hi, lo) weight parts.
// k-steps: a K of n tiles is consumed as n/2 k16 steps plus one k8 step if n is odd.
template <int NSW, int W = 25>
struct EmbedNetFragH {
    static constexpr int HNT2 = HW<W>::HNT2, HNT3 = HW<W>::HNT3;
    float w1[32], b1[32];                    // natural order e (zero padded)
    float b2[HNT2 * 8];                      // by position nt*8 + 2r + j
    float b3[HNT3 * 8];
    uint32_t W2f[NSW][2][HNT2][32][2];       // K = 32 (y1 slots, natural order e): 2 k16 steps
    uint32_t W3f[NSW][4][HNT3][32][2];       // K = HNT2 tiles: 3 k16 + 1 k8 (W = 25) / 4 k16 (W = 32)
    uint32_t W3Tf[NSW][HNT3 / 2][HNT2][32][2];   // K = HNT3 tiles: HNT3 / 2 k16 steps
    uint32_t W2Tf[NSW][4][4][32][2];         // K = HNT2 tiles: 3 k16 + 1 k8 / 4 k16 ; N = 32 y1 slots (4 tiles)
};

#ifdef __CUDACC__
__device__ __forceinline__ void mma16816(float (&c)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3,
                                         uint32_t b0, uint32_t b1) {
    asm("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
        : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
        : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}
__device__ __forceinline__ void mma1688(float (&c)[4], uint32_t a0, uint32_t a1, uint32_t b0) {
    asm("mma.sync.aligned.m16n8k8.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5}, {%6}, {%0,%1,%2,%3};"
        : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
        : "r"(a0), "r"(a1), "r"(b0));
}
__device__ __forceinline__ uint32_t pack_h2(float x, float y) {
    __half2 h = __floats2half2_rn(x, y);
    return *reinterpret_cast<uint32_t *>(&h);
}
// x = hi + lo with hi = fp16(x), lo = fp16(x - hi)
// hi is x truncated to 11 significant bits (exactly representable in fp16 for normal-range values), so the
// fp32 -> fp16 conversion of hi is exact and no conversion back is needed to form the remainder.
__device__ __forceinline__ void split_h2(float x, float y, uint32_t &hi, uint32_t &lo) {
    const float xh = __int_as_float(__float_as_int(x) & 0xFFFFE000), yh = __int_as_float(__float_as_int(y) & 0xFFFFE000);
    hi = pack_h2(xh, yh);
    lo = pack_h2(x - xh, y - yh);
}
__device__ __forceinline__ uint32_t movmatrix_trans(uint32_t x) {
    uint32_t y;
    asm("movmatrix.sync.aligned.m8n8.trans.b16 %0, %1;" : "=r"(y) : "r"(x));
    return y;
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

// NS encodes which operands of a product are split into hi + lo fp16 parts:
//   1: none (1 MMA)   2: activations only (2 MMAs)   4: weights only (2 MMAs)   3: both (3 MMAs, lo*lo dropped)
__host__ __device__ constexpr bool ns_asplit(int ns) { return ns == 2 || ns == 3; }
__host__ __device__ constexpr bool ns_wsplit(int ns) { return ns == 3 || ns == 4; }
__host__ __device__ constexpr int ns_wparts(int ns) { return ns_wsplit(ns) ? 2 : 1; }

// An A operand for one k-step: hi (and lo when NS == 3) parts of a 16x16 (or 16x8) fp16 fragment.
template <int NS>
struct AFrag {
    uint32_t hi[4];
    uint32_t lo[4];
};
// Build from C-layout values: v0a,v0b = row g cols 2r,2r+1 ; v1a,v1b = row g+8 (first 8-wide tile),
// w.. the second tile (k + 8).
template <int NS>
__device__ __forceinline__ void make_afrag(AFrag<NS> &f, float v0a, float v0b, float v1a, float v1b, float w0a,
                                           float w0b, float w1a, float w1b) {
    if (!ns_asplit(NS)) {
        f.hi[0] = pack_h2(v0a, v0b); f.hi[1] = pack_h2(v1a, v1b); f.hi[2] = pack_h2(w0a, w0b); f.hi[3] = pack_h2(w1a, w1b);
    } else {
        split_h2(v0a, v0b, f.hi[0], f.lo[0]); split_h2(v1a, v1b, f.hi[1], f.lo[1]);
        split_h2(w0a, w0b, f.hi[2], f.lo[2]); split_h2(w1a, w1b, f.hi[3], f.lo[3]);
    }
}
template <int NS>
__device__ __forceinline__ void make_afrag8(AFrag<NS> &f, float v0a, float v0b, float v1a, float v1b) {
    if (!ns_asplit(NS)) { f.hi[0] = pack_h2(v0a, v0b); f.hi[1] = pack_h2(v1a, v1b); }
    else { split_h2(v0a, v0b, f.hi[0], f.lo[0]); split_h2(v1a, v1b, f.hi[1], f.lo[1]); }
}
// c += A * B for a k16 step; B fragment registers bh (hi part) and bl (lo part, NS == 3 only)
template <int NS>
__device__ __forceinline__ void mma_k16(float (&c)[4], const AFrag<NS> &a, const uint32_t *bh, const uint32_t *bl) {
    mma16816(c, a.hi[0], a.hi[1], a.hi[2], a.hi[3], bh[0], bh[1]);
    if (ns_wsplit(NS)) mma16816(c, a.hi[0], a.hi[1], a.hi[2], a.hi[3], bl[0], bl[1]);
    if (ns_asplit(NS)) mma16816(c, a.lo[0], a.lo[1], a.lo[2], a.lo[3], bh[0], bh[1]);
}
template <int NS>
__device__ __forceinline__ void mma_k8(float (&c)[4], const AFrag<NS> &a, const uint32_t *bh, const uint32_t *bl) {
    mma1688(c, a.hi[0], a.hi[1], bh[0]);
    if (ns_wsplit(NS)) mma1688(c, a.hi[0], a.hi[1], bl[0]);
    if (ns_asplit(NS)) mma1688(c, a.lo[0], a.lo[1], bh[0]);
}
#endif
