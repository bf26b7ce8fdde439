// tcgen05 / TMEM version of the mixed-precision embedding kernels (sm_100a): shared definitions.
//
// A tile is 128 neighbour rows (TMEM lane = row).  Two threads own a row: thread (row, h) handles the feature half h.
// The feature order inside the MMA K / N dimensions is permuted so that every residual "(x,x) + tanh" is thread-local:
//   layer-1 position p1 (K of layer 2, 32)  : h = p1/16, t = p1%16          -> e  = e0(h) + t           (t < ce(h))
//   layer-2 column n    (N of layer 2, 64)  : h = n/32, j = (n/16)%2, t     -> f  = e0(h) + t + 25 j
//   layer-3 column c3   (N of layer 3, 128) : h = c3/64, j3 = (c3/32)%2, u  -> m  = f(32h + u) + 50 j3
// with e0 = {0, 13}, ce = {13, 12}; all other positions are zero padding.
// Shared-memory operand images are "chunk-major": for every 16-byte chunk (8 fp16 along the contiguous dimension) a
// column of ROWS x 16 B.  The same image is a K-major operand (rows = M/N, LBO = ROWS*16, SBO = 128) or an MN-major
// operand (rows = K, SBO = ROWS*16, LBO = 128) of tcgen05.mma (no swizzle).
#pragma once
#include <cuda_fp16.h>
#include "dp_internal.h"

constexpr int TC_ROWS = 128;
constexpr int TC_K1 = 32, TC_N2 = 64, TC_N3 = 128;
constexpr int TC_NSLOT = 6;       // atoms (contraction slots) per contraction pass: N = 8 * TC_NSLOT = 48

// widths (W, 2 W, 4 W), W = 25 or 32: e0 = {0, 13} / {0, 16}, ce = {13, 12} / {16, 16}
template <int W> __host__ __device__ inline int tc_e0(int h) { return h ? (W + 1) / 2 : 0; }
template <int W> __host__ __device__ inline int tc_ce(int h) { return h ? W / 2 : (W + 1) / 2; }
template <int W> __host__ __device__ inline int tc_e_of_p1(int p1) { int h = p1 >> 4, t = p1 & 15; return t < tc_ce<W>(h) ? tc_e0<W>(h) + t : -1; }
template <int W> __host__ __device__ inline int tc_f_of_n(int n) {
    int h = n >> 5, j = (n >> 4) & 1, t = n & 15;
    return t < tc_ce<W>(h) ? tc_e0<W>(h) + t + W * j : -1;
}
template <int W> __host__ __device__ inline int tc_m_of_c3(int c3) {
    int h = c3 >> 6, j3 = (c3 >> 5) & 1, u = c3 & 31;
    int f = tc_f_of_n<W>(32 * h + u);
    return f < 0 ? -1 : f + 2 * W * j3;
}

// One (centre type, neighbour type) embedding net as tcgen05 operand images.  NSW weight parts (hi [, lo]).
template <int NSW>
struct EmbedNetTC {
    float w1[TC_K1], b1[TC_K1], b2[TC_N2], b3[TC_N3];
    __half W2[NSW][TC_K1 / 8][TC_N2][8];     // B of layer 2 fwd: (n, k)   = W2[e(k)][f(n)]
    __half W3[NSW][TC_N2 / 8][TC_N3][8];     // B of layer 3 fwd: (c3, k)  = W3[f(k)][m(c3)]
    __half W3T[NSW][TC_N3 / 8][TC_N2][8];    // B of layer 3 bwd: (n, k=c3) = W3[f(n)][m(c3)]
    __half W2T[NSW][TC_N2 / 8][TC_K1][8];    // B of layer 2 bwd: (p1, k=n) = W2[e(p1)][f(n)]
};
