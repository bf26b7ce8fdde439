// Second-generation tcgen05 embedding kernels (MIX-16): shared layout definitions.
//
// One warpgroup (128 threads) owns one 128-row tile; thread = neighbour row = TMEM lane.  Several warpgroups per CTA keep
// several tiles in flight so that one tile's MUFU/ALU phases overlap the others' tensor-core phases.
//
// The residual layers are folded into the contractions, so only tanh outputs are ever stored (PAPER.md:134 rule
// y = (x,x) + tanh(xW+b) restated):   y1 = t1,  y2 = (t1,t1) + t2,  G = (y2,y2) + t3   with t_l = tanh(z_l), hence
//   z3 = y2 W3 + b3 = t2 W3 + t1 (W3[0:W] + W3[W:2W]) + b3
//   A  = R^T G / Nm = fold(R^T [t1 | t2 | t3]) / Nm,   fold(C)[c][m] = C3[c][m] + C2[c][m mod 2W] + C1[c][m mod W]
// and the biases ride in the GEMMs: multiplied by a constant-one column.
//
// Embedding widths (W, 2 W, 4 W), W = 25 (BASELINE configs) or W = 32 (the paper's networks).
// T row layout (fp16 columns): t1 block cols [0,32), t2 block cols [32,96), t3 block cols [96, 96 + K3).
//   W = 25: t1 e < 25 real, cols 25 and 26 hold 1.0 (bias hi / lo rows of the weight images), t2 f < 50 real, t3 m < 100
//           real of K3 = 112: 26 chunks of 8 columns.
//   W = 32: every column is real (K3 = 128, 28 chunks); the biases enter through one extra K = 16 step per layer whose A
//           operand is a constant "ones" image (columns 0 and 1 = 1.0) and whose B operand holds the bias hi / lo rows.
#pragma once
#include <cuda_fp16.h>
#include "dp_internal.h"

constexpr int T2_ROWS = 128;
constexpr int T2_K1 = 32, T2_K2 = 64;                      // padded block widths of t1, t2 (both shapes)
constexpr int T2_O1 = 0, T2_O2 = 32, T2_O3 = 96;           // block column offsets
constexpr int T2_ONE_HI = 25, T2_ONE_LO = 26;             // W = 25: constant-one columns of the t1 block
constexpr int T2_NSLOT = 2;                               // atoms accumulated side by side in the contraction (N = 16)

template <int W>
struct T2 {
    static constexpr int M0 = W, M1 = 2 * W, M2E = 4 * W;
    static constexpr int K3 = W == 25 ? 112 : 128;         // padded t3 block width
    static constexpr int COLS = T2_O3 + K3;                // 208 / 224
    static constexpr int CHUNKS = COLS / 8;                // 26 / 28
    static constexpr bool ONES_STEP = W != 25;             // biases through a separate K = 16 ones step
};
constexpr int T2_COLS = T2<25>::COLS;                     // (fit_tc.cu, dp_api.cu: the W = 25 sizes)

// One (centre type, neighbour type) embedding net as tcgen05 K-major B operand images [K/8][N][8] (fp16).
template <int W>
struct EmbedNetTC2 {
    float w1[32], b1[32];
    __half W2[T2_K1 / 8][64][8];                     // layer 2: A = t1 block (K = 32), N = 64
    __half W3[(T2_K2 + T2_K1) / 8][T2<W>::K3][8];    // layer 3: A = t2 block then t1 block (K = 96), N = K3
    // backward (A operands dz3 [K = K3], dz2 [K = 64])
    __half W3T[T2<W>::K3 / 8][96][8];                // n = e < 32: dy1[e] += dz3[m] (W3[e][m] + W3[e+W][m]);  n = 32 + f: dy2[f] += dz3[m] W3[f][m]
    __half W2T[T2_K2 / 8][32][8];                    // dy1[e] += dz2[f] W2[e][f]
    // W = 32 only (ONES_STEP): bias rows k = 0 (hi part), k = 1 (lo part), k = 2..7 zero; one 8-deep K chunk each (the second
    // chunk of the K = 16 step aliases the first through a zero leading-dimension stride: the ones image is zero there)
    __half Bb2[64][8];
    __half Bb3[T2<W>::K3][8];
};
