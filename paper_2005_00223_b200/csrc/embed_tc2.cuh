// Second-generation tcgen05 embedding kernels (MIX-16): shared layout definitions.
//
// One warpgroup (128 threads) owns one 128-row tile; thread = neighbour row = TMEM lane.  Several warpgroups per CTA keep
// several tiles in flight so that one tile's MUFU/ALU phases overlap the others' tensor-core phases.
//
// The residual layers are folded into the contractions, so only tanh outputs are ever stored (PAPER.md:134 rule
// y = (x,x) + tanh(xW+b) restated):   y1 = t1,  y2 = (t1,t1) + t2,  G = (y2,y2) + t3   with t_l = tanh(z_l), hence
//   z3 = y2 W3 + b3 = t2 W3 + t1 (W3[0:25] + W3[25:50]) + b3
//   A  = R^T G / Nm = fold(R^T [t1 | t2 | t3]) / Nm,   fold(C)[c][m] = C3[c][m] + C2[c][m mod 50] + C1[c][m mod 25]
// and the biases ride in the GEMMs through a constant-one column of the t1 block.
//
// T row layout (fp16 columns): t1 block cols [0,32): e < 25 real, cols 25 and 26 hold 1.0 (bias hi / lo rows), rest 0;
// t2 block cols [32,96): f < 50 real; t3 block cols [96,208): m < 100 real.  26 chunks of 8 columns.
#pragma once
#include <cuda_fp16.h>
#include "dp_internal.h"

constexpr int T2_ROWS = 128;
constexpr int T2_K1 = 32, T2_K2 = 64, T2_K3 = 112;        // padded block widths
constexpr int T2_O1 = 0, T2_O2 = 32, T2_O3 = 96;           // block column offsets
constexpr int T2_COLS = 208;
constexpr int T2_CHUNKS = T2_COLS / 8;                    // 26
constexpr int T2_ONE_HI = 25, T2_ONE_LO = 26;             // constant-one columns of the t1 block
constexpr int T2_NSLOT = 2;                               // atoms accumulated side by side in the contraction (N = 16)

// One (centre type, neighbour type) embedding net as tcgen05 K-major B operand images [K/8][N][8] (fp16).
struct EmbedNetTC2 {
    float w1[32], b1[32];
    __half W2[T2_K1 / 8][64][8];                 // layer 2: A = t1 block (K = 32), N = 64 (50 real)
    __half W3[(T2_K2 + T2_K1) / 8][112][8];      // layer 3: A = t2 block then t1 block (K = 96), N = 112 (100 real)
    // backward (A operands dz3 [K = 112], dz2 [K = 64])
    __half W3T[T2_K3 / 8][96][8];                // n = e < 32: dy1[e] += dz3[m] (W3[e][m] + W3[e+25][m]);  n = 32 + f: dy2[f] += dz3[m] W3[f][m]
    __half W2T[T2_K2 / 8][32][8];                // dy1[e] += dz2[f] W2[e][f]
};
