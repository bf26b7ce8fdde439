// Internal declarations of the CUDA path (never included by oracle/).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include <atomic>
#include "../../include/dp.h"

// One-time opt-in of a kernel to more than 48 KB of dynamic shared memory.  The attribute belongs to the device context,
// so the "done" flag is per device (bit = device ordinal) and per call site; the return code is checked.
#define DP_SMEM_OPTIN(kern, bytes)                                                                                      \
    do {                                                                                                                \
        static std::atomic<unsigned long long> done_{0ull};                                                             \
        int dev_ = 0;                                                                                                   \
        if (cudaGetDevice(&dev_) != cudaSuccess) return cudaErrorInvalidDevice;                                         \
        if (!((done_.load(std::memory_order_acquire) >> (dev_ & 63)) & 1ull)) {                                         \
            const cudaError_t e_ = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(bytes)); \
            if (e_ != cudaSuccess) return e_;                                                                           \
            done_.fetch_or(1ull << (dev_ & 63), std::memory_order_release);                                             \
        }                                                                                                               \
    } while (0)

#define DP_MAX_TYPES 16
#define DP_NEVENTS 8
#define DP_WARPS_PER_CTA 8

// ---------------------------------------------------------------- shapes fixed by this build (dp.h: widths (25,50,100))
constexpr int M0 = 25, M1 = 50, M2E = 100;   // embedding widths
// bytes of one 128-row hi + lo fp16 operand image of gz1 (fit_tc.cu: k_fit_chain -> k_fit_tc<6>)
constexpr size_t FIT_GZ_TILE_BYTES = 3 * 2 * 10 * (128 * 16 + 16);
constexpr int KC1 = 7;                       // ceil(M0/4) k-chunks of layer-1 output
constexpr int NT2 = 7;                       // 8-wide tiles of layer-2 output (56 positions, 50 real)
constexpr int NT3 = 14;                      // 8-wide tiles of layer-3 output (112 positions, 100 real)
constexpr int M2P = NT3 * 8;                 // padded G width
constexpr int ROWCHUNK = 64;                 // neighbour rows staged per pre-pass / post-pass

// Width-dependent constants of the register-chained (mma.sync) kernels for embedding widths (W, 2 W, 4 W); W = 25 is the
// BASELINE shape, W = 32 the paper's ("the embedding nets are of size (32, 64, 128)").
template <int W>
struct EmbW {
    static constexpr int M0 = W, M1 = 2 * W, M2E = 4 * W;
    static constexpr int KC1 = (W + 3) / 4;          // k-chunks of 4 of the layer-1 output
    static constexpr int NT2 = KC1;                  // 8-wide tiles of the layer-2 output
    static constexpr int NT3 = 2 * KC1;              // 8-wide tiles of the layer-3 output
    static constexpr int NT1 = (KC1 + 1) / 2;        // 8-wide tiles of the layer-1 slots (backward of layer 2)
};

// Fragment-ordered embedding net (one per (centre type, neighbour type)), element type TW.
// Logical feature <-> internal position maps:
//   layer-1 slot (kc,r)        : e  = 4*kc + r                       (valid if < 25)
//   layer-2 position (nt,r,j)  : f2 = (4*nt + r) + 25*j              (valid if 4*nt+r < 25)
//   layer-3 position (nt3,r,j3): f3 = f2(nt3/2, r, nt3%2) + 50*j3    (valid if f2 valid)
template <typename TW, int W = 25>
struct EmbedNetFrag {
    using E = EmbW<W>;
    TW w1[E::KC1 * 4];                      // by slot
    TW b1[E::KC1 * 4];
    TW b2[E::NT2 * 8];                      // by position nt*8 + 2r + j
    TW b3[E::NT3 * 8];
    TW W2f[E::KC1 * E::NT2 * 32];           // forward B fragments  [kc][nt][lane]
    TW W3f[E::NT3 * E::NT3 * 32];           // forward B fragments  [kc'=2nt2+j2][nt3][lane]
    TW W3Tf[2 * E::NT3 * E::NT2 * 32];      // backward B fragments [kc=2nt3+j3][nt2][lane]
    TW W2Tf[E::NT3 * E::NT1 * 32];          // backward B fragments [kc=2nt2+j2][nt1][lane]
};

struct dp_model {
    int T;
    int sel[DP_MAX_TYPES];
    int off[DP_MAX_TYPES + 1];
    int Nm;
    int m0, m1, m2;                 // embedding widths (W, 2 W, 4 W): (25, 50, 100), (32, 64, 128), or wide: W = 64 ... 512
    int wide;                       // W >= 64: layer-by-layer GEMM path with activations in HBM (MIX-16: wide.cu; else wide_gen.cu)
    int wide_gen;                   // wide and FP64 / MIX-32: DMMA / 3xTF32 GEMMs on row-major activations (wide_gen.cu)
    void *wide_vec_dev;             // wide: [T*T][8 W] floats w1, b1, b2, b3; wide_gen: [T*T] parameter blocks (8 W + 20 W^2 elements)
    void *wide_img_dev;             // wide: [T*T][20 W^2] fp16 weight images W2, W3, W3^T, W2^T
    int axis;                       // 16
    int F;                          // fitting width 240
    double rc, rc_smth;
    dp_precision prec;
    int n_type_map;
    int *type_map_dev;
    // device weights
    void *embed_frag_dev;           // T*T EmbedNetFrag<double> (FP64) / EmbedNetFragH<2> (MIX-32 backward, mma.sync)
    void *embed_tc_dev;             // T*T EmbedNetTC<2> (MIX-32 forward, tcgen05) / EmbedNetTC<1> (MIX-16 with fwd_split)
    int fwd_split;                  // MIX-16, Nm < 128: forward with hi + lo activations (embed_tc.cu) instead of embed_tc2.cu
    void *embed_tc2_dev;            // T*T EmbedNetTC2 (MIX-16, warpgroup-per-tile tcgen05 kernels)
    void *fit_tc_img_dev;           // MIX-16: T x six fp16 weight images (fit_tc.cu)
    int device;                     // CUDA device the model was created on (dp_compute checks it)
    double *avg_dev, *std_dev;      // [T][4]
    double *ebias_dev;              // [T]
    // fitting nets (per type): V1 [1600][240], V2, V3 [240][240] row-major in x out, biases, v4, c4
    void *fitV1_dev, *fitV2_dev, *fitV3_dev;   // TW
    void *fitc1_dev, *fitc2_dev, *fitc3_dev, *fitv4_dev, *fitc4_dev;  // TW / float
    int num_sms;
    // state of the last compute
    long last_natoms;
    long last_next;                 // capacity of the extended atom arrays of the last compute (= last_natoms without ghosts)
    void *last_ws;
    cudaStream_t last_stream;
    int sort_cap;
    int profile;
    int last_cuda_error, last_cuda_step;   // first failing CUDA call of the last dp_compute (dp_last_cuda_error)
    // buffered neighbour list of the MD loop (md.cu sets these around its dp_compute calls; 0 / null otherwise)
    int list_mode;                  // 0: search the cells every call; 1: search with rc + skin and store candidates; 2: reuse them
    int keep_flags;                 // dp_md_run, evaluations after the first: device error flags accumulate over the whole run
    double md_skin;
    int *md_cand, *md_candcnt;      // [T][N][sort_cap], [T][N] in the MD part of the workspace
    double *md_xref;                // [N][3] coordinates at the last list build (user order)
    cudaEvent_t ev[8];                // ev[0..5]: phase boundaries; ev[6], ev[7]: around the MIX-16 tcgen05 backward kernel
};

// Workspace carve-up (all offsets 256-byte aligned), filled by dp_ws_layout().
struct WsLayout {
    size_t total;
    size_t status;      // int[8]: [0] error flags, [1] n_truncated, [2] rows_fwd(lo) ... as unsigned long long at [2],[4]
    size_t bin_count;   // int[nbins+1]
    size_t bin_start;   // int[nbins+1]
    size_t bin_cursor;  // int[nbins]
    size_t atom_bin;    // int[N]
    size_t tmp_order;   // int[N]
    size_t perm;        // int[N]  sorted -> user
    size_t inv;         // int[N]  user -> sorted
    size_t xs;          // double[N][3] wrapped coords, sorted order
    size_t xsf;         // float4[N] the same, rounded to fp32 (conservative pre-filter of the neighbour search)
    size_t xw;          // double[N][3] wrapped coords, user order
    size_t nlist;       // int[N][Nm] sorted-space indices
    size_t nreal;       // int[N][T]
    size_t scan_tmp;    // scratch of the two-level scans
    size_t rowcnt;      // int[T][N]   rows per (neighbour type, atom): real + one padded-row representative (mixed modes)
    size_t rowstart;    // int[T][N+1] exclusive prefix of rowcnt over the sorted atoms
    size_t rows_rh;     // float4[T][N*sel_b...] compact env rows R^ (mixed modes, tcgen05 path)
    size_t rows_id;     // int2 {atom, neighbour j} ; {atom, -npad} for the padded-row representative
    size_t rows_g;      // float4 dE/dR~ per compact row (MIX-16 tcgen05 backward -> ProdForce / ProdViral)
    size_t fj32;        // float4[NE] MIX-16: the neighbours' force shares, accumulated by 16-byte fp32 vector reductions
    size_t multi_cnt;   // int[16][16] MIX-16 backward: 1 if a tile of the (centre, neighbour) type block spans more than two atoms
    size_t A;           // double[N][4][100]   (float for mixed modes)
    size_t gAf;         // gA fragments [N][42][32] doubles (fp64) / [N][NSW][28][32] words (mixed)
    size_t gscale;      // float[N] power-of-two scale of the mixed gA fragments
    size_t fit_act;     // 7 activation buffers [N][240]
    size_t gD;          // [N][1600]
    size_t eatom;       // double[N] sorted order
    size_t fsorted;     // double[N][3] sorted order
    size_t virial;      // double[9] + energy accumulators
    // ghost mode: extended atom arrays (the per-atom arrays above that are indexed by a neighbour are sized cap_ext)
    size_t ext_owner;   // int[cap_ext] user index of the owner of unsorted item u (u < N: the atom itself)
    size_t ext_code;    // int[cap_ext] packed image shift of unsorted item u
    size_t ext_base;    // int[cap_ext] sorted index of the owner of sorted item e
    size_t ext_scode;   // int[cap_ext] packed image shift of sorted item e
    size_t gcnt;        // int[N] ghosts per atom
    size_t gstart;      // int[N+1]
    // wide networks (wide.cu): tile table and the activation images, per 128-row tile [columns / 8][128][8] fp16
    size_t wide_tab;    // int4[T*T + 1]
    size_t wide_t1, wide_y2, wide_t2, wide_t3;      // W, 2 W, 2 W, 4 W columns (wide_gen.cu: row-major [N Nm][columns], fp64 / fp32)
    size_t wide_rh, wide_gr;                        // wide_gen.cu: R^ and dE/dR~ per compact row, [N Nm][4]
};

// the compact rows (rowcnt, rowstart, rows_id) exist in the mixed modes and on every wide path
inline bool dp_uses_rows(const dp_model *m) { return m->prec != DP_FP64 || m->wide; }

// FP64 fitting net, first layer (K = 16 m2): split K over four CTAs per output tile when the row tiles (64 rows x 80 columns)
// are too few to fill the GPU (fit_f64.cu; one more launch per evaluation: dp_launches_per_compute)
inline bool fit_f64_splitk(const dp_model *m, long N) {
    return ((N + 63) / 64) * 3 * 2 <= m->num_sms && (m->m2 * 16 / 16) % 4 == 0;
}

// neighbour capacities per type and their prefix sums, passed to kernels by value (a __grid_constant__ parameter: indexed
// dynamically straight from constant memory)
struct TypeTab {
    int sel[DP_MAX_TYPES];
    int off[DP_MAX_TYPES + 1];
};
inline TypeTab make_typetab(const dp_model *m) {
    TypeTab t{};
    for (int b = 0; b < DP_MAX_TYPES; ++b) { t.sel[b] = b < m->T ? m->sel[b] : 0; t.off[b] = b <= m->T ? m->off[b] : m->off[m->T]; }
    t.off[DP_MAX_TYPES] = m->off[m->T];
    return t;
}

struct Grid3 {
    int nc[3];          // cells per axis
    double L[3];        // box lengths (ghost mode: 1e300, which switches the minimum image off in every kernel)
    double inv_cw[3];   // nc / L
    int ncell;
    int reach;          // neighbour cells searched per direction: 1 (cell edge >= rc) or 2 (cell edge >= rc/2)
    // ---- ghost mode (ghost.cu): general cell or a cell edge shorter than 2 rc; periodic images are explicit ghost atoms
    int ghost;          // 0: orthorhombic box with every length >= 2 rc (minimum image, nlist.cu)
    int ortho;          // ghost mode: the box is diagonal (reading N2: per-axis wrap and shift) or general (reading N2t)
    double H[9];        // box rows a, b, c
    double Hinv[9];     // x = f H, f = x Hinv
    int nimg[3];        // images per axis: ceil(rc / h_k)
    double flo[3];      // fractional coordinate of the low edge of the extended region: -(rc / h_k) (1 + 1e-9)
    double fcw[3];      // cells per unit fractional length
    long cap_ext;       // capacity of the extended (local + ghost) atom arrays
};

// launchers (each returns cudaGetLastError())
void dp_launch_scan(int n, const int *cnt, int *start, int *tmp, cudaStream_t st);
cudaError_t launch_build_ghost(const dp_model *m, long N, const double *coords, const int *types, const Grid3 &g, char *ws,
                               const WsLayout &L, cudaStream_t st);
cudaError_t launch_nlist_ghost(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st);
cudaError_t launch_fold_ghost(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st);
cudaError_t launch_build_cells(const dp_model *m, long N, const double *coords, const int *types, const Grid3 &g,
                               char *ws, const WsLayout &L, cudaStream_t st);
cudaError_t launch_regather(const dp_model *m, long N, const double *coords, const Grid3 &g, char *ws, const WsLayout &L,
                            cudaStream_t st);
cudaError_t launch_nlist(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st);
cudaError_t launch_get_nlist(const dp_model *m, long N, char *ws, const WsLayout &L, int *out, cudaStream_t st);
cudaError_t launch_embed_fwd_f64(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st);
cudaError_t launch_embed_bwd_f64(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st);
cudaError_t launch_fit_f64(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st);
cudaError_t launch_finalize(const dp_model *m, long N, char *ws, const WsLayout &L, double *energy, double *eatom,
                            double *forces, double *virial, cudaStream_t st);
cudaError_t launch_embed_bwd_mix(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st);
cudaError_t launch_embed_fwd_tc(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st);
cudaError_t launch_embed_fwd_tc2(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st);
cudaError_t launch_embed_bwd_tc2(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st);
cudaError_t launch_fit_tc(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st);
cudaError_t launch_prod_force_virial(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st);
// wide networks (wide.cu)
cudaError_t launch_embed_fwd_wide(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st);
cudaError_t launch_embed_bwd_wide(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st);
size_t wide_net_img_elems(int W);
void wide_build_net(int W, const double *net, float *vec, struct __half *img);
long wide_tiles_cap(const dp_model *m, long N);
cudaError_t launch_wide_tiles(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st);
// wide networks in FP64 and MIX-32 (wide_gen.cu)
cudaError_t launch_embed_fwd_wide_gen(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st);
cudaError_t launch_embed_bwd_wide_gen(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st);
size_t wide_gen_net_elems(int W, bool f64);
void wide_gen_build_net(int W, bool f64, const double *net, void *out);
size_t fit_tc32_type_elems(int nd);
void fit_tc32_build_type(int nd, const double *V1, struct __half *out);
cudaError_t launch_fit_tc32_first(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st);
cudaError_t launch_fit_tc32_last(const dp_model *m, long N, const float *gz1, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st);
size_t fit_tc_type_elems(int nd);
void fit_tc_build_type(int nd, const double *V1, const double *V2, const double *V3, struct __half *out);
cudaError_t launch_env_rows(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st);
cudaError_t launch_fit_mix(const dp_model *m, long N, const Grid3 &g, char *ws, const WsLayout &L, cudaStream_t st);
