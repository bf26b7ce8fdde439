/*
 * dp.h -- C ABI of the B200-native Deep Potential (smooth edition, se_a) evaluator.
 *
 * One call, dp_compute, evaluates energy, per-atom energy, forces and virial of a periodic system:
 * the per-step "key function" of DeePMD-kit (section IV: "the calculation of atomic
 * energies and forces predicted by the DP model") with the model structure of PAPER.md:51 (section
 * III-B, Fig. 1), the neighbour-list layout of PAPER.md:109-119 (section V-B1/2), the Environment /
 * ProdForce / ProdViral operators of PAPER.md:121 and the precision schemes of PAPER.md:125.
 * Every formula the paper leaves to its references is the reading listed in DESIGN.md ("Readings").
 *
 * Conventions
 *   - extern "C", plain pointers and sizes only.  "_dev" pointers are CUDA device pointers (caller
 *     owned, e.g. torch tensors' data_ptr()); "_host" / unmarked struct members are host pointers.
 *   - All functions return DP_OK (0) or a negative dp_error; nothing throws or aborts across the ABI.
 *   - dp_compute only ENQUEUES work on the caller's CUDA stream: no host synchronisation, no allocation
 *     (the paper's "trunk of GPU memory allocated at the initialisation stage", is the
 *     caller-owned workspace).  Outputs are valid after the stream is synchronised.
 *   - Units: Angstrom, eV, eV/Angstrom; virial in eV.  Outputs are fp64 in every precision mode
 *     ("outputs of the fitting net ... converted back to double precision").
 *   - There is no CPU fallback: without a CUDA device every compute entry point returns DP_ECUDA.
 */
#ifndef DP_B200_H
#define DP_B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dp_model dp_model; /* opaque; owns device copies of the (re-laid-out, converted) weights */

/* PAPER.md:125.  DP_FP64: everything double.  DP_MIX32: nets in fp32, coordinates / environment matrix /
 * force and virial accumulation in fp64.  DP_MIX16: embedding net and fitting layers 1-2 with fp16 operands
 * on tensor cores and fp32 accumulation, tanh and the last fitting layer in fp32, fp64 accumulation of
 * forces and virial. */
typedef enum { DP_FP64 = 0, DP_MIX32 = 1, DP_MIX16 = 2 } dp_precision;

typedef enum {
    DP_OK = 0,
    DP_EINVAL = -1,   /* null pointer, natoms <= 0 or > 2^24, natoms * max(sel) >= 2^31, rc_smth >= rc, rc*rc >= 128, sel <= 0 */
    DP_EBOX = -2,     /* degenerate box: zero volume, or so small that more than 7 images per axis lie inside rc   */
    DP_ENOMEM = -3,   /* workspace_bytes < dp_workspace_bytes(model, natoms, box); or (dp_status) more periodic
                         images than the extended atom arrays hold (strongly non-uniform density in a small cell)   */
    DP_ETYPE = -4,    /* an atom type outside type_map (detected on device, reported by dp_status)            */
    DP_ECUDA = -5,    /* CUDA runtime error, no device, or the current device is not the one the model was created on */
    DP_ENEIGH = -6,   /* an atom has more candidates inside rc than the sort buffer holds (dp_status)         */
    DP_EUNSUPPORTED = -7, /* precision mode / shape not built                                                */
    DP_ESKIN = -8     /* dp_md_run with a buffered list: an atom moved > skin/2 since the list was built (dp_status) */
} dp_error;

/* Host-side description of one model; read only during dp_create (weights are copied and converted once,
 * round-to-nearest-even: "trained in double precision, and cast").
 * Dense layers are y = x W + b with W row-major [in][out].
 * Layer rule (Fig. 1(e),(f)): out == 2*in -> y = (x,x) + tanh(xW+b); out == in -> y = x + tanh(xW+b);
 * otherwise y = tanh(xW+b).  The last fitting layer is linear. */
typedef struct {
    int ntypes;              /* T, 1..16 (the type field of the sort key has 4 bits)          */
    int embed_widths[3];     /* (m0, m1, m2) = (W, 2 W, 4 W): (25, 50, 100), or the paper's (32, 64, 128);
                                or W = 64, 128, 256, 512, the network-size study of PAPER.md:273-279 (Fig. 7), in every
                                precision.  The wide nets keep their activations in the workspace: dp_workspace_bytes
                                grows by 18 W (DP_MIX16), 36 W (DP_MIX32) or 72 W (DP_FP64) bytes per neighbour-list slot   */
    int axis;                /* M2 (16): D = A^T A[:, :M2]                                                   */
    int fit_widths[3];       /* (240, 240, 240)                                                             */
    const double *embed;     /* T*T nets, index a*T+b (a centre type, b neighbour type):
                                W1[1*m0] b1[m0] W2[m0*m1] b2[m1] W3[m1*m2] b3[m2]                           */
    const double *fit;       /* T nets: V1[(m2*axis)*f0] c1[f0] V2[f0*f1] c2[f1] V3[f1*f2] c3[f2] v4[f2] c4[1] */
    const double *ebias;     /* [T] per-type energy bias added to E_i                                       */
    const double *avg;       /* [T][4] per CENTRE type: R^ = (R~ - avg) / std                               */
    const double *std;       /* [T][4]                                                                      */
} dp_weights;

/* Create a model.  type_map[user_type] -> model type in [0,T) or -1 (unmapped -> DP_ETYPE at compute time);
 * n_type_map entries.  sel[b] = neighbour capacity of type b ("cut-off number of neighbors").
 * rc_smth < rc, rc*rc < 128 (distance field of the 64-bit sort key).  *out is set on DP_OK. */
int dp_create(dp_model **out, const dp_weights *w, const int *type_map, int n_type_map, double rc,
              double rc_smth, const int *sel, dp_precision prec);

/* Bytes of device workspace dp_compute needs for natoms atoms in the box box_host[9] (0 on invalid arguments).
 * box_host == NULL: any orthorhombic box with every length >= 2 rc (the minimum-image path).  A general (triclinic) cell or
 * an edge shorter than 2 rc makes the periodic images explicit ghost atoms (Fig. 1(a)) and needs room for them:
 * pass the box. */
size_t dp_workspace_bytes(const dp_model *m, long natoms, const double *box_host);

/* One evaluation.  coords_dev [natoms][3] fp64 (may lie outside the box; wrapped canonically),
 * types_dev [natoms] int32 USER types, box_host[9] row-major rows a,b,c: any non-degenerate cell (orthorhombic boxes with
 * every length >= 2 rc use the minimum image; general cells and shorter edges use explicit ghost images),
 * workspace_dev: >= dp_workspace_bytes(m, natoms, box_host), 256-byte aligned, contents undefined on entry and exit,
 * cuda_stream: a cudaStream_t (NULL = default stream).
 * Outputs (device, fp64): energy_dev[1]; atom_energy_dev[natoms] or NULL; forces_dev[natoms][3];
 * virial_dev[9] row-major, Xi_ab = -sum d_a (dE/dd_b) = -dE/d(strain_ab), or NULL.
 * A neighbour block that exceeds its capacity keeps the nearest sel[b]; this is counted,
 * not an error. */
int dp_compute(dp_model *m, long natoms, const double *coords_dev, const int *types_dev,
               const double *box_host, void *workspace_dev, size_t workspace_bytes, void *cuda_stream,
               double *energy_dev, double *atom_energy_dev, double *forces_dev, double *virial_dev);

/* The formatted neighbour list of the LAST dp_compute on this model (workspace must still be alive):
 * nlist_dev [natoms][Nm] int32, user indices, rows in user order, type-blocked, each block sorted by
 * (quantised r^2, j), -1 padded.  Enqueued on cuda_stream. */
int dp_get_nlist(dp_model *m, int *nlist_dev, void *cuda_stream);

/* Synchronises the stream of the last dp_compute and reports device-detected conditions:
 * returns DP_OK, DP_ETYPE or DP_ENEIGH; *n_truncated_atoms (may be NULL) = atoms with an over-full block. */
int dp_status(dp_model *m, long *n_truncated_atoms);

/* Number of kernels dp_compute enqueues for this model (for launch accounting in benchmarks). */
int dp_launches_per_compute(const dp_model *m);

/* Neighbour rows actually pushed through the embedding net by the last dp_compute (after dp_status):
 * forward and backward counts; padded rows of a block collapse to one representative row. */
int dp_last_row_counts(dp_model *m, long *rows_forward, long *rows_backward);

/* Optional per-phase device timing of dp_compute (CUDA events recorded on the caller's stream; off by default).
 * dp_profile_read synchronises the last compute and returns DP_NPHASES durations in milliseconds:
 * [0] cell binning + neighbour list (S1,S2), [1] embedding forward + contraction (S3-S5), [2] fitting net
 * forward + backward (S6), [3] embedding backward + ProdForce + ProdViral (S7-S9), [4] finalize,
 * [5] the embedding-backward kernel alone (a part of [3]; equal to [3] where one kernel does all of S7-S9). */
#define DP_NPHASES 6
int dp_profile_enable(dp_model *m, int on);
int dp_profile_read(dp_model *m, double *ms_host);

#define DP_MD_NTHERMO 4   /* doubles per thermo record of dp_md_run */
/* Velocity-Verlet MD loop around dp_compute (section VI-A: "the MD equations are numerically
 * integrated by the velocity-Verlet scheme for 500 steps (the energy and forces are evaluated for 501 times)").
 * One evaluation at the input coordinates, then nsteps times: v += (dt/2) a; x += dt v; evaluate; v += (dt/2) a,
 * with a = F / m * 9.648533216e-3 A/fs^2 per (eV/A)/amu (CODATA 2018 e / amu * 1e-10).  nsteps + 1 evaluations.
 *   coords_dev [natoms][3] fp64, in: x(0), out: x(nsteps dt) (not wrapped);  vel_dev [natoms][3] fp64 in A/fs, in/out;
 *   types_dev as dp_compute;  mass_host[n_mass] amu per USER type (1 <= n_mass <= 8, all > 0);
 *   dt_fs > 0 in femtoseconds;  box / stream as dp_compute;
 *   skin (A) and rebuild_every: with skin > 0 and rebuild_every > 1 the neighbour search keeps, per atom and type, the
 *   candidates within rc + skin of the last cell search and repeats that search every rebuild_every evaluations
 *   ("The neighbor list with a 2 A buffer region is updated every 50 steps"); in between a step re-tests the
 *   candidates exactly, re-sorts and truncates, so the formatted list is the same as without the buffer as long as no atom
 *   moved more than skin/2 since the last search (checked on the device: DP_ESKIN from dp_status).  skin = 0 or
 *   rebuild_every <= 1: every evaluation searches the cells.
 *   workspace_dev: >= dp_md_workspace_bytes(m, natoms, skin, box_host) bytes (skin = 0 if not buffered), 256-byte aligned;
 *   (the buffered list needs the minimum-image path: in a general cell or with an edge < 2 rc every evaluation searches);
 *   forces_dev [natoms][3]: forces at the final coordinates;  thermo_dev [nsteps + 1][DP_MD_NTHERMO] fp64, one record per
 *   evaluation 0 .. nsteps ("kinetic energy, potential energy, temperature, pressure, are collected"):
 *   [0] potential energy E (eV), [1] kinetic energy sum 1/2 m v^2 (eV), [2] temperature 2 KE / ((3 natoms - 3) kB) (K),
 *   [3] pressure (2 KE + trace(virial)) / (3 V) (bar);  virial_dev [9] or NULL: virial of the last evaluation.
 *   Only enqueues on cuda_stream (no host synchronisation, no allocation).  dp_status afterwards reports the device-detected
 *   conditions of the WHOLE run (the flags of all nsteps + 1 evaluations are OR-ed: DP_ETYPE, DP_ENEIGH, DP_ESKIN) and the
 *   truncation count of the last evaluation.  Errors as dp_compute; DP_EINVAL for bad masses, dt_fs, skin < 0, nsteps < 0 or
 *   rebuild_every < 0. */
size_t dp_md_workspace_bytes(const dp_model *m, long natoms, double skin, const double *box_host);
int dp_md_run(dp_model *m, long natoms, double *coords_dev, double *vel_dev, const int *types_dev,
              const double *mass_host, int n_mass, const double *box_host, double dt_fs, int nsteps,
              double skin, int rebuild_every, void *workspace_dev, size_t workspace_bytes, void *cuda_stream,
              double *forces_dev, double *thermo_dev, double *virial_dev);

/* Measured peaks of the arithmetic pipes the path is bound by, for the roofline fractions of the benchmark (
 * the paper reports its own GEMM efficiency against the hardware limit): a few milliseconds of synthetic
 * single-instruction-kind kernels on the current device, timed with CUDA events on cuda_stream (synchronises; allocates 64
 * bytes).  out_host[DP_NPEAKS]: [0] fp64 FMA TFLOP/s (DFMA), [1] fp64 tensor TFLOP/s (mma.sync m8n8k4), [2] fp32 FMA
 * TFLOP/s (FFMA), [3] tanh.approx.f32 in 1e12 per second (MUFU), [4] fp16 mma.sync m16n8k16 TFLOP/s, [5] number of SMs.
 * Not part of the evaluation path. */
#define DP_NPEAKS 6
int dp_measure_peaks(double *out_host, int n_out, void *cuda_stream);

/* Diagnostic for DP_ECUDA: the CUDA runtime's message for the first failing call of the last dp_compute on this model and,
 * in *step (may be NULL), the ordinal of that call inside dp_compute.  The string is static. */
const char *dp_last_cuda_error(const dp_model *m, int *step);

/* ---- Exclusive prefix sum of the neighbour-list build (bin and row offsets), callable alone.
 * start_dev[0 .. n] = exclusive prefix sums of cnt_dev[0 .. n) (n + 1 outputs; start_dev[n] = the total), 32-bit integers,
 * exact.  Three launches on cuda_stream; returns without synchronising.  DP_EINVAL: n <= 0 or a null pointer; DP_ECUDA.
 *
 * dp_scan_exclusive: the path dp_compute runs.  scratch_dev: caller-owned device scratch of at least
 * dp_scan_scratch_bytes(n) bytes (DP_ENOMEM if scratch_bytes is smaller).
 *
 * dp_scan_exclusive_static: the same result from an entry point that ALLOCATES NOTHING and needs no scratch from the caller,
 * for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it).  Its
 * scratch is a static device array inside the library (32,784 bytes, held by every GPU that loads the library until exit),
 * which limits n to DP_SCAN_STATIC_MAX (more: DP_ENOMEM, nothing is launched).  The first call on a device looks the array up
 * (no allocation; make that call before starting a graph capture).  All calls share the array, which keeps the last call's
 * contents (the kernels write every word they read, so no clearing is needed): calls that OVERLAP on the GPU (different
 * streams) race and give wrong sums; calls on one stream are ordered and safe.  It calls no cudaMalloc / cudaFree. */
#define DP_SCAN_STATIC_MAX 16777216
size_t dp_scan_scratch_bytes(int n);
int dp_scan_exclusive(int n, const int *cnt_dev, int *start_dev, void *scratch_dev, size_t scratch_bytes, void *cuda_stream);
int dp_scan_exclusive_static(int n, const int *cnt_dev, int *start_dev, void *cuda_stream);

void dp_destroy(dp_model *m);
const char *dp_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* DP_B200_H */
