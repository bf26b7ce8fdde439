// Velocity-Verlet MD loop around dp_compute ("the MD equations are numerically
// integrated by the velocity-Verlet scheme for 500 steps (the energy and forces are evaluated for 501 times)").
// Everything is enqueued on the caller's stream: no host synchronisation, no allocation; the neighbour list is rebuilt by
// every evaluation, or (skin > 0, rebuild_every > 1) kept as a buffered candidate list for rebuild_every evaluations as in the
// paper (2 A buffer, update every 50 steps); then a step only re-tests, re-sorts and truncates (nlist.cu).
#include <cmath>
#include "dp_internal.h"

namespace {

// acceleration of 1 eV/A on 1 amu in A/fs^2: (e / amu) * 1e-10 (CODATA 2018: e = 1.602176634e-19 C, amu = 1.66053906660e-27 kg)
constexpr double ACC = 1.602176634e-19 / 1.66053906660e-27 * 1.0e-10;
constexpr int MD_MAX_MASS = 8;
struct Masses {
    int n;
    double m[MD_MAX_MASS];
};

// v += hk F / m  (hk = dt/2 * ACC, 0 for none);  x += dt v  (DRIFT);  kinetic energy sum 1/2 m v^2 / ACC in eV (KE)
template <bool DRIFT, bool KE>
__global__ void __launch_bounds__(256) k_md(long N, double *__restrict__ x, double *__restrict__ v,
                                            const double *__restrict__ F, const int *__restrict__ types, Masses ms,
                                            double hk, double dt, double *__restrict__ ke_out) {
    double ke = 0.0;
    for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < N; i += (long)gridDim.x * blockDim.x) {
        const int ty = types[i];
        if (ty < 0 || ty >= ms.n) continue;                 // dp_compute flags the type (DP_ETYPE); the atom stays put
        const double mass = ms.m[ty], c = hk / mass;
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            double vb = v[3 * i + b];
            if (hk != 0.0) vb = fma(c, F[3 * i + b], vb);
            v[3 * i + b] = vb;
            if (DRIFT) x[3 * i + b] = fma(dt, vb, x[3 * i + b]);
            if (KE) ke = fma(0.5 * mass * vb, vb, ke);
        }
    }
    if (KE) {
        __shared__ double red[8];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) ke += __shfl_xor_sync(0xffffffffu, ke, o);
        if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = ke;
        __syncthreads();
        if (threadIdx.x == 0) {
            double s = 0.0;
            for (int w = 0; w < 8; ++w) s += red[w];
            atomicAdd(ke_out, s / ACC);
        }
    }
}

// temperature (K) and pressure (bar) of one evaluation from its kinetic energy and virial ("kinetic energy,
// potential energy, temperature, pressure, are collected"): T = 2 KE / ((3 N - 3) kB) (three momentum constraints, as
// LAMMPS counts them), P = (2 KE + tr Xi) / (3 V) with Xi = -dE/d(strain); 1 eV/A^3 = 1.602176634e6 bar.
__global__ void k_thermo(double *__restrict__ rec, const double *__restrict__ virial, double dof, double volume) {
    const double ke = rec[1];
    rec[2] = 2.0 * ke / (dof * 8.617333262e-5);
    rec[3] = (2.0 * ke + virial[0] + virial[4] + virial[8]) / (3.0 * volume) * 1.602176634e6;
}

}  // namespace

namespace {
struct MdWs { size_t base, vir, cand, candcnt, xref, total; };
MdWs md_layout(const dp_model *m, long N, double skin, const double *box) {
    MdWs w{};
    auto al = [](size_t x) { return (x + 255) & ~(size_t)255; };
    w.base = al(dp_workspace_bytes(m, N, box));
    w.vir = w.base;
    w.total = al(w.vir + 16 * sizeof(double));
    if (skin > 0.0) {
        w.cand = w.total; w.total = al(w.total + sizeof(int) * (size_t)m->T * (size_t)N * (size_t)m->sort_cap);
        w.candcnt = w.total; w.total = al(w.total + sizeof(int) * (size_t)m->T * (size_t)N);
        w.xref = w.total; w.total = al(w.total + sizeof(double) * 3 * (size_t)N);
    }
    return w;
}
}  // namespace

extern "C" size_t dp_md_workspace_bytes(const dp_model *m, long natoms, double skin, const double *box_host) {
    if (!m || natoms <= 0 || !(skin >= 0.0) || dp_workspace_bytes(m, natoms, box_host) == 0) return 0;
    return md_layout(m, natoms, skin, box_host).total;
}

extern "C" int dp_md_run(dp_model *m, long natoms, double *coords_dev, double *vel_dev, const int *types_dev,
                         const double *mass_host, int n_mass, const double *box_host, double dt_fs, int nsteps,
                         double skin, int rebuild_every, void *workspace_dev, size_t workspace_bytes, void *cuda_stream,
                         double *forces_dev, double *thermo_dev, double *virial_dev) {
    if (!m || natoms <= 0 || !coords_dev || !vel_dev || !types_dev || !mass_host || n_mass <= 0 || n_mass > MD_MAX_MASS ||
        !box_host || !(dt_fs > 0.0) || nsteps < 0 || !forces_dev || !thermo_dev || !(skin >= 0.0) || rebuild_every < 0 ||
        !workspace_dev)
        return DP_EINVAL;
    Masses ms;
    ms.n = n_mass;
    for (int k = 0; k < MD_MAX_MASS; ++k) ms.m[k] = k < n_mass ? mass_host[k] : 1.0;
    for (int k = 0; k < n_mass; ++k) if (!(ms.m[k] > 0.0)) return DP_EINVAL;
    // the buffered list lives on the minimum-image path: a general cell or an edge shorter than 2 rc searches every step
    // (a stored candidate is re-tested at its nearest image, which is the only image that can be inside rc when L >= 2 rc)
    bool mi_box = box_host[1] == 0 && box_host[2] == 0 && box_host[3] == 0 && box_host[5] == 0 && box_host[6] == 0 && box_host[7] == 0;
    for (int a = 0; a < 3; ++a) mi_box = mi_box && box_host[4 * a] >= 2.0 * m->rc;
    const bool buffered = skin > 0.0 && rebuild_every > 1 && mi_box;
    const MdWs W = md_layout(m, natoms, buffered ? skin : 0.0, box_host);
    if (W.base == 0) return DP_EINVAL;
    if (workspace_bytes < W.total) return DP_ENOMEM;
    char *ws = (char *)workspace_dev;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const unsigned grid = (unsigned)((natoms + 255) / 256 < 148L * 8 ? (natoms + 255) / 256 : 148L * 8);
    const double hk = 0.5 * dt_fs * ACC;
    if (cudaMemsetAsync(thermo_dev, 0, sizeof(double) * DP_MD_NTHERMO * ((size_t)nsteps + 1), st) != cudaSuccess) return DP_ECUDA;
    const double *bx = box_host;
    const double volume = std::fabs(bx[0] * (bx[4] * bx[8] - bx[5] * bx[7]) - bx[1] * (bx[3] * bx[8] - bx[5] * bx[6]) +
                                    bx[2] * (bx[3] * bx[7] - bx[4] * bx[6]));
    const double dof = natoms > 1 ? 3.0 * (double)natoms - 3.0 : 3.0;
    double *vir = virial_dev ? virial_dev : (double *)(ws + W.vir);
    if (buffered) {
        m->md_skin = skin;
        m->md_cand = (int *)(ws + W.cand); m->md_candcnt = (int *)(ws + W.candcnt); m->md_xref = (double *)(ws + W.xref);
    }
    int rc = DP_OK;
    for (int s = 0; s <= nsteps && rc == DP_OK; ++s) {
        if (s > 0)
            k_md<true, false><<<grid, 256, 0, st>>>(natoms, coords_dev, vel_dev, forces_dev, types_dev, ms, hk, dt_fs, nullptr);
        if (buffered) {
            m->list_mode = (s % rebuild_every == 0) ? 1 : 2;
            if (m->list_mode == 1 &&
                cudaMemcpyAsync(m->md_xref, coords_dev, sizeof(double) * 3 * (size_t)natoms, cudaMemcpyDeviceToDevice, st) != cudaSuccess)
                rc = DP_ECUDA;
        }
        m->keep_flags = s > 0;          // device error flags accumulate over the run (dp_status reports all of it)
        if (rc == DP_OK)
            rc = dp_compute(m, natoms, coords_dev, types_dev, box_host, workspace_dev, W.base, cuda_stream,
                            thermo_dev + DP_MD_NTHERMO * s, nullptr, forces_dev, vir);
        if (rc == DP_OK) {
            k_md<false, true><<<grid, 256, 0, st>>>(natoms, coords_dev, vel_dev, forces_dev, types_dev, ms, s > 0 ? hk : 0.0,
                                                     dt_fs, thermo_dev + DP_MD_NTHERMO * s + 1);
            k_thermo<<<1, 1, 0, st>>>(thermo_dev + DP_MD_NTHERMO * s, vir, dof, volume);
        }
    }
    m->keep_flags = 0;
    m->list_mode = 0; m->md_skin = 0.0; m->md_cand = nullptr; m->md_candcnt = nullptr; m->md_xref = nullptr;
    if (rc != DP_OK) return rc;
    return cudaGetLastError() == cudaSuccess ? DP_OK : DP_ECUDA;
}
