// dg_energy.cu — dg_drag_update_energy (include/dg.h): the fused drag update plus the gas energy with frictional heating
// (Eq. 4 and the third entry of Eq. 11; reading R20).
//
// The paper gives no discrete formula for E_g in the EXP step.  Along the exact momenta p(t) = exp(t Omega) p(0) the
// drag terms of Eq. 4 integrate exactly: the work term is the change of the gas kinetic energy, the heating term is
// w times the kinetic energy the drag dissipates (dK/dt = -sum_i rho_d,i |v_d,i - v_g|^2 / T_s,i by Eq. 3, 6), so
//     E_g(t+dt) = E_g(t) + [KE_g(t+dt) - KE_g(t)] + w [K(t) - K(t+dt)],    K = |M_g|^2/(2 rho_g) + sum_i |M_d,i|^2/(2 rho_d,i).
// N <= 12: ONE launch — the sorted-tile kernel (dg_tps_kernels.cu) holds rho_g, rho_d, p_in and p_out of a tile in shared
// memory anyway and forms the two kinetic-energy sums on the way (one more tile row for E).
// N >= 13: three launches on the caller's stream: k_energy_pre (the terms at t, from p_in — before the update, so that
// p_out may alias p_in), the fused drag update (dg_drag_update's kernel for this N), k_energy_post (the terms at t+dt,
// from p_out).  Both energy kernels are one thread per cell, every field row read coalesced: O(N) flops, HBM-bound;
// they add 7-12 % to a 10-14 ms update.
#include <cmath>
#include <cstdint>

#include "../../include/dg.h"
#include "dg_internal.h"

namespace dg {
dg_status cuda_status(cudaError_t e);
cudaError_t launch_update(int N, int variant, const UpdateArgs& a, cudaStream_t st);
bool has_fused_energy(int N);
cudaError_t launch_update_energy(int N, const UpdateArgs& a, const double* E_in, double* E_out, double w, cudaStream_t st);

namespace {
constexpr int kThreads = 256;

// KE_g and K of one cell from momenta p[3][n][nc]; a species with rho_d = 0 carries nothing
__device__ __forceinline__ void kinetic(const double* rho_g, const double* rho_d, const double* p, int N, long long nc,
                                        long long c, double& keg, double& k) {
    const int n = N + 1;
    double g2 = 0.0;
#pragma unroll
    for (int comp = 0; comp < 3; ++comp) {
        const double v = p[(long long)(comp * n) * nc + c];
        g2 = fma(v, v, g2);
    }
    keg = g2 / (2.0 * rho_g[c]);
    double kd = 0.0;
    for (int i = 0; i < N; ++i) {
        const double rd = rho_d[(long long)i * nc + c];
        double d2 = 0.0;
#pragma unroll
        for (int comp = 0; comp < 3; ++comp) {
            const double v = p[(long long)(comp * n + 1 + i) * nc + c];
            d2 = fma(v, v, d2);
        }
        if (rd > 0.0) kd += d2 / (2.0 * rd);
    }
    k = keg + kd;
}

__global__ void __launch_bounds__(kThreads) k_energy_pre(const double* rho_g, const double* rho_d, const double* p_in,
                                                         const double* E_in, double w, int N, long long nc,
                                                         double* E_out) {
    const long long c = (long long)blockIdx.x * kThreads + threadIdx.x;
    if (c >= nc) return;
    double keg, k;
    kinetic(rho_g, rho_d, p_in, N, nc, c, keg, k);
    E_out[c] = E_in[c] + fma(w, k, -keg);
}
__global__ void __launch_bounds__(kThreads) k_energy_post(const double* rho_g, const double* rho_d, const double* p_out,
                                                          double w, int N, long long nc, double* E_out) {
    const long long c = (long long)blockIdx.x * kThreads + threadIdx.x;
    if (c >= nc) return;
    double keg, k;
    kinetic(rho_g, rho_d, p_out, N, nc, c, keg, k);
    E_out[c] += fma(-w, k, keg);
}
}  // namespace
}  // namespace dg

using namespace dg;

extern "C" dg_status dg_drag_update_energy(const double* rho_g, const double* rho_d, const double* t_s, double dt,
                                           const double* p_in, const double* E_in, double w, int N, long long ncells,
                                           double* p_out, double* E_out, void* stream) {
    if (N < 1 || N > DG_NMAX || ncells < 0) return DG_ERANGE;
    if (!(dt >= 0.0) || !std::isfinite(dt) || !(w >= 0.0 && w <= 1.0)) return DG_EINVAL;
    if (ncells == 0) return DG_OK;
    const void* ptrs[] = {rho_g, rho_d, t_s, p_in, E_in, p_out, E_out};
    for (const void* p : ptrs) {
        if (p == nullptr) return DG_ENULL;
        if (reinterpret_cast<uintptr_t>(p) & 7u) return DG_EALIGN;
    }
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (has_fused_energy(N)) {  // N <= 12: one launch, the sums are formed inside the sorted-tile kernel
        UpdateArgs a{rho_g, rho_d, t_s, dt, p_in, ncells, p_out, nullptr, nullptr};
        return cuda_status(launch_update_energy(N, a, E_in, E_out, w, st));
    }
    const unsigned grid = (unsigned)((ncells + kThreads - 1) / kThreads);
    k_energy_pre<<<grid, kThreads, 0, st>>>(rho_g, rho_d, p_in, E_in, w, N, ncells, E_out);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_status(e);
    UpdateArgs a{rho_g, rho_d, t_s, dt, p_in, ncells, p_out, nullptr, nullptr};
    e = launch_update(N, DG_VARIANT_DEFAULT, a, st);
    if (e != cudaSuccess) return cuda_status(e);
    k_energy_post<<<grid, kThreads, 0, st>>>(rho_g, rho_d, p_out, w, N, ncells, E_out);
    return cuda_status(cudaGetLastError());
}
