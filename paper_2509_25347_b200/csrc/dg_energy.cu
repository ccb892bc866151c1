// dg_energy.cu — dg_drag_update_energy (include/dg.h): the fused drag update plus the gas energy with frictional heating
// (Eq. 4 and the third entry of Eq. 11; reading R20).
//
// The paper gives no discrete formula for E_g in the EXP step.  Along the exact momenta p(t) = exp(t Omega) p(0) the
// drag terms of Eq. 4 integrate exactly: the work term is the change of the gas kinetic energy, the heating term is
// w times the kinetic energy the drag dissipates (dK/dt = -sum_i rho_d,i |v_d,i - v_g|^2 / T_s,i by Eq. 3, 6), so
//     E_g(t+dt) = E_g(t) + [KE_g(t+dt) - KE_g(t)] + w [K(t) - K(t+dt)],    K = |M_g|^2/(2 rho_g) + sum_i |M_d,i|^2/(2 rho_d,i).
// ONE launch for every N: the default kernel for N forms the two kinetic-energy sums on the way.  The sorted-tile kernel
// (dg_tps_kernels.cu, N <= 12) holds rho_g, rho_d, p_in and p_out of a tile in shared memory anyway (one more tile row
// for E); the pair-per-cell kernel (dg_ppc_kernels.cu, N >= 13) sums over the rows each lane applies and stores, re-reads
// its rho_d row (an L2 hit) and adds the two lanes' sums with one shuffle.  Until round 3 N >= 13 took three launches
// (an O(N) kernel before and after the update: +7-12 % time and twice the field traffic).
#include <cmath>
#include <cstdint>

#include "../../include/dg.h"
#include "dg_internal.h"

namespace dg {
dg_status cuda_status(cudaError_t e);
cudaError_t launch_update_energy(int N, const UpdateArgs& a, const double* E_in, double* E_out, double w, cudaStream_t st);
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
    UpdateArgs a{rho_g, rho_d, t_s, dt, p_in, ncells, p_out, nullptr, nullptr};
    return cuda_status(launch_update_energy(N, a, E_in, E_out, w, static_cast<cudaStream_t>(stream)));
}
