// dg_f32_kernels.cu — the fused drag update in SINGLE precision for ONE species count N = DG_N.
//
// Eq. B.8 offers the scaling thresholds theta_m for other unit round-offs than 2^-53; this is the
// u = 2^-24 instantiation: the same thread-per-cell arithmetic as the fp64 path (dg_tpc.cuh, Tpc<N, float>: symmetrised
// arrowhead, factored Horner recurrence, cancellation-free squarings with the diagonal from conservation) with every
// quantity a float and the (m, s) choice made against the single-precision column of thresholds (dg_params.cuh
// c_theta32).  Inputs and outputs are float SoA arrays in the layouts of include/dg.h.
// One thread per cell, rows read and written coalesced (128 bytes per warp and row); not persistent, no staging: at
// 4 (8N + 7) bytes per cell this kernel is bound by its fp32 arithmetic and by latency, not by HBM, and it is a widened
// row, not the timed path.
#include "dg_internal.h"
#include "dg_tpc.cuh"

#ifndef DG_N
#error "compile with -DDG_N=<number of dust species>"
#endif

namespace dg {
namespace {

constexpr int N = DG_N;
constexpr int n = N + 1;
using Core = Tpc<N, float>;
constexpr int SZ = Core::SZ;
constexpr int kThreads = 128;

__global__ void __launch_bounds__(kThreads) k_update_f32(UpdateArgsF32 g) {
    const long long nc = g.ncells;
    const long long c = (long long)blockIdx.x * kThreads + threadIdx.x;
    const bool valid = c < nc;  // no early return: the lanes of a warp choose the Taylor degree together
    // a1: eps_i (Eq. 14), a_i = dt alpha_i (Eq. 15), symmetrising weights; a lane without a cell gets the identity
    float a[N], w[N], iw[N];
    if (valid) {
        const float irg = fast_rcp(__ldg(g.rho_g + c));
        static_for<0, N>([&](auto I) {
            constexpr int i = I;
            a[i] = g.dt * fast_rcp(__ldg(g.t_s + (long long)i * nc + c));
            sym_weights(__ldg(g.rho_d + (long long)i * nc + c) * irg, w[i], iw[i]);
        });
    } else {
        static_for<0, N>([&](auto I) {
            a[I] = 0.0f;
            w[I] = iw[I] = 1.0f;
        });
    }
    // a2-a4
    float P[SZ];
    int m, s;
    Core::template expm<0>(a, w, iw, P, m, s);
    if (!valid) return;
    if (g.s_out) g.s_out[c] = s;
    if (g.m_out) g.m_out[c] = m;
    // a5: p_out = p_in + W P W^-1 p_in, one component at a time
#pragma unroll 1
    for (int comp = 0; comp < 3; ++comp) {
        const float* pi = g.p_in + (long long)comp * n * nc + c;
        float* po = g.p_out + (long long)comp * n * nc + c;
        float p[n], q[n];
        static_for<0, n>([&](auto K) { p[K] = __ldg(pi + (long long)K * nc); });
        static_for<0, n>([&](auto K) {
            constexpr int k = K;
            if constexpr (k == 0) q[k] = p[k];
            else q[k] = p[k] * iw[k - 1];
        });
        static_for<0, n>([&](auto I) {
            constexpr int i = I;
            float y = 0.0f;
            static_for<0, n>([&](auto K) {
                constexpr int k = K;
                y = fmaf(P[Core::sx(i, k)], q[k], y);
            });
            if constexpr (i == 0) po[0] = p[0] + y;
            else po[(long long)i * nc] = fmaf(w[i - 1], y, p[i]);
        });
    }
}

cudaError_t launch_update(const UpdateArgsF32& a, cudaStream_t st) {
    k_update_f32<<<(unsigned)((a.ncells + kThreads - 1) / kThreads), kThreads, 0, st>>>(a);
    return cudaGetLastError();
}

}  // namespace

#define DG_CAT_(a, b) a##b
#define DG_CAT(a, b) DG_CAT_(a, b)
extern const F32Launchers DG_CAT(f32_launchers_N, DG_N) = {launch_update};

}  // namespace dg
