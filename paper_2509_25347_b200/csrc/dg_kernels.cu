// dg_kernels.cu — the kernels of libdg for ONE species count N = DG_N (compiled once per N, -DDG_N=<N>).
//
// Thread-per-cell kernels: every field is structure-of-arrays with the cell index fastest, so a warp's loads and
// stores of one field row are 256 contiguous bytes.  The fused kernel k_update never writes a matrix to HBM.
#include "dg_internal.h"
#include "dg_tpc.cuh"

#ifndef DG_N
#error "compile with -DDG_N=<number of dust species>"
#endif

namespace dg {
namespace {

constexpr int N = DG_N;
constexpr int n = N + 1;
using Core = Tpc<N>;
constexpr int SZ = Core::SZ;
constexpr int kThreads = 128;

// ---------------------------------------------------------------------------------------------- fused a1..a5
__global__ void __launch_bounds__(kThreads) k_update(UpdateArgs g) {
    const long long c = (long long)blockIdx.x * kThreads + threadIdx.x;
    if (c >= g.ncells) return;
    const long long nc = g.ncells;

    // a1: eps_i (Eq. 14), a_i = dt alpha_i (Eq. 15), symmetrising weights
    double a[N], w[N], iw[N];
    {
        const double irg = 1.0 / __ldg(g.rho_g + c);
#pragma unroll
        for (int i = 0; i < N; ++i) {
            a[i] = g.dt / __ldg(g.t_s + i * nc + c);
            sym_weights(__ldg(g.rho_d + i * nc + c) * irg, w[i], iw[i]);
        }
    }
    // a2-a4
    double P[SZ];
    int m, s;
    Core::expm(a, w, iw, P, m, s);
    if (g.s_out) g.s_out[c] = s;
    if (g.m_out) g.m_out[c] = m;

    // a5: p_out = p_in + W P W^-1 p_in, one component at a time
#pragma unroll 1
    for (int comp = 0; comp < 3; ++comp) {
        const double* pi = g.p_in + (long long)comp * n * nc + c;
        double* po = g.p_out + (long long)comp * n * nc + c;
        double p[n], q[n];
#pragma unroll
        for (int k = 0; k < n; ++k) {
            p[k] = __ldg(pi + k * nc);
            q[k] = (k == 0) ? p[k] : p[k] * iw[k == 0 ? 0 : k - 1];
        }
#pragma unroll
        for (int i = 0; i < n; ++i) {
            double y = 0.0;
#pragma unroll
            for (int k = 0; k < n; ++k) y = fma(P[Core::sx(i, k)], q[k], y);
            po[i * nc] = (i == 0) ? p[i] + y : fma(w[i == 0 ? 0 : i - 1], y, p[i]);
        }
    }
}

// ---------------------------------------------------------------------------------------------- staged a1
__global__ void __launch_bounds__(kThreads) k_build(BuildArgs g) {
    const long long c = (long long)blockIdx.x * kThreads + threadIdx.x;
    if (c >= g.ncells) return;
    const long long nc = g.ncells;
    const double rg = __ldg(g.rho_g + c);
    double* A = g.A + c;
    double sb = 0.0;
#pragma unroll
    for (int i = 1; i < n; ++i) {
        const double ai = g.dt / __ldg(g.t_s + (i - 1) * nc + c);
        const double bi = (__ldg(g.rho_d + (i - 1) * nc + c) / rg) * ai;
        sb += bi;
#pragma unroll
        for (int k = 1; k < n; ++k) A[(long long)(i * n + k) * nc] = (k == i) ? -ai : 0.0;
        A[(long long)(0 * n + i) * nc] = ai;  // row 0: gas gains from dust i
        A[(long long)(i * n + 0) * nc] = bi;  // column 0: dust i gains from gas
    }
    A[0] = -sb;
}

// ---------------------------------------------------------------------------------------------- staged a2-a4
__global__ void __launch_bounds__(kThreads) k_expm(ExpmArgs g) {
    const long long c = (long long)blockIdx.x * kThreads + threadIdx.x;
    if (c >= g.ncells) return;
    const long long nc = g.ncells;
    const double* A = g.A + c;
    double a[N], w[N], iw[N];
#pragma unroll
    for (int i = 1; i < n; ++i) {
        const double ai = __ldg(A + (long long)(0 * n + i) * nc);
        const double bi = __ldg(A + (long long)(i * n + 0) * nc);
        a[i - 1] = ai;
        sym_weights(ai > 0.0 ? bi / ai : 1.0, w[i - 1], iw[i - 1]);
    }
    double P[SZ];
    int m, s;
    Core::expm(a, w, iw, P, m, s);
    if (g.s_out) g.s_out[c] = s;
    double* E = g.E + c;
#pragma unroll
    for (int i = 0; i < n; ++i)
#pragma unroll
        for (int k = 0; k < n; ++k) {
            double v = P[Core::sx(i, k)];
            if (i > 0) v *= w[i == 0 ? 0 : i - 1];
            if (k > 0) v *= iw[k == 0 ? 0 : k - 1];
            if (i == k) v = 1.0 + P[Core::ix(i, i)];
            E[(long long)(i * n + k) * nc] = v;
        }
}

// ---------------------------------------------------------------------------------------------- staged a5
__global__ void __launch_bounds__(kThreads) k_apply(ApplyArgs g) {
    const long long c = (long long)blockIdx.x * kThreads + threadIdx.x;
    if (c >= g.ncells) return;
    const long long nc = g.ncells;
    double p[3][n];
#pragma unroll
    for (int comp = 0; comp < 3; ++comp)
#pragma unroll
        for (int k = 0; k < n; ++k) p[comp][k] = __ldg(g.p_in + (long long)(comp * n + k) * nc + c);
#pragma unroll 1
    for (int i = 0; i < n; ++i) {
        double y0 = 0.0, y1 = 0.0, y2 = 0.0;
#pragma unroll
        for (int k = 0; k < n; ++k) {
            const double e = __ldg(g.E + (long long)(i * n + k) * nc + c);
            y0 = fma(e, p[0][k], y0);
            y1 = fma(e, p[1][k], y1);
            y2 = fma(e, p[2][k], y2);
        }
        g.p_out[(long long)(0 * n + i) * nc + c] = y0;
        g.p_out[(long long)(1 * n + i) * nc + c] = y1;
        g.p_out[(long long)(2 * n + i) * nc + c] = y2;
    }
}

inline unsigned grid_for(long long ncells) { return (unsigned)((ncells + kThreads - 1) / kThreads); }

cudaError_t launch_update(const UpdateArgs& a, cudaStream_t st) {
    k_update<<<grid_for(a.ncells), kThreads, 0, st>>>(a);
    return cudaGetLastError();
}
cudaError_t launch_build(const BuildArgs& a, cudaStream_t st) {
    k_build<<<grid_for(a.ncells), kThreads, 0, st>>>(a);
    return cudaGetLastError();
}
cudaError_t launch_expm(const ExpmArgs& a, cudaStream_t st) {
    k_expm<<<grid_for(a.ncells), kThreads, 0, st>>>(a);
    return cudaGetLastError();
}
cudaError_t launch_apply(const ApplyArgs& a, cudaStream_t st) {
    k_apply<<<grid_for(a.ncells), kThreads, 0, st>>>(a);
    return cudaGetLastError();
}

}  // namespace

#define DG_CAT_(a, b) a##b
#define DG_CAT(a, b) DG_CAT_(a, b)
extern const Launchers DG_CAT(launchers_N, DG_N) = {launch_update, launch_build, launch_expm, launch_apply,
                                                    "thread-per-cell, symmetric packed registers"};

}  // namespace dg
