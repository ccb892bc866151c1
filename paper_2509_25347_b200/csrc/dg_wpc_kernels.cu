// dg_wpc_kernels.cu — warp-per-cell DMMA kernels for ONE species count N = DG_N (compiled once per N).
//
// Each warp walks the cells assigned to it (consecutive cells go to the warps of one block, so the 32-byte sectors a
// warp touches are shared through L1/L2 with its neighbours).  Lane j < N is the "canonical" lane of dust species j:
// it loads that species' fields, does the divisions / rsqrt once, and stores that species' results; a per-warp
// shared-memory table hands the values to the lanes that need them in the tensor-core fragment layout.
#include "dg_internal.h"
#include "dg_wpc.cuh"

#ifndef DG_N
#error "compile with -DDG_N=<number of dust species>"
#endif

namespace dg {
namespace {

constexpr int N = DG_N;
constexpr int n = N + 1;
using Core = Wpc<N>;
constexpr int TL = Core::TL;
constexpr int ND = Core::ND;
constexpr int kWarps = 8;
constexpr int kThreads = 32 * kWarps;

struct WarpSmem {
    double al[ND], be[ND], w[ND], iw[ND];  // per dust species: a 2^-s, beta, sqrt(eps), 1/sqrt(eps)
    double q[3][ND], q0[3];                // W^-1 p_in per component
    double y[3][ND], y0[3];                // P W^-1 p_in per component
};

__device__ __forceinline__ double warp_sum(double x) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(kFull, x, o);
    return x;
}
__device__ __forceinline__ double warp_max(double x) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x = fmax(x, __shfl_xor_sync(kFull, x, o));
    return x;
}

// Everything between "the a_j, eps_j of this cell are known in the canonical lanes" and "P = exp(S) - I is in the
// fragment registers".  a, eps: this lane's species (lanes >= N: a = 0, eps = 1).
struct CellState {
    double T[TL][TL][2];
    Core::VecR rR, wR, iwR;
    Core::VecC rC, iwC;
    double d0;
    double w, iw;  // canonical lane's own weights
    int m, s;
};

__device__ __forceinline__ void cell_expm(const Core::Lane& L, WarpSmem& sm, int lane, double a, double eps,
                                          CellState& st) {
    double w = 1.0, iw = 1.0;
    if (lane < N) sym_weights(eps, w, iw);
    const double aw = a * w;
    const double sb = warp_sum(aw * w);
    const double amax = warp_max(a);
    choose_m_s(2.0 * fmax(sb, amax), Core::hcost(), st.m, st.s);
    const double sc = pow2neg(st.s);
    __syncwarp();
    if (lane < ND) {
        sm.al[lane] = a * sc;
        sm.be[lane] = aw * sc;
        sm.w[lane] = w;
        sm.iw[lane] = iw;
    }
    __syncwarp();
    Core::VecR alR, beR;
    Core::VecC beC, wC;
#pragma unroll
    for (int I = 0; I < TL; ++I) {
        const int row = 8 * I + L.g;
        alR.v[I] = sm.al[row];
        beR.v[I] = sm.be[row];
        st.wR.v[I] = sm.w[row];
        st.iwR.v[I] = sm.iw[row];
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            const int col = 8 * I + 2 * L.t + e;
            beC.v[I][e] = sm.be[col];
            wC.v[I][e] = sm.w[col];
            st.iwC.v[I][e] = sm.iw[col];
        }
    }
    st.w = w;
    st.iw = iw;
    Core::expm(L, st.m, st.s, alR, beR, beC, -sb * sc, st.wR, wC, st.iwR, st.T, st.rR, st.rC, st.d0);
}

// ---------------------------------------------------------------------------------------------- fused a1..a5
__global__ void __launch_bounds__(kThreads) k_update_wpc(UpdateArgs g) {
    __shared__ WarpSmem smem[kWarps];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    WarpSmem& sm = smem[warp];
    const Core::Lane L;
    const long long nc = g.ncells;
    const long long stride = (long long)gridDim.x * kWarps;
    for (long long c = (long long)blockIdx.x * kWarps + warp; c < nc; c += stride) {
        // a1: canonical lanes load their species (lane 31 doubles as the gas lane for the momenta)
        double a = 0.0, eps = 1.0;
        if (lane < N) {
            a = g.dt / __ldg(g.t_s + lane * nc + c);
            eps = __ldg(g.rho_d + lane * nc + c) / __ldg(g.rho_g + c);
        }
        double p[3] = {0.0, 0.0, 0.0};
        const int k = (lane < N) ? lane + 1 : 0;  // momentum row of this lane
        const bool has_p = (lane < N) || (lane == 31);
        if (has_p) {
#pragma unroll
            for (int comp = 0; comp < 3; ++comp) p[comp] = __ldg(g.p_in + (long long)(comp * n + k) * nc + c);
        }
        // a2-a4
        CellState st;
        cell_expm(L, sm, lane, a, eps, st);
        if (lane == 0) {
            if (g.s_out) g.s_out[c] = st.s;
            if (g.m_out) g.m_out[c] = st.m;
        }
        // a5: y = P W^-1 p_in, p_out = p_in + W y
#pragma unroll
        for (int comp = 0; comp < 3; ++comp) {
            if (lane < ND) sm.q[comp][lane] = p[comp] * st.iw;  // padding lanes: p = 0
            if (lane == 31) sm.q0[comp] = p[comp];
        }
        __syncwarp();
#pragma unroll
        for (int comp = 0; comp < 3; ++comp) {
            Core::VecC qC;
            Core::VecR yR;
            const double q0 = sm.q0[comp];
            double acc = 0.0;
#pragma unroll
            for (int I = 0; I < TL; ++I) {
#pragma unroll
                for (int e = 0; e < 2; ++e) qC.v[I][e] = sm.q[comp][8 * I + 2 * L.t + e];
                acc = fma(st.rR.v[I], sm.q[comp][8 * I + L.g], acc);
            }
            Core::matvec(st.T, qC, yR);
            const double y0 = fma(st.d0, q0, oct_sum(acc));
#pragma unroll
            for (int I = 0; I < TL; ++I)
                if (L.t == 0) sm.y[comp][8 * I + L.g] = fma(st.rR.v[I], q0, yR.v[I]);
            if (lane == 0) sm.y0[comp] = y0;
        }
        __syncwarp();
        if (has_p) {
#pragma unroll
            for (int comp = 0; comp < 3; ++comp) {
                const double y = (lane < N) ? sm.y[comp][lane] : sm.y0[comp];
                g.p_out[(long long)(comp * n + k) * nc + c] = fma(st.w, y, p[comp]);
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------- staged a2-a4
__global__ void __launch_bounds__(kThreads) k_expm_wpc(ExpmArgs g) {
    __shared__ WarpSmem smem[kWarps];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    WarpSmem& sm = smem[warp];
    const Core::Lane L;
    const long long nc = g.ncells;
    const long long stride = (long long)gridDim.x * kWarps;
    for (long long c = (long long)blockIdx.x * kWarps + warp; c < nc; c += stride) {
        double a = 0.0, eps = 1.0;
        if (lane < N) {
            a = __ldg(g.A + (long long)(0 * n + lane + 1) * nc + c);
            const double b = __ldg(g.A + (long long)((lane + 1) * n + 0) * nc + c);
            eps = a > 0.0 ? b / a : 1.0;
        }
        CellState st;
        cell_expm(L, sm, lane, a, eps, st);
        if (lane == 0 && g.s_out) g.s_out[c] = st.s;
        double* E = g.E + c;
        // E = I + W P W^-1
#pragma unroll
        for (int I = 0; I < TL; ++I) {
            const int row = 8 * I + L.g;
#pragma unroll
            for (int J = 0; J < TL; ++J)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int col = 8 * J + 2 * L.t + e;
                    if (row < N && col < N) {
                        const double v = (row == col) ? 1.0 + st.T[I][J][e] : st.wR.v[I] * st.T[I][J][e] * st.iwC.v[J][e];
                        E[(long long)((row + 1) * n + col + 1) * nc] = v;
                    }
                }
            if (L.t == 0 && row < N) E[(long long)((row + 1) * n) * nc] = st.wR.v[I] * st.rR.v[I];  // column 0
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int col = 8 * I + 2 * L.t + e;
                if (L.g == 0 && col < N) E[(long long)(col + 1) * nc] = st.rC.v[I][e] * st.iwC.v[I][e];  // row 0
            }
        }
        if (lane == 0) E[0] = 1.0 + st.d0;
        __syncwarp();
    }
}

unsigned persistent_grid(const void* kernel, long long ncells) {
    int dev = 0, sms = 148, per_sm = 1;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, kThreads, 0);
    if (per_sm < 1) per_sm = 1;
    long long want = (ncells + kWarps - 1) / kWarps;
    long long cap = (long long)sms * per_sm;
    return (unsigned)(want < cap ? want : cap);
}

cudaError_t launch_update(const UpdateArgs& a, cudaStream_t st) {
    k_update_wpc<<<persistent_grid((const void*)k_update_wpc, a.ncells), kThreads, 0, st>>>(a);
    return cudaGetLastError();
}
cudaError_t launch_expm(const ExpmArgs& a, cudaStream_t st) {
    k_expm_wpc<<<persistent_grid((const void*)k_expm_wpc, a.ncells), kThreads, 0, st>>>(a);
    return cudaGetLastError();
}

}  // namespace

#define DG_CAT_(a, b) a##b
#define DG_CAT(a, b) DG_CAT_(a, b)
extern const WpcLaunchers DG_CAT(wpc_launchers_N, DG_N) = {launch_update, launch_expm,
                                                           "warp-per-cell, DMMA m8n8k4 symmetric tiles"};

}  // namespace dg
