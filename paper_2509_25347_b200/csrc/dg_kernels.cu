// dg_kernels.cu — the kernels of libdg for ONE species count N = DG_N (compiled once per N, -DDG_N=<N>).
//
// Thread-per-cell kernels: every field is structure-of-arrays with the cell index fastest, so a warp's loads and
// stores of one field row are 256 contiguous bytes.  The fused kernel k_update never writes a matrix to HBM.
#include "dg_async.cuh"
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
// Persistent over cells: thread t of the grid walks cells t, t + T, t + 2T, ... (T = threads in the grid), so a warp
// always owns 32 consecutive cells and every row access is 256 contiguous bytes.  All global reads go through
// cp.async (LDGSTS) into the thread's own column of a shared-memory staging tile [row][thread]:
//   * the momenta of the current cell are requested BEFORE the matrix work and read after it,
//   * the densities / stopping times of the NEXT cell are requested before the matrix work of the current one,
// so the few resident warps (the matrices occupy up to 255 registers per thread) never wait on HBM latency.
// A thread only ever reads shared memory that its own cp.async wrote: cp.async.wait_group is the only
// synchronisation needed, there is no barrier.
constexpr int kMinBlocks = N <= 2 ? 8 : N <= 4 ? 4 : N <= 7 ? 3 : 2;  // register budget 64 / 128 / 168 / 255 per thread
constexpr int kRowsIn = 1 + 2 * N;  // rho_g, rho_d[N], t_s[N]
constexpr int kRowsP = 3 * n;       // p_in[3][n]
constexpr size_t kSmemBytes = (size_t)(kRowsIn + kRowsP) * kThreads * sizeof(double);

__global__ void __launch_bounds__(kThreads, kMinBlocks) k_update(UpdateArgs g) {
    extern __shared__ double stage[];
    double* s_in = stage + threadIdx.x;                      // [kRowsIn][kThreads]
    double* sp = stage + kRowsIn * kThreads + threadIdx.x;  // [kRowsP][kThreads]
    const long long nc = g.ncells;
    const long long stride = (long long)gridDim.x * kThreads;
    long long c = (long long)blockIdx.x * kThreads + threadIdx.x;
    long long cw = c - (threadIdx.x & 31);  // first cell of this warp: the loop is warp-uniform (the lanes take the
                                            // Taylor degree together, dg_params.cuh); lanes past the end idle

    // row addresses by running pointers (one 64-bit add per row instead of a 64-bit multiply-add chain)
    auto request_inputs = [&](long long cc) {
        if (cc < nc) {
            cp_async8(s_in, g.rho_g + cc);
            const double* pd = g.rho_d + cc;
            const double* pt = g.t_s + cc;
            static_for<0, N>([&](auto I) {
                constexpr int i = I;
                cp_async8(s_in + (1 + i) * kThreads, pd);
                cp_async8(s_in + (1 + N + i) * kThreads, pt);
                pd += nc;
                pt += nc;
            });
        }
        cp_async_commit();
    };
    request_inputs(c);
    while (cw < nc) {
        const bool valid = c < nc;
        if (valid) {
            const double* pp = g.p_in + c;
            static_for<0, kRowsP>([&](auto R) {
                constexpr int r = R;
                cp_async8(sp + r * kThreads, pp);
                pp += nc;
            });
        }
        cp_async_commit();
        cp_async_wait<1>();  // the inputs of cell c have landed (its momenta may still be in flight)

        // a1: eps_i (Eq. 14), a_i = dt alpha_i (Eq. 15), symmetrising weights; a lane without a cell gets the
        // identity (a = 0)
        double a[N], w[N], iw[N];
        if (valid) {
            const double irg = fast_rcp(s_in[0]);
            static_for<0, N>([&](auto I) {
                constexpr int i = I;
                a[i] = g.dt * fast_rcp(s_in[(1 + N + i) * kThreads]);
                sym_weights(s_in[(1 + i) * kThreads] * irg, w[i], iw[i]);
            });
        } else {
            static_for<0, N>([&](auto I) {
                constexpr int i = I;
                a[i] = 0.0;
                w[i] = iw[i] = 1.0;
            });
        }
        const long long cn = c + stride;
        request_inputs(cn);  // always commits a group (an empty one past the end) so the wait counts stay uniform

        // a2-a4
        double P[SZ];
        int m, s;
        Core::template expm<Core::kDefer>(a, w, iw, P, m, s);
        if (valid) {
            if (g.s_out) g.s_out[c] = s;
            if (g.m_out) g.m_out[c] = m;
        }

        // a5: p_out = p_in + W P W^-1 p_in, one component at a time; applied 2^k times where the last k squarings were
        // left out (dg_tpc.cuh kDefer)
        cp_async_wait<1>();  // the momenta of cell c have landed (the next cell's inputs may still be in flight)
        if (valid) {
            const int napply = 1 << min(Core::kDefer, s);
#pragma unroll 1
            for (int comp = 0; comp < 3; ++comp) {
                const double* pi = sp + comp * n * kThreads;
                double* po = g.p_out + (long long)comp * n * nc + c;
                double p[n], q[n];
                static_for<0, n>([&](auto K) { p[K] = pi[K * kThreads]; });
                auto apply_once = [&]() {
                    static_for<0, n>([&](auto K) {
                        constexpr int k = K;
                        if constexpr (k == 0) q[k] = p[k];
                        else q[k] = p[k] * iw[k - 1];
                    });
                    static_for<0, n>([&](auto I) {
                        constexpr int i = I;
                        double y = 0.0;
                        static_for<0, n>([&](auto K) {
                            constexpr int k = K;
                            y = fma(P[Core::sx(i, k)], q[k], y);
                        });
                        if constexpr (i == 0) p[0] = p[0] + y;
                        else p[i] = fma(w[i - 1], y, p[i]);
                    });
                };
#pragma unroll 1
                for (int rep = 0; rep < napply; ++rep) apply_once();
                static_for<0, n>([&](auto I) {
                    *po = p[I];
                    po += nc;
                });
            }
        }
        c = cn;
        cw += stride;
    }
    cp_async_wait<0>();
}

// ---------------------------------------------------------------------------------------------- RK1 (App. A.2)
// First-order implicit drag step  U^(n+1) = (I - dt Omega)^-1 U^(n)  by the O(N) closed form of Eq. A.8-A.9
// (PAPER.md:468-482), per component b -> q:
//     g_i = 1 / (1 + a_i),  c_i = a_i g_i,   A = 1 + sum_i eps_i c_i,   B = sum_i c_i b_i      (a_i = dt / t_s,i)
//     q_0 = (b_0 + B) / A,      q_i = g_i b_i + eps_i c_i q_0.
// The paper's speed reference for the EXP solver (Fig. 6-7).  Same fields, same bytes per cell as the fused EXP
// kernel, O(N) flops: bound by HBM.  Same persistent cp.async staging as k_update (the next cell's fields travel
// while this cell's momenta are worked on), more blocks per SM because the state is two vectors, not two matrices.
constexpr int kRk1MinBlocks = N <= 4 ? 6 : N <= 8 ? 4 : 2;

__global__ void __launch_bounds__(kThreads, kRk1MinBlocks) k_rk1(UpdateArgs g) {
    extern __shared__ double stage[];
    double* s_in = stage + threadIdx.x;                      // [kRowsIn][kThreads]
    double* sp = stage + kRowsIn * kThreads + threadIdx.x;  // [kRowsP][kThreads]
    const long long nc = g.ncells;
    const long long stride = (long long)gridDim.x * kThreads;
    long long c = (long long)blockIdx.x * kThreads + threadIdx.x;

    // row addresses by running pointers (one 64-bit add per row instead of a 64-bit multiply-add chain)
    auto request_inputs = [&](long long cc) {
        if (cc < nc) {
            cp_async8(s_in, g.rho_g + cc);
            const double* pd = g.rho_d + cc;
            const double* pt = g.t_s + cc;
            static_for<0, N>([&](auto I) {
                constexpr int i = I;
                cp_async8(s_in + (1 + i) * kThreads, pd);
                cp_async8(s_in + (1 + N + i) * kThreads, pt);
                pd += nc;
                pt += nc;
            });
        }
        cp_async_commit();
    };
    request_inputs(c);
    while (c < nc) {
        const double* pp = g.p_in + c;
        static_for<0, kRowsP>([&](auto R) {
            constexpr int r = R;
            cp_async8(sp + r * kThreads, pp);
            pp += nc;
        });
        cp_async_commit();
        cp_async_wait<1>();  // the fields of cell c have landed
        double gi[N], ci[N], ei[N];
        double A = 1.0;
        {
            const double irg = fast_rcp(s_in[0]);
            static_for<0, N>([&](auto I) {
                constexpr int i = I;
                const double a = g.dt * fast_rcp(s_in[(1 + N + i) * kThreads]);  // Eq. 15 times dt
                gi[i] = fast_rcp(1.0 + a);
                ci[i] = a * gi[i];
                ei[i] = (s_in[(1 + i) * kThreads] * irg) * ci[i];                // eps_i c_i (Eq. 14)
                A += ei[i];
            });
        }
        const double iA = fast_rcp(A);
        const long long cn = c + stride;
        request_inputs(cn);
        cp_async_wait<1>();  // the momenta of cell c have landed
#pragma unroll
        for (int comp = 0; comp < 3; ++comp) {
            const double* pi = sp + comp * n * kThreads;
            double* po = g.p_out + (long long)comp * n * nc + c;
            double b[n];
            static_for<0, n>([&](auto K) { b[K] = pi[K * kThreads]; });
            double B = b[0];
            static_for<0, N>([&](auto I) { B = fma(ci[I], b[I + 1], B); });
            const double q0 = B * iA;
            *po = q0;
            static_for<0, N>([&](auto I) {
                constexpr int i = I;
                po += nc;
                *po = fma(ei[i], q0, gi[i] * b[i + 1]);
            });
        }
        c = cn;
    }
    cp_async_wait<0>();
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
    const bool valid = c < g.ncells;  // no early return: the lanes of a warp choose the Taylor degree together
    const long long nc = g.ncells;
    const double* A = g.A + c;
    double a[N], w[N], iw[N];
#pragma unroll
    for (int i = 1; i < n; ++i) {
        a[i - 1] = 0.0;
        w[i - 1] = iw[i - 1] = 1.0;
        if (valid) {
            const double ai = __ldg(A + (long long)(0 * n + i) * nc);
            const double bi = __ldg(A + (long long)(i * n + 0) * nc);
            a[i - 1] = ai;
            sym_weights(ai > 0.0 ? bi * fast_rcp(ai) : 1.0, w[i - 1], iw[i - 1]);
        }
    }
    double P[SZ];
    int m, s;
    Core::expm(a, w, iw, P, m, s);
    if (!valid) return;
    if (g.s_out) g.s_out[c] = s;
    double* E = g.E + c;
    static_for<0, n>([&](auto I) {
        constexpr int i = I;
        static_for<0, n>([&](auto K) {
            constexpr int k = K;
            double v = P[Core::sx(i, k)];
            if constexpr (i > 0) v *= w[i - 1];
            if constexpr (k > 0) v *= iw[k - 1];
            if constexpr (i == k) v = 1.0 + P[Core::ix(i, i)];
            E[(long long)(i * n + k) * nc] = v;
        });
    });
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

// Persistent grid: as many blocks as fit on the device at once (or fewer, if there are not enough cells).
template <class Kernel>
cudaError_t launch_persistent(Kernel kernel, int (&blocks_per_sm)[64], const UpdateArgs& a, cudaStream_t st) {
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
    if (blocks_per_sm[dev] == 0) {
        e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes);
        if (e != cudaSuccess) return e;
        int per_sm = 0;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, kThreads, kSmemBytes);
        if (e != cudaSuccess) return e;
        blocks_per_sm[dev] = per_sm > 0 ? per_sm : 1;
    }
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return e;
    const long long want = (a.ncells + kThreads - 1) / kThreads;
    const long long cap = (long long)sms * blocks_per_sm[dev];
    kernel<<<(unsigned)(want < cap ? want : cap), kThreads, kSmemBytes, st>>>(a);
    return cudaGetLastError();
}
cudaError_t launch_update(const UpdateArgs& a, cudaStream_t st) {
    static int blocks_per_sm[64] = {0};  // per device; 0 = not yet queried
    return launch_persistent(k_update, blocks_per_sm, a, st);
}
cudaError_t launch_rk1(const UpdateArgs& a, cudaStream_t st) {
    static int blocks_per_sm[64] = {0};
    return launch_persistent(k_rk1, blocks_per_sm, a, st);
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
                                                    launch_rk1, "thread-per-cell, symmetric packed registers"};

}  // namespace dg
