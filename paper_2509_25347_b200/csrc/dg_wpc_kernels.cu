// dg_wpc_kernels.cu — warp-per-cell DMMA kernels for ONE species count N = DG_N (compiled once per N).
//
// A warp walks GROUPS of kGroup = 4 consecutive cells: one field row of a group is 32 contiguous bytes — exactly one
// DRAM sector when the row is 32-byte aligned — so every byte the kernel moves is a byte the method needs (a warp
// that loaded its single cell's fields lane by lane fetched 4-5x the algorithmic bytes, ncu round 1).  All rows of
// the NEXT group are requested with cp.async into the warp's private double-buffered staging tile before the
// matrix work of the current group starts; results are staged in shared memory (over the group's own momenta rows)
// and written back as whole sectors.
// There is no block-level synchronisation: warps are independent, __syncwarp is the only barrier.
#include <atomic>

#include "dg_async.cuh"
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
constexpr int kGroup = 4;             // cells per staged group
constexpr int kRowsIn = 1 + 2 * N;    // rho_g, rho_d[N], t_s[N]
constexpr int kRowsP = 3 * n;         // p[3][n]
constexpr int kRows = kRowsIn + kRowsP;
constexpr int kPerPass = 32 / ND;     // cells whose species fit the 32 lanes of one prologue pass

struct alignas(16) WarpSmem {
    double in[2][kRows][kGroup];   // staged inputs, double buffered: [stage][row][cell of the group]; a cell's
                                   // results overwrite its own momenta rows once they have been consumed
    Core::Cell cell[kGroup];       // per-cell vectors prepared by the prologue
    double q[3][ND], q0[4];        // W^-1 p_in of the current cell, per component (q0[3] pads to 16 bytes)
};
static_assert(sizeof(WarpSmem) % 16 == 0, "cp.async 16-byte destinations need 16-byte aligned per-warp tiles");
constexpr size_t kSmemBytes = sizeof(WarpSmem) * kWarps;

__device__ __forceinline__ const double* row_ptr(const UpdateArgs& g, int r) {
    const long long nc = g.ncells;
    if (r == 0) return g.rho_g;
    if (r < 1 + N) return g.rho_d + (long long)(r - 1) * nc;
    if (r < kRowsIn) return g.t_s + (long long)(r - 1 - N) * nc;
    return g.p_in + (long long)(r - kRowsIn) * nc;
}

// Requests all rows of the group starting at cell c0 into `dst`.  vec16: every row start is 16-byte aligned
// (ncells even) and the group is complete, so a row is two 16-byte copies; otherwise element by element.
__device__ __forceinline__ void request_group(const UpdateArgs& g, double (*dst)[kGroup], long long c0, int lane,
                                              bool vec16) {
    const long long nc = g.ncells;
    if (c0 < nc) {
        if (vec16 && c0 + kGroup <= nc) {
            for (int it = lane; it < 2 * kRows; it += 32) {
                const int r = it >> 1, h = it & 1;
                cp_async16(&dst[r][2 * h], row_ptr(g, r) + c0 + 2 * h);
            }
        } else {
            for (int it = lane; it < kGroup * kRows; it += 32) {
                const int r = it >> 2, k = it & 3;
                if (c0 + k < nc) cp_async8(&dst[r][k], row_ptr(g, r) + c0 + k);
            }
        }
    }
    cp_async_commit();
}

// Segmented (ND lanes) sum and max.
__device__ __forceinline__ double seg_sum(double x) {
#pragma unroll
    for (int o = 1; o < ND; o <<= 1) x += __shfl_xor_sync(kFull, x, o);
    return x;
}
__device__ __forceinline__ double seg_max(double x) {
#pragma unroll
    for (int o = 1; o < ND; o <<= 1) x = fmax(x, __shfl_xor_sync(kFull, x, o));
    return x;
}

// a1 for one lane's (cell, species): eps (Eq. 14), a = dt alpha (Eq. 15), the symmetrising weights; fills the
// cell's vectors.  Lanes of padding species (sp >= N) or absent cells contribute a = 0, w = 1.
__device__ __forceinline__ void prepare(Core::Cell& cv, int sp, bool live, double dt, double rho_g, double rho_d,
                                        double t_s) {
    double a = 0.0, w = 1.0, iw = 1.0;
    if (live) {
        a = dt * fast_rcp(t_s);
        sym_weights(rho_d * fast_rcp(rho_g), w, iw);
    }
    const double be = a * w;
    const double sb = seg_sum(be * w);
    const double amax = seg_max(a);
    cv.a[sp] = a;
    cv.be[sp] = be;
    cv.w[sp] = w;
    cv.iw[sp] = iw;
    if (sp == 0) {
        cv.sb = sb;
        cv.amax = amax;
    }
}

// ---------------------------------------------------------------------------------------------- fused a1..a5
__global__ void __launch_bounds__(kThreads, 3) k_update_wpc(UpdateArgs g) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    WarpSmem& sm = reinterpret_cast<WarpSmem*>(smem_raw)[warp];
    const Core::Lane L;
    const long long nc = g.ncells;
    const long long ngroups = (nc + kGroup - 1) / kGroup;
    const long long gstride = (long long)gridDim.x * kWarps;
    // 16-byte copies need every row start 16-byte aligned: an even cell count AND 16-byte aligned base pointers (the ABI
    // only asks for 8: include/dg.h); otherwise the element-by-element path
    const bool vec16 = (nc & 1) == 0 &&
                       ((reinterpret_cast<unsigned long long>(g.rho_g) | reinterpret_cast<unsigned long long>(g.rho_d) |
                         reinterpret_cast<unsigned long long>(g.t_s) | reinterpret_cast<unsigned long long>(g.p_in) |
                         reinterpret_cast<unsigned long long>(g.p_out)) & 15ull) == 0;
    long long grp = (long long)blockIdx.x * kWarps + warp;
    int stage = 0;
    request_group(g, sm.in[0], grp * kGroup, lane, vec16);
    for (; grp < ngroups; grp += gstride, stage ^= 1) {
        const long long c0 = grp * kGroup;
        // the next group's rows travel while this group is worked on (an empty commit past the end keeps the
        // wait count uniform)
        request_group(g, sm.in[stage ^ 1], (grp + gstride) * kGroup, lane, vec16);
        cp_async_wait<1>();
        __syncwarp();
        double (*in)[kGroup] = sm.in[stage];
        const int ncell = (nc - c0 < kGroup) ? (int)(nc - c0) : kGroup;

        // a1 for the whole group: lane <-> (cell, species)
#pragma unroll
        for (int pass = 0; pass < kGroup / kPerPass; ++pass) {
            const int k = pass * kPerPass + lane / ND, sp = lane % ND;
            const bool live = (sp < N) && (k < ncell);
            double rg = 1.0, rd = 1.0, ts = 1.0;
            if (live) {
                rg = in[0][k];
                rd = in[1 + sp][k];
                ts = in[1 + N + sp][k];
            }
            prepare(sm.cell[k], sp, live, g.dt, rg, rd, ts);
        }
        __syncwarp();

        for (int k = 0; k < ncell; ++k) {
            const Core::Cell& cv = sm.cell[k];
            // a2-a4
            Core::Result R;
            Core::expm(L, cv, R);
            if (lane == 0) {
                if (g.s_out) g.s_out[c0 + k] = R.s;
                if (g.m_out) g.m_out[c0 + k] = R.m;
            }
            // a5: y = P W^-1 p_in, p_out = p_in + W y
            if (lane < ND) {
                const double iw = cv.iw[lane];
#pragma unroll
                for (int comp = 0; comp < 3; ++comp)
                    sm.q[comp][lane] = (lane < N) ? in[kRowsIn + comp * n + 1 + lane][k] * iw : 0.0;
            } else if (lane < ND + 3) {
                sm.q0[lane - ND] = in[kRowsIn + (lane - ND) * n][k];
            }
            __syncwarp();
            {
                // Dust rows, all three components in ONE tensor-core product: Y = r q0^T + T Q with Q[j][comp] as the
                // B operand (lane (g, t) supplies Q[8K + 2t + e][g], zero for g >= 3).  The accumulator hands lane
                // (g, t) the entries Y[8I + g][2t], Y[8I + g][2t + 1]: components 0, 1 to t = 0, component 2 to t = 1,
                // with no cross-lane reduction.
                double Bq[TL][2];
#pragma unroll
                for (int K = 0; K < TL; ++K)
#pragma unroll
                    for (int e = 0; e < 2; ++e) Bq[K][e] = (L.g < 3) ? sm.q[L.g][8 * K + 2 * L.t + e] : 0.0;
                const double q0a = (L.t < 2) ? sm.q0[2 * L.t] : 0.0;       // q0[2t]     (t = 0, 1)
                const double q0b = (L.t == 0) ? sm.q0[1] : 0.0;             // q0[2t + 1] (t = 0)
                double Y[TL][2];
#pragma unroll
                for (int I = 0; I < TL; ++I) {
                    Y[I][0] = R.rR.v[I] * q0a;
                    Y[I][1] = R.rR.v[I] * q0b;
                }
#pragma unroll
                for (int K = 0; K < TL; ++K)
#pragma unroll
                    for (int e = 0; e < 2; ++e)
#pragma unroll
                        for (int I = 0; I < TL; ++I) dmma884(Y[I][0], Y[I][1], R.T[I][K][e], Bq[K][e]);
                // gas row: y0 = d0 q0 + r . q, per component (quad reductions, independent of the product above)
                double y0[3];
#pragma unroll
                for (int comp = 0; comp < 3; ++comp) {
                    Core::VecC qC;
#pragma unroll
                    for (int I = 0; I < TL; ++I)
#pragma unroll
                        for (int e = 0; e < 2; ++e) qC.v[I][e] = sm.q[comp][8 * I + 2 * L.t + e];
                    y0[comp] = fma(R.d0, sm.q0[comp], Core::dotC(R.rC, qC));
                }
#pragma unroll
                for (int I = 0; I < TL; ++I) {
                    const int row = 8 * I + L.g;
                    if (row < N && L.t < 2) {
                        const double w = cv.w[row];
                        double* slot = &in[kRowsIn + 2 * L.t * n + 1 + row][k];  // component 2t
                        *slot = fma(w, Y[I][0], *slot);
                        if (L.t == 0) slot[n * kGroup] = fma(w, Y[I][1], slot[n * kGroup]);  // component 1
                    }
                }
                if (lane < 3) in[kRowsIn + lane * n][k] = sm.q0[lane] + (lane == 0 ? y0[0] : lane == 1 ? y0[1] : y0[2]);
            }
            __syncwarp();
        }

        // write the group's results: whole 32-byte sectors when aligned and complete
        if (vec16 && ncell == kGroup) {
            for (int it = lane; it < 2 * kRowsP; it += 32) {
                const int r = it >> 1, h = it & 1;
                const double2 v = *reinterpret_cast<const double2*>(&in[kRowsIn + r][2 * h]);
                *reinterpret_cast<double2*>(g.p_out + (long long)r * nc + c0 + 2 * h) = v;
            }
        } else {
            for (int it = lane; it < kGroup * kRowsP; it += 32) {
                const int r = it >> 2, k = it & 3;
                if (k < ncell) g.p_out[(long long)r * nc + c0 + k] = in[kRowsIn + r][k];
            }
        }
        __syncwarp();
    }
    cp_async_wait<0>();
}

// ---------------------------------------------------------------------------------------------- staged a2-a4
__global__ void __launch_bounds__(kThreads) k_expm_wpc(ExpmArgs g) {
    __shared__ Core::Cell cells[kWarps];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    Core::Cell& cv = cells[warp];
    const Core::Lane L;
    const long long nc = g.ncells;
    const long long stride = (long long)gridDim.x * kWarps;
    for (long long c = (long long)blockIdx.x * kWarps + warp; c < nc; c += stride) {
        // recover a_j and eps_j from the staged matrix: A_0j = a_j, A_j0 = eps_j a_j (Eq. 17)
        if (lane < ND) {
            double a = 0.0, w = 1.0, iw = 1.0;
            if (lane < N) {
                a = __ldg(g.A + (long long)(0 * n + lane + 1) * nc + c);
                const double b = __ldg(g.A + (long long)((lane + 1) * n + 0) * nc + c);
                sym_weights(a > 0.0 ? b * fast_rcp(a) : 1.0, w, iw);
            }
            cv.a[lane] = a;
            cv.be[lane] = a * w;
            cv.w[lane] = w;
            cv.iw[lane] = iw;
        }
        __syncwarp();
        if (lane == 0) {
            double sb = 0.0, amax = 0.0;
            for (int j = 0; j < N; ++j) {
                sb = fma(cv.be[j], cv.w[j], sb);
                amax = fmax(amax, cv.a[j]);
            }
            cv.sb = sb;
            cv.amax = amax;
        }
        __syncwarp();
        Core::Result R;
        Core::expm(L, cv, R);
        if (lane == 0 && g.s_out) g.s_out[c] = R.s;
        double* E = g.E + c;
        // E = I + W P W^-1
#pragma unroll
        for (int I = 0; I < TL; ++I) {
            const int row = 8 * I + L.g;
            const double wr = cv.w[row];
#pragma unroll
            for (int J = 0; J < TL; ++J)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int col = 8 * J + 2 * L.t + e;
                    if (row < N && col < N) {
                        const double v = (row == col) ? 1.0 + R.T[I][J][e] : wr * R.T[I][J][e] * cv.iw[col];
                        E[(long long)((row + 1) * n + col + 1) * nc] = v;
                    }
                }
            if (L.t == 0 && row < N) E[(long long)((row + 1) * n) * nc] = wr * R.rR.v[I];  // column 0
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int col = 8 * I + 2 * L.t + e;
                if (L.g == 0 && col < N) E[(long long)(col + 1) * nc] = R.rC.v[I][e] * cv.iw[col];  // row 0
            }
        }
        if (lane == 0) E[0] = 1.0 + R.d0;
        __syncwarp();
    }
}

// Persistent grid: as many blocks as fit on the device at once (or fewer, if there is not enough work).  The
// occupancy query and the shared-memory opt-in are done once per device and cached (`cap` = blocks per device; atomic,
// because the entry points may be called from several host threads at once: two threads may both do the query, which is
// harmless, but neither may see a torn value).
using CapTable = std::atomic<long long>[64];
cudaError_t persistent_grid(const void* kernel, size_t smem, CapTable& cap, long long units, unsigned* grid) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
    long long blocks = cap[dev].load(std::memory_order_acquire);
    if (blocks == 0) {
        int sms = 0, per_sm = 0;
        if (smem > 0) {
            e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e != cudaSuccess) return e;
        }
        e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return e;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, kThreads, smem);
        if (e != cudaSuccess) return e;
        blocks = (long long)sms * (per_sm > 0 ? per_sm : 1);
        cap[dev].store(blocks, std::memory_order_release);
    }
    const long long want = (units + kWarps - 1) / kWarps;
    *grid = (unsigned)(want < blocks ? want : blocks);
    return cudaSuccess;
}

cudaError_t launch_update(const UpdateArgs& a, cudaStream_t st) {
    static CapTable cap;  // per device; 0 = not yet queried
    unsigned grid = 0;
    const long long ngroups = (a.ncells + kGroup - 1) / kGroup;
    cudaError_t e = persistent_grid((const void*)k_update_wpc, kSmemBytes, cap, ngroups, &grid);
    if (e != cudaSuccess) return e;
    k_update_wpc<<<grid, kThreads, kSmemBytes, st>>>(a);
    return cudaGetLastError();
}
cudaError_t launch_expm(const ExpmArgs& a, cudaStream_t st) {
    static CapTable cap;
    unsigned grid = 0;
    cudaError_t e = persistent_grid((const void*)k_expm_wpc, 0, cap, a.ncells, &grid);
    if (e != cudaSuccess) return e;
    k_expm_wpc<<<grid, kThreads, 0, st>>>(a);
    return cudaGetLastError();
}

}  // namespace

#define DG_CAT_(a, b) a##b
#define DG_CAT(a, b) DG_CAT_(a, b)
extern const WpcLaunchers DG_CAT(wpc_launchers_N, DG_N) = {launch_update, launch_expm,
                                                           "warp-per-cell, DMMA m8n8k4 symmetric tiles"};

}  // namespace dg
