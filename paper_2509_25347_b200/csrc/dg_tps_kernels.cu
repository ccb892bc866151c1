// dg_tps_kernels.cu — thread-per-cell fused kernel over SORTED TILES, for ONE species count N = DG_N (N <= 12).
//
// Same arithmetic as k_update of dg_kernels.cu (the Tpc core of dg_tpc.cuh: one thread owns one cell, the packed
// symmetric iterate in its registers).  What differs is which 32 cells share a warp.  The lanes of a warp run the
// Horner loop for the warp's common Taylor degree m and the squaring loop for the warp's LARGEST s (R8), so a
// warp of 32 consecutive cells of a stiff field (s = 3..17 side by side, BASELINE.json configs[4]) executes far more
// than its cells need — the divergence the paper rewrites Alg. 1 into the branch-reduced Alg. 2 for.
// Here a block stages a TILE of kTile consecutive cells in shared memory, counting-sorts it by the binary exponent of
// the norm bound (stiffest first, stable, deterministic) and hands the warps CHUNKS of 32 cells of similar stiffness:
//
//   1. every field row of the tile (rho_g, rho_d[N], t_s[N], p_in[3][n]: 5N + 4 rows of kTile doubles) travels global ->
//      shared with ONE bulk copy per row (cp.async.bulk, the TMA engine; completion on an mbarrier) — no per-thread
//      address arithmetic or LDGSTS, whole 128-byte lines whatever the order the cells are processed in;
//   2. each thread forms the sort key of its cells (conflict-free column reads), a stable counting sort over 64 keys
//      (MATCH.ANY ranks inside a warp, per-segment counters, one warp scans them) writes the permutation;
//   3. the warps take chunks of 32 sorted cells in serpentine order; a lane reads ITS cell's column of the tile (permuted
//      shared-memory reads), runs a1..a4 in registers, applies the result to the cell's momenta in place in the tile;
//   4. the 3n momentum rows leave shared -> global with one bulk copy per row.
// One tile per block, several blocks per SM: the copies of one block overlap the arithmetic of the others.
// The same kernel, instantiated with kEnergy, is dg_drag_update_energy for N <= 12: the tile already holds rho_g, rho_d,
// p_in and p_out, so the kinetic energies before and after the update (Eq. 4, R20) cost one more row (E) and a few
// FMAs per species instead of two further passes over the momenta in HBM.
// Unaligned pointers (8 but not 16 bytes), odd row strides and the ragged last tile take per-thread 8-byte copies.
#include <atomic>
#include <cstdint>

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
// -DDG_TPS_F32: the same kernel in single precision (dg_drag_update_f32: float arrays, the u = 2^-24 thresholds of Eq. B.8)
#ifdef DG_TPS_F32
using Real = float;
using Args = UpdateArgsF32;
#else
using Real = double;
using Args = UpdateArgs;
#endif
using Core = Tpc<N, Real>;
constexpr int SZ = Core::SZ;
constexpr int kThreads = 128;
constexpr int kWarps = kThreads / 32;
// Tile size and resident blocks per SM, measured on B200 (2^22 stiff cells): 128-thread blocks with ONE
// tile each beat larger blocks, larger tiles at fewer blocks per SM and blocks that walk several tiles with the next
// tile's copies under way: what hides a block's load / sort / store phases is the other blocks on the SM.
#if defined(DG_TPS_F32)  // half the bytes and about half the registers per cell
constexpr int kTile = N <= 1 ? 128 : 256;
constexpr int kMinBlocks = N <= 1 ? 16 : N <= 2 ? 14 : N <= 6 ? 6 : N <= 8 ? 4 : 3;
#else
// (N = 11, 12: two 256-cell tiles do not fit one SM.  N = 7: with 128-cell tiles THREE blocks fit at 162 registers without
// spills — 5 % faster on smooth fields, equal on stiff ones; at N = 8 the third block needs a 168-register build: 6 % slower.)
constexpr int kTile = (N <= 1 || N == 7) ? 128 : N <= 10 ? 256 : 128;
constexpr int kMinBlocks = N <= 1 ? 16 : N <= 2 ? 7 : N <= 4 ? 4 : N <= 7 ? 3 : 2;
#endif
static_assert(kTile % kThreads == 0 && kTile <= 2048 && 2048 % kTile == 0, "tile: whole rounds of the block; divides 2048");
constexpr int kPerThread = kTile / kThreads;
constexpr int kSegs = kTile / 32;
constexpr int kKeys = 64;
constexpr int kRowsIn = 1 + 2 * N;  // rho_g, rho_d[N], t_s[N]
constexpr int kRowsP = 3 * n;       // p[3][n]
constexpr unsigned kFull = 0xffffffffu;

template <bool kEnergy>
struct SmemT {
    Real F[kRowsIn][kTile];               // fields of the tile
    Real PM[kRowsP][kTile];               // momenta of the tile: p_in, overwritten in place by p_out
    double EN[kEnergy ? kTile : 2];       // (energy variant) gas energy of the tile: E_in, overwritten in place by E_out
    unsigned long long mbar[2];           // [0] fields landed, [1] momenta landed
    unsigned short seg[kSegs][kKeys];     // counting sort: per 32-cell segment and key, count -> offset inside the key
    unsigned short base[kKeys];           // first sorted position of each key
    unsigned short order[kTile];          // sorted position -> cell of the tile
};
struct EnergyArgs {  // dg_drag_update_energy: E_in, E_out [ncells], heating fraction w
    const double* E_in;
    double* E_out;
    double w;
};
template <bool kEnergy>
constexpr size_t kSmemBytesT = sizeof(SmemT<kEnergy>);

__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
    unsigned done;
    do {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n"
            : "=r"(done)
            : "r"(smem_u32(bar)), "r"(parity)
            : "memory");
    } while (!done);
}
// global -> shared bulk copy (16-byte aligned on both sides, bytes a multiple of 16), completion counted on `bar`
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src_gmem, unsigned bytes, unsigned long long* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n" ::"r"(
                     smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
// shared -> global bulk copy
__device__ __forceinline__ void bulk_s2g(void* dst_gmem, const void* src_smem, unsigned bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;\n" ::"l"(dst_gmem), "r"(smem_u32(src_smem)),
                 "r"(bytes)
                 : "memory");
}

// Sort key of a cell, 1..63, monotone in the norm bound max_i a_i + sum_i eps_i a_i (R5); key 0 is reserved for
// the slots past the end of a ragged tile; the sort is descending; a non-finite norm gets 63: stiffest.
//   N <= 8: the binary exponent of the norm (2^-30 .. 2^31, clamped).
//   N >= 9: above the last threshold of Table B.1 the key IS the number of squarings the cell needs with the m = 30 row
//   (the row stiff cells end up with): s = e - t + [f > g] (dg_params.cuh) changes with the mantissa INSIDE a binade, so
//   a sort by the exponent alone leaves cells of s and s + 1 interleaved in every chunk of that binade (4 % more
//   squarings per chunk); below the threshold (s = 0, where the lower rows compete) it is the binary exponent.
//   Measured: -1.8 % at N = 12, -0.7 % at N = 8 on the stiff recipe, but +0.3-1 % at N <= 8 wherever the squarings are not
//   most of the time (the key costs a few more integer instructions per cell), hence the split.
constexpr bool kSquaringsKey = N >= 9;
__device__ __forceinline__ int sort_key(Real norm) {
    int e;  // unbiased binary exponent (NaN / Inf: large)
    if constexpr (sizeof(Real) == 8) e = (int)(((unsigned)__double2hiint((double)norm) >> 20) & 0x7ffu) - 1023;
    else e = (int)(((unsigned)__float_as_int((float)norm) >> 23) & 0xffu) - 127;
    if constexpr (!kSquaringsKey) {
        return min(max(e + 32, 1), kKeys - 1);
    } else {
        const Real theta = Num<Real>::theta(kRows - 1);  // 3.54 (double), 6.32 (float): exponent 1, 2
        // s = 0.  A valid norm here has e <= theta's exponent, so the key is at most 20; the upper clamp is for a NEGATIVE
        // norm (a cell that breaks the preconditions: t_s < 0, rho < 0), whose exponent can be anything: its key must stay
        // inside seg[][] / base[] so that the damage stays in that cell (include/dg.h, "Pre-conditions").
        if (norm <= theta) return min(max(20 + e - (sizeof(Real) == 8 ? 1 : 2), 1), 20);
        if (!(norm > theta)) return kKeys - 1;                                    // NaN
        return 20 + min(scaling_exponent(norm, theta), kKeys - 1 - 20);
    }
}

template <bool kEnergy>
__global__ void __launch_bounds__(kThreads, kMinBlocks) k_update_tps(Args g, EnergyArgs eg, int bulk_ok) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    SmemT<kEnergy>& sm = *reinterpret_cast<SmemT<kEnergy>*>(smem_raw);
    const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
    const long long nc = g.ncells;
    const long long tile_base = (long long)blockIdx.x * kTile;
    const long long left = nc - tile_base;
    const int count = left < kTile ? (int)left : kTile;
    const bool bulk = bulk_ok && count == kTile;  // block-uniform
    constexpr unsigned kRowBytes = kTile * sizeof(Real);
    Real(&F)[kRowsIn][kTile] = sm.F;
    Real(&PM)[kRowsP][kTile] = sm.PM;
    // ---- 1. the tile's rows: global -> shared ------------------------------------------------------------------
    if (bulk) {
        if (t == 0) {
            mbar_init(&sm.mbar[0], 1);
            mbar_init(&sm.mbar[1], 1);
            asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
        }
        __syncthreads();
        if (warp == 0) {
            if (lane == 0) {
                mbar_expect_tx(&sm.mbar[0], (kRowsIn + (kEnergy ? 1 : 0)) * kRowBytes);
                mbar_expect_tx(&sm.mbar[1], kRowsP * kRowBytes);
            }
            __syncwarp();
            for (int r = lane; r < kRowsIn; r += 32) {
                const Real* src = (r == 0 ? g.rho_g : r <= N ? g.rho_d + (long long)(r - 1) * nc
                                                               : g.t_s + (long long)(r - 1 - N) * nc) +
                                    tile_base;
                bulk_g2s(F[r], src, kRowBytes, &sm.mbar[0]);
            }
            if (kEnergy && lane == 31) bulk_g2s(sm.EN, eg.E_in + tile_base, kRowBytes, &sm.mbar[0]);
            for (int r = lane; r < kRowsP; r += 32)
                bulk_g2s(PM[r], g.p_in + (long long)r * nc + tile_base, kRowBytes, &sm.mbar[1]);
        }
    } else {
#pragma unroll
        for (int j = 0; j < kPerThread; ++j) {
            const int idx = t + j * kThreads;
            if (idx < count) {
                const long long c = tile_base + idx;
                cp_async8(&F[0][idx], g.rho_g + c);
                if constexpr (kEnergy) cp_async8(&sm.EN[idx], eg.E_in + c);
                const Real* pd = g.rho_d + c;
                const Real* pt = g.t_s + c;
#pragma unroll
                for (int i = 0; i < N; ++i) {
                    cp_async8(&F[1 + i][idx], pd);
                    cp_async8(&F[1 + N + i][idx], pt);
                    pd += nc;
                    pt += nc;
                }
            }
        }
        cp_async_commit();
#pragma unroll
        for (int j = 0; j < kPerThread; ++j) {
            const int idx = t + j * kThreads;
            if (idx < count) {
                const Real* pp = g.p_in + tile_base + idx;
#pragma unroll
                for (int r = 0; r < kRowsP; ++r) {
                    cp_async8(&PM[r][idx], pp);
                    pp += nc;
                }
            }
        }
        cp_async_commit();
    }
    // (meanwhile) clear the segment counters
    {
        unsigned* z = reinterpret_cast<unsigned*>(&sm.seg[0][0]);
        for (int i = t; i < kSegs * kKeys / 2; i += kThreads) z[i] = 0u;
    }
    // (only warp 0 polls the mbarrier; the others sleep at the block barrier instead of spending issue slots on the poll:
    // 1 % at N = 1, where the kernel is issue-bound)
    if (bulk) {
        if (warp == 0) mbar_wait(&sm.mbar[0], 0);
    } else {
        cp_async_wait<1>();
    }
    __syncthreads();  // fields visible to every thread; counters cleared

    // ---- 2. keys and the stable counting sort -----------------------------------------------------------------
    int key[kPerThread], rank[kPerThread];
#pragma unroll
    for (int j = 0; j < kPerThread; ++j) {
        const int idx = t + j * kThreads;
        int kk = 0;
        if (idx < count) {
            // (1 / rho_g and a_i = dt / t_s,i replace rho_g and t_s,i in the tile: step 3 reads them back)
            const Real irg = fast_rcp(F[0][idx]);
            F[0][idx] = irg;
            Real sb = Real(0), amax = Real(0);
#pragma unroll
            for (int i = 0; i < N; ++i) {
                const Real a = g.dt * fast_rcp(F[1 + N + i][idx]);
                F[1 + N + i][idx] = a;
                sb = fma(F[1 + i][idx] * irg, a, sb);
                amax = fmax(amax, a);
            }
            kk = sort_key(sb + amax);
        }
        key[j] = kk;
        const unsigned peers = __match_any_sync(kFull, kk);
        rank[j] = __popc(peers & ((1u << lane) - 1u));
        if (rank[j] == 0) sm.seg[j * kWarps + warp][kk] = (unsigned short)__popc(peers);
    }
    __syncthreads();
    if (warp == 0) {
        // lane l owns the keys 63 - 2l and 62 - 2l (descending order of stiffness); segments in cell order
        const int ka = kKeys - 1 - 2 * lane, kb = ka - 1;
        int sa = 0, sb = 0;
#pragma unroll 4
        for (int sg = 0; sg < kSegs; ++sg) {
            const int ca = sm.seg[sg][ka], cb = sm.seg[sg][kb];
            sm.seg[sg][ka] = (unsigned short)sa;
            sm.seg[sg][kb] = (unsigned short)sb;
            sa += ca;
            sb += cb;
        }
        int incl = sa + sb;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int v = __shfl_up_sync(kFull, incl, d);
            if (lane >= d) incl += v;
        }
        const int excl = incl - (sa + sb);
        sm.base[ka] = (unsigned short)excl;
        sm.base[kb] = (unsigned short)(excl + sa);
    }
    __syncthreads();
#pragma unroll
    for (int j = 0; j < kPerThread; ++j) {
        const int idx = t + j * kThreads;
        const int pos = sm.base[key[j]] + sm.seg[j * kWarps + warp][key[j]] + rank[j];
        sm.order[pos] = (unsigned short)idx;
    }
    // The momenta are first needed by the apply step, a whole matrix exponential later.  For N <= 4 (bulk path) they are
    // not waited for here: each warp checks their mbarrier before its first apply (measured: -6.5 % at N = 1, -1.6 % at
    // N = 4, neutral at N = 2, 3; from N = 5 the per-warp poll costs more than the earlier start gains, +0.2-2 %).
    constexpr bool kLateP = N <= 4;
    if (bulk) {
        if (!kLateP && warp == 0) mbar_wait(&sm.mbar[1], 0);
    } else {
        cp_async_wait<0>();
    }
    __syncthreads();  // permutation (and, unless deferred, the momenta) visible
    bool p_landed = !(bulk && kLateP);

    // ---- 3. chunks of 32 sorted cells ------------------------------------------------------------------------------
    // Chunks are dealt to the warps in serpentine order (0 1 2 3 | 3 2 1 0 | ..): the tile is sorted stiffest first, so
    // every warp gets about the same number of squarings without a shared counter.
#pragma unroll 1
    for (int round = 0;; ++round) {
        const int j = round * kWarps + ((round & 1) ? kWarps - 1 - warp : warp);
        if (round * kWarps * 32 >= count) break;
        if (j * 32 >= count) continue;
        const int pos = j * 32 + lane;
        const bool valid = pos < count;
        const int cell = sm.order[valid ? pos : j * 32];

        // a1: eps_i (Eq. 14), a_i = dt alpha_i (Eq. 15), symmetrising weights; a lane without a cell gets the identity
        Real a[N], w[N], iw[N];
        {
            const Real irg = F[0][cell];
            static_for<0, N>([&](auto I) {
                constexpr int i = I;
                a[i] = F[1 + N + i][cell];
                const Real rd = F[1 + i][cell];
                sym_weights(rd * irg, w[i], iw[i]);
                if (!valid) {
                    a[i] = Real(0);
                    w[i] = iw[i] = Real(1);
                }
                if constexpr (kEnergy) {
                    // 1 / (2 rho_d,i) replaces rho_d,i in the cell's column of the tile (a species with rho_d = 0 carries
                    // no energy); true division: one per species and cell, off the critical path
                    if (valid) F[1 + i][cell] = rd > Real(0) ? Real(0.5) / rd : Real(0);
                }
            });
        }
        // a2-a4
        Real P[SZ];
        int m, s;
        Core::template expm<Core::kDefer>(a, w, iw, P, m, s);
        if (valid) {
            if (g.s_out) g.s_out[tile_base + cell] = s;
            if (g.m_out) g.m_out[tile_base + cell] = m;
        }
        // a5: p_out = p_in + W P W^-1 p_in, in place in the tile, one component at a time
        if (!p_landed) {  // warp-uniform
            mbar_wait(&sm.mbar[1], 0);
            p_landed = true;
        }
        if (valid) {
            const int napply = 1 << min(Core::kDefer, s);
            // (energy variant) sums over the components of |M_g|^2 and of sum_i |M_d,i|^2 / (2 rho_d,i), before and after
            double g2_in = 0.0, kd_in = 0.0, g2_out = 0.0, kd_out = 0.0;
            auto kinetic = [&](const Real (&pv)[n], double& g2, double& kd) {
                g2 = fma((double)pv[0], (double)pv[0], g2);
                static_for<1, n>([&](auto K) { kd = fma((double)pv[K] * (double)pv[K], (double)F[K][cell], kd); });
            };
#pragma unroll 1
            for (int comp = 0; comp < 3; ++comp) {
                Real* pc = &PM[comp * n][cell];
                Real p[n], q[n];
                static_for<0, n>([&](auto K) { p[K] = pc[K * kTile]; });
                if constexpr (kEnergy) kinetic(p, g2_in, kd_in);
                auto apply_once = [&]() {
                    static_for<0, n>([&](auto K) {
                        constexpr int kq = K;
                        if constexpr (kq == 0) q[kq] = p[kq];
                        else q[kq] = p[kq] * iw[kq - 1];
                    });
                    static_for<0, n>([&](auto I) {
                        constexpr int i = I;
                        Real y = Real(0);
                        static_for<0, n>([&](auto K) {
                            constexpr int kq = K;
                            y = fma(P[Core::sx(i, kq)], q[kq], y);
                        });
                        if constexpr (i == 0) p[0] = p[0] + y;
                        else p[i] = fma(w[i - 1], y, p[i]);
                    });
                };
#pragma unroll 1
                for (int rep = 0; rep < napply; ++rep) apply_once();
                static_for<0, n>([&](auto K) { pc[K * kTile] = p[K]; });
                if constexpr (kEnergy) kinetic(p, g2_out, kd_out);
            }
            if constexpr (kEnergy) {
                // E_g(t+dt) = E_g(t) + [KE_g(t+dt) - KE_g(t)] + w [K(t) - K(t+dt)],  K = KE_g + sum_i |M_d,i|^2 / (2 rho_d,i)
                const double h = 0.5 * F[0][cell];  // 1 / (2 rho_g)
                const double keg_in = g2_in * h, keg_out = g2_out * h;
                const double k_in = keg_in + kd_in, k_out = keg_out + kd_out;
                sm.EN[cell] = sm.EN[cell] + ((keg_out - keg_in) + eg.w * (k_in - k_out));
            }
        }
    }

    // ---- 4. the momentum rows: shared -> global --------------------------------------------------------------------
    if (bulk) {
        asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");  // generic-proxy writes before async-proxy reads
        __syncthreads();
        if (warp == 0) {
            for (int r = lane; r < kRowsP; r += 32) bulk_s2g(g.p_out + (long long)r * nc + tile_base, PM[r], kRowBytes);
            if (kEnergy && lane == 31) bulk_s2g(eg.E_out + tile_base, sm.EN, kRowBytes);
            asm volatile("cp.async.bulk.commit_group;\n" ::: "memory");
            asm volatile("cp.async.bulk.wait_group.read 0;\n" ::: "memory");  // the tile must outlive the reads
        }
    } else {
        __syncthreads();
#pragma unroll
        for (int j = 0; j < kPerThread; ++j) {
            const int idx = t + j * kThreads;
            if (idx < count) {
                Real* po = g.p_out + tile_base + idx;
#pragma unroll
                for (int r = 0; r < kRowsP; ++r) {
                    *po = PM[r][idx];
                    po += nc;
                }
                if constexpr (kEnergy) eg.E_out[tile_base + idx] = sm.EN[idx];
            }
        }
    }
}

template <bool kEnergy>
cudaError_t launch(const Args& a, const EnergyArgs& eg, cudaStream_t st) {
    // Per device: has the kernel been given its dynamic shared-memory size.  Atomic: the entry points may be called from
    // several host threads at once (include/dg.h); setting the attribute twice is harmless, a torn flag is not.
    static std::atomic<bool> configured[64];
    constexpr size_t smem = kSmemBytesT<kEnergy>;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
    if (!configured[dev].load(std::memory_order_acquire)) {
        e = cudaFuncSetAttribute(k_update_tps<kEnergy>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        configured[dev].store(true, std::memory_order_release);
    }
    const long long ntiles = (a.ncells + kTile - 1) / kTile;
    if (ntiles > 0x7fffffffLL) return cudaErrorInvalidValue;
    // bulk copies need 16-byte aligned rows: 16-byte aligned base pointers and an even row stride
    uintptr_t bits = reinterpret_cast<uintptr_t>(a.rho_g) | reinterpret_cast<uintptr_t>(a.rho_d) |
                     reinterpret_cast<uintptr_t>(a.t_s) | reinterpret_cast<uintptr_t>(a.p_in) |
                     reinterpret_cast<uintptr_t>(a.p_out);
    if (kEnergy) bits |= reinterpret_cast<uintptr_t>(eg.E_in) | reinterpret_cast<uintptr_t>(eg.E_out);
    constexpr long long kPer16 = 16 / sizeof(Real);  // elements per 16 bytes: the row stride must be a multiple of it
    const int bulk_ok = ((bits & 15u) == 0 && a.ncells % kPer16 == 0) ? 1 : 0;
    k_update_tps<kEnergy><<<(unsigned)ntiles, kThreads, smem, st>>>(a, eg, bulk_ok);
    return cudaGetLastError();
}
#ifdef DG_TPS_F32
cudaError_t launch_update(const UpdateArgsF32& a, cudaStream_t st) { return launch<false>(a, EnergyArgs{nullptr, nullptr, 0.0}, st); }
#else
cudaError_t launch_update(const UpdateArgs& a, cudaStream_t st) { return launch<false>(a, EnergyArgs{nullptr, nullptr, 0.0}, st); }
cudaError_t launch_update_energy(const UpdateArgs& a, const double* E_in, double* E_out, double w, cudaStream_t st) {
    return launch<true>(a, EnergyArgs{E_in, E_out, w}, st);
}
#endif

}  // namespace

#define DG_CAT_(a, b) a##b
#define DG_CAT(a, b) DG_CAT_(a, b)
#ifdef DG_TPS_F32
extern const TpsF32Launchers DG_CAT(tps_f32_launchers_N, DG_N) = {launch_update, kTile};
#else
extern const TpsLaunchers DG_CAT(tps_launchers_N, DG_N) = {launch_update, launch_update_energy, kTile,
                                                           "thread-per-cell over stiffness-sorted shared-memory tiles"};
#endif

}  // namespace dg
