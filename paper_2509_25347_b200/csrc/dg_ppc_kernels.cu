// dg_ppc_kernels.cu — pair-per-cell fused kernel for NP = DG_NP dust slots (NP even; serves N = NP and N = NP - 1, the
// odd count running with one inert slot: a = 0, w = 1).  Core and layout: dg_ppc.cuh.
//
// One block per SM, 8 warps; a warp works on CHUNKS of 16 cells (two lanes per cell), the cell's matrix in the warp's
// private shared-memory tile.  Cells are handed out in TILES of kTile consecutive cells:
//   1. the block computes the norm bound of every cell of the tile (the fields are read once more for this: 33 of the
//      84 doubles a cell moves, from L2 the second time) and sorts the tile by the norm's binary exponent, stiffest
//      first (bitonic sort on (key, cell) words: deterministic);
//   2. warps claim chunks of 16 sorted cells from a shared counter.  The lanes of a warp run the largest s and the common
//      Taylor degree m of their 16 cells (R8), so after the sort a chunk holds cells of (nearly) one s and
//      nothing is executed for lanes that are already done — the divergence Alg. 2 is written to avoid.
// Loads and stores of the fields are therefore gathers inside a 2048-cell window (16 KB per field row, L1/L2-resident);
// at N >= 13 the kernel is bound by the fp64 pipe by a factor of ~20 over HBM, so the gathers do not show.
#include "dg_internal.h"
#include "dg_ppc.cuh"

#ifndef DG_NP
#error "compile with -DDG_NP=<even number of dust slots>"
#endif

namespace dg {
namespace {

constexpr int NP = DG_NP;
using Core = Ppc<NP>;
constexpr int C = Core::C, g = Core::g, CW = Core::CW;
constexpr int kWarps = 8;
constexpr int kThreads = 32 * kWarps;
constexpr int kTile = 2048;
constexpr int kPerThread = kTile / kThreads;
constexpr unsigned kFullMask = 0xffffffffu;

constexpr size_t kTilesBytes = Core::kWarpBytes * kWarps;
constexpr size_t kSortBytes = sizeof(unsigned) * kTile;  // aliases the warp tiles (idle while the block sorts)
constexpr size_t kMatBytes = kTilesBytes > kSortBytes ? kTilesBytes : kSortBytes;
constexpr size_t kSmemBytes = kMatBytes + sizeof(unsigned short) * kTile + 16;

__constant__ const Core::Tab c_tab = Core::make_tab();

__device__ __forceinline__ void prefetch_l2(const double* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }
// A load the compiler may not sink towards its first use: the gathers of a chunk are issued back to back (one round
// trip to L2 / HBM for all of them), not one per dependent reciprocal.
__device__ __forceinline__ double ldg_now(const double* p) {
    double v;
    asm volatile("ld.global.nc.f64 %0, [%1];" : "=d"(v) : "l"(p));
    return v;
}
// Emits nothing; placed after a batch of ldg_now() it keeps every use of v behind the LAST load of the batch (volatile
// asm statements keep their order), so that no dependent instruction stalls the warp before all loads have been issued.
__device__ __forceinline__ void after_loads(double& v) { asm volatile("" : "+d"(v)); }

// Sort keys of the kPerThread cells base + threadIdx.x + j kThreads: the binary exponent of the norm bound
// max_i a_i + sum_i eps_i a_i (R5), stiffest first, non-finite first of all; cells past the end last.
// Species-major so that the loads of all the thread's cells for one species are in flight together.
__device__ __forceinline__ void sort_keys(const UpdateArgs& G, int N, long long base, int count, unsigned* keys) {
    const long long nc = G.ncells;
    long long cell[kPerThread];
    double irg[kPerThread], sb[kPerThread], amax[kPerThread];
#pragma unroll
    for (int j = 0; j < kPerThread; ++j) {
        const int idx = threadIdx.x + j * kThreads;
        cell[j] = base + (idx < count ? idx : 0);
        irg[j] = ldg_now(G.rho_g + cell[j]);
        sb[j] = 0.0;
        amax[j] = 0.0;
    }
#pragma unroll
    for (int j = 0; j < kPerThread; ++j) irg[j] = fast_rcp(irg[j]);
#pragma unroll 2
    for (int i = 0; i < N; ++i) {
        double ts[kPerThread], rd[kPerThread];
#pragma unroll
        for (int j = 0; j < kPerThread; ++j) {
            ts[j] = ldg_now(G.t_s + (long long)i * nc + cell[j]);
            rd[j] = ldg_now(G.rho_d + (long long)i * nc + cell[j]);
        }
#pragma unroll
        for (int j = 0; j < kPerThread; ++j) {
            const double a = G.dt * fast_rcp(ts[j]);
            sb[j] = fma(rd[j] * irg[j], a, sb[j]);
            amax[j] = fmax(amax[j], a);
        }
    }
#pragma unroll
    for (int j = 0; j < kPerThread; ++j) {
        const int idx = threadIdx.x + j * kThreads;
        const unsigned e = ((unsigned)__double2hiint(sb[j] + amax[j]) >> 20) & 0x7ffu;  // 0x7ff: Inf / NaN
        const unsigned key = (idx < count) ? 0x7ffu - e : 0xfffu;
        keys[idx] = (key << 16) | (unsigned)idx;
    }
}

__device__ __forceinline__ void sort_tile(unsigned* keys) {
#pragma unroll 1
    for (int k = 2; k <= kTile; k <<= 1) {
#pragma unroll 1
        for (int j = k >> 1; j > 0; j >>= 1) {
#pragma unroll
            for (int t = threadIdx.x; t < kTile / 2; t += kThreads) {
                const int i = ((t & ~(j - 1)) << 1) | (t & (j - 1));
                const int l = i | j;
                const unsigned x = keys[i], y = keys[l];
                const bool up = (i & k) == 0;
                if ((x > y) == up) {
                    keys[i] = y;
                    keys[l] = x;
                }
            }
            __syncthreads();
        }
    }
}

__global__ void __launch_bounds__(kThreads, 1) k_update_ppc(UpdateArgs G, int N) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double* tiles = reinterpret_cast<double*>(smem_raw);
    unsigned* keys = reinterpret_cast<unsigned*>(smem_raw);
    unsigned short* order = reinterpret_cast<unsigned short*>(smem_raw + kMatBytes);
    int* next_chunk = reinterpret_cast<int*>(smem_raw + kMatBytes + sizeof(unsigned short) * kTile);

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int r = lane >> 4, c = lane & 15;
    const long long nc = G.ncells;
    const int n = N + 1;
    const long long ntiles = (nc + kTile - 1) / kTile;
    const typename Core::View V = Core::view(tiles + (size_t)warp * Core::CELL * CW, lane);

    for (long long tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const long long base = tile * kTile;
        const int count = (nc - base < kTile) ? (int)(nc - base) : kTile;
        // ---- 1. sort the tile by stiffness
        sort_keys(G, N, base, count, keys);
        if (threadIdx.x == 0) *next_chunk = 0;
        __syncthreads();
        // (a tile whose cells all carry one key is already in order)
        const unsigned k0 = keys[0] >> 16;
        int differs = 0;
#pragma unroll
        for (int j = 0; j < kPerThread; ++j) {
            const int idx = threadIdx.x + j * kThreads;
            differs |= (idx < count) && ((keys[idx] >> 16) != k0);
        }
        if (__syncthreads_or(differs)) sort_tile(keys);
        unsigned mine[kPerThread];
#pragma unroll
        for (int j = 0; j < kPerThread; ++j) mine[j] = keys[threadIdx.x + j * kThreads];
        __syncthreads();  // keys (aliasing the warp tiles) are dead from here on
#pragma unroll
        for (int j = 0; j < kPerThread; ++j) order[threadIdx.x + j * kThreads] = (unsigned short)(mine[j] & 0xffffu);
        __syncthreads();
        const int nchunks = (count + CW - 1) / CW;

        // ---- 2. chunks of 16 sorted cells
        auto claim = [&]() {
            int j = 0;
            if (lane == 0) j = atomicAdd(next_chunk, 1);
            return __shfl_sync(kFullMask, j, 0);
        };
        int jnext = claim();
        while (jnext < nchunks) {
            const int j = jnext;
            jnext = claim();  // the chunk after this one (its fields are prefetched into L2 before this one's apply step)
            const int pos = j * CW + c;
            const bool valid = pos < count;
            const long long cell = base + (valid ? (int)order[pos] : 0);

            // a1: eps_i (Eq. 14), a_i = dt / t_s,i (Eq. 15), symmetrising weights, for the species at my own positions
            double av[g], wv[g], iwv[g];
            double sbp = 0.0, amx = 0.0;
            {
                double ts[g], rd[g];
                const double rg = ldg_now(G.rho_g + cell);  // (an absent cell reads the tile's first cell)
                static_for<0, g>([&](auto a) {  // all loads first: one round trip
                    const int k = 2 * a + r;    // dust species at my own position a (an inert slot re-reads species 0)
                    const long long row = (long long)(k < N ? k : 0) * nc + cell;
                    ts[a] = ldg_now(G.t_s + row);
                    rd[a] = ldg_now(G.rho_d + row);
                });
                static_for<0, g>([&](auto a) {
                    after_loads(ts[a]);
                    after_loads(rd[a]);
                });
                const double irg = fast_rcp(rg);
                static_for<0, g>([&](auto a) {
                    const int k = 2 * a + r;
                    const bool live = valid && k < N;
                    double w, iw;
                    sym_weights(rd[a] * irg, w, iw);
                    double aa = G.dt * fast_rcp(ts[a]);
                    aa = live ? aa : 0.0;
                    w = live ? w : 1.0;
                    iw = live ? iw : 1.0;
                    av[a] = aa;
                    wv[a] = w;
                    iwv[a] = iw;
                    sbp = fma(aa * w, w, sbp);
                    amx = fmax(amx, aa);
                });
            }
            // a2: norm bound of the pair's cell (both lanes form it identically), Table B.1 row for the warp, s per cell
            const double sbo = __shfl_xor_sync(kFullMask, sbp, 16);
            const double amo = __shfl_xor_sync(kFullMask, amx, 16);
            const double sb = (r ? sbo : sbp) + (r ? sbp : sbo);
            const double norm = sb + fmax(amx, amo);
            int m, s;
            choose_m_s_warp(norm, Core::hcost(), m, s);
            m = __reduce_max_sync(kFullMask, m);  // already uniform; REDUX puts it in a uniform register
            const double sc = pow2neg(s);
            {
                static_for<0, g>([&](auto a) {
                    const double als = av[a] * sc;
                    Core::at(V, 2 * a, Core::CAL) = als;
                    Core::at(V, 2 * a, Core::CBE) = als * wv[a];
                    Core::at(V, 2 * a, Core::CWT) = wv[a];
                    Core::at(V, 2 * a, Core::CIW) = iwv[a];
                    if constexpr (a == 0) {
                        if (r == 0) {  // position 0 once more in row C (read by role 1)
                            Core::at(V, C, Core::CAL) = als;
                            Core::at(V, C, Core::CBE) = als * wv[a];
                            Core::at(V, C, Core::CWT) = wv[a];
                            Core::at(V, C, Core::CIW) = iwv[a];
                        }
                    }
                });
            }
            __syncwarp();

            // a3: Taylor polynomial; a4: squarings (the last one is replaced by a second apply)
            typename Core::Acc A;
            Core::horner(V, m, -sb * sc, A);
            const int nsq = max(s - Core::kDefer, 0);
            const int napply = 1 << min(Core::kDefer, s);
            Core::conserve_store(V, A, true, nsq == 0);
            const int smax = __reduce_max_sync(kFullMask, nsq);
            // Prefetches into L2, issued one phase ahead of their use — early enough to cover the HBM latency, late enough
            // that the lines are still there (the tiles in flight on all SMs are larger than L2): this cell's momenta
            // before the last squaring, the next chunk's fields before the apply step.
            auto prefetch_momenta = [&]() {
                if (valid) {
                    static_for<0, 3>([&](auto cp) {
                        static_for<0, g>([&](auto a) {
                            const int k = 2 * a + r;
                            if (k < N) prefetch_l2(G.p_in + ((long long)cp * n + 1 + k) * nc + cell);
                        });
                        if (r == 0) prefetch_l2(G.p_in + ((long long)cp * n) * nc + cell);
                    });
                }
            };
            if (smax == 0) prefetch_momenta();
            for (int it = 0; it < smax; ++it) {
                if (it == smax - 1) prefetch_momenta();
                Core::square(V, c_tab, A);
                Core::conserve_store(V, A, it < nsq, it == nsq - 1);
            }
            if (valid && r == 0) {
                if (G.s_out) G.s_out[cell] = s;
                if (G.m_out) G.m_out[cell] = m;
            }

            if (jnext < nchunks && jnext * CW + c < count) {
                const long long cn = base + (int)order[jnext * CW + c];
                if (r == 0) prefetch_l2(G.rho_g + cn);
                static_for<0, g>([&](auto a) {
                    const int k = 2 * a + r;
                    if (k < N) {
                        prefetch_l2(G.t_s + (long long)k * nc + cn);
                        prefetch_l2(G.rho_d + (long long)k * nc + cn);
                    }
                });
            }

            // a5: p_out = p_in + W P W^-1 p_in (Eq. 18), applied 2^min(defer, s) times
            {
                double pu[3][g], p0[3], wu[g], iwu[g];
                static_for<0, g>([&](auto a) {
                    const int k = 2 * a + r;
                    wu[a] = Core::at(V, 2 * a, Core::CWT);
                    iwu[a] = Core::at(V, 2 * a, Core::CIW);
                    static_for<0, 3>([&](auto cp) {
                        pu[cp][a] = (valid && k < N) ? __ldg(G.p_in + ((long long)cp * n + 1 + k) * nc + cell) : 0.0;
                    });
                });
                static_for<0, 3>([&](auto cp) { p0[cp] = valid ? __ldg(G.p_in + ((long long)cp * n) * nc + cell) : 0.0; });
                const int amax_w = __reduce_max_sync(kFullMask, napply);
                for (int rep = 0; rep < amax_w; ++rep) {
                    const bool doit = rep < napply;
                    double q[3][C];
                    static_for<0, 3>([&](auto cp) {
                        double qu[g], qo[g];
                        static_for<0, g>([&](auto a) { qu[a] = pu[cp][a] * iwu[a]; });
                        static_for<0, g>([&](auto a) { qo[a] = __shfl_xor_sync(kFullMask, qu[a], 16); });
                        static_for<0, g>([&](auto a) {
                            q[cp][2 * a] = qu[a];
                            q[cp][2 * a + 1] = r ? qo[(a + 1) % g] : qo[a];  // my other position a is the partner's own
                        });
                    });
                    double y0[3];
                    Core::apply(V, q, p0, y0, [&](auto a, const double (&y)[3]) {
                        static_for<0, 3>([&](auto cp) { pu[cp][a] = doit ? fma(wu[a], y[cp], pu[cp][a]) : pu[cp][a]; });
                    });
                    static_for<0, 3>([&](auto cp) { p0[cp] = doit ? p0[cp] + y0[cp] : p0[cp]; });
                }
                if (valid) {
                    static_for<0, 3>([&](auto cp) {
                        static_for<0, g>([&](auto a) {
                            const int k = 2 * a + r;
                            if (k < N) G.p_out[((long long)cp * n + 1 + k) * nc + cell] = pu[cp][a];
                        });
                        if (r == 0) G.p_out[((long long)cp * n) * nc + cell] = p0[cp];
                    });
                }
            }
            __syncwarp();  // both lanes of a pair are done with the tile before the next chunk's scratch overwrites it
        }
        __syncthreads();  // all chunks of this tile are done: the tiles may be reused as the sort buffer
    }
}

cudaError_t launch_update(const UpdateArgs& a, int N, cudaStream_t st) {
    static long long cap[64] = {0};  // blocks per device (one per SM: the shared-memory tile fills it); 0 = not queried
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
    if (cap[dev] == 0) {
        int sms = 0, per_sm = 0;
        e = cudaFuncSetAttribute(k_update_ppc, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes);
        if (e != cudaSuccess) return e;
        e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return e;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_update_ppc, kThreads, kSmemBytes);
        if (e != cudaSuccess) return e;
        cap[dev] = (long long)sms * (per_sm > 0 ? per_sm : 1);
    }
    const long long ntiles = (a.ncells + kTile - 1) / kTile;
    k_update_ppc<<<(unsigned)(ntiles < cap[dev] ? ntiles : cap[dev]), kThreads, kSmemBytes, st>>>(a, N);
    return cudaGetLastError();
}

}  // namespace

#define DG_CAT_(a, b) a##b
#define DG_CAT(a, b) DG_CAT_(a, b)
extern const PpcLaunchers DG_CAT(ppc_launchers_NP, DG_NP) = {launch_update, kTile,
                                                             "pair-per-cell, circulant shared-memory tile, sorted chunks"};

}  // namespace dg
