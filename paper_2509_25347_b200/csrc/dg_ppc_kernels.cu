// dg_ppc_kernels.cu — pair-per-cell fused kernel for NP = DG_NP dust slots (NP even; serves N = NP and N = NP - 1, the
// odd count running with one inert slot: a = 0, w = 1).  Core and layout: dg_ppc.cuh.
//
// One block per SM, 8 warps; a warp works on CHUNKS of 16 cells (two lanes per cell), the cells' matrices in the warp's
// private shared-memory tile.  The lanes of a warp run the largest s and the common Taylor degree m of their 16 cells
// (R8), so cells are handed out sorted by stiffness — the divergence Alg. 2 is written to avoid
// (PAPER.md:646):
//   * the block walks TILES of kTile consecutive cells (tile k of block b is tile b + k gridDim.x of the array);
//   * ONE warp sorts a tile: it computes the norm bound of every cell (reading the 2N + 1 field rows of the tile,
//     coalesced) and sorts (key, cell) words, stiffest first, with a bitonic network in its own shared-memory tile —
//     deterministic, no block barrier;
//   * all warps claim chunks of 16 sorted cells from the tile's counter; the warp that claims the FIRST chunk of tile k
//     sorts tile k + 1 before it starts on its chunk, so the next tile is ready long before this one runs out
//     (three order buffers: the one being overwritten belongs to tile k - 2, and a warp that comes back to a buffer
//     after it has moved on to a later tile sees that from the sequence number in the buffer's state word).  No warp
//     waits for another one except at the very start.
// Loads and stores of the fields are gathers inside a tile.  A tile is small (128 cells, 86 KB of fields) so that the
// tiles in flight on all SMs stay L2-resident: with 2048-cell tiles they did not (5.6 KB of DRAM reads per cell for
// 0.94 KB needed, ncu round 2), because a 32-byte sector fetched for one cell was evicted before its three neighbours
// were processed.
#include <atomic>

#include "dg_async.cuh"
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
constexpr int kTile = 128;
constexpr int kPerLane = kTile / 32;
constexpr int kBufs = 3;
constexpr unsigned kFullMask = 0xffffffffu;

struct Sched {  // block-wide scheduling state
    unsigned short order[kBufs][kTile];  // sorted cell offsets of the tiles in flight
    // per buffer: ((sequence number of the tile whose order is in the buffer) + 1) << 8 | chunks claimed so far; 0 = none.
    // One word, so that publishing a tile, claiming a chunk (compare-and-swap) and noticing that the buffer has moved on
    // to a later tile are each a single atomic access.
    unsigned state[kBufs];
    // per buffer: how many claimed chunks of the tile in the buffer have READ their order[] entries.  A buffer is sorted
    // into again only when every chunk of its previous tile has been counted here (sort_and_publish), so a claimer can
    // never find a later tile's order under its feet, however long it is held up between its claim and its read.
    unsigned done[kBufs];
};
static_assert(kTile / 16 < 256, "the chunk counter lives in the low byte of Sched::state");
constexpr size_t kTilesBytes = Core::kWarpBytes * kWarps;
static_assert(Core::kWarpBytes >= sizeof(unsigned) * kTile, "a warp sorts a tile inside its own shared-memory tile");
constexpr size_t kSmemBytes = kTilesBytes + sizeof(Sched);

__constant__ const Core::Tab c_tab = Core::make_tab();

__device__ __forceinline__ void prefetch_l2(const double* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }
// A load the compiler's front end may not sink towards its first use (the sort keys: all loads of a species together).
__device__ __forceinline__ double ldg_now(const double* p) {
    double v;
    asm volatile("ld.global.nc.f64 %0, [%1];" : "=d"(v) : "l"(p));
    return v;
}
// (cp_async8 of dg_async.cuh: asynchronous 8-byte copy global -> shared, LDGSTS.)  The gathers of a chunk are issued
// back to back through it and waited for ONCE: with plain loads ptxas places each dependent reciprocal right behind its load, and the warp
// (in-order issue) then pays one round trip to L2 per field row — 17 of them per chunk (ncu, round 2).

// One warp sorts the tile starting at cell `base` (count cells) into order[]: key = the squarings the norm bound
// max_i a_i + sum_i eps_i a_i (R5) needs with the m = 30 row (its binary exponent below the last threshold), stiffest first, non-finite first of all, ties in cell order; entries
// past `count` sort last.  keys: kTile words of scratch in the warp's own tile.  Species-major loads: all the lane's
// cells for one species are in flight together.
__device__ __noinline__ void sort_tile_warp(const double* rho_g, const double* rho_d, const double* t_s, double dt,
                                            long long nc, int N, long long base, int count, unsigned* keys,
                                            unsigned short* order, int lane) {
    long long cell[kPerLane];
    double irg[kPerLane], sb[kPerLane], amax[kPerLane];
#pragma unroll
    for (int j = 0; j < kPerLane; ++j) {
        const int idx = lane + j * 32;
        cell[j] = base + (idx < count ? idx : 0);
        irg[j] = ldg_now(rho_g + cell[j]);
        sb[j] = 0.0;
        amax[j] = 0.0;
    }
#pragma unroll
    for (int j = 0; j < kPerLane; ++j) irg[j] = fast_rcp(irg[j]);
#pragma unroll 2
    for (int i = 0; i < N; ++i) {
        double ts[kPerLane], rd[kPerLane];
#pragma unroll
        for (int j = 0; j < kPerLane; ++j) {
            ts[j] = ldg_now(t_s + (long long)i * nc + cell[j]);
            rd[j] = ldg_now(rho_d + (long long)i * nc + cell[j]);
        }
#pragma unroll
        for (int j = 0; j < kPerLane; ++j) {
            const double a = dt * fast_rcp(ts[j]);
            sb[j] = fma(rd[j] * irg[j], a, sb[j]);
            amax[j] = fmax(amax[j], a);
        }
    }
    unsigned mine[kPerLane];
    bool differs = false;
#pragma unroll
    for (int j = 0; j < kPerLane; ++j) {
        const int idx = lane + j * 32;
        // Above the last threshold of Table B.1 the key is the number of squarings the cell needs with the m = 30 row:
        // s = e - t + [f > g] (dg_params.cuh) changes with the mantissa INSIDE a binade, and sorted by the binary exponent
        // alone cells of s and s + 1 sit interleaved in every chunk of that binade (4 % more squarings per chunk).  Below
        // it (s = 0) the key is the binary exponent.  Inf / NaN: largest.  Monotone in the norm; the sort is descending.
        const double nrm = sb[j] + amax[j];
        const unsigned e = ((unsigned)__double2hiint(nrm) >> 20) & 0x7ffu;
        const unsigned v = (nrm > c_theta[kRows - 1]) ? 0x800u + (unsigned)min(scaling_exponent(nrm, c_theta[kRows - 1]), 0x7fe)
                                                      : (e == 0x7ffu ? 0xfffu : e);
        const unsigned key = (idx < count) ? 0xfffu - v : 0x1000u;
        mine[j] = (key << 16) | (unsigned)idx;
    }
    const unsigned k0 = __shfl_sync(kFullMask, mine[0], 0) >> 16;
#pragma unroll
    for (int j = 0; j < kPerLane; ++j) differs |= (lane + j * 32 < count) && ((mine[j] >> 16) != k0);
    if (__any_sync(kFullMask, differs)) {  // (a tile whose cells all carry one key is already in order)
#pragma unroll
        for (int j = 0; j < kPerLane; ++j) keys[lane + j * 32] = mine[j];
        __syncwarp();
#pragma unroll 1
        for (int k = 2; k <= kTile; k <<= 1) {
#pragma unroll 1
            for (int j = k >> 1; j > 0; j >>= 1) {
#pragma unroll
                for (int q = 0; q < kPerLane / 2; ++q) {
                    const int t = lane + q * 32;
                    const int i = ((t & ~(j - 1)) << 1) | (t & (j - 1));
                    const int l = i | j;
                    const unsigned x = keys[i], y = keys[l];
                    const bool up = (i & k) == 0;
                    if ((x > y) == up) {
                        keys[i] = y;
                        keys[l] = x;
                    }
                }
                __syncwarp();
            }
        }
#pragma unroll
        for (int j = 0; j < kPerLane; ++j) mine[j] = keys[lane + j * 32];
        __syncwarp();
    }
#pragma unroll
    for (int j = 0; j < kPerLane; ++j) order[lane + j * 32] = (unsigned short)(mine[j] & 0xffffu);
}

// kEnergy: dg_drag_update_energy in the same launch — the two kinetic-energy sums of Eq. 4's drag part (dg_energy.cu) are
// formed in the apply step, where a lane holds p_in and p_out of its own rows anyway; the plain instantiation carries
// none of it.
struct EnergyArgs {  // E_in, E_out [ncells], heating fraction w
    const double* E_in;
    double* E_out;
    double w;
};
template <bool kEnergy>
__global__ void __launch_bounds__(kThreads, 1) k_update_ppc(UpdateArgs G, int N, EnergyArgs eg) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double* tiles = reinterpret_cast<double*>(smem_raw);
    Sched& sch = *reinterpret_cast<Sched*>(smem_raw + kTilesBytes);

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int r = lane >> 4, c = lane & 15;
    const long long nc = G.ncells;
    const int n = N + 1;
    const long long ntiles = (nc + kTile - 1) / kTile;
    const int ktiles = (int)((ntiles - blockIdx.x + gridDim.x - 1) / gridDim.x);  // tiles of this block
    double* my_tile = tiles + (size_t)warp * Core::CELL * CW;
    const typename Core::View V = Core::view(my_tile, lane);

    auto tile_base = [&](int k) { return ((long long)blockIdx.x + (long long)k * gridDim.x) * kTile; };
    auto tile_count = [&](int k) {
        const long long left = nc - tile_base(k);
        return left < kTile ? (int)left : kTile;
    };
    // sorts tile k into its buffer and publishes it (called by ONE warp, whose own tile is free at that moment)
    auto chunks_of = [&](int k) { return (tile_count(k) + CW - 1) / CW; };
    auto sort_and_publish = [&](int k) {
        const int b = k % kBufs;
        if (k >= kBufs) {
            // The buffer still belongs to tile k - kBufs until all its chunks have read their cells from it.  (They were
            // claimed at least a whole tile ago, so this wait is over before it starts; it is here so that the recycling
            // is correct by construction and not by timing.  No deadlock: a warp counts its read before it claims again,
            // and only a warp that has claimed chunk 0 of tile k - 1 gets here.)
            if (lane == 0) {
                const unsigned need = (unsigned)chunks_of(k - kBufs);
                while (*reinterpret_cast<volatile unsigned*>(&sch.done[b]) < need) __nanosleep(32);
                *reinterpret_cast<volatile unsigned*>(&sch.done[b]) = 0;  // nobody counts again before the publish below
            }
            __syncwarp();
        }
        sort_tile_warp(G.rho_g, G.rho_d, G.t_s, G.dt, nc, N, tile_base(k), tile_count(k),
                       reinterpret_cast<unsigned*>(my_tile), sch.order[b], lane);
        __syncwarp();
        __threadfence_block();
        if (lane == 0) *reinterpret_cast<volatile unsigned*>(&sch.state[b]) = (unsigned)(k + 1) << 8;
        __syncwarp();
    };

    if (threadIdx.x < kBufs) {
        sch.state[threadIdx.x] = 0;
        sch.done[threadIdx.x] = 0;
    }
    __syncthreads();  // the only block-wide barrier
    if (warp == 0) sort_and_publish(0);

    // Claims the next chunk of this block: tile sequence number kc (advanced when a tile runs out), chunk index in the
    // tile, and this lane's cell.  false when the block's tiles are exhausted.
    int kc = 0;
    auto claim = [&](long long& cell, bool& valid) {
        for (;;) {
            if (kc >= ktiles) return false;
            const int b = kc % kBufs;
            const int count = tile_count(kc);
            const int nchunks = (count + CW - 1) / CW;
            int j = 0;
            if (lane == 0) {
                volatile unsigned* st = &sch.state[b];
                for (;;) {
                    const unsigned v = *st;
                    const int seq = (int)(v >> 8) - 1;
                    if (seq < kc) {  // not sorted yet (only at the very start, or behind a slow sorter)
                        __nanosleep(64);
                        continue;
                    }
                    j = (int)(v & 0xffu);
                    if (seq > kc) j = nchunks;  // the buffer already holds a later tile: this one ran out long ago
                    if (j >= nchunks) break;
                    if (atomicCAS(&sch.state[b], v, v + 1) == v) break;
                }
            }
            j = __shfl_sync(kFullMask, j, 0);
            if (j < nchunks) {
                const int pos = j * CW + c;
                valid = pos < count;
                // Invariant: between a successful claim of a chunk of tile kc and the count below, buffer b holds tile
                // kc's order — sort_and_publish(kc + kBufs) waits for done[b] to reach the tile's chunk count first.
                __threadfence_block();  // the order[] entries were written before the state word this claim observed
                cell = tile_base(kc) + (valid ? (int)*reinterpret_cast<volatile unsigned short*>(&sch.order[b][pos]) : 0);
                __threadfence_block();  // ... and are read before this chunk is counted as done with the buffer
                __syncwarp();
                if (lane == 0) atomicAdd(&sch.done[b], 1u);
                // the first claimer of a tile sorts the next one before it starts on its chunk
                if (j == 0 && kc + 1 < ktiles) sort_and_publish(kc + 1);
                return true;
            }
            ++kc;
        }
    };

    long long cell_n = 0;
    bool valid_n = false;
    bool have = claim(cell_n, valid_n);
    while (have) {
        const long long cell = cell_n;
        const bool valid = valid_n;
        {
            // the chunk after this one is claimed now (its fields are prefetched into L2 before this one's apply step)
            have = claim(cell_n, valid_n);

            // a1: eps_i (Eq. 14), a_i = dt / t_s,i (Eq. 15), symmetrising weights, for the species at my own positions
            double av[g], wv[g], iwv[g];
            double sbp = 0.0, amx = 0.0;
            {
                // the fields travel into the (still unused) table: t_s -> col 2, rho_d -> col 3 of my own rows, rho_g ->
                // my copy of the zz slot; a lane reads back only what it requested itself
                {
                    // my own positions hold the dust species k = 2a + r: rows r, r + 2, ... of t_s and rho_d (running
                    // pointers; an inert slot re-reads the last live row)
                    const int r0 = r < N ? r : N - 1;  // (N = 1: role 1 owns no live species; row 1 does not exist)
                    const double* pt = G.t_s + (long long)r0 * nc + cell;
                    const double* pd = G.rho_d + (long long)r0 * nc + cell;
                    const long long step = 2 * nc;
                    static_for<0, g>([&](auto a) {
                        cp_async8(&Core::at(V, 2 * a, 2), pt);
                        cp_async8(&Core::at(V, 2 * a, 3), pd);
                        if (2 * (a + 1) + r < N) {
                            pt += step;
                            pd += step;
                        }
                    });
                }
                cp_async8(&V.x[Core::ZZ * CW], G.rho_g + cell);  // (an absent cell reads the tile's first cell)
                cp_async_wait_all();
                double ts[g], rd[g];
                const double rg = V.x[Core::ZZ * CW];
                static_for<0, g>([&](auto a) {
                    ts[a] = Core::at(V, 2 * a, 2);
                    rd[a] = Core::at(V, 2 * a, 3);
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
            // Every cell of the chunk runs the LARGEST s among its 16 cells: any s' >= s satisfies Theorem 1's premise
            // a fortiori, the lanes would idle through those squarings otherwise, and with one s per
            // warp no store is predicated.  After the sort the chunk's cells differ by at most one in s anyway.
            s = __reduce_max_sync(kFullMask, s);
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

            // a3: Taylor polynomial; a4: s squarings.  One loop: its first pass stores the polynomial, every later one
            // squares first (one copy of the conservation / store code).
            typename Core::Acc A;
            Core::horner(V, m, -sb * sc, A);
            const int smax = s;
            for (int it = 0; it <= smax; ++it) {
                if (it > 0) Core::square(V, c_tab, A);
                if (it == smax) {
                    // This cell's momenta (never touched so far) start their way from HBM to L2 one squaring ahead of the
                    // apply step.  (The fields of the next chunk need no prefetch: the warp that sorted the tile read them.)
                    if (valid) {
                        const long long step = 2 * nc;
                        const double* pg = G.p_in + cell;
#pragma unroll 1
                        for (int cp = 0; cp < 3; ++cp) {
                            if (r == 0) prefetch_l2(pg);
                            const double* pd = pg + (long long)(1 + r) * nc;
#pragma unroll 4
                            for (int k = r; k < N; k += 2) {
                                prefetch_l2(pd);
                                pd += step;
                            }
                            pg += (long long)n * nc;
                        }
                    }
                }
                Core::conserve_store(V, A, it == smax);
            }
            if (valid && r == 0) {
                if (G.s_out) G.s_out[cell] = s;
                if (G.m_out) G.m_out[cell] = m;
            }

            // a5: p_out = p_in + W P W^-1 p_in (Eq. 18).  q = W^-1 p_in for all positions (own: loaded, other: from the
            // partner lane), then one pass over the rows, each row's result going straight to global memory.
            {
                double q[3][C], q0[3];
                {
                    const double* pp = G.p_in + (long long)(1 + r) * nc + cell;
                    static_for<0, 3>([&](auto cp) {
                        double qu[g], qo[g];
                        q0[cp] = valid ? G.p_in[(long long)cp * n * nc + cell] : 0.0;
                        static_for<0, g>([&](auto a) {
                            const int k = 2 * a + r;
                            qu[a] = (valid && k < N) ? pp[(long long)(2 * a) * nc] : 0.0;
                        });
                        static_for<0, g>([&](auto a) { qu[a] *= Core::at(V, 2 * a, Core::CIW); });
                        static_for<0, g>([&](auto a) { qo[a] = __shfl_xor_sync(kFullMask, qu[a], 16); });
                        static_for<0, g>([&](auto a) {
                            q[cp][2 * a] = qu[a];
                            q[cp][2 * a + 1] = r ? qo[(a + 1) % g] : qo[a];  // my other position a is the partner's own
                        });
                        pp += (long long)n * nc;
                    });
                }
                const double* pin = G.p_in + (long long)(1 + r) * nc + cell;
                double* pout = G.p_out + (long long)(1 + r) * nc + cell;
                const long long comp_stride = (long long)n * nc;
                // my own dust rows, species k = 2a + r; the row's p_in values are requested two rows ahead (they were read
                // once for q, but a gather of 27 rows does not survive in what is left of L1 beside the 217 KB of tiles)
                // (energy variant: rho_d of the row travels with its momenta, `prd` below)
                const double* prd = G.rho_d + (long long)r * nc + cell;  // rho_d of my own row a: prd[2a nc]
                auto load_p = [&](int a, double (&pv)[3], double& rv) {
                    const bool live = valid && 2 * a + r < N;
                    static_for<0, 3>([&](auto cp) { pv[cp] = live ? pin[(long long)(2 * a) * nc + cp * comp_stride] : 0.0; });
                    if constexpr (kEnergy) rv = live ? prd[(long long)(2 * a) * nc] : 0.0;
                };
                double pa[3], pb[3], ra = 0.0, rb = 0.0;
                load_p(0, pa, ra);
                load_p(g > 1 ? 1 : 0, pb, rb);
                // (energy variant) this lane's share of sum_i |M_d,i|^2 / (2 rho_d,i) before and after the step
                double kd_in = 0.0, kd_out = 0.0;
                auto row = [&](int a, const double (&pc)[3], double rd, const double (&y)[3]) {
                    const double w = V.x[((2 * a) * Core::ROW + Core::CWT) * CW];
                    if (valid && 2 * a + r < N) {
                        double po[3];
                        static_for<0, 3>([&](auto cp) {
                            po[cp] = fma(w, y[cp], pc[cp]);
                            pout[cp * comp_stride] = po[cp];
                        });
                        if constexpr (kEnergy) {
                            // 1 / (2 rho_d): true division, once per species and cell; a species with rho_d = 0 carries
                            // no energy
                            const double h = rd > 0.0 ? 0.5 / rd : 0.0;
                            kd_in = fma(fma(pc[0], pc[0], fma(pc[1], pc[1], pc[2] * pc[2])), h, kd_in);
                            kd_out = fma(fma(po[0], po[0], fma(po[1], po[1], po[2] * po[2])), h, kd_out);
                        }
                    }
                    pout += 2 * nc;
                };
                // two rows per iteration: twelve independent FMA chains instead of six
#pragma unroll 1
                for (int a = 0; a + 1 < g; a += 2) {
                    double pc0[3], pc1[3], y0[3], y1[3];
                    static_for<0, 3>([&](auto cp) {
                        pc0[cp] = pa[cp];
                        pc1[cp] = pb[cp];
                    });
                    const double rc0 = ra, rc1 = rb;
                    load_p(a + 2 < g ? a + 2 : g - 1, pa, ra);
                    load_p(a + 3 < g ? a + 3 : g - 1, pb, rb);
                    Core::apply_row(V, c_tab.ap[a], q, q0, y0);
                    Core::apply_row(V, c_tab.ap[a + 1], q, q0, y1);
                    row(a, pc0, rc0, y0);
                    row(a + 1, pc1, rc1, y1);
                }
                if constexpr (g % 2 == 1) {
                    double y[3];
                    Core::apply_row(V, c_tab.ap[g - 1], q, q0, y);
                    row(g - 1, pa, ra, y);
                }
                {  // the gas row (both lanes compute it, role 0 stores it)
                    double rgv = 1.0;
                    if constexpr (kEnergy) rgv = G.rho_g[cell];  // (requested before the row's arithmetic)
                    double y[3];
                    Core::apply_row(V, c_tab.ap[g], q, q0, y);
                    if (valid && r == 0) {
                        static_for<0, 3>([&](auto cp) {
                            G.p_out[cp * comp_stride + cell] = q0[cp] + y[cp];  // q0 is the gas momentum itself (w_z = 1)
                        });
                    }
                    if constexpr (kEnergy) {
                        // E_g(t+dt) = E_g(t) + [KE_g(t+dt) - KE_g(t)] + w [K(t) - K(t+dt)],  K = KE_g + sum_i |M_d,i|^2 / (2 rho_d,i)
                        // (dg_energy.cu).  The dust sums of the two lanes are added in role order; role 0 stores.
                        const double oi = __shfl_xor_sync(kFullMask, kd_in, 16), oo = __shfl_xor_sync(kFullMask, kd_out, 16);
                        if (valid && r == 0) {
                            const double h = 0.5 / rgv;
                            double g2_in = 0.0, g2_out = 0.0;
                            static_for<0, 3>([&](auto cp) {
                                const double po = q0[cp] + y[cp];
                                g2_in = fma(q0[cp], q0[cp], g2_in);
                                g2_out = fma(po, po, g2_out);
                            });
                            const double keg_in = g2_in * h, keg_out = g2_out * h;
                            const double k_in = keg_in + (kd_in + oi), k_out = keg_out + (kd_out + oo);
                            eg.E_out[cell] = eg.E_in[cell] + ((keg_out - keg_in) + eg.w * (k_in - k_out));
                        }
                    }
                }
            }
            __syncwarp();  // both lanes of a pair are done with the tile before the next chunk's scratch overwrites it
        }
    }
}

template <bool kEnergy>
cudaError_t launch(const UpdateArgs& a, int N, const EnergyArgs& eg, cudaStream_t st) {
    // blocks per device (one per SM: the shared-memory tile fills it); 0 = not queried.  Atomic: the entry points may be
    // called from several host threads at once (two may both run the query: harmless; a torn value is not).
    static std::atomic<long long> cap[64];
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
    long long blocks = cap[dev].load(std::memory_order_acquire);
    if (blocks == 0) {
        int sms = 0, per_sm = 0;
        e = cudaFuncSetAttribute(k_update_ppc<kEnergy>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes);
        if (e != cudaSuccess) return e;
        e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return e;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_update_ppc<kEnergy>, kThreads, kSmemBytes);
        if (e != cudaSuccess) return e;
        blocks = (long long)sms * (per_sm > 0 ? per_sm : 1);
        cap[dev].store(blocks, std::memory_order_release);
    }
    const long long ntiles = (a.ncells + kTile - 1) / kTile;
    k_update_ppc<kEnergy><<<(unsigned)(ntiles < blocks ? ntiles : blocks), kThreads, kSmemBytes, st>>>(a, N, eg);
    return cudaGetLastError();
}
cudaError_t launch_update(const UpdateArgs& a, int N, cudaStream_t st) {
    return launch<false>(a, N, EnergyArgs{nullptr, nullptr, 0.0}, st);
}
cudaError_t launch_update_energy(const UpdateArgs& a, int N, const double* E_in, double* E_out, double w, cudaStream_t st) {
    return launch<true>(a, N, EnergyArgs{E_in, E_out, w}, st);
}

}  // namespace

#define DG_CAT_(a, b) a##b
#define DG_CAT(a, b) DG_CAT_(a, b)
extern const PpcLaunchers DG_CAT(ppc_launchers_NP, DG_NP) = {launch_update, launch_update_energy, kTile,
                                                             "pair-per-cell, circulant shared-memory tile, sorted chunks"};

}  // namespace dg
