// dg_ppc.cuh — pair-per-cell core: TWO lanes own one cell; the symmetrised iterate X lives in shared memory, the
// accumulators of a squaring in the two lanes' registers.  This is the "hierarchical" mapping with shared-memory
// staging that the paper suggests but does not build, sized for N = 13..16 where one thread can no
// longer hold the matrices in registers (the register cliff the paper measures at N = 8 -> 9).
//
// Same arithmetic as dg_tpc.cuh: symmetrised arrowhead S = W^-1 (dt Omega) W of Eq. 17
// (PAPER.md:117-126), X = exp(S) carried as off-diagonals O >= 0 plus a diagonal that is never computed by the
// recurrences but re-derived from conservation of total momentum, the Taylor polynomial of Eq. 19
// by the factored Horner recurrence, s cancellation-free squarings (Eq. 23-24).
//
// Why two lanes and why this layout.  A squaring of the symmetric n x n iterate is  C_ik = sum_l X_li X_lk  for the
// n(n-1)/2 pairs i < k (the diagonal comes from conservation): 2312 FMAs at n = 17.  B200 moves 16 doubles per clock
// per SM out of shared memory against 64 fp64 FMAs per clock, so every operand fetched must feed >= 4 FMAs; with all
// 136 accumulators of one cell in ONE thread that ratio would be 8 but they do not fit (272 registers), and fp64
// shared-memory loads are served per half-warp, so two lanes reading the same word do not share a wavefront.  Two
// lanes with 68 accumulators each, both streaming the whole row l (17 loads for 68 FMAs), is the register-feasible
// point; what remains is to give both lanes THE SAME CODE with no selects or predicates in the hot loop:
//
//   * The NP (even) dust species sit on a circle of C = NP positions, the gas is the extra index z.  Role r in {0,1}
//     "owns" the positions p = 2a + r (a = 0..g-1, g = C/2) and computes the pairs
//         T: {2a+r, 2b+r}               a < b                 (own, own)
//         M: {2a+r, 2((a+dd) mod g)+1+r}  dd = 0..D-1, D = ceil(g/2)   (own, other)
//         Z: {z, 2a+r}                                        (gas, own)
//     Role 1's pairs are role 0's rotated by one position; together they are all pairs exactly once (for odd g the
//     antipodal class is computed by both and stored by role 0).
//   * The matrix is stored by circle DIAGONALS: pair {p, p+d} at table[p][d], d = 0..g, with X[z][p], w[p] and 1/w[p]
//     in three more columns of row p, plus row C = a copy of row 0, plus X[z][z] once per role.  Rotating every index
//     by one position then moves every address by the same constant (one table row), so role 1 runs role 0's code on
//     a base pointer shifted by one row: no select and no predicate in the hot loop.
//   * The squaring loops over the rows l of X (two per iteration, operands double-buffered) with the row's operand
//     offsets in a constant-memory table (LDCU.128 + LDS [R + UR]): 2 KB of loop instead of 29 KB of unrolled code.
//
// Measured on B200 (N = 16, ncu, profiles/): in the squaring loop the fp64 pipe and the shared-memory pipe are
// co-limiting (17 eight-byte loads per lane per 68 FMAs = one wavefront per 4 FMAs of the SM, exactly the ratio of the
// two peaks); whole kernel: fp64 pipe ~62 % busy, shared-memory wavefronts ~73 % of peak.
#pragma once
#include "dg_params.cuh"
#include "dg_tpc.cuh"  // static_for, Idx

namespace dg {

template <int NP>
struct Ppc {
    static_assert(NP >= 2 && NP % 2 == 0, "pair-per-cell core: even number of dust slots");
    static constexpr int C = NP;            // circle size = dust slots
    static constexpr int g = NP / 2;        // positions per role
    static constexpr int D = (g + 1) / 2;   // (own, other) diagonals per role
    static constexpr int n = NP + 1;
    static constexpr int CW = 16;           // cells per warp
    static constexpr int NT = g * (g - 1) / 2;
    static constexpr bool kDupClass = (g & 1) != 0;  // the antipodal class {p, p+g} is computed by both roles

    // ---- shared-memory layout of one cell (in doubles; the cell index is the fastest dimension, stride CW) ----
    // One table, row p = circle position p (rows 0..C-1, row C = a copy of row 0 for role 1's rotated reads):
    //     col d = 0..g : X[p][p+d]      col g+1 : X[z][p]      col g+2 : w[p] = sqrt(eps_p)      col g+3 : 1 / w[p]
    // then X[z][z], once per role (each role reads and writes its own copy through its shifted base pointer).
    static constexpr int ROW = g + 4;
    static constexpr int CZ = g + 1, CWT = g + 2, CIW = g + 3;
    static constexpr int ZZ = (C + 1) * ROW;      // role 0's copy; role 1's is one row further
    static constexpr int CELL = ZZ + ROW + 1;     // doubles per cell
    // Horner-phase scratch (dead before the first matrix store): cols 0, 1 of row p
    static constexpr int CAL = 0;                 // alpha[p] 2^-s
    static constexpr int CBE = 1;                 // beta[p] 2^-s

    static constexpr size_t kWarpBytes = (size_t)CELL * CW * sizeof(double);

    __host__ __device__ static constexpr int md(int x) { return ((x % C) + C) % C; }
    // slot of the pair of circle positions {p, q} (role-0 coordinates); the antipodal pair has a second slot
    __host__ __device__ static constexpr int slot(int p, int q) {
        const int d = md(q - p);
        return d <= g ? p * ROW + d : q * ROW + (C - d);
    }
    __host__ __device__ static constexpr int slot2(int p, int q) { return md(q - p) == g ? q * ROW + g : -1; }
    __host__ __device__ static constexpr int tix(int a, int b) { return a * g - (a * (a + 1)) / 2 + (b - a - 1); }
    __host__ __device__ static constexpr int opos(int b) { return md(2 * b + 1); }  // other position b, role 0

    // fp64-pipe instructions of one Horner step and one squaring per lane: prices the polynomial in choose_m_s
    static constexpr int kHornerOps = NT + g * D + 2 * g + 5;
    static constexpr int kSquareOps = n * (NT + g * D + g) + 2 * (NT + g * D + g) + 3 * g;
    __host__ __device__ static constexpr float hcost() { return (float)kHornerOps / (float)kSquareOps; }

    // (No "apply X_{s-1} twice instead of the last squaring" here, unlike dg_tpc.cuh for N = 6..10: with the iterate in
    // shared memory a second apply costs this mapping as much time as the squaring it would save — measured.)

    struct Acc {  // the off-diagonal entries one lane computes
        double T[NT > 0 ? NT : 1];
        double M[g][D];
        double Z[g];
    };

    // Byte offsets (from a lane's base pointer) of the n operands of every row l of a squaring, l = 0..C-1 the circle
    // positions and l = C the gas row: sq[l][2a] = X[l][own a], sq[l][2a+1] = X[l][other a], sq[l][C] = X[l][z].
    // The squaring loops over l with this table in constant memory: the loop body is 68 FMAs + 17 loads whatever l,
    // 2 KB of code instead of the 29 KB of the unrolled form (which did not fit the 32 KB instruction cache next to
    // the other phases: 18 % of the squaring's issue slots went to instruction fetch, ncu round 2).
    // ap[a][j]: the operands of row a of the apply step, a = 0..g-1 the lane's own positions and a = g the gas row:
    // ap[a][j] = X[own a][position j], j = 0..C-1 (j = 2a: the diagonal), ap[a][C] = X[own a][z]; for the gas row
    // ap[g][j] = X[z][position j], ap[g][C] = X[z][z].
    static constexpr int RW = ((C + 1 + 3) / 4) * 4;  // table rows padded to 16 bytes: four offsets per constant load
    struct alignas(16) Tab {
        int sq[C + 1][RW];
        int ap[g + 1][RW];
    };
    // the C + 1 offsets of one table row, fetched four at a time (LDCU.128)
    __device__ __forceinline__ static void row_offsets(const int* row, int (&off)[RW]) {
        const int4* r4 = reinterpret_cast<const int4*>(row);
        static_for<0, RW / 4>([&](auto i) {
            const int4 v = r4[i];
            off[4 * i] = v.x;
            off[4 * i + 1] = v.y;
            off[4 * i + 2] = v.z;
            off[4 * i + 3] = v.w;
        });
    }
    __host__ __device__ static constexpr Tab make_tab() {
        Tab t{};
        for (int l = 0; l < C; ++l) {
            for (int a = 0; a < g; ++a) {
                t.sq[l][2 * a] = slot(l, 2 * a) * CW * 8;
                t.sq[l][2 * a + 1] = slot(l, opos(a)) * CW * 8;
            }
            t.sq[l][C] = (l * ROW + CZ) * CW * 8;
        }
        for (int a = 0; a < g; ++a) {
            t.sq[C][2 * a] = ((2 * a) * ROW + CZ) * CW * 8;
            t.sq[C][2 * a + 1] = ((2 * a + 1) * ROW + CZ) * CW * 8;
        }
        t.sq[C][C] = ZZ * CW * 8;
        for (int a = 0; a < g; ++a) {
            for (int j = 0; j < C; ++j) t.ap[a][j] = slot(2 * a, j) * CW * 8;
            t.ap[a][C] = ((2 * a) * ROW + CZ) * CW * 8;
        }
        for (int j = 0; j < C; ++j) t.ap[g][j] = (j * ROW + CZ) * CW * 8;
        t.ap[g][C] = ZZ * CW * 8;
        return t;
    }

    // A lane's view of its cell: the base pointer with the role shift (one table row) folded in.
    struct View {
        double* x;
        int r;
    };
    __device__ __forceinline__ static View view(double* warp_tile, int lane) {
        const int r = lane >> 4, c = lane & 15;
        View v;
        v.x = warp_tile + c + r * ROW * CW;
        v.r = r;
        return v;
    }
    __device__ __forceinline__ static double& at(const View& V, int row, int col) { return V.x[(row * ROW + col) * CW]; }

    __device__ __forceinline__ static double lds(const double* base, int byte_off) {
        return *reinterpret_cast<const volatile double*>(reinterpret_cast<const char*>(base) + byte_off);
    }

    // ---- one squaring: A <- off-diagonals of X X (own share) -----------------------------------------------------
    // volatile loads: every row is fetched when it is used.
    struct RowOps {  // the n operands of one row l
        double u[g], o[g], z;
    };
    __device__ __forceinline__ static void load_row(const View& V, const int* row, RowOps& R) {
        int off[RW];
        row_offsets(row, off);
        static_for<0, g>([&](auto a) {
            R.u[a] = lds(V.x, off[2 * a]);
            R.o[a] = lds(V.x, off[2 * a + 1]);
        });
        R.z = lds(V.x, off[C]);
    }
    template <bool First>
    __device__ __forceinline__ static void fma_row(const RowOps& R, Acc& A) {
        static_for<0, g>([&](auto a) {
            static_for<a + 1, g>([&](auto b) {
                if constexpr (First) A.T[tix(a, b)] = R.u[a] * R.u[b];
                else A.T[tix(a, b)] = fma(R.u[a], R.u[b], A.T[tix(a, b)]);
            });
            static_for<0, D>([&](auto dd) {
                if constexpr (First) A.M[a][dd] = R.u[a] * R.o[(a + dd) % g];
                else A.M[a][dd] = fma(R.u[a], R.o[(a + dd) % g], A.M[a][dd]);
            });
            if constexpr (First) A.Z[a] = R.z * R.u[a];
            else A.Z[a] = fma(R.z, R.u[a], A.Z[a]);
        });
    }
    // Rows 0..C (C + 1 of them, an odd number), two per loop iteration with the operands double-buffered: the loads of
    // the next row are in flight while the FMAs of the current one issue.
    __device__ __forceinline__ static void square(const View& V, const Tab& tab, Acc& A) {
        RowOps Ra, Rb;
        load_row(V, tab.sq[0], Ra);
        load_row(V, tab.sq[1], Rb);
        fma_row<true>(Ra, A);
#pragma unroll 1
        for (int l = 1; l < C; l += 2) {
            load_row(V, tab.sq[l + 1], Ra);
            fma_row<false>(Rb, A);
            load_row(V, tab.sq[l + 2 <= C ? l + 2 : C], Rb);  // (the last iteration re-reads row C: never used)
            fma_row<false>(Ra, A);
        }
    }

    // ---- conservation + store ------------------------------------------------------------------------------------
    // The diagonal from conservation of total momentum:  d_j = -(sum_{i != j} w_i O_ij) / w_j  (w_z = 1).  Every lane
    // sums its own entries into the columns they touch; the partner's share of a lane's own columns comes by shuffle.
    // Writes the off-diagonals, the diagonal (X_jj = 1 + d_j, or d_j itself when `fin`: the matrix handed to the apply
    // step is P = X - I) and the copies the rotated addressing needs.  `fin` is warp-uniform.
    __device__ __forceinline__ static void conserve_store(const View& V, const Acc& A, bool fin) {
        constexpr bool active = true;  // every lane of the warp runs the same number of squarings (see the kernel)
        const int r = V.r;
        const bool r0 = (r == 0);
        double wu[g], wo[g];
        static_for<0, g>([&](auto a) {
            wu[a] = at(V, 2 * a, CWT);
            wo[a] = at(V, 2 * a + 1, CWT);
        });
        __syncwarp();  // every lane has finished reading the old matrix (or the Horner scratch)
        // The off-diagonal stores come FIRST in program order and are unconditional (but for the role-0 copies), so that
        // the scheduler can interleave them with the sums below: 96 back-to-back STS.64 cost a lane ~6 issue cycles
        // each with nothing else to do (9 % of the kernel, ncu round 2); the sums keep the fp64 pipe busy meanwhile.
        auto st = [&](int idx, double v, bool pred) {
            if (pred) V.x[idx * CW] = v;
        };
        static_for<0, g>([&](auto a) {
            static_for<a + 1, g>([&](auto b) {
                constexpr int s1 = slot(2 * a, 2 * b), s2 = slot2(2 * a, 2 * b);
                const double v = A.T[tix(a, b)];
                st(s1, v, active);
                if constexpr (s2 >= 0) st(s2, v, active);
                if constexpr (s1 / ROW == 0) st(s1 + C * ROW, v, active && r0);  // row C = copy of row 0 (role 0's)
            });
            static_for<0, D>([&](auto dd) {
                constexpr int q = opos((a + dd) % g);
                constexpr int s1 = slot(2 * a, q), s2 = slot2(2 * a, q);
                const double v = A.M[a][dd];
                if constexpr (kDupClass && dd == D - 1) {  // antipodal class: role 0 stores both slots
                    st(s1, v, active && r0);
                    st(s2, v, active && r0);
                    if constexpr (s1 / ROW == 0) st(s1 + C * ROW, v, active && r0);
                    if constexpr (s2 / ROW == 0) st(s2 + C * ROW, v, active && r0);
                } else {
                    st(s1, v, active);
                    if constexpr (s2 >= 0) st(s2, v, active);
                    if constexpr (s1 / ROW == 0) st(s1 + C * ROW, v, active && r0);
                }
            });
            st((2 * a) * ROW + CZ, A.Z[a], active);
            if constexpr (a == 0) st(C * ROW + CZ, A.Z[a], active && r0);
        });
        // (three short independent chains per own column — own pairs above, own pairs below, mixed pairs — so that the
        // fp64 pipe's 8-cycle dependent latency is hidden inside the lane)
        double cu[g], co[g], cz = 0.0;
        {
            double ca[g], cb[g], cm[g];
            static_for<0, g>([&](auto a) {
                ca[a] = A.Z[a];  // the gas row's entry: w_z = 1
                cb[a] = 0.0;
                cm[a] = 0.0;
                co[a] = 0.0;
            });
            static_for<0, g>([&](auto a) {
                static_for<a + 1, g>([&](auto b) {
                    const double v = A.T[tix(a, b)];
                    ca[a] = fma(wu[b], v, ca[a]);
                    cb[b] = fma(wu[a], v, cb[b]);
                });
                static_for<0, D>([&](auto dd) {
                    constexpr int b = (a + dd) % g;
                    double v = A.M[a][dd];
                    if constexpr (kDupClass && dd == D - 1) v = r ? 0.0 : v;  // counted by role 0 only
                    cm[a] = fma(wo[b], v, cm[a]);
                    co[b] = fma(wu[a], v, co[b]);
                });
            });
            double cza = 0.0, czb = 0.0;
            static_for<0, g>([&](auto a) {
                cu[a] = (ca[a] + cb[a]) + cm[a];
                if constexpr (a % 2 == 0) cza = fma(wu[a], A.Z[a], cza);
                else czb = fma(wu[a], A.Z[a], czb);
            });
            cz = cza + czb;
        }
        // partner's sums for MY own columns: its other-position b is my own position a = b + 1 - r_partner
        static_for<0, g>([&](auto b) { co[b] = __shfl_xor_sync(0xffffffffu, co[b], 16); });
        static_for<0, g>([&](auto a) {
            const double pv = r ? co[a] : co[(a + g - 1) % g];
            const double d = -(cu[a] + pv) * at(V, 2 * a, CIW);
            const double dgl = fin ? d : 1.0 + d;
            st((2 * a) * ROW, dgl, active);
            if constexpr (a == 0) st(C * ROW, dgl, active && r0);
        });
        {
            const double other = __shfl_xor_sync(0xffffffffu, cz, 16);
            const double lo = r ? other : cz, hi = r ? cz : other;  // same order in both lanes
            cz = -(lo + hi);
            st(ZZ, fin ? cz : 1.0 + cz, active);  // each role its own copy
        }
        __syncwarp();
    }

    // ---- Taylor polynomial T_m(S / 2^s) - I  (Eq. 19), factored Horner recurrence of dg_tpc.cuh ----------------------
    // Q_j = (m!/j!) P_j,  Q_0k = beta_k v_k,  Q_ik = beta_i beta_k U_ik:
    //     U_ik <- v_k - alpha_i U_ik,   v_k <- (kappa_j + Q_00) - alpha_k v_k,   Q_00 <- b00 (kappa_j + Q_00) + sum_l beta_l^2 v_l
    // (right-hand sides: old values).  The lane owns U for its pairs (T: own a, own b; M: own a, other b) and v at its
    // own positions; the only cross-lane traffic of a step is the partner's half of the sum (one 64-bit shuffle).
    // For an M pair the recurrence is used in its mirrored form U <- v_own - alpha_other U (B Q is symmetric).
    // alpha, beta (already scaled by 2^-s) are read from the Horner scratch in shared memory.  m is warp-uniform.
    __device__ __forceinline__ static void horner(const View& V, int m, double b00, Acc& A) {
        double alu[g], alo[g], b2u[g], vu[g];
        static_for<0, g>([&](auto a) {
            alu[a] = at(V, 2 * a, CAL);
            alo[a] = at(V, 2 * a + 1, CAL);
            const double bu = at(V, 2 * a, CBE);
            b2u[a] = bu * bu;
            vu[a] = 1.0;
            static_for<0, D>([&](auto dd) { A.M[a][dd] = 0.0; });
        });
        static_for<0, (NT > 0 ? NT : 1)>([&](auto K) { A.T[K] = 0.0; });
        double q00 = b00, kap = 1.0;
        for (int j = m - 1; j >= 1; --j) {
            kap *= c_dbl[j + 1];
            // sum_l beta_l^2 v_l: my own positions here (two chains), the partner's half by shuffle; the U updates below
            // do not depend on it and cover the shuffle's latency
            double ta = b2u[0] * vu[0], tb = 0.0;
            static_for<1, g>([&](auto a) {
                if constexpr (a % 2 == 1) tb = fma(b2u[a], vu[a], tb);
                else ta = fma(b2u[a], vu[a], ta);
            });
            const double tmine = ta + tb;
            const double tother = __shfl_xor_sync(0xffffffffu, tmine, 16);
            static_for<0, g>([&](auto a) {
                static_for<a + 1, g>([&](auto b) { A.T[tix(a, b)] = fma(-alu[a], A.T[tix(a, b)], vu[b]); });
                static_for<0, D>([&](auto dd) {
                    constexpr int b = (a + dd) % g;
                    A.M[a][dd] = fma(-alo[b], A.M[a][dd], vu[a]);
                });
            });
            const double t00 = (V.r ? tother : tmine) + (V.r ? tmine : tother);  // same order in both lanes
            const double x00 = kap + q00;
            static_for<0, g>([&](auto a) { vu[a] = fma(-alu[a], vu[a], x00); });
            q00 = fma(b00, x00, t00);
        }
        // P_0k = beta_k v_k / m!,  P_ik = beta_i beta_k U_ik / m!; off-diagonals are >= 0 in exact arithmetic
        const double inv = c_ifact[m];
        static_for<0, g>([&](auto a) {
            const double bs = at(V, 2 * a, CBE) * inv;
            A.Z[a] = clamp_below(bs * vu[a], 0.0);
            static_for<a + 1, g>([&](auto b) {
                A.T[tix(a, b)] = clamp_below(A.T[tix(a, b)] * (bs * at(V, 2 * b, CBE)), 0.0);
            });
            static_for<0, D>([&](auto dd) {
                constexpr int b = (a + dd) % g;
                A.M[a][dd] = clamp_below(A.M[a][dd] * (bs * at(V, 2 * b + 1, CBE)), 0.0);
            });
        });
    }

    // ---- apply: one row of y = P q ---------------------------------------------------------------------------------
    // q[comp][j] (j = 0..C-1 in role-rotated order: index j <-> position j + r) and q0[comp] are the three W^-1 p_in
    // vectors; `off` = tab.ap[row].  Returns y[comp] = P[row][z] q0 + sum_j P[row][j] q_j.  Two partial sums per
    // component (six independent FMA chains).  The caller loops over the rows: the code is the same for every row.
    __device__ __forceinline__ static void apply_row(const View& V, const int* row, const double (&q)[3][C],
                                                     const double (&q0)[3], double (&y)[3]) {
        int off[RW];
        row_offsets(row, off);
        double e[C + 1];
        static_for<0, C + 1>([&](auto j) { e[j] = lds(V.x, off[j]); });
        double ya[3], yb[3];
        static_for<0, 3>([&](auto cp) {
            ya[cp] = e[C] * q0[cp];
            yb[cp] = e[0] * q[cp][0];
        });
        static_for<1, C>([&](auto j) {
            static_for<0, 3>([&](auto cp) {
                if constexpr (j % 2 == 1) ya[cp] = fma(e[j], q[cp][j], ya[cp]);
                else yb[cp] = fma(e[j], q[cp][j], yb[cp]);
            });
        });
        static_for<0, 3>([&](auto cp) { y[cp] = ya[cp] + yb[cp]; });
    }
};

}  // namespace dg
