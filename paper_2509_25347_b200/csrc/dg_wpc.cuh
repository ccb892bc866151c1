// dg_wpc.cuh — warp-per-cell core: one warp owns one cell; the dust block of the symmetrised matrix lives in the
// warp's registers in the fp64 tensor-core accumulator layout and is squared with DMMA (mma.sync m8n8k4 f64).
//
// Same arithmetic as dg_tpc.cuh (symmetrised arrowhead S = W^-1 (dt Omega) W, P = exp(S) - I = O + diag(d), Taylor
// recurrence P <- (B + B P)/j with B P = P B, cancellation-free squarings with the diagonal re-derived from
// conservation of total momentum); only the mapping differs.  This is the "hierarchical" kernel the paper suggests
// but does not build.
//
// Layout.  The symmetric matrix X = [[x00, r^T], [r, D]] is split into the gas entry x00, the gas-dust vector r and
// the ND x ND dust block D (ND = 8 or 16, species beyond N are zero padding that stays decoupled).  With lane
// coordinates g = lane >> 2 (0..7) and t = lane & 3, D is held as TL x TL tiles of 8 x 8 in the DMMA accumulator
// layout:   T[I][J][e] = D[8 I + g][8 J + 2 t + e],  e = 0, 1.
// Because D is symmetric, T[I][K][e] is at the same time the A fragment (rows 8I.., k-set {8K + 2t + e}) and T[J][K][e]
// the B fragment (k-set {8K + 2t + e}, columns 8J..) of mma.m8n8k4 — the k index may be permuted freely as long as A
// and B agree — so    (D D)[tile I, J] = sum_{K, e} mma(T[I][K][e], T[J][K][e])    lands directly in the layout the
// next squaring consumes: no fragment re-layout between squarings.  The rank-one border r r^T initialises the
// accumulators (two DMUL per tile: cheaper than a DMMA whose k-slots would be three-quarters empty).  Tile (1,0) is the
// transpose of tile (0,1), fetched with shuffles instead of four more DMMAs.
// Vectors come in two replicated forms: row-indexed vR[I] = v[8 I + g] and column-indexed vC[J][e] = v[8 J + 2 t + e].
//
// Measured on B200: DMMA.8x8x4 issues every 16 cycles per SM sub-partition (the same 64 FMA/clk/SM as
// DFMA) with a dependent-accumulator latency of 26 cycles; m16n8k{4,8,16} compile to sequences of DMMA.8x8x4.
#pragma once
#include "dg_params.cuh"

namespace dg {

__device__ __forceinline__ void dmma884(double& d0, double& d1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(d0), "+d"(d1)
                 : "d"(a), "d"(b));
}

constexpr unsigned kFull = 0xffffffffu;

__device__ __forceinline__ double quad_sum(double x) {  // over t (lanes 4g .. 4g+3)
    x += __shfl_xor_sync(kFull, x, 1);
    x += __shfl_xor_sync(kFull, x, 2);
    return x;
}

// Per-cell quantities the canonical lanes prepare in shared memory (species j < N; padding: a = be = 0, w = iw = 1).
template <int ND>
struct CellVecs {
    double a[ND];   // dt / t_s,j                       (Eq. 15)
    double be[ND];  // a_j sqrt(eps_j)
    double w[ND];   // sqrt(eps_j)                      (Eq. 14)
    double iw[ND];  // 1 / sqrt(eps_j)
    double sb;      // sum_j eps_j a_j
    double amax;    // max_j a_j
};

template <int N>
struct Wpc {
    static constexpr int n = N + 1;
    static constexpr int TL = (N <= 8) ? 1 : 2;
    static constexpr int ND = 8 * TL;
    // Price of one Horner step in units of one squaring for choose_m_s (R8): about 23 fp64 instructions
    // and one quad reduction against 12 DMMA (16 pipe cycles each) + ~33 fp64 instructions + 32 SHFL for a squaring.
    // The optimum is flat (config 4 timed within 1 % for prices between 0.2 and 0.45).
    __host__ __device__ static constexpr float hcost() { return TL == 1 ? 0.4f : 0.22f; }

    struct VecR { double v[TL]; };
    struct VecC { double v[TL][2]; };
    using Cell = CellVecs<ND>;

    struct Lane {
        int g, t;
        bool dg[2];  // this lane holds a diagonal entry of tile (I, I) in slot e
        __device__ __forceinline__ Lane() {
            const int lane = threadIdx.x & 31;
            g = lane >> 2;
            t = lane & 3;
            dg[0] = (g == 2 * t);
            dg[1] = (g == 2 * t + 1);
        }
    };

    // column-indexed copy of a row-indexed vector: vC[J][e] = v[8J + 2t + e], held (row-indexed) by quad 2t + e
    __device__ __forceinline__ static void row_to_col(const Lane& L, const VecR& r, VecC& c) {
#pragma unroll
        for (int J = 0; J < TL; ++J)
#pragma unroll
            for (int e = 0; e < 2; ++e) c.v[J][e] = __shfl_sync(kFull, r.v[J], 4 * (2 * L.t + e));
    }

    // y[8I + g] = sum_col D[8I + g][col] x[col], partial sums reduced over the quad
    __device__ __forceinline__ static void matvec(const double (&T)[TL][TL][2], const VecC& x, VecR& y) {
#pragma unroll
        for (int I = 0; I < TL; ++I) {
            double acc = T[I][0][0] * x.v[0][0];
            acc = fma(T[I][0][1], x.v[0][1], acc);
#pragma unroll
            for (int J = 1; J < TL; ++J)
#pragma unroll
                for (int e = 0; e < 2; ++e) acc = fma(T[I][J][e], x.v[J][e], acc);
            y.v[I] = quad_sum(acc);
        }
    }
    // sum_col x[col] y[col] for column-indexed vectors (every lane receives the full sum)
    __device__ __forceinline__ static double dotC(const VecC& x, const VecC& y) {
        double acc = x.v[0][0] * y.v[0][0];
        acc = fma(x.v[0][1], y.v[0][1], acc);
#pragma unroll
        for (int J = 1; J < TL; ++J)
#pragma unroll
            for (int e = 0; e < 2; ++e) acc = fma(x.v[J][e], y.v[J][e], acc);
        return quad_sum(acc);
    }

    // Conservation of total momentum: with O the off-diagonal part (T with zeroed diagonal, r) returns
    //   dR[I] = -(r[row] + sum_col O[row][col] w[col]) / w[row]   and   d0 = -sum_j w_j r_j.
    __device__ __forceinline__ static void conserve(const double (&T)[TL][TL][2], const VecR& rR, const VecC& rC,
                                                    const VecC& wC, const VecR& iwR, VecR& dR, double& d0) {
        VecR s;
        matvec(T, wC, s);
#pragma unroll
        for (int I = 0; I < TL; ++I) dR.v[I] = -(rR.v[I] + s.v[I]) * iwR.v[I];
        d0 = -dotC(wC, rC);
    }

    __device__ __forceinline__ static void set_diag(const Lane& L, double (&T)[TL][TL][2], const VecR& d, double add) {
#pragma unroll
        for (int I = 0; I < TL; ++I) {
            const double v = add + d.v[I];
#pragma unroll
            for (int e = 0; e < 2; ++e)
                if (L.dg[e]) T[I][I][e] = v;
        }
    }
    __device__ __forceinline__ static void zero_diag(const Lane& L, double (&T)[TL][TL][2]) {
#pragma unroll
        for (int I = 0; I < TL; ++I)
#pragma unroll
            for (int e = 0; e < 2; ++e)
                if (L.dg[e]) T[I][I][e] = 0.0;
    }

    __device__ __forceinline__ static void load_weights(const Lane& L, const Cell& cv, VecC& wC, VecR& iwR) {
#pragma unroll
        for (int I = 0; I < TL; ++I) {
            iwR.v[I] = cv.iw[8 * I + L.g];
#pragma unroll
            for (int e = 0; e < 2; ++e) wC.v[I][e] = cv.w[8 * I + 2 * L.t + e];
        }
    }

    // One squaring of X = [[x00, r^T], [r, D]] held as (T with its diagonal, rR/rC, x00).  Project = true re-derives
    // the diagonal (dR, d0) from conservation and writes 1 + d back; Project = false keeps the diagonal of X X.
    template <bool Project>
    __device__ __forceinline__ static void square(const Lane& L, const Cell& cv, double (&T)[TL][TL][2], VecR& rR,
                                                  VecC& rC, double& x00, VecR& dR, double& d0) {
        // the weights are re-read from shared memory where they are needed instead of living in registers across
        // the DMMA phase (the kernel runs at 80 registers per thread: three blocks per SM)
        VecC wC;
        VecR iwR;
        if (Project) load_weights(L, cv, wC, iwR);
        // gas row of X X: x00 r + D r
        VecR rn;
        matvec(T, rC, rn);
        // dust block of X X: r r^T + D D, upper tiles by DMMA on top of the rank-one border
        double C[TL][TL][2];
#pragma unroll
        for (int I = 0; I < TL; ++I)
#pragma unroll
            for (int J = I; J < TL; ++J) {
                C[I][J][0] = rR.v[I] * rC.v[J][0];
                C[I][J][1] = rR.v[I] * rC.v[J][1];
            }
#pragma unroll
        for (int K = 0; K < TL; ++K)
#pragma unroll
            for (int e = 0; e < 2; ++e)
#pragma unroll
                for (int I = 0; I < TL; ++I)
#pragma unroll
                    for (int J = I; J < TL; ++J) dmma884(C[I][J][0], C[I][J][1], T[I][K][e], T[J][K][e]);
        if (TL == 2) {  // tile (1,0)[g][2t+e] = tile (0,1)[2t+e][g], held by lane 4 (2t+e) + g/2 in slot g & 1
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int src = 4 * (2 * L.t + e) + (L.g >> 1);
                const double v0 = __shfl_sync(kFull, C[0][TL - 1][0], src);
                const double v1 = __shfl_sync(kFull, C[0][TL - 1][1], src);
                C[TL - 1][0][e] = (L.g & 1) ? v1 : v0;
            }
        }
        double x00n = 0.0;
        if (!Project) x00n = fma(x00, x00, dotC(rC, rC));  // (X X)_00 = x00^2 + r.r
#pragma unroll
        for (int I = 0; I < TL; ++I) {
#pragma unroll
            for (int J = 0; J < TL; ++J) T[I][J][0] = C[I][J][0], T[I][J][1] = C[I][J][1];
            rR.v[I] = fma(x00, rR.v[I], rn.v[I]);
        }
        row_to_col(L, rR, rC);
        if (Project) {
            zero_diag(L, T);
            conserve(T, rR, rC, wC, iwR, dR, d0);
            set_diag(L, T, dR, 1.0);
            x00 = 1.0 + d0;
        } else {
            x00 = x00n;
        }
    }

    // What the apply step needs once P = exp(S) - I is known: the dust block T (diagonal slots = d), the gas-dust
    // vector r in both forms, the gas entry d0.
    struct Result {
        double T[TL][TL][2];
        VecR rR;
        VecC rC;
        double d0;
        int m, s;
    };

    // cv: this cell's vectors in shared memory (read-only here).  All 32 lanes call it together.
    __device__ __forceinline__ static void expm(const Lane& L, const Cell& cv, Result& R) {
        // ||S||_2 <= max_j a_j + sum_j eps_j a_j (dg_tpc.cuh gives the argument; R5)
        const double norm = cv.sb + cv.amax;
        choose_m_s(norm, hcost(), R.m, R.s);
        // every lane holds the same (m, s); passing them through REDUX puts them in uniform registers, so the compiler
        // knows the Horner and squaring loops are warp-uniform and drops the divergence guards around their shuffles
        const int m = __reduce_max_sync(kFull, R.m), s = __reduce_max_sync(kFull, R.s);
        const double sc = pow2neg(s);

        VecR alR, beR;
        VecC beC;
#pragma unroll
        for (int I = 0; I < TL; ++I) {
            const int row = 8 * I + L.g;
            alR.v[I] = cv.a[row] * sc;
            beR.v[I] = cv.be[row] * sc;
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int col = 8 * I + 2 * L.t + e;
                beC.v[I][e] = cv.be[col] * sc;
            }
        }
        const double b00 = -cv.sb * sc;
        double (&T)[TL][TL][2] = R.T;
        VecR& rR = R.rR;
        VecC& rC = R.rC;

        // The polynomial, in the factored unscaled form of dg_tpc.cuh: Q_j = (m!/j!) P_j with Q_0k = beta_k v_k and
        // Q_ik = beta_i beta_k U_ik, so that one Horner step is
        //     U_ik <- v_k - alpha_i U_ik,   v_k <- (kappa_j + Q_00) - alpha_k v_k,
        //     Q_00 <- b00 (kappa_j + Q_00) + sum_l beta_l^2 v_l          (right-hand sides: OLD values),
        // one fused multiply-add per entry.  T holds U during the loop; v is carried in both replicated forms (vR,
        // vC) elementwise, so the only cross-lane traffic of a step is the quad reduction of the sum.  The dust
        // diagonal is never carried: the diagonal slots of T hold bounded don't-care values until zero_diag() below.
        VecC alC, be2C, vC;
        VecR vR;
#pragma unroll
        for (int I = 0; I < TL; ++I) {
#pragma unroll
            for (int J = 0; J < TL; ++J) T[I][J][0] = T[I][J][1] = 0.0;
            vR.v[I] = 1.0;
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                alC.v[I][e] = cv.a[8 * I + 2 * L.t + e] * sc;
                be2C.v[I][e] = beC.v[I][e] * beC.v[I][e];
                vC.v[I][e] = 1.0;
            }
        }
        double p00 = b00, kap = 1.0;
        for (int j = m - 1; j >= 1; --j) {
            kap *= c_dbl[j + 1];
#pragma unroll
            for (int I = 0; I < TL; ++I)
#pragma unroll
                for (int J = 0; J < TL; ++J)
#pragma unroll
                    for (int e = 0; e < 2; ++e) T[I][J][e] = fma(-alR.v[I], T[I][J][e], vC.v[J][e]);
            const double t00 = dotC(be2C, vC);
            const double x00 = kap + p00;
#pragma unroll
            for (int I = 0; I < TL; ++I) {
                vR.v[I] = fma(-alR.v[I], vR.v[I], x00);
#pragma unroll
                for (int e = 0; e < 2; ++e) vC.v[I][e] = fma(-alC.v[I][e], vC.v[I][e], x00);
            }
            p00 = fma(b00, x00, t00);
        }
        // P_0k = beta_k v_k / m!,  P_ik = beta_i beta_k U_ik / m!; clamp the off-diagonals (non-negative in exact
        // arithmetic), re-derive the diagonal from conservation
        zero_diag(L, T);
        {
            const double inv = c_ifact[m];
#pragma unroll
            for (int I = 0; I < TL; ++I) {
                const double bs = beR.v[I] * inv;
#pragma unroll
                for (int J = 0; J < TL; ++J)
#pragma unroll
                    for (int e = 0; e < 2; ++e) T[I][J][e] = clamp_below(T[I][J][e] * (bs * beC.v[J][e]), 0.0);
                rR.v[I] = clamp_below(bs * vR.v[I], 0.0);
            }
        }
        row_to_col(L, rR, rC);
        VecR dR;
        double d0;
        {
            VecC wC;
            VecR iwR;
            load_weights(L, cv, wC, iwR);
            conserve(T, rR, rC, wC, iwR, dR, d0);
        }

        // s squarings of X = O + diag(1 + d).  The diagonal is re-derived from conservation on every OTHER squaring
        // only (always on the last one): in between, the diagonal of X X that the DMMAs deliver anyway, a sum of
        // squares, serves as the multiplicand.  A diagonal entry enters the off-diagonals of the next X X only as a
        // factor (relative error ~n u), and the component of that error along the conserved mode — the one that
        // doubles per squaring — is removed again one step later, so it never exceeds ~2 n u.
        set_diag(L, T, dR, 1.0);
        double x00 = 1.0 + d0;
        int it = 0;
        if (s & 1) {
            square<true>(L, cv, T, rR, rC, x00, dR, d0);
            it = 1;
        }
        for (; it < s; it += 2) {
            square<false>(L, cv, T, rR, rC, x00, dR, d0);
            square<true>(L, cv, T, rR, rC, x00, dR, d0);
        }
        set_diag(L, T, dR, 0.0);
        R.d0 = d0;
    }
};

}  // namespace dg
