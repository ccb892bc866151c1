// dg_wpc.cuh — warp-per-cell core: one warp owns one cell; the dust block of the symmetrised matrix lives in the
// warp's registers in the fp64 tensor-core accumulator layout and is squared with DMMA (mma.sync m8n8k4 f64).
//
// Same arithmetic as dg_tpc.cuh (symmetrised arrowhead S = W^-1 (dt Omega) W, P = exp(S) - I = O + diag(d), Taylor
// recurrence P <- (B + B P)/j, cancellation-free squarings with the diagonal re-derived from conservation of total
// momentum); only the mapping differs.  This is the "hierarchical" kernel the paper suggests but does not build
// (PAPER.md:329, 343).
//
// Layout.  The symmetric matrix X = [[x00, r^T], [r, D]] is split into the gas entry x00, the gas-dust vector r and
// the ND x ND dust block D (ND = 8 or 16, species beyond N are zero padding that stays decoupled).  With lane
// coordinates g = lane >> 2 (0..7) and t = lane & 3, D is held as TL x TL tiles of 8 x 8 in the DMMA accumulator
// layout:   T[I][J][e] = D[8 I + g][8 J + 2 t + e],  e = 0, 1.
// Because D is symmetric, T[I][K][e] is at the same time the A fragment (rows 8I.., k-set {8K + 2t + e}) and T[J][K][e]
// the B fragment (k-set {8K + 2t + e}, columns 8J..) of mma.m8n8k4 — the k index may be permuted freely as long as A
// and B agree — so    (D D)[tile I, J] = sum_{K, e} mma(T[I][K][e], T[J][K][e])    lands directly in the layout the
// next squaring consumes: no fragment re-layout between squarings.  The rank-one border r r^T is one more mma whose
// k = 0 slot carries r.  Tile (1,0) is the transpose of tile (0,1), fetched with shuffles instead of five more DMMAs.
// Vectors come in two replicated forms: row-indexed vR[I] = v[8 I + g] and column-indexed vC[J][e] = v[8 J + 2 t + e].
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
__device__ __forceinline__ double oct_sum(double x) {  // over g (lanes with equal t)
    x += __shfl_xor_sync(kFull, x, 4);
    x += __shfl_xor_sync(kFull, x, 8);
    x += __shfl_xor_sync(kFull, x, 16);
    return x;
}

template <int N>
struct Wpc {
    static constexpr int n = N + 1;
    static constexpr int TL = (N <= 8) ? 1 : 2;
    static constexpr int ND = 8 * TL;
    // one Horner step costs about a third of a squaring in this mapping (measured)
    __host__ __device__ static constexpr float hcost() { return TL == 1 ? 0.6f : 0.33f; }

    struct VecR { double v[TL]; };
    struct VecC { double v[TL][2]; };

    struct Lane {
        int g, t;
        bool dg[2];  // this lane holds a diagonal entry of tile (I, I) in slot e
        __device__ __forceinline__ Lane() {
            const int lane = threadIdx.x & 31;
            g = lane >> 2;
            t = lane & 3;
            dg[0] = (t == (g >> 1)) && ((g & 1) == 0);
            dg[1] = (t == (g >> 1)) && ((g & 1) == 1);
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
            double acc = 0.0;
#pragma unroll
            for (int J = 0; J < TL; ++J)
#pragma unroll
                for (int e = 0; e < 2; ++e) acc = fma(T[I][J][e], x.v[J][e], acc);
            y.v[I] = quad_sum(acc);
        }
    }

    // Conservation of total momentum: with O the off-diagonal part (T with zeroed diagonal, r) returns
    //   dR[I] = -(r[row] + sum_col O[row][col] w[col]) / w[row]   and   d0 = -sum_j w_j r_j.
    __device__ __forceinline__ static void conserve(const double (&T)[TL][TL][2], const VecR& rR, const VecR& wR,
                                                    const VecC& wC, const VecR& iwR, VecR& dR, double& d0) {
        VecR s;
        matvec(T, wC, s);
        double acc = 0.0;
#pragma unroll
        for (int I = 0; I < TL; ++I) {
            dR.v[I] = -(rR.v[I] + s.v[I]) * iwR.v[I];
            acc = fma(wR.v[I], rR.v[I], acc);
        }
        d0 = -oct_sum(acc);
    }

    __device__ __forceinline__ static void set_diag(const Lane& L, double (&T)[TL][TL][2], const VecR& d, double add) {
#pragma unroll
        for (int I = 0; I < TL; ++I)
#pragma unroll
            for (int e = 0; e < 2; ++e)
                if (L.dg[e]) T[I][I][e] = add + d.v[I];
    }
    __device__ __forceinline__ static void zero_diag(const Lane& L, double (&T)[TL][TL][2]) {
#pragma unroll
        for (int I = 0; I < TL; ++I)
#pragma unroll
            for (int e = 0; e < 2; ++e)
                if (L.dg[e]) T[I][I][e] = 0.0;
    }

    // On entry: alR/beR/beC = a_j 2^-s, beta_j = a_j w_j 2^-s (row / column indexed), b00 = -sum_j beta_j w_j,
    // wR/wC/iwR the symmetrising weights.  On return T (diagonal slots = d), rR, rC, d0 hold P = exp(S) - I.
    __device__ __forceinline__ static void expm(const Lane& L, int m, int s, const VecR& alR, const VecR& beR,
                                                const VecC& beC, double b00, const VecR& wR, const VecC& wC,
                                                const VecR& iwR, double (&T)[TL][TL][2], VecR& rR, VecC& rC,
                                                double& d0) {
        // P = B / m
        double p00;
        {
            const double r = c_inv[m];
#pragma unroll
            for (int I = 0; I < TL; ++I) {
#pragma unroll
                for (int J = 0; J < TL; ++J) T[I][J][0] = T[I][J][1] = 0.0;
                rR.v[I] = beR.v[I] * r;
            }
            VecR dinit;
#pragma unroll
            for (int I = 0; I < TL; ++I) dinit.v[I] = -alR.v[I] * r;
            set_diag(L, T, dinit, 0.0);
#pragma unroll
            for (int J = 0; J < TL; ++J)
#pragma unroll
                for (int e = 0; e < 2; ++e) rC.v[J][e] = beC.v[J][e] * r;
            p00 = b00 * r;
        }
        // P <- (B + B P) / j
        for (int j = m - 1; j >= 1; --j) {
            const double r = c_inv[j];
            VecR t0;  // row 0 of B P (dust part): b00 r_k + sum_l beta_l P_lk
            matvec(T, beC, t0);
            double acc = 0.0;
#pragma unroll
            for (int I = 0; I < TL; ++I) acc = fma(beR.v[I], rR.v[I], acc);
            const double t00 = fma(b00, p00, oct_sum(acc));
#pragma unroll
            for (int I = 0; I < TL; ++I) {  // rows >= 1: (B P)_ik = beta_i P_0k - alpha_i P_ik (+ B_ii on the diagonal)
#pragma unroll
                for (int J = 0; J < TL; ++J)
#pragma unroll
                    for (int e = 0; e < 2; ++e) {
                        double v = fma(beR.v[I], rC.v[J][e], -alR.v[I] * T[I][J][e]);
                        if (I == J && L.dg[e]) v -= alR.v[I];
                        T[I][J][e] = v * r;
                    }
            }
#pragma unroll
            for (int I = 0; I < TL; ++I) rR.v[I] = (beR.v[I] + fma(b00, rR.v[I], t0.v[I])) * r;
            row_to_col(L, rR, rC);
            p00 = (b00 + t00) * r;
        }
        // clamp the off-diagonals (non-negative in exact arithmetic), re-derive the diagonal from conservation
        zero_diag(L, T);
#pragma unroll
        for (int I = 0; I < TL; ++I) {
#pragma unroll
            for (int J = 0; J < TL; ++J)
#pragma unroll
                for (int e = 0; e < 2; ++e) T[I][J][e] = fmax(T[I][J][e], 0.0);
            rR.v[I] = fmax(rR.v[I], 0.0);
        }
        row_to_col(L, rR, rC);
        VecR dR;
        conserve(T, rR, wR, wC, iwR, dR, d0);

        // s squarings of X = O + diag(1 + d)
        for (int it = 0; it < s; ++it) {
            set_diag(L, T, dR, 1.0);
            const double x00 = 1.0 + d0;
            // gas row of X X: x00 r + D r
            VecR rn;
            matvec(T, rC, rn);
            // dust block of X X: r r^T + D D, upper tiles by DMMA
            double C[TL][TL][2];
            VecR rb;
#pragma unroll
            for (int I = 0; I < TL; ++I) rb.v[I] = (L.t == 0) ? rR.v[I] : 0.0;
#pragma unroll
            for (int I = 0; I < TL; ++I)
#pragma unroll
                for (int J = I; J < TL; ++J) {
                    C[I][J][0] = C[I][J][1] = 0.0;
#pragma unroll
                    for (int K = 0; K < TL; ++K)
#pragma unroll
                        for (int e = 0; e < 2; ++e) dmma884(C[I][J][0], C[I][J][1], T[I][K][e], T[J][K][e]);
                    dmma884(C[I][J][0], C[I][J][1], rb.v[I], rb.v[J]);
                }
            if (TL == 2) {  // tile (1,0)[g][2t+e] = tile (0,1)[2t+e][g], held by lane 4 (2t+e) + g/2 in slot g & 1
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int src = 4 * (2 * L.t + e) + (L.g >> 1);
                    const double v0 = __shfl_sync(kFull, C[0][TL - 1][0], src);
                    const double v1 = __shfl_sync(kFull, C[0][TL - 1][1], src);
                    C[TL - 1][0][e] = (L.g & 1) ? v1 : v0;
                }
            }
#pragma unroll
            for (int I = 0; I < TL; ++I) {
#pragma unroll
                for (int J = 0; J < TL; ++J) T[I][J][0] = C[I][J][0], T[I][J][1] = C[I][J][1];
                rR.v[I] = fma(x00, rR.v[I], rn.v[I]);
            }
            zero_diag(L, T);
            row_to_col(L, rR, rC);
            conserve(T, rR, wR, wC, iwR, dR, d0);
        }
        set_diag(L, T, dR, 0.0);
    }
};

}  // namespace dg
