// dg_tpc.cuh — thread-per-cell core: one thread owns one cell; every matrix lives in that thread's registers.
//
// The arithmetic (DESIGN.md §3 gives the derivation and the error argument):
//   * Eq. 17 satisfies detailed balance, Omega * diag(rho) is symmetric, so with
//     w_0 = 1, w_i = sqrt(eps_i) the matrix  S = W^-1 (dt Omega) W  is a SYMMETRIC arrowhead:
//         S_0i = S_i0 = a_i w_i =: beta_i,   S_ii = -a_i,   S_00 = -sum_i beta_i w_i,     a_i = dt / t_s,i ,
//     and exp(dt Omega) = W exp(S) W^-1.  Only the upper triangle is stored (n(n+1)/2 doubles) and a squaring
//     costs n^2(n+1)/2 FMAs instead of n^3.
//   * X = exp(S) is carried as P = X - I = O + diag(d) with O >= 0 off-diagonal and d <= 0 the diagonal, which is
//     never computed by the recurrences but re-derived from conservation of total momentum (columns of Eq. 17 sum
//     to zero):   d_j = -(sum_{i != j} w_i O_ij) / w_j.
//     - Taylor polynomial (Eq. 19) without ever adding I:   P <- (B + B P) / j,  j = m .. 1,
//       B = S / 2^s, exploiting that B has 3N+1 non-zeros (one Horner step is O(n^2)).
//     - Squaring (Eq. 23-24):  O <- offdiag((O + diag(1+d))^2), a sum of non-negative products,
//       so the s squarings amplify no cancellation error and total momentum is conserved to rounding at every step.
//   * Apply (Eq. 18):  p_out = p_in + W P W^-1 p_in.
#pragma once
#include "dg_params.cuh"

namespace dg {

template <int N>
struct Tpc {
    static constexpr int n = N + 1;
    static constexpr int SZ = n * (n + 1) / 2;
    // packed upper triangle, i <= j
    __host__ __device__ static constexpr int ix(int i, int j) { return i * n - (i * (i - 1)) / 2 + (j - i); }
    __host__ __device__ static constexpr int sx(int i, int j) { return i <= j ? ix(i, j) : ix(j, i); }

    // Cost of one Horner step in units of one squaring (for choose_m_s): ~(n^2 + 3n) FMAs vs ~n^2 (n+1)/2 + n^2.
    __host__ __device__ static constexpr float hcost() { return (float)(n * n + 3 * n) / (float)(n * n * (n + 1) / 2 + n * n); }

    // d_j = -(sum_{i != j} w_i O_ij) / w_j   (w_0 = 1); writes the diagonal slots of P.
    __device__ __forceinline__ static void conserve(double (&P)[SZ], const double (&w)[N], const double (&iw)[N]) {
#pragma unroll
        for (int j = 0; j < n; ++j) {
            double acc = 0.0;
#pragma unroll
            for (int i = 0; i < n; ++i)
                if (i != j) acc = (i == 0) ? acc + P[sx(i, j)] : fma(w[i - 1], P[sx(i, j)], acc);
            P[ix(j, j)] = (j == 0) ? -acc : -acc * iw[j - 1];
        }
    }

    // a[i] = dt/t_s,i (unscaled), w[i] = sqrt(eps_i), iw[i] = 1/w[i].  On return P holds exp(S) - I (packed, diagonal
    // slots = d) and m, s are the chosen Taylor degree and scaling exponent.
    __device__ __forceinline__ static void expm(const double (&a)[N], const double (&w)[N], const double (&iw)[N],
                                                double (&P)[SZ], int& m, int& s) {
        // ||A||_1 of Eq. 17 in closed form: column 0 sums to 2 sum_i eps_i a_i, column i to 2 a_i (R5)
        double sb = 0.0, amax = 0.0;
#pragma unroll
        for (int i = 0; i < N; ++i) {
            sb = fma(a[i] * w[i], w[i], sb);
            amax = fmax(amax, a[i]);
        }
        const double norm = 2.0 * fmax(sb, amax);
        choose_m_s(norm, hcost(), m, s);
        const double sc = pow2neg(s);

        double al[N], be[N];
        double b00 = 0.0;
#pragma unroll
        for (int i = 0; i < N; ++i) {
            al[i] = a[i] * sc;
            be[i] = al[i] * w[i];
            b00 = fma(be[i], w[i], b00);
        }
        b00 = -b00;

        // P = B / m
        {
            const double r = c_inv[m];
#pragma unroll
            for (int k = 0; k < SZ; ++k) P[k] = 0.0;
            P[ix(0, 0)] = b00 * r;
#pragma unroll
            for (int i = 1; i < n; ++i) {
                P[ix(0, i)] = be[i - 1] * r;
                P[ix(i, i)] = -al[i - 1] * r;
            }
        }
        // P <- (B + B P) / j
        for (int j = m - 1; j >= 1; --j) {
            const double r = c_inv[j];
            double t[n];
#pragma unroll
            for (int k = 0; k < n; ++k) {  // row 0 of B P, from the old P
                double acc = b00 * P[ix(0, k)];
#pragma unroll
                for (int l = 1; l < n; ++l) acc = fma(be[l - 1], P[sx(l, k)], acc);
                t[k] = acc;
            }
#pragma unroll
            for (int i = 1; i < n; ++i)  // rows i >= 1: (B P)_ik = beta_i P_0k - alpha_i P_ik
#pragma unroll
                for (int k = i; k < n; ++k) {
                    double v = fma(be[i - 1], P[ix(0, k)], -al[i - 1] * P[ix(i, k)]);
                    if (k == i) v -= al[i - 1];
                    P[ix(i, k)] = v * r;
                }
            P[ix(0, 0)] = (b00 + t[0]) * r;
#pragma unroll
            for (int k = 1; k < n; ++k) P[ix(0, k)] = (be[k - 1] + t[k]) * r;
        }
        // off-diagonals are non-negative in exact arithmetic; clamp the rounding noise, then re-derive the diagonal
#pragma unroll
        for (int i = 0; i < n; ++i)
#pragma unroll
            for (int k = i + 1; k < n; ++k) P[ix(i, k)] = fmax(P[ix(i, k)], 0.0);
        conserve(P, w, iw);

        // s squarings: O <- offdiag(X X), X = O + diag(1 + d) >= 0 entrywise, X symmetric
        for (int it = 0; it < s; ++it) {
            double X[SZ];
#pragma unroll
            for (int k = 0; k < SZ; ++k) X[k] = P[k];
#pragma unroll
            for (int i = 0; i < n; ++i) X[ix(i, i)] = 1.0 + P[ix(i, i)];
#pragma unroll
            for (int i = 0; i < n; ++i)
#pragma unroll
                for (int k = i + 1; k < n; ++k) {
                    double acc = X[sx(i, 0)] * X[sx(0, k)];
#pragma unroll
                    for (int l = 1; l < n; ++l) acc = fma(X[sx(i, l)], X[sx(l, k)], acc);
                    P[ix(i, k)] = acc;
                }
            conserve(P, w, iw);
        }
    }
};

}  // namespace dg
