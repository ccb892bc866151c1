// dg_tpc.cuh — thread-per-cell core: one thread owns one cell; every matrix lives in that thread's registers.
//
// The arithmetic (DESIGN.md §3 gives the derivation and the error argument):
//   * Eq. 17 satisfies detailed balance, Omega * diag(rho) is symmetric, so with
//     w_0 = 1, w_i = sqrt(eps_i) the matrix  S = W^-1 (dt Omega) W  is a SYMMETRIC arrowhead:
//         S_0i = S_i0 = a_i w_i =: beta_i,   S_ii = -a_i,   S_00 = -sum_i beta_i w_i,     a_i = dt / t_s,i ,
//     and exp(dt Omega) = W exp(S) W^-1.  Only the upper triangle is stored (n(n+1)/2 doubles) and a squaring
//     costs n^2(n-1)/2 FMAs instead of n^3.
//   * X = exp(S) is carried as P = X - I = O + diag(d) with O >= 0 off-diagonal and d <= 0 the diagonal, which is
//     never computed by the recurrences but re-derived from conservation of total momentum (columns of Eq. 17 sum
//     to zero):   d_j = -(sum_{i != j} w_i O_ij) / w_j.
//     - Taylor polynomial (Eq. 19) without ever adding I:   P <- B_j + B_j P,  B_j = B / j,  j = m .. 1,
//       B = S / 2^s.  B has 3N+1 non-zeros, and P is a polynomial in B, so B P = P B is symmetric: row 0 of B P is
//       its column 0, (B P)_0k = (B P)_k0 = beta_k P_00 - alpha_k P_0k, and only (B P)_00 needs a dot product.  One
//       Horner step is N(N-1)/2 + 2N + 3 fp64-pipe instructions (see expm() for the two further rewritings).
//     - Squaring (Eq. 23-24):  O <- offdiag((O + diag(1+d))^2), a sum of non-negative products,
//       so the s squarings amplify no cancellation error and total momentum is conserved to rounding at every step.
//   * Apply (Eq. 18):  p_out = p_in + W P W^-1 p_in.
//
// Every loop over matrix indices is a static_for over integral constants, so each P[...] subscript is a compile-time
// constant and the arrays are guaranteed to be registers (a "#pragma unroll" the front end declines leaves them in
// local memory).
#pragma once
#include "dg_params.cuh"

namespace dg {

template <int V>
struct Idx {  // a compile-time index: "constexpr int i = I;" inside a static_for body
    __host__ __device__ constexpr operator int() const { return V; }
};

template <int B, int E, class F>
__device__ __forceinline__ void static_for(F&& f) {
    if constexpr (B < E) {
        f(Idx<B>{});
        static_for<B + 1, E>(f);
    }
}

template <int N, class Real = double>
struct Tpc {
    static constexpr int n = N + 1;
    static constexpr int SZ = n * (n + 1) / 2;
    // packed upper triangle, i <= j
    __host__ __device__ static constexpr int ix(int i, int j) { return i * n - (i * (i - 1)) / 2 + (j - i); }
    __host__ __device__ static constexpr int sx(int i, int j) { return i <= j ? ix(i, j) : ix(j, i); }

    // fp64-pipe instructions of one Horner step and of one squaring (with its conservation sums) as coded below;
    // their ratio prices the polynomial in choose_m_s (R8).
    static constexpr int kHornerOps = N * (N - 1) / 2 + 2 * N + 3;
    static constexpr int kSquareOps = n * n * (n - 1) / 2 + n * n + n;
    __host__ __device__ static constexpr float hcost() { return (float)kHornerOps / (float)kSquareOps; }

    // d_j = -(sum_{i != j} w_i O_ij) / w_j   (w_0 = 1); writes the diagonal slots of P.
    __device__ __forceinline__ static void conserve(Real (&P)[SZ], const Real (&w)[N], const Real (&iw)[N]) {
        static_for<0, n>([&](auto J) {
            constexpr int j = J;
            if constexpr (j == 0) {
                Real acc = w[0] * P[ix(0, 1)];
                static_for<2, n>([&](auto I) {
                    constexpr int i = I;
                    acc = fma(w[i - 1], P[ix(0, i)], acc);
                });
                P[ix(0, 0)] = -acc;
            } else {
                Real acc = P[ix(0, j)];  // w_0 = 1
                static_for<1, n>([&](auto I) {
                    constexpr int i = I;
                    if constexpr (i != j) acc = fma(w[i - 1], P[sx(i, j)], acc);
                });
                P[ix(j, j)] = -acc * iw[j - 1];
            }
        });
    }

    // The fused kernel does not need exp(S) itself, only exp(S) applied to three vectors.  A squaring costs ~n^3/2
    // fp64 instructions, an apply 3 n^2: for n > 6 it is cheaper to leave the LAST squaring out and apply X_{s-1}
    // twice, exp(S) q = X_{s-1} (X_{s-1} q).  Measured: 2-4 % faster for N = 6..10; from N = 11, where P spills, the
    // second apply costs what it saves (and leaving two squarings out for four applies is 5 % slower), so not there.
    // Every X_k has had its diagonal re-derived from conservation, so each apply conserves total momentum to rounding.
    static constexpr int kDefer = (N >= 6 && N <= 10) ? 1 : 0;

    // a[i] = dt/t_s,i (unscaled), w[i] = sqrt(eps_i), iw[i] = 1/w[i].  On return m, s are the chosen Taylor degree and
    // scaling exponent and P holds X - I (packed, diagonal slots = d) with X = exp(S / 2^min(defer, s)): exp(S) itself
    // for defer = 0, the iterate min(defer, s) squarings short of it otherwise.
    template <int defer = 0>
    __device__ __forceinline__ static void expm(const Real (&a)[N], const Real (&w)[N], const Real (&iw)[N],
                                                Real (&P)[SZ], int& m, int& s) {
        // The scaling exponent is chosen on ||S||_2 (Theorem 1, holds in any consistent norm; S is
        // symmetric and the whole iteration runs in S's basis).  S is negative semi-definite and its eigenvalues
        // -mu solve the secular equation 1 = sum_i eps_i a_i / (mu - a_i) (Eq. 29's lambda), whose
        // largest root obeys  mu <= max_i a_i + sum_i eps_i a_i  =: norm  (<= ||A||_1 = 2 max(sum eps a, max a);
        // DESIGN.md R5).
        Real sb = Real(0), amax = Real(0);
        static_for<0, N>([&](auto I) {
            constexpr int i = I;
            sb = fma(a[i] * w[i], w[i], sb);
            amax = fmax(amax, a[i]);
        });
        const Real norm = sb + amax;
        choose_m_s_warp(norm, hcost(), m, s);  // m is warp-uniform, s is this cell's own
        const Real sc = Num<Real>::pow2(s);

        Real al[N], be[N];
        Real b00 = Real(0);
        static_for<0, N>([&](auto I) {
            constexpr int i = I;
            al[i] = a[i] * sc;
            be[i] = al[i] * w[i];
            b00 = fma(be[i], w[i], b00);
        });
        b00 = -b00;

        // The polynomial.  Three rewritings of Horner's  P_j = (B + B P_{j+1}) / j  make a step N(N-1)/2 + 2N + 3 fused
        // multiply-adds and nothing else:
        //  (i)   Q_j = (m!/j!) P_j satisfies  Q_j = kappa_j B + B Q_{j+1},  kappa_j = m!/j!  — B is never rescaled;
        //  (ii)  Q_j is a polynomial in B, so B Q = Q B is symmetric: its row 0 is its column 0,
        //        (B Q)_0k = beta_k Q_00 - alpha_k Q_0k, and the dust block is (B Q)_ik = beta_i Q_0k - alpha_i Q_ik;
        //  (iii) every entry of Q outside (0,0) carries its beta's as plain factors, Q_0k = beta_k v_k and
        //        Q_ik = beta_i beta_k U_ik, and in (v, U) the recurrences lose their multiplications:
        //            U_ik <- v_k - alpha_i U_ik,   v_k <- (kappa_j + Q_00) - alpha_k v_k,
        //            Q_00 <- b00 (kappa_j + Q_00) + sum_l beta_l^2 v_l        (all right-hand sides: OLD values).
        //        No division is ever performed (Q_m = B is v = 1, U = 0), so beta_k = 0 needs no special case.
        // The dust DIAGONAL is not carried at all: a step feeds P_ii only back into P_ii, and the final diagonal is
        // re-derived from conservation below.  P = Q_1 / m! is put back together at the end.
        // Storage: P[ix(0,k)] holds v_k, P[ix(i,k)] (1 <= i < k) holds U_ik, P[ix(0,0)] holds Q_00.
        Real be2[N];
        static_for<0, N>([&](auto I) { be2[I] = be[I] * be[I]; });
        static_for<0, SZ>([&](auto K) { P[K] = Real(0); });
        P[ix(0, 0)] = b00;
        static_for<1, n>([&](auto I) { P[ix(0, I)] = Real(1); });
        Real kap = Real(1);
        auto horner_step = [&](int j) {
            kap *= Num<Real>::num(j + 1);
            static_for<1, n>([&](auto I) {
                constexpr int i = I;
                static_for<i + 1, n>([&](auto K) {
                    constexpr int k = K;
                    P[ix(i, k)] = fma(-al[i - 1], P[ix(i, k)], P[ix(0, k)]);
                });
            });
            Real t00 = be2[0] * P[ix(0, 1)];
            static_for<2, n>([&](auto L) {
                constexpr int l = L;
                t00 = fma(be2[l - 1], P[ix(0, l)], t00);
            });
            const Real x00 = kap + P[ix(0, 0)];
            static_for<1, n>([&](auto K) {
                constexpr int k = K;
                P[ix(0, k)] = fma(-al[k - 1], P[ix(0, k)], x00);
            });
            P[ix(0, 0)] = fma(b00, x00, t00);
        };
        {
            int j = m - 1;
            // two steps per trip where the loop overhead is a large part of a step (N = 2..4, measured: 1-2 %)
            if constexpr (N >= 2 && N <= 4) {
                for (; j >= 2; j -= 2) {
                    horner_step(j);
                    horner_step(j - 1);
                }
            }
            for (; j >= 1; --j) horner_step(j);
        }
        {
            // P_0k = beta_k v_k / m!,  P_ik = beta_i beta_k U_ik / m!
            const Real inv = Num<Real>::ifact(m);
            Real bs[N];
            static_for<0, N>([&](auto I) { bs[I] = be[I] * inv; });
            static_for<1, n>([&](auto I) {
                constexpr int i = I;
                P[ix(0, i)] *= bs[i - 1];
                static_for<i + 1, n>([&](auto K) {
                    constexpr int k = K;
                    P[ix(i, k)] *= bs[i - 1] * be[k - 1];
                });
            });
        }
        // off-diagonals are non-negative in exact arithmetic; clamp the rounding noise, then re-derive the diagonal
        static_for<0, n>([&](auto I) {
            constexpr int i = I;
            static_for<i + 1, n>([&](auto K) {
                constexpr int k = K;
                P[ix(i, k)] = clamp_below(P[ix(i, k)], Real(0));
            });
        });
        conserve(P, w, iw);

        // s squarings: O <- offdiag(X X), X = O + diag(1 + d) >= 0 entrywise, X symmetric
        for (int it = min(defer, s); it < s; ++it) {
            Real X[SZ];
            static_for<0, SZ>([&](auto K) { X[K] = P[K]; });
            static_for<0, n>([&](auto I) {
                constexpr int i = I;
                X[ix(i, i)] = Real(1) + P[ix(i, i)];
            });
            static_for<0, n>([&](auto I) {
                constexpr int i = I;
                static_for<i + 1, n>([&](auto K) {
                    constexpr int k = K;
                    Real acc = X[sx(i, 0)] * X[sx(0, k)];
                    static_for<1, n>([&](auto L) {
                        constexpr int l = L;
                        acc = fma(X[sx(i, l)], X[sx(l, k)], acc);
                    });
                    P[ix(i, k)] = acc;
                });
            });
            conserve(P, w, iw);
        }
    }
};

}  // namespace dg
