// dg_params.cuh — Table B.1 constants and the norm-based choice of (m, s).
//
// theta_m: backward-error thresholds of Eq. B.4-B.8 for u = 2^-53, the nine rows of Table B.1
// (PAPER.md:619-631), m = 2, 4, 6, 9, 12, 16, 20, 25, 30.  Rows 5 and 6 are garbled in the extracted table; all nine
// values were recomputed from the definition in 80-digit arithmetic (reading R3,
// tests/test_host_logic.py repeats the computation) and are rounded DOWN here.
#pragma once
#include <cuda_runtime.h>

namespace dg {

constexpr int kRows = 9;
__constant__ const int c_m[kRows] = {2, 4, 6, 9, 12, 16, 20, 25, 30};
__constant__ const double c_theta[kRows] = {2.5809568029e-8, 3.3971688399e-4, 9.0656564075e-3,
                                            8.9577602032e-2, 2.9961589138e-1, 7.8028742566e-1,
                                            1.4382525967,    2.4285825244,    3.5396663487};
// 1/i!, i = 0..30: the Taylor coefficients b_i of Eq. 19
__constant__ const double c_ifact[31] = {
    1.0, 1.0, 1.0 / 2, 1.0 / 6, 1.0 / 24, 1.0 / 120, 1.0 / 720, 1.0 / 5040, 1.0 / 40320, 1.0 / 362880, 1.0 / 3628800,
    1.0 / 39916800, 1.0 / 479001600, 1.0 / 6227020800.0, 1.0 / 87178291200.0, 1.0 / 1307674368000.0,
    1.0 / 20922789888000.0, 1.0 / 355687428096000.0, 1.0 / 6402373705728000.0, 1.0 / 121645100408832000.0,
    1.0 / 2432902008176640000.0, 1.0 / 51090942171709440000.0, 1.0 / 1124000727777607680000.0,
    1.0 / 25852016738884976640000.0, 1.0 / 620448401733239439360000.0, 1.0 / 15511210043330985984000000.0,
    1.0 / 403291461126605635584000000.0, 1.0 / 10888869450418352160768000000.0,
    1.0 / 304888344611713860501504000000.0, 1.0 / 8841761993739701954543616000000.0,
    1.0 / 265252859812191058636308480000000.0};
// j as a double, j = 0..30 (the running factor m!/j! of the unscaled Horner recurrence)
__constant__ const double c_dbl[31] = {0,  1,  2,  3,  4,  5,  6,  7,  8,  9,  10, 11, 12, 13, 14, 15,
                                       16, 17, 18, 19, 20, 21, 22, 23, 24, 25, 26, 27, 28, 29, 30};

constexpr int kSMax = 1000;  // 2^-s must stay a normal double

// 2^-s exactly, 0 <= s <= kSMax
__device__ __forceinline__ double pow2neg(int s) { return __hiloint2double((1023 - s) << 20, 0); }

// Smallest s >= 0 with norm * 2^-s <= theta (reading R6: the ceil form of Eq. B.10), exact
// and in integer arithmetic.  With norm = f 2^e and theta = g 2^t (f, g in [1, 2)) the answer is e - t + (f > g),
// which is the carry of the bit patterns' difference: ceil((bits(norm) - bits(theta)) / 2^52).  No rounded log2 and
// no fp64 instruction.  norm >= 0 and finite; subnormal norms give 0.
__device__ __forceinline__ int scaling_exponent(double norm, double theta) {
    const long long d = __double_as_longlong(norm) - __double_as_longlong(theta) + 0xFFFFFFFFFFFFFLL;
    return max((int)(d >> 52), 0);
}

// Choice of the Table B.1 row: minimise the cost  hcost * m_k + s_k  over the nine rows (B.11, PAPER.md:635-638,
// with the polynomial priced by this implementation's sparse Horner recurrence, hcost = cost of one Horner step in
// units of one squaring, instead of Pi_m dense products; reading R8).  Ties go to the lower row.
// Non-finite norms give row 8 (m = 30).
//
// The decision is always taken by a WHOLE, CONVERGED warp for one norm: lane k < 9 prices row k in fixed point
// (1/256 of a squaring), one REDUX picks the minimum of (cost, row) packed into an int.  Every lane must call it.
__device__ __forceinline__ int choose_row_warp(double norm, float hcost) {
    const int lane = threadIdx.x & 31;
    int packed = 0x7fffffff;
    if (lane < kRows) {
        const int sk = scaling_exponent(norm, c_theta[lane]);
        const int cost = (int)(hcost * 256.0f + 0.5f) * c_m[lane] + (min(sk, 4000) << 8);
        packed = (cost << 4) | lane;
    }
    const int best = __reduce_min_sync(0xffffffffu, packed);
    return (norm <= 1.7e308) ? (best & 15) : kRows - 1;
}

// s for a given row; a non-finite norm gives s = 0 (the NaN/Inf then propagates through the polynomial into that
// cell's output only).
__device__ __forceinline__ int s_for_row(double norm, int row) {
    if (!(norm <= 1.7e308)) return 0;
    return min(scaling_exponent(norm, c_theta[row]), kSMax);
}

// Warp-per-cell mapping: the whole warp holds the same norm.
__device__ __forceinline__ void choose_m_s(double norm, float hcost, int& m, int& s) {
    const int row = choose_row_warp(norm, hcost);
    m = c_m[row];
    s = s_for_row(norm, row);
}

// Thread-per-cell mapping: the lanes of a warp run the Horner loop in lock step, so a per-lane degree would cost
// max(m) steps anyway.  The row is therefore chosen ONCE per warp, for the largest norm among its lanes (the paper
// rewrites Alg. 1 as the branch-reduced Alg. 2 for the same reason), and every lane then takes the
// smallest s that satisfies Theorem 1's premise for ITS OWN norm with that row.  Any row is admissible for any
// cell, so correctness never depends on the other lanes.  The warp maximum is taken on the high word of the double
// (one REDUX instruction) and rounded up: an upper bound within 2^-20, which can only cost, never break.
// All 32 lanes must call it (lanes without a cell pass norm = 0).
__device__ __forceinline__ void choose_m_s_warp(double norm, float hcost, int& m, int& s) {
    const unsigned hi = __reduce_max_sync(0xffffffffu, (unsigned)__double2hiint(norm));  // NaN / Inf / negative win
    const double nmax = (hi >= 0x7ff00000u) ? __longlong_as_double(0x7ff0000000000000LL) : __hiloint2double((int)hi + 1, 0);
    const int row = choose_row_warp(nmax, hcost);
    m = c_m[row];
    s = s_for_row(norm, row);
}

// 1/x and 1/sqrt(x) to about one ulp for normal positive x: the hardware seed (MUFU.RCP64H / MUFU.RSQ64H, relative
// error < 2^-22) and two Newton steps, without the IEEE routines' exponent fix-ups and slow paths.  The drag matrix
// takes a_i = dt/t_s,i and eps_i as DATA: an ulp of relative error in them is the same perturbation as the
// rounding of the inputs themselves, and it keeps Eq. 17's structure (zero column sums) exactly.  Zero, subnormal,
// infinite or NaN arguments give a non-finite result (the contract: non-finite output in that cell only); arguments
// above 2^1022 give 0.
__device__ __forceinline__ double fast_rcp(double x) {
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    double e = fma(-x, y, 1.0);
    y = fma(y, e, y);
    e = fma(-x, y, 1.0);
    return fma(y, e, y);
}
__device__ __forceinline__ double fast_rsqrt(double x) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    double e = fma(-(x * y), y, 1.0);
    y = fma(0.5 * y, e, y);
    e = fma(-(x * y), y, 1.0);
    return fma(0.5 * y, e, y);
}

// max(x, lo) that lets a NaN through (fmax would return lo): the clamps of rounding noise must not hide a non-finite
// input (include/dg.h: non-finite input gives non-finite output in that cell)
__device__ __forceinline__ double clamp_below(double x, double lo) { return (x < lo) ? lo : x; }

// 1/sqrt(eps) and sqrt(eps) with eps clamped away from zero so that rho_d = 0 stays finite (R12).
__device__ __forceinline__ void sym_weights(double eps, double& w, double& iw) {
    eps = clamp_below(eps, 1e-200);
    iw = fast_rsqrt(eps);
    w = eps * iw;
}

}  // namespace dg
