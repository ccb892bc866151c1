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
// The same thresholds for SINGLE precision, u = 2^-24: Eq. B.8 "one can take another value depending on
// the desired accuracy: 2^-11, 2^-24, 2^-113 and 2^-237 for half, single, quadruple and octuple precision".  Computed
// from the definition (Eq. B.4-B.8) by the same 60-digit routine that reproduces the u = 2^-53 column
// (tests/test_host_logic.py repeats it), rounded DOWN to floats the kernels compare against.
__constant__ const float c_theta32[kRows] = {0.00059788581f, 0.051166188f, 0.249528915f, 0.779511273f, 1.46166134f,
                                             2.47828054f,    3.55092597f,  4.92689896f,  6.32108164f};
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

// 32-bit twins of pow2neg / scaling_exponent (same carry trick on the float bit pattern)
constexpr int kSMax32 = 120;  // 2^-s must stay a normal float
__device__ __forceinline__ float pow2neg32(int s) { return __int_as_float((127 - s) << 23); }
__device__ __forceinline__ int scaling_exponent(float norm, float theta) {
    const int d = __float_as_int(norm) - __float_as_int(theta) + 0x7FFFFF;
    return max(d >> 23, 0);
}

// What the (m, s) choice and the recurrences need to know about the arithmetic type.
template <class Real>
struct Num;
template <>
struct Num<double> {
    __device__ __forceinline__ static double theta(int row) { return c_theta[row]; }
    __device__ __forceinline__ static double ifact(int m) { return c_ifact[m]; }
    __device__ __forceinline__ static double num(int j) { return c_dbl[j]; }  // j as a Real, 0 <= j <= 30
    __device__ __forceinline__ static double pow2(int s) { return pow2neg(s); }
    __device__ __forceinline__ static bool finite(double x) { return x <= 1.7e308; }
    __device__ __forceinline__ static unsigned key(double x) { return (unsigned)__double2hiint(x); }  // order-preserving, x >= 0
    __device__ __forceinline__ static double from_key_up(unsigned hi) {
        return (hi >= 0x7ff00000u) ? __longlong_as_double(0x7ff0000000000000LL) : __hiloint2double((int)hi + 1, 0);
    }
    static constexpr int smax = kSMax;
};
template <>
struct Num<float> {
    __device__ __forceinline__ static float theta(int row) { return c_theta32[row]; }
    __device__ __forceinline__ static float ifact(int m) { return (float)c_ifact[m]; }
    __device__ __forceinline__ static float num(int j) { return (float)j; }
    __device__ __forceinline__ static float pow2(int s) { return pow2neg32(s); }
    __device__ __forceinline__ static bool finite(float x) { return x <= 3.4e38f; }
    __device__ __forceinline__ static unsigned key(float x) { return (unsigned)__float_as_int(x); }
    __device__ __forceinline__ static float from_key_up(unsigned b) {
        return (b >= 0x7f800000u) ? __int_as_float(0x7f800000) : __int_as_float((int)b + 1);
    }
    static constexpr int smax = kSMax32;
};

// Choice of the Table B.1 row: minimise the cost  hcost * m_k + s_k  over the nine rows (B.11, PAPER.md:635-638,
// with the polynomial priced by this implementation's sparse Horner recurrence, hcost = cost of one Horner step in
// units of one squaring, instead of Pi_m dense products; reading R8).  Ties go to the lower row.
// Non-finite norms give row 8 (m = 30).
//
// The decision is always taken by a WHOLE, CONVERGED warp for one norm: lane k < 9 prices row k in fixed point
// (1/256 of a squaring), one REDUX picks the minimum of (cost, row) packed into an int.  Every lane must call it.
template <class Real>
__device__ __forceinline__ int choose_row_warp(Real norm, float hcost) {
    const int lane = threadIdx.x & 31;
    int packed = 0x7fffffff;
    if (lane < kRows) {
        const int sk = scaling_exponent(norm, Num<Real>::theta(lane));
        const int cost = (int)(hcost * 256.0f + 0.5f) * c_m[lane] + (min(sk, 4000) << 8);
        packed = (cost << 4) | lane;
    }
    const int best = __reduce_min_sync(0xffffffffu, packed);
    return Num<Real>::finite(norm) ? (best & 15) : kRows - 1;
}

// s for a given row; a non-finite norm gives s = 0 (the NaN/Inf then propagates through the polynomial into that
// cell's output only).
template <class Real>
__device__ __forceinline__ int s_for_row(Real norm, int row) {
    if (!Num<Real>::finite(norm)) return 0;
    return min(scaling_exponent(norm, Num<Real>::theta(row)), Num<Real>::smax);
}

// Warp-per-cell mapping: the whole warp holds the same norm.
template <class Real>
__device__ __forceinline__ void choose_m_s(Real norm, float hcost, int& m, int& s) {
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
template <class Real>
__device__ __forceinline__ void choose_m_s_warp(Real norm, float hcost, int& m, int& s) {
    const unsigned hi = __reduce_max_sync(0xffffffffu, Num<Real>::key(norm));  // NaN / Inf / negative win
    const Real nmax = Num<Real>::from_key_up(hi);
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

// Single precision: the correctly rounded hardware reciprocal / reciprocal square root are one instruction each.
__device__ __forceinline__ float fast_rcp(float x) { return __frcp_rn(x); }
__device__ __forceinline__ float fast_rsqrt(float x) { return __frsqrt_rn(x); }

// max(x, lo) that lets a NaN through (fmax would return lo): the clamps of rounding noise must not hide a non-finite
// input (include/dg.h: non-finite input gives non-finite output in that cell)
__device__ __forceinline__ double clamp_below(double x, double lo) { return (x < lo) ? lo : x; }
__device__ __forceinline__ float clamp_below(float x, float lo) { return (x < lo) ? lo : x; }

// 1/sqrt(eps) and sqrt(eps) with eps clamped away from zero so that rho_d = 0 stays finite (R12).
__device__ __forceinline__ void sym_weights(double eps, double& w, double& iw) {
    eps = clamp_below(eps, 1e-200);
    iw = fast_rsqrt(eps);
    w = eps * iw;
}
__device__ __forceinline__ void sym_weights(float eps, float& w, float& iw) {
    eps = clamp_below(eps, 1e-30f);
    iw = fast_rsqrt(eps);
    w = eps * iw;
}

}  // namespace dg
