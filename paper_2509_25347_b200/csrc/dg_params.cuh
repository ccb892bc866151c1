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
// 1/theta_m (rounded; scaling_exponent() re-checks its result against theta_m itself)
__constant__ const double c_inv_theta[kRows] = {1.0 / 2.5809568029e-8, 1.0 / 3.3971688399e-4, 1.0 / 9.0656564075e-3,
                                                1.0 / 8.9577602032e-2, 1.0 / 2.9961589138e-1, 1.0 / 7.8028742566e-1,
                                                1.0 / 1.4382525967,    1.0 / 2.4285825244,    1.0 / 3.5396663487};
// 1/j for the Horner recurrence P <- (B + B P)/j, j = 1..30 (index 0 unused)
__constant__ const double c_inv[31] = {
    0.0,        1.0 / 1.0,  1.0 / 2.0,  1.0 / 3.0,  1.0 / 4.0,  1.0 / 5.0,  1.0 / 6.0,  1.0 / 7.0,
    1.0 / 8.0,  1.0 / 9.0,  1.0 / 10.0, 1.0 / 11.0, 1.0 / 12.0, 1.0 / 13.0, 1.0 / 14.0, 1.0 / 15.0,
    1.0 / 16.0, 1.0 / 17.0, 1.0 / 18.0, 1.0 / 19.0, 1.0 / 20.0, 1.0 / 21.0, 1.0 / 22.0, 1.0 / 23.0,
    1.0 / 24.0, 1.0 / 25.0, 1.0 / 26.0, 1.0 / 27.0, 1.0 / 28.0, 1.0 / 29.0, 1.0 / 30.0};

constexpr int kSMax = 1000;  // 2^-s must stay a normal double

// 2^-s exactly, 0 <= s <= kSMax
__device__ __forceinline__ double pow2neg(int s) { return __hiloint2double((1023 - s) << 20, 0); }

// Smallest s >= 0 with norm * 2^-s <= theta (reading R6: the ceil form of Eq. B.10), found
// from the exponent field of norm/theta plus one compare instead of a rounded log2.
__device__ __forceinline__ int scaling_exponent(double norm, double theta, double inv_theta) {
    double r = norm * inv_theta;
    int e = ((__double2hiint(r) >> 20) & 0x7ff) - 1022;  // r = f * 2^e, f in [0.5, 1), for normal r
    int s = max(e - 1, 0);                                // norm/2^(e-1) = 2 f theta: may still exceed theta
    if (norm * pow2neg(min(s, kSMax)) > theta) ++s;
    return s;
}

// Choice of the Table B.1 row: minimise the cost  hcost * m_k + s_k  over the nine rows (B.11, PAPER.md:635-638,
// with the polynomial priced by this implementation's sparse Horner recurrence, hcost = cost of one Horner step in
// units of one squaring, instead of Pi_m dense products; reading R8).  Ties go to the lower row.
// Non-finite norms give s = 0 (the NaN/Inf then propagates through the polynomial into that cell's output only).
__device__ __forceinline__ void choose_m_s(double norm, float hcost, int& m, int& s) {
    m = c_m[kRows - 1];
    s = 0;
    if (!(norm <= 1.7e308)) return;
    float best = 3.0e38f;
#pragma unroll
    for (int k = 0; k < kRows; ++k) {
        int sk = scaling_exponent(norm, c_theta[k], c_inv_theta[k]);
        float cost = hcost * (float)c_m[k] + (float)sk;
        if (cost < best) { best = cost; m = c_m[k]; s = sk; }
    }
    s = min(s, kSMax);
}

// 1/sqrt(eps) and sqrt(eps) with eps clamped away from zero so that rho_d = 0 stays finite (R12).
__device__ __forceinline__ void sym_weights(double eps, double& w, double& iw) {
    eps = fmax(eps, 1e-200);
    iw = rsqrt(eps);
    w = eps * iw;
}

}  // namespace dg
