// dg_internal.h — declarations shared by the translation units of libdg (not installed, not part of the ABI).
#pragma once
#include <cuda_runtime.h>

namespace dg {

struct UpdateArgs {  // dg_drag_update / dg_drag_update_ex
    const double* rho_g;
    const double* rho_d;
    const double* t_s;
    double dt;
    const double* p_in;
    long long ncells;
    double* p_out;
    int* s_out;
    int* m_out;
};
struct BuildArgs {  // dg_drag_matrix_build
    const double* rho_g;
    const double* rho_d;
    const double* t_s;
    double dt;
    long long ncells;
    double* A;
};
struct ExpmArgs {  // dg_expm_scale_square
    const double* A;
    long long ncells;
    double* E;
    int* s_out;
};
struct ApplyArgs {  // dg_drag_apply
    const double* E;
    const double* p_in;
    long long ncells;
    double* p_out;
};

struct UpdateArgsF32 {  // dg_drag_update_f32
    const float* rho_g;
    const float* rho_d;
    const float* t_s;
    float dt;
    const float* p_in;
    long long ncells;
    float* p_out;
    int* s_out;
    int* m_out;
};

// One set of launchers per N (a translation unit each, compiled from dg_kernels.cu with -DDG_N=<N>).
struct Launchers {
    cudaError_t (*update)(const UpdateArgs&, cudaStream_t);
    cudaError_t (*build)(const BuildArgs&, cudaStream_t);
    cudaError_t (*expm)(const ExpmArgs&, cudaStream_t);
    cudaError_t (*apply)(const ApplyArgs&, cudaStream_t);
    cudaError_t (*rk1)(const UpdateArgs&, cudaStream_t);  // dg_drag_rk1 (s_out / m_out unused)
    const char* variant;
};

// Warp-per-cell DMMA variant (dg_wpc_kernels.cu, one translation unit per N).
struct WpcLaunchers {
    cudaError_t (*update)(const UpdateArgs&, cudaStream_t);
    cudaError_t (*expm)(const ExpmArgs&, cudaStream_t);
    const char* variant;
};

// The paper's scheme as printed (dg_paper_kernels.cu, one translation unit per N): a measured reference, not the product.
struct PaperLaunchers {
    cudaError_t (*update[3])(const UpdateArgs&, cudaStream_t);  // [0] min(Pi_m + s); [1] Alg. 2; [2] Alg. 2 + Alg. 8/9
    const char* variant;
};

// Pair-per-cell kernel (dg_ppc_kernels.cu, one translation unit per EVEN number of dust slots NP; serves N = NP - 1, NP).
struct PpcLaunchers {
    cudaError_t (*update)(const UpdateArgs&, int N, cudaStream_t);
    // dg_drag_update_energy in ONE launch (s_out / m_out unused), as TpsLaunchers::update_energy
    cudaError_t (*update_energy)(const UpdateArgs&, int N, const double* E_in, double* E_out, double w, cudaStream_t);
    int tile;  // cells per sorted tile: launches over sub-ranges that start on a multiple of it give the same bits
    const char* variant;
};
extern const PpcLaunchers ppc_launchers_NP2, ppc_launchers_NP4, ppc_launchers_NP6, ppc_launchers_NP8, ppc_launchers_NP10,
    ppc_launchers_NP12, ppc_launchers_NP14, ppc_launchers_NP16;

// Thread-per-cell kernel over stiffness-sorted shared-memory tiles (dg_tps_kernels.cu, one translation unit per N <= 12).
struct TpsLaunchers {
    cudaError_t (*update)(const UpdateArgs&, cudaStream_t);
    // dg_drag_update_energy in ONE launch: the update plus E_out = E_in + [KE_g] + w [K(t) - K(t+dt)] (s_out / m_out unused)
    cudaError_t (*update_energy)(const UpdateArgs&, const double* E_in, double* E_out, double w, cudaStream_t);
    int tile;  // cells per sorted tile: launches over sub-ranges that start on a multiple of it give the same bits
    const char* variant;
};
constexpr int kTpsMaxN = 12;
extern const TpsLaunchers tps_launchers_N1, tps_launchers_N2, tps_launchers_N3, tps_launchers_N4, tps_launchers_N5,
    tps_launchers_N6, tps_launchers_N7, tps_launchers_N8, tps_launchers_N9, tps_launchers_N10, tps_launchers_N11,
    tps_launchers_N12;

// The sorted-tile kernel in single precision (dg_tps_kernels.cu compiled with -DDG_TPS_F32, one translation unit per N <= 12).
struct TpsF32Launchers {
    cudaError_t (*update)(const UpdateArgsF32&, cudaStream_t);
    int tile;
};
extern const TpsF32Launchers tps_f32_launchers_N1, tps_f32_launchers_N2, tps_f32_launchers_N3, tps_f32_launchers_N4,
    tps_f32_launchers_N5, tps_f32_launchers_N6, tps_f32_launchers_N7, tps_f32_launchers_N8, tps_f32_launchers_N9,
    tps_f32_launchers_N10, tps_f32_launchers_N11, tps_f32_launchers_N12;

// Single-precision thread-per-cell kernel (dg_f32_kernels.cu, one translation unit per N).
struct F32Launchers {
    cudaError_t (*update)(const UpdateArgsF32&, cudaStream_t);
};

#define DG_DECL_LAUNCHERS(NN)                       \
    extern const Launchers launchers_N##NN;         \
    extern const F32Launchers f32_launchers_N##NN;  \
    extern const WpcLaunchers wpc_launchers_N##NN;  \
    extern const PaperLaunchers paper_launchers_N##NN;
DG_DECL_LAUNCHERS(1)
DG_DECL_LAUNCHERS(2)
DG_DECL_LAUNCHERS(3)
DG_DECL_LAUNCHERS(4)
DG_DECL_LAUNCHERS(5)
DG_DECL_LAUNCHERS(6)
DG_DECL_LAUNCHERS(7)
DG_DECL_LAUNCHERS(8)
DG_DECL_LAUNCHERS(9)
DG_DECL_LAUNCHERS(10)
DG_DECL_LAUNCHERS(11)
DG_DECL_LAUNCHERS(12)
DG_DECL_LAUNCHERS(13)
DG_DECL_LAUNCHERS(14)
DG_DECL_LAUNCHERS(15)
DG_DECL_LAUNCHERS(16)
#undef DG_DECL_LAUNCHERS

}  // namespace dg
