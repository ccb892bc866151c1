// dg_api.cu — the C ABI of include/dg.h: argument validation and dispatch on N.  No arithmetic here.
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstring>

#include "../../include/dg.h"
#include "dg_internal.h"

namespace dg {

static const Launchers* const kTable[DG_NMAX + 1] = {
    nullptr,        &launchers_N1,  &launchers_N2,  &launchers_N3,  &launchers_N4,  &launchers_N5,
    &launchers_N6,  &launchers_N7,  &launchers_N8,  &launchers_N9,  &launchers_N10, &launchers_N11,
    &launchers_N12, &launchers_N13, &launchers_N14, &launchers_N15, &launchers_N16};

static const WpcLaunchers* const kWpcTable[DG_NMAX + 1] = {
    nullptr,            &wpc_launchers_N1,  &wpc_launchers_N2,  &wpc_launchers_N3,  &wpc_launchers_N4,
    &wpc_launchers_N5,  &wpc_launchers_N6,  &wpc_launchers_N7,  &wpc_launchers_N8,  &wpc_launchers_N9,
    &wpc_launchers_N10, &wpc_launchers_N11, &wpc_launchers_N12, &wpc_launchers_N13, &wpc_launchers_N14,
    &wpc_launchers_N15, &wpc_launchers_N16};

static const PaperLaunchers* const kPaperTable[DG_NMAX + 1] = {
    nullptr,              &paper_launchers_N1,  &paper_launchers_N2,  &paper_launchers_N3,  &paper_launchers_N4,
    &paper_launchers_N5,  &paper_launchers_N6,  &paper_launchers_N7,  &paper_launchers_N8,  &paper_launchers_N9,
    &paper_launchers_N10, &paper_launchers_N11, &paper_launchers_N12, &paper_launchers_N13, &paper_launchers_N14,
    &paper_launchers_N15, &paper_launchers_N16};

static const F32Launchers* const kF32Table[DG_NMAX + 1] = {
    nullptr,            &f32_launchers_N1,  &f32_launchers_N2,  &f32_launchers_N3,  &f32_launchers_N4,
    &f32_launchers_N5,  &f32_launchers_N6,  &f32_launchers_N7,  &f32_launchers_N8,  &f32_launchers_N9,
    &f32_launchers_N10, &f32_launchers_N11, &f32_launchers_N12, &f32_launchers_N13, &f32_launchers_N14,
    &f32_launchers_N15, &f32_launchers_N16};

static const PpcLaunchers* const kPpcTable[DG_NMAX + 1] = {
    nullptr,
    &ppc_launchers_NP2,  &ppc_launchers_NP2,  &ppc_launchers_NP4,  &ppc_launchers_NP4,  &ppc_launchers_NP6,  &ppc_launchers_NP6,
    &ppc_launchers_NP8,  &ppc_launchers_NP8,  &ppc_launchers_NP10, &ppc_launchers_NP10, &ppc_launchers_NP12, &ppc_launchers_NP12,
    &ppc_launchers_NP14, &ppc_launchers_NP14, &ppc_launchers_NP16, &ppc_launchers_NP16};

static const TpsLaunchers* const kTpsTable[DG_NMAX + 1] = {
    nullptr,           &tps_launchers_N1,  &tps_launchers_N2,  &tps_launchers_N3, &tps_launchers_N4,
    &tps_launchers_N5, &tps_launchers_N6,  &tps_launchers_N7,  &tps_launchers_N8, &tps_launchers_N9,
    &tps_launchers_N10, &tps_launchers_N11, &tps_launchers_N12, nullptr,           nullptr,
    nullptr,           nullptr};

static const TpsF32Launchers* const kTpsF32Table[DG_NMAX + 1] = {
    nullptr,                &tps_f32_launchers_N1,  &tps_f32_launchers_N2,  &tps_f32_launchers_N3, &tps_f32_launchers_N4,
    &tps_f32_launchers_N5,  &tps_f32_launchers_N6,  &tps_f32_launchers_N7,  &tps_f32_launchers_N8, &tps_f32_launchers_N9,
    &tps_f32_launchers_N10, &tps_f32_launchers_N11, &tps_f32_launchers_N12, nullptr,               nullptr,
    nullptr,                nullptr};

// The mapping dg_drag_update uses for each N, chosen from measurements on B200.  One thread per cell
// with the packed symmetric matrices in its registers up to N = 12 (mild spills from N = 10), run over stiffness-sorted
// shared-memory tiles (dg_tps_kernels.cu): 3-25 % faster than the same core over 32 consecutive cells (dg_kernels.cu,
// kept as DG_VARIANT_TPC) on every workload of BASELINE.json.  From N = 13 the thread-per-cell spills take over and the
// pair-per-cell kernel (two lanes per cell, the iterate in a shared-memory tile) wins (2^22 stiff cells, ms: N = 12:
// 5.7 sorted thread / 7.9 pair; N = 13: 16.2 thread / 10.8 pair; N = 16: 13.9 pair, warp-per-cell DMMA 23.1).
constexpr int kFirstPpcN = 13;
static_assert(kFirstPpcN == kTpsMaxN + 1, "every N has a default kernel");
static inline int default_variant(int N) { return N >= kFirstPpcN ? DG_VARIANT_PPC : DG_VARIANT_TPS; }
// The staged dg_expm_scale_square has no pair-per-cell form (it writes dense matrices to HBM: a test path); it keeps the
// warp-per-cell DMMA kernel from N = 14 and the thread-per-cell one below.
static inline int expm_variant(int N) { return N >= 14 ? DG_VARIANT_WPC : DG_VARIANT_TPC; }

static thread_local char g_cuda_err[256] = "";

dg_status cuda_status(cudaError_t e) {
    if (e == cudaSuccess) return DG_OK;
    snprintf(g_cuda_err, sizeof g_cuda_err, "%s: %s", cudaGetErrorName(e), cudaGetErrorString(e));
    return DG_ECUDA;
}

static inline bool misaligned(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 7u) != 0; }

// Common checks.  Returns DG_OK with *noop = true when there is nothing to do.
static dg_status check_common(int N, long long ncells, bool* noop) {
    *noop = false;
    if (N < 1 || N > DG_NMAX || ncells < 0) return DG_ERANGE;
    if (ncells == 0) *noop = true;
    return DG_OK;
}

cudaError_t launch_update(int N, int variant, const UpdateArgs& a, cudaStream_t st) {
    if (variant == DG_VARIANT_DEFAULT) variant = default_variant(N);
    if (variant == DG_VARIANT_PAPER) return kPaperTable[N]->update[0](a, st);
    if (variant == DG_VARIANT_PAPER_ALG2) return kPaperTable[N]->update[1](a, st);
    if (variant == DG_VARIANT_PAPER_BOUND) return kPaperTable[N]->update[2](a, st);
    if (variant == DG_VARIANT_PPC) return kPpcTable[N]->update(a, N, st);
    if (variant == DG_VARIANT_TPS) return kTpsTable[N]->update(a, st);
    return variant == DG_VARIANT_WPC ? kWpcTable[N]->update(a, st) : kTable[N]->update(a, st);
}

// dg_drag_update_energy: one launch of the default kernel for N, which forms the kinetic-energy sums on the way
cudaError_t launch_update_energy(int N, const UpdateArgs& a, const double* E_in, double* E_out, double w, cudaStream_t st) {
    if (default_variant(N) == DG_VARIANT_PPC) return kPpcTable[N]->update_energy(a, N, E_in, E_out, w, st);
    return kTpsTable[N]->update_energy(a, E_in, E_out, w, st);
}

}  // namespace dg

using namespace dg;

#define DG_CHECK_PTR(p)                  \
    do {                                 \
        if ((p) == nullptr) return DG_ENULL; \
        if (misaligned(p)) return DG_EALIGN; \
    } while (0)
#define DG_CHECK_OPT_PTR(p)                            \
    do {                                               \
        if ((p) != nullptr && (reinterpret_cast<uintptr_t>(p) & 3u)) return DG_EALIGN; \
    } while (0)

extern "C" {

dg_status dg_drag_matrix_build(const double* rho_g, const double* rho_d, const double* t_s, double dt, int N,
                               long long ncells, double* A, void* stream) {
    bool noop;
    dg_status st = check_common(N, ncells, &noop);
    if (st != DG_OK) return st;
    if (!(dt >= 0.0) || !std::isfinite(dt)) return DG_EINVAL;
    if (noop) return DG_OK;
    DG_CHECK_PTR(rho_g);
    DG_CHECK_PTR(rho_d);
    DG_CHECK_PTR(t_s);
    DG_CHECK_PTR(A);
    BuildArgs a{rho_g, rho_d, t_s, dt, ncells, A};
    return cuda_status(kTable[N]->build(a, static_cast<cudaStream_t>(stream)));
}

dg_status dg_expm_scale_square(const double* A, int N, long long ncells, double* E, int* s_out, void* stream) {
    bool noop;
    dg_status st = check_common(N, ncells, &noop);
    if (st != DG_OK) return st;
    if (noop) return DG_OK;
    DG_CHECK_PTR(A);
    DG_CHECK_PTR(E);
    DG_CHECK_OPT_PTR(s_out);
    ExpmArgs a{A, ncells, E, s_out};
    cudaStream_t cs = static_cast<cudaStream_t>(stream);
    return cuda_status(expm_variant(N) == DG_VARIANT_WPC ? kWpcTable[N]->expm(a, cs) : kTable[N]->expm(a, cs));
}

dg_status dg_drag_apply(const double* E, const double* p_in, int N, long long ncells, double* p_out, void* stream) {
    bool noop;
    dg_status st = check_common(N, ncells, &noop);
    if (st != DG_OK) return st;
    if (noop) return DG_OK;
    DG_CHECK_PTR(E);
    DG_CHECK_PTR(p_in);
    DG_CHECK_PTR(p_out);
    ApplyArgs a{E, p_in, ncells, p_out};
    return cuda_status(kTable[N]->apply(a, static_cast<cudaStream_t>(stream)));
}

dg_status dg_drag_update_variant(const double* rho_g, const double* rho_d, const double* t_s, double dt,
                                 const double* p_in, int N, long long ncells, double* p_out, int* s_out, int* m_out,
                                 int variant, void* stream) {
    bool noop;
    dg_status st = check_common(N, ncells, &noop);
    if (st != DG_OK) return st;
    if (!(dt >= 0.0) || !std::isfinite(dt)) return DG_EINVAL;
    if (variant < DG_VARIANT_DEFAULT || variant > DG_VARIANT_TPS) return DG_EINVAL;
    if (variant == DG_VARIANT_TPS && N > kTpsMaxN) return DG_EINVAL;
    if (noop) return DG_OK;
    DG_CHECK_PTR(rho_g);
    DG_CHECK_PTR(rho_d);
    DG_CHECK_PTR(t_s);
    DG_CHECK_PTR(p_in);
    DG_CHECK_PTR(p_out);
    DG_CHECK_OPT_PTR(s_out);
    DG_CHECK_OPT_PTR(m_out);
    UpdateArgs a{rho_g, rho_d, t_s, dt, p_in, ncells, p_out, s_out, m_out};
    return cuda_status(launch_update(N, variant, a, static_cast<cudaStream_t>(stream)));
}

dg_status dg_drag_update_ex(const double* rho_g, const double* rho_d, const double* t_s, double dt,
                            const double* p_in, int N, long long ncells, double* p_out, int* s_out, int* m_out,
                            void* stream) {
    return dg_drag_update_variant(rho_g, rho_d, t_s, dt, p_in, N, ncells, p_out, s_out, m_out, DG_VARIANT_DEFAULT,
                                  stream);
}

dg_status dg_drag_update(const double* rho_g, const double* rho_d, const double* t_s, double dt, const double* p_in,
                         int N, long long ncells, double* p_out, void* stream) {
    return dg_drag_update_ex(rho_g, rho_d, t_s, dt, p_in, N, ncells, p_out, nullptr, nullptr, stream);
}

dg_status dg_drag_update_steps(const double* rho_g, const double* rho_d, const double* t_s, double dt,
                               const double* p_in, int N, long long ncells, int nsteps, double* p_out, void* stream) {
    if (nsteps < 0) return DG_EINVAL;
    if (nsteps == 0) {
        bool noop;
        dg_status st = check_common(N, ncells, &noop);
        if (st != DG_OK || noop) return st;
        DG_CHECK_PTR(p_in);
        DG_CHECK_PTR(p_out);
        if (p_in == p_out) return DG_OK;
        return cuda_status(cudaMemcpyAsync(p_out, p_in, sizeof(double) * 3 * (size_t)(N + 1) * (size_t)ncells,
                                           cudaMemcpyDeviceToDevice, static_cast<cudaStream_t>(stream)));
    }
    dg_status st = dg_drag_update(rho_g, rho_d, t_s, dt, p_in, N, ncells, p_out, stream);
    for (int k = 1; k < nsteps && st == DG_OK; ++k)
        st = dg_drag_update(rho_g, rho_d, t_s, dt, p_out, N, ncells, p_out, stream);
    return st;
}

dg_status dg_drag_update_f32(const float* rho_g, const float* rho_d, const float* t_s, float dt, const float* p_in,
                             int N, long long ncells, float* p_out, int* s_out, int* m_out, void* stream) {
    bool noop;
    dg_status st = check_common(N, ncells, &noop);
    if (st != DG_OK) return st;
    if (!(dt >= 0.0f) || !std::isfinite(dt)) return DG_EINVAL;
    if (noop) return DG_OK;
    const void* ptrs[] = {rho_g, rho_d, t_s, p_in, p_out};
    for (const void* p : ptrs) {
        if (p == nullptr) return DG_ENULL;
        if (reinterpret_cast<uintptr_t>(p) & 3u) return DG_EALIGN;
    }
    DG_CHECK_OPT_PTR(s_out);
    DG_CHECK_OPT_PTR(m_out);
    UpdateArgsF32 a{rho_g, rho_d, t_s, dt, p_in, ncells, p_out, s_out, m_out};
    // same choice of mapping as in double precision: sorted tiles up to N = 12, the consecutive-cell kernel above
    if (N <= kTpsMaxN) return cuda_status(kTpsF32Table[N]->update(a, static_cast<cudaStream_t>(stream)));
    return cuda_status(kF32Table[N]->update(a, static_cast<cudaStream_t>(stream)));
}

dg_status dg_drag_rk1(const double* rho_g, const double* rho_d, const double* t_s, double dt, const double* p_in,
                      int N, long long ncells, double* p_out, void* stream) {
    bool noop;
    dg_status st = check_common(N, ncells, &noop);
    if (st != DG_OK) return st;
    if (!(dt >= 0.0) || !std::isfinite(dt)) return DG_EINVAL;
    if (noop) return DG_OK;
    DG_CHECK_PTR(rho_g);
    DG_CHECK_PTR(rho_d);
    DG_CHECK_PTR(t_s);
    DG_CHECK_PTR(p_in);
    DG_CHECK_PTR(p_out);
    UpdateArgs a{rho_g, rho_d, t_s, dt, p_in, ncells, p_out, nullptr, nullptr};
    return cuda_status(kTable[N]->rk1(a, static_cast<cudaStream_t>(stream)));
}

int dg_launches_per_update(int N, long long ncells) {
    if (N < 1 || N > DG_NMAX || ncells <= 0) return 0;
    return 1;
}

const char* dg_variant_name(int N) {
    if (N < 1 || N > DG_NMAX) return "";
    return default_variant(N) == DG_VARIANT_PPC ? kPpcTable[N]->variant : kTpsTable[N]->variant;
}

const char* dg_status_string(dg_status st) {
    switch (st) {
        case DG_OK: return "DG_OK";
        case DG_EINVAL: return "DG_EINVAL: scalar argument out of range (dt negative or not finite)";
        case DG_ENULL: return "DG_ENULL: required pointer is NULL";
        case DG_EALIGN: return "DG_EALIGN: pointer is not 8-byte aligned";
        case DG_ERANGE: return "DG_ERANGE: N outside [1, 16] or ncells < 0";
        case DG_ECUDA: return "DG_ECUDA: CUDA runtime error (see dg_last_cuda_error)";
        case DG_ECAPACITY:
            return "DG_ECAPACITY: ncells * 8 * (8N + 7) bytes exceed the fixed 32 MiB staging array of "
                   "dg_drag_update_host_static (it never allocates; split the cells or use dg_drag_update_host)";
    }
    return "unknown dg_status";
}

const char* dg_last_cuda_error(void) { return g_cuda_err; }

int dg_version(void) { return DG_VERSION; }

}  // extern "C"
