// dg_host_static.cu — dg_drag_update_host_static (include/dg.h): the fused update on HOST buffers for callers that must
// not allocate device memory.
//
// Why it exists.  dg_drag_update_host needs device memory to stage a chunk of cells next to the kernel, and gets it
// with cudaMalloc (and creates three streams).  Some programs that embed this library cannot afford that call: a hydro
// code whose own pool has already taken the whole card at start-up (the cudaMalloc then fails), a time-step loop that
// must not stall (cudaMalloc and cudaFree synchronise the whole device), a process running under a fixed device-memory
// quota, or a plug-in whose host application forbids allocation after initialisation.  For them the staging area is
// not requested at run time at all: it is the file-scope array `g_stage` below, part of the library image, which the
// driver places on the device when this translation unit's module is loaded and keeps there until the process exits.
// The price is a hard upper limit on the problem size (DG_STATIC_STAGE_BYTES) and 32 MiB of every GPU that loads the
// module, used or not.
//
// What it does.  One chunk, one stream (the caller's): four contiguous host-to-device copies into the array (the host
// rows have pitch ncells, exactly the staging layout, so every field is a single 1-D copy), the kernel dg_drag_update
// launches for this N, one device-to-host copy of the result, and a cudaStreamSynchronize so that p_out is complete on
// return.  No cudaMalloc, cudaFree, cudaMallocAsync, stream or event creation anywhere on this path.
//
// The array's name in host code.  `g_stage` written in a host function names a host-side shadow object the runtime uses
// as a look-up key — NOT device memory.  Handing that to a kernel or a cudaMemcpy would fault, or on a system where the
// GPU can reach host memory it would quietly work on the wrong bytes.  The device address comes from
// cudaGetSymbolAddress, asked once per device with that device current (stage_address() below), and only that pointer
// goes to the copies and the kernel.
#include <cmath>
#include <cstdint>
#include <mutex>

#include "../../include/dg.h"
#include "dg_internal.h"

namespace dg {
dg_status cuda_status(cudaError_t e);
cudaError_t launch_update(int N, int variant, const UpdateArgs& a, cudaStream_t st);

namespace {

constexpr size_t kStageDoubles = (size_t)DG_STATIC_STAGE_BYTES / sizeof(double);
// The staging area.  256-byte aligned so that, with an even ncells, every staged row starts on a 16-byte boundary and
// the kernels move whole tile rows per bulk copy.  Never initialised and never cleared: see "stale contents" below.
static __device__ __align__(256) double g_stage[kStageDoubles];

constexpr int kMaxDevices = 64;
std::mutex g_mu;
double* g_stage_ptr[kMaxDevices];  // device address of g_stage on each device; nullptr until first asked

// One-time set-up per device: resolve the device address of g_stage.  `device` must be the current device (the
// answer is the address in the current device's copy of the module).  The first call loads this module on the device,
// which is when the driver actually places the 32 MiB; later calls return the cached pointer.
cudaError_t stage_address(int device, double** out) {
    std::lock_guard<std::mutex> lock(g_mu);
    if (g_stage_ptr[device] == nullptr) {
        double* ptr = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void**)&ptr, g_stage);
        if (e != cudaSuccess) return e;
        if (ptr == nullptr) return cudaErrorInvalidSymbol;
        g_stage_ptr[device] = ptr;
    }
    *out = g_stage_ptr[device];
    return cudaSuccess;
}

#define DG_TRY(x)                         \
    do {                                  \
        cudaError_t e_ = (x);             \
        if (e_ != cudaSuccess) return e_; \
    } while (0)

cudaError_t run(double* stage, const double* rho_g, const double* rho_d, const double* t_s, double dt,
                const double* p_in, int N, long long ncells, double* p_out, cudaStream_t st) {
    const size_t nc = (size_t)ncells, n = (size_t)N + 1;
    // Layout inside the array (doubles): rho_g [nc] | rho_d [N][nc] | t_s [N][nc] | p_in [3n][nc] | p_out [3n][nc].
    // Stale contents: the array still holds whatever the previous call left.  Nothing here has to start at zero — the
    // four copies overwrite every double the kernel reads, and the kernel writes every double of the p_out region that
    // is copied back — so nothing is cleared.
    double* d_rho_g = stage;
    double* d_rho_d = d_rho_g + nc;
    double* d_t_s = d_rho_d + (size_t)N * nc;
    double* d_p_in = d_t_s + (size_t)N * nc;
    double* d_p_out = d_p_in + 3 * n * nc;
    const size_t w = nc * sizeof(double);
    DG_TRY(cudaMemcpyAsync(d_rho_g, rho_g, w, cudaMemcpyHostToDevice, st));
    DG_TRY(cudaMemcpyAsync(d_rho_d, rho_d, w * (size_t)N, cudaMemcpyHostToDevice, st));
    DG_TRY(cudaMemcpyAsync(d_t_s, t_s, w * (size_t)N, cudaMemcpyHostToDevice, st));
    DG_TRY(cudaMemcpyAsync(d_p_in, p_in, w * 3 * n, cudaMemcpyHostToDevice, st));
    UpdateArgs a{d_rho_g, d_rho_d, d_t_s, dt, d_p_in, ncells, d_p_out, nullptr, nullptr};
    DG_TRY(launch_update(N, DG_VARIANT_DEFAULT, a, st));
    DG_TRY(cudaMemcpyAsync(p_out, d_p_out, w * 3 * n, cudaMemcpyDeviceToHost, st));
    return cudaSuccess;
}

}  // namespace
}  // namespace dg

using namespace dg;

extern "C" dg_status dg_drag_update_host_static(const double* rho_g, const double* rho_d, const double* t_s, double dt,
                                                const double* p_in, int N, long long ncells, double* p_out,
                                                void* stream) {
    if (N < 1 || N > DG_NMAX || ncells < 0) return DG_ERANGE;
    if (!(dt >= 0.0) || !std::isfinite(dt)) return DG_EINVAL;
    if (ncells == 0) return DG_OK;
    if (!rho_g || !rho_d || !t_s || !p_in || !p_out) return DG_ENULL;
    const uintptr_t bits = reinterpret_cast<uintptr_t>(rho_g) | reinterpret_cast<uintptr_t>(rho_d) |
                           reinterpret_cast<uintptr_t>(t_s) | reinterpret_cast<uintptr_t>(p_in) |
                           reinterpret_cast<uintptr_t>(p_out);
    if (bits & 7u) return DG_EALIGN;
    // 8N + 7 doubles of staging per cell: 1 + N + N inputs, 3(N+1) momenta in, 3(N+1) momenta out.  Checked before any
    // CUDA call, so an oversized request costs nothing and touches nothing.
    const unsigned long long per_cell = 8ull * (unsigned long long)N + 7ull;
    if ((unsigned long long)ncells > (unsigned long long)kStageDoubles / per_cell) return DG_ECAPACITY;
    int device = 0;
    cudaError_t e = cudaGetDevice(&device);
    if (e != cudaSuccess) return cuda_status(e);
    if (device < 0 || device >= kMaxDevices) return DG_EINVAL;
    double* stage = nullptr;
    e = stage_address(device, &stage);
    if (e != cudaSuccess) return cuda_status(e);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    e = run(stage, rho_g, rho_d, t_s, dt, p_in, N, ncells, p_out, st);
    // Drain the stream also after a failed enqueue: no copy out of or into the caller's host buffers may still be in
    // flight when this call returns.
    const cudaError_t es = cudaStreamSynchronize(st);
    return cuda_status(e != cudaSuccess ? e : es);
}
