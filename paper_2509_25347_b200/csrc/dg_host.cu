// dg_host.cu — dg_drag_update_host (include/dg.h): the fused update on HOST buffers.
//
// The cells are cut into chunks; each chunk's field rows are copied with one strided 2-D copy per array into a
// compact device staging slot, the fused kernel runs on the slot, and the result rows are copied back.  Three slots
// with a stream each keep the H2D copy of chunk k+1, the kernel of chunk k and the D2H copy of chunk k-1 in flight
// together (the GPU has separate copy engines per direction).  No arithmetic here: the kernel is the one
// dg_drag_update launches.
#include <atomic>
#include <cmath>
#include <cstdint>
#include <mutex>

#include "../../include/dg.h"
#include "dg_internal.h"

namespace dg {
dg_status cuda_status(cudaError_t e);
cudaError_t launch_update(int N, int variant, const UpdateArgs& a, cudaStream_t st);

namespace {

constexpr int kSlots = 3;
constexpr int kMaxDevices = 64;
constexpr long long kDefaultChunk = 1LL << 19;

struct Slot {
    cudaStream_t stream = nullptr;
    double* buf = nullptr;
    size_t cap = 0;  // bytes
};
struct Ctx {
    bool streams = false;
    size_t max_pitch = 0;  // cudaDevAttrMaxPitch: the largest row pitch a 2-D copy accepts
    Slot slot[kSlots];
    std::mutex mu;         // one caller at a time per device; callers on different devices do not wait for each other
};
Ctx g_ctx[kMaxDevices];
std::atomic<size_t> g_pitch_cap{0};  // dg_host_set_max_pitch: 0 = the device's own limit

#define DG_TRY(x)                           \
    do {                                    \
        cudaError_t e_ = (x);               \
        if (e_ != cudaSuccess) return e_;   \
    } while (0)

cudaError_t ensure(Ctx& c, int device, size_t bytes) {
    if (!c.streams) {
        int mp = 0;
        DG_TRY(cudaDeviceGetAttribute(&mp, cudaDevAttrMaxPitch, device));
        c.max_pitch = (size_t)(mp > 0 ? mp : 0);
        for (int k = 0; k < kSlots; ++k) DG_TRY(cudaStreamCreateWithFlags(&c.slot[k].stream, cudaStreamNonBlocking));
        c.streams = true;
    }
    for (int k = 0; k < kSlots; ++k) {
        Slot& s = c.slot[k];
        if (s.cap >= bytes) continue;
        DG_TRY(cudaStreamSynchronize(s.stream));
        if (s.buf) DG_TRY(cudaFree(s.buf));
        s.buf = nullptr;
        s.cap = 0;
        DG_TRY(cudaMalloc(&s.buf, bytes));
        s.cap = bytes;
    }
    return cudaSuccess;
}

// `rows` rows of `width` bytes between a pitched host array and a compact device slot: one strided 2-D copy, or one 1-D
// copy per row when the host pitch (ncells * 8 bytes) exceeds what a 2-D copy accepts (2^31 - 1 bytes: ncells >= 2^28).
cudaError_t copy_rows(const Ctx& c, void* dst, size_t dpitch, const void* src, size_t spitch, size_t width, size_t rows,
                      cudaMemcpyKind kind, cudaStream_t st) {
    // (dg_host_set_max_pitch lowers the limit: the tests use it to reach the per-row path at small sizes)
    size_t limit = c.max_pitch;
    const size_t cap = g_pitch_cap.load(std::memory_order_relaxed);
    if (cap != 0 && cap < limit) limit = cap;
    if (dpitch <= limit && spitch <= limit) return cudaMemcpy2DAsync(dst, dpitch, src, spitch, width, rows, kind, st);
    for (size_t r = 0; r < rows; ++r)
        DG_TRY(cudaMemcpyAsync(static_cast<char*>(dst) + r * dpitch, static_cast<const char*>(src) + r * spitch, width, kind, st));
    return cudaSuccess;
}

cudaError_t enqueue(Ctx& c, const double* rho_g, const double* rho_d, const double* t_s, double dt, const double* p_in,
                    int N, long long ncells, double* p_out, long long chunk) {
    const int n = N + 1;
    const size_t hpitch = (size_t)ncells * sizeof(double);
    int k = 0;
    for (long long c0 = 0; c0 < ncells; c0 += chunk, k = (k + 1) % kSlots) {
        const long long cc = (ncells - c0 < chunk) ? ncells - c0 : chunk;
        Slot& s = c.slot[k];
        const size_t w = (size_t)cc * sizeof(double);
        double* d_rho_g = s.buf;
        double* d_rho_d = d_rho_g + cc;
        double* d_t_s = d_rho_d + (size_t)N * cc;
        double* d_p_in = d_t_s + (size_t)N * cc;
        double* d_p_out = d_p_in + (size_t)3 * n * cc;
        DG_TRY(cudaMemcpyAsync(d_rho_g, rho_g + c0, w, cudaMemcpyHostToDevice, s.stream));
        DG_TRY(copy_rows(c, d_rho_d, w, rho_d + c0, hpitch, w, (size_t)N, cudaMemcpyHostToDevice, s.stream));
        DG_TRY(copy_rows(c, d_t_s, w, t_s + c0, hpitch, w, (size_t)N, cudaMemcpyHostToDevice, s.stream));
        DG_TRY(copy_rows(c, d_p_in, w, p_in + c0, hpitch, w, (size_t)3 * n, cudaMemcpyHostToDevice, s.stream));
        UpdateArgs a{d_rho_g, d_rho_d, d_t_s, dt, d_p_in, cc, d_p_out, nullptr, nullptr};
        DG_TRY(launch_update(N, DG_VARIANT_DEFAULT, a, s.stream));
        DG_TRY(copy_rows(c, p_out + c0, hpitch, d_p_out, w, w, (size_t)3 * n, cudaMemcpyDeviceToHost, s.stream));
    }
    return cudaSuccess;
}

cudaError_t run(Ctx& c, int device, const double* rho_g, const double* rho_d, const double* t_s, double dt,
                const double* p_in, int N, long long ncells, double* p_out, long long chunk) {
    const int n = N + 1;
    const size_t doubles_per_cell = (size_t)(1 + 2 * N + 3 * n + 3 * n);
    DG_TRY(ensure(c, device, doubles_per_cell * (size_t)chunk * sizeof(double)));
    const cudaError_t e = enqueue(c, rho_g, rho_d, t_s, dt, p_in, N, ncells, p_out, chunk);
    // Always drain the three streams, also after a failed enqueue: no copy into or out of the caller's host buffers may
    // still be in flight when this call returns.
    cudaError_t first = e;
    for (int j = 0; j < kSlots; ++j) {
        const cudaError_t es = cudaStreamSynchronize(c.slot[j].stream);
        if (first == cudaSuccess) first = es;
    }
    return first;
}

}  // namespace
}  // namespace dg

using namespace dg;

extern "C" dg_status dg_drag_update_host(const double* rho_g, const double* rho_d, const double* t_s, double dt,
                                         const double* p_in, int N, long long ncells, double* p_out,
                                         long long chunk_cells, int device) {
    if (N < 1 || N > DG_NMAX || ncells < 0) return DG_ERANGE;
    if (!(dt >= 0.0) || !std::isfinite(dt) || chunk_cells < 0) return DG_EINVAL;
    if (ncells == 0) return DG_OK;
    if (!rho_g || !rho_d || !t_s || !p_in || !p_out) return DG_ENULL;
    const uintptr_t bits = reinterpret_cast<uintptr_t>(rho_g) | reinterpret_cast<uintptr_t>(rho_d) |
                           reinterpret_cast<uintptr_t>(t_s) | reinterpret_cast<uintptr_t>(p_in) |
                           reinterpret_cast<uintptr_t>(p_out);
    if (bits & 7u) return DG_EALIGN;
    int prev = 0;
    cudaError_t e = cudaGetDevice(&prev);
    if (e != cudaSuccess) return cuda_status(e);
    if (device < 0) device = prev;
    if (device >= kMaxDevices) return DG_EINVAL;
    std::lock_guard<std::mutex> lock(g_ctx[device].mu);  // the staging slots of this device have one user at a time
    if (device != prev) {
        e = cudaSetDevice(device);
        if (e != cudaSuccess) return cuda_status(e);
    }
    // Chunks are whole multiples of 2048 cells: the kernels take one decision (the Taylor degree) per group of cells that
    // share a warp — 32 (or 16) cells of a stiffness-sorted tile of 128 or 256 consecutive cells — so every chunk must
    // start on a tile boundary of a single launch over all cells for the two entry points to agree bit for bit; it also
    // keeps every staged row 16 KiB-aligned (bulk copies need 16 bytes).
    long long chunk = chunk_cells > 0 ? chunk_cells : kDefaultChunk;
    chunk = (chunk + 2047) & ~2047LL;
    if (chunk > ncells) chunk = ncells;
    e = run(g_ctx[device], device, rho_g, rho_d, t_s, dt, p_in, N, ncells, p_out, chunk);
    if (device != prev) cudaSetDevice(prev);
    return cuda_status(e);
}

extern "C" dg_status dg_host_release(void) {
    int prev = 0;
    if (cudaGetDevice(&prev) != cudaSuccess) return DG_OK;  // no CUDA context: nothing was ever allocated
    cudaError_t first = cudaSuccess;
    for (int d = 0; d < kMaxDevices; ++d) {
        Ctx& c = g_ctx[d];
        std::lock_guard<std::mutex> lock(c.mu);
        if (!c.streams) continue;
        cudaSetDevice(d);
        for (int k = 0; k < kSlots; ++k) {
            Slot& s = c.slot[k];
            cudaError_t e = cudaStreamSynchronize(s.stream);
            if (s.buf) e = cudaFree(s.buf);
            cudaStreamDestroy(s.stream);
            if (e != cudaSuccess && first == cudaSuccess) first = e;
            s = Slot();
        }
        c.streams = false;
    }
    cudaSetDevice(prev);
    return cuda_status(first);
}

extern "C" dg_status dg_host_set_max_pitch(long long bytes) {
    if (bytes < 0) return DG_EINVAL;
    g_pitch_cap.store((size_t)bytes, std::memory_order_relaxed);
    return DG_OK;
}
