// dg_async.cuh — the asynchronous global -> shared copy instructions (cp.async / LDGSTS) every kernel file stages its
// fields with, spelled once.  A thread waits for its OWN copies with cp_async_wait; data another thread copied needs a
// barrier on top.
#pragma once

namespace dg {

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

// one fp64 element (8 bytes)
__device__ __forceinline__ void cp_async8(double* dst_smem, const double* src_gmem) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"(smem_u32(dst_smem)), "l"(src_gmem) : "memory");
}
// one fp32 element (4 bytes; same name so that the kernels templated on the element type stay one source)
__device__ __forceinline__ void cp_async8(float* dst_smem, const float* src_gmem) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;\n" ::"r"(smem_u32(dst_smem)), "l"(src_gmem) : "memory");
}
// two fp64 elements (16 bytes, both sides 16-byte aligned)
__device__ __forceinline__ void cp_async16(double* dst_smem, const double* src_gmem) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(smem_u32(dst_smem)), "l"(src_gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
// waits until at most `Pending` of this thread's committed groups are still in flight
template <int Pending>
__device__ __forceinline__ void cp_async_wait() {
    asm volatile("cp.async.wait_group %0;\n" ::"n"(Pending) : "memory");
}
// commits whatever was issued and waits for everything
__device__ __forceinline__ void cp_async_wait_all() {
    asm volatile("cp.async.commit_group;\ncp.async.wait_group 0;\n" ::: "memory");
}

}  // namespace dg
