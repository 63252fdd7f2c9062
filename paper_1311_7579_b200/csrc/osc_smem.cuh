// osc_smem.cuh -- explicit shared-memory accesses through 32-bit shared-window addresses.
//
// The hot loops index shared-memory tables with data-dependent offsets.  Going through generic
// pointers makes the compiler rebuild the shared-window base (S2UR + ULEA) at many uses; a 32-bit
// address obtained once with cvta and used with ld.shared / st.shared keeps the address arithmetic to a
// single integer add.  The loads are declared non-volatile: the tables they read are written once before
// a barrier; the histogram read-modify-writes use the volatile forms so that their order is preserved.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace oscb {

// A loop-invariant 32-bit value the compiler must keep in a register: without this it prefers to recompute shared-window
// addresses, lane masks and table offsets inside the event loop (a dozen integer instructions per iteration that all
// compete with the fp64 instructions for issue slots and register-file reads).
__device__ __forceinline__ uint32_t pin_u32(uint32_t v)
{
    uint32_t r;
    asm volatile("mov.u32 %0, %1;" : "=r"(r) : "r"(v));
    return r;
}

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ unsigned long long lds_u64(uint32_t a)
{
    unsigned long long v;
    asm("ld.shared.u64 %0, [%1];" : "=l"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ uint32_t lds_u16(uint32_t a)
{
    unsigned short v;
    asm("ld.shared.u16 %0, [%1];" : "=h"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ double lds_f64(uint32_t a)
{
    double v;
    asm("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ double2 lds_f64x2(uint32_t a)
{
    double2 v;
    asm("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(a));
    return v;
}
__device__ __forceinline__ double lds_f64_volatile(uint32_t a)
{
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a) : "memory");
    return v;
}
__device__ __forceinline__ void sts_f64_volatile(uint32_t a, double v)
{
    asm volatile("st.shared.f64 [%0], %1;" ::"r"(a), "d"(v) : "memory");
}

// Programmatic dependent launch (PTX griddepcontrol): the fused kernels are launched with the programmatic-stream-
// serialization attribute, so a launch may be set up -- blocks scheduled, shared memory initialised -- while the kernel
// before it on the stream is still draining; pdl_wait() returns once that kernel has completed and its memory is
// visible, and nothing before it may touch global memory.  Without the attribute, or after a kernel that never
// triggers, both are no-ops and the launch is ordered as usual.
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

} // namespace oscb
