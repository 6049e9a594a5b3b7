// mr_tmem.cuh -- Tensor Memory (TMEM, 256 KB per SM on sm_100a) used as a per-thread parking lot.
//
// The streaming step kernels are bound by registers: a node carries ~16 fp64 values from one z-plane to the next
// and the stage that forms the Jacobian / area vectors needs ~40 more registers of temporaries, so a thread that
// owns two nodes does not fit into the 128 registers that two CTAs (16 warps) per SM allow.  The tensor cores are
// idle in this stencil, and so is their 256 KB accumulator memory.  tcgen05.st / tcgen05.ld in the 32x32b shape
// move N 32-bit registers of every thread of a warp to / from N columns of the warp's own 32 TMEM lanes: a
// private, conflict-free scratchpad on a data path of its own (measured here: ~280 B/clk/SM store, >440 B/clk/SM
// load, ~45 clk load latency), which does not touch the shared-memory crossbar the stencil exchange saturates.
//
// Layout: TMEM is 128 lanes x 512 columns x 32 bit.  Warp w of a CTA may only touch lanes 32 (w % 4) .. +31; the
// warps that share a lane quarter split the CTA's columns.  Address = (lane << 16) | column.
#pragma once
#include <cstdint>

namespace mr {
namespace tmem {

// one warp allocates `NCOLS` columns (power of two >= 32) and publishes the base address through shared memory
template <int NCOLS>
__device__ __forceinline__ void alloc(uint32_t* base_in_smem)
{
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(
                     (uint32_t)__cvta_generic_to_shared(base_in_smem)),
                 "n"(NCOLS)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
template <int NCOLS>
__device__ __forceinline__ void dealloc(uint32_t base)
{
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(base), "n"(NCOLS) : "memory");
}
__device__ __forceinline__ void fence_before_sync() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void fence_after_sync() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

// 16 / 8 registers of every thread of the warp -> 16 / 8 consecutive columns (asynchronous: wait_st before re-reading)
__device__ __forceinline__ void st16(uint32_t taddr, const uint32_t (&r)[16])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};" ::"r"(taddr),
                 "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]), "r"(r[9]),
                 "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]));
}
__device__ __forceinline__ void st8(uint32_t taddr, const uint32_t (&r)[8])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"r"(taddr), "r"(r[0]), "r"(r[1]),
                 "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]));
}
__device__ __forceinline__ void st4(uint32_t taddr, const uint32_t (&r)[4])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1,%2,%3,%4};" ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]));
}
// asynchronous loads: the registers are valid only after wait_ld over the same registers
__device__ __forceinline__ void ld16(uint32_t taddr, uint32_t (&r)[16])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
                   "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
                 : "r"(taddr));
}
__device__ __forceinline__ void ld8(uint32_t taddr, uint32_t (&r)[8])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
                 : "r"(taddr));
}
__device__ __forceinline__ void ld4(uint32_t taddr, uint32_t (&r)[4])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0,%1,%2,%3}, [%4];" : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(taddr));
}
// Wait for every earlier tcgen05.ld of this thread.  The registers go through the statement as in/out operands so
// that the compiler cannot move a use of them above the wait.
__device__ __forceinline__ void wait_ld(uint32_t (&r)[16])
{
    asm volatile("tcgen05.wait::ld.sync.aligned;"
                 : "+r"(r[0]), "+r"(r[1]), "+r"(r[2]), "+r"(r[3]), "+r"(r[4]), "+r"(r[5]), "+r"(r[6]), "+r"(r[7]), "+r"(r[8]),
                   "+r"(r[9]), "+r"(r[10]), "+r"(r[11]), "+r"(r[12]), "+r"(r[13]), "+r"(r[14]), "+r"(r[15]));
}
__device__ __forceinline__ void wait_ld(uint32_t (&r)[8])
{
    asm volatile("tcgen05.wait::ld.sync.aligned;"
                 : "+r"(r[0]), "+r"(r[1]), "+r"(r[2]), "+r"(r[3]), "+r"(r[4]), "+r"(r[5]), "+r"(r[6]), "+r"(r[7]));
}
__device__ __forceinline__ void wait_ld(uint32_t (&r)[4])
{
    asm volatile("tcgen05.wait::ld.sync.aligned;" : "+r"(r[0]), "+r"(r[1]), "+r"(r[2]), "+r"(r[3]));
}
// N = 16 / 8 / 4 words by one operation
template <int N> __device__ __forceinline__ void st(uint32_t taddr, const uint32_t (&r)[N])
{
    if constexpr (N == 16) st16(taddr, r); else if constexpr (N == 8) st8(taddr, r); else st4(taddr, r);
}
template <int N> __device__ __forceinline__ void ld(uint32_t taddr, uint32_t (&r)[N])
{
    if constexpr (N == 16) ld16(taddr, r); else if constexpr (N == 8) ld8(taddr, r); else ld4(taddr, r);
}

__device__ __forceinline__ void wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

// value <-> 32-bit words (a double is a register pair: no instruction is spent on the conversion)
template <typename T> struct Words;
template <> struct Words<double> {
    static constexpr int N = 2;
    static __device__ __forceinline__ void put(uint32_t* w, double v) { w[0] = (uint32_t)__double2loint(v); w[1] = (uint32_t)__double2hiint(v); }
    static __device__ __forceinline__ double get(const uint32_t* w) { return __hiloint2double((int)w[1], (int)w[0]); }
};
template <> struct Words<float> {
    static constexpr int N = 1;
    static __device__ __forceinline__ void put(uint32_t* w, float v) { w[0] = __float_as_uint(v); }
    static __device__ __forceinline__ float get(const uint32_t* w) { return __uint_as_float(w[0]); }
};

}  // namespace tmem
}  // namespace mr
