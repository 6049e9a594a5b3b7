// mr_lanes.cuh -- what one thread of the streaming mimetic kernel owns along i.
//
// fp64: one node per thread (V = double).  fp32: TWO adjacent nodes per thread, V = f2 = a packed pair of floats: the
// shared-memory accesses are 64-bit like the fp64 kernel's (half the load instructions per node) and the arithmetic
// uses Blackwell's packed fp32 pipe (add / mul / fma .f32x2 -> FADD2 / FMUL2 / FFMA2: half the math instructions per
// node).  The fp32 variant at 36 B per update is bound by instruction issue, not by HBM (profiles/r2_sym_f32_*), so
// instructions per node are what counts there.  Lanes<T> hides the difference from mr_sym.cuh: loads, stores, the
// central difference along i (the only place where the two nodes of a pair see different neighbours), per-node
// access for the rare one-sided face formulas and the reductions.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace mr {

struct __align__(8) f2 {
    float x, y;
};

__device__ __forceinline__ unsigned long long f2_bits(f2 a) { return *reinterpret_cast<unsigned long long*>(&a); }
__device__ __forceinline__ f2 f2_from(unsigned long long a) { return *reinterpret_cast<f2*>(&a); }
__device__ __forceinline__ f2 operator+(f2 a, f2 b)
{
    unsigned long long r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(f2_bits(a)), "l"(f2_bits(b)));
    return f2_from(r);
}
__device__ __forceinline__ f2 operator-(f2 a, f2 b)
{
    unsigned long long r;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(f2_bits(a)), "l"(f2_bits(b)));
    return f2_from(r);
}
__device__ __forceinline__ f2 operator*(f2 a, f2 b)
{
    unsigned long long r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(f2_bits(a)), "l"(f2_bits(b)));
    return f2_from(r);
}
using ::fma;      // (the overload below must not hide the scalar ones inside namespace mr)
__device__ __forceinline__ f2 fma(f2 a, f2 b, f2 c)
{
    unsigned long long r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(f2_bits(a)), "l"(f2_bits(b)), "l"(f2_bits(c)));
    return f2_from(r);
}
__device__ __forceinline__ f2 operator-(f2 a) { return f2{ -a.x, -a.y }; }      // (ptxas folds it into the FFMA2 operand)
__device__ __forceinline__ f2& operator+=(f2& a, f2 b) { a = a + b; return a; }

template <typename T> struct Lanes;

template <> struct Lanes<double> {
    using V = double;
    static constexpr int NV = 1;
    static __device__ __forceinline__ V ld(const double* p) { return *p; }
    static __device__ __forceinline__ void st(double* p, V v) { *p = v; }
    // central difference along i of the node(s) at p; own = ld(p)
    static __device__ __forceinline__ V di(const double* p, V) { return p[1] - p[-1]; }
    static __device__ __forceinline__ V bc(double s) { return s; }
    static __device__ __forceinline__ double get(V v, int) { return v; }
    static __device__ __forceinline__ void set(V& v, int, double s) { v = s; }
    static __device__ __forceinline__ V rcp(V d);      // defined in mr_sym.cuh (fast_rcp)
};

template <> struct Lanes<float> {
    using V = f2;
    static constexpr int NV = 2;
    static __device__ __forceinline__ V ld(const float* p) { return *reinterpret_cast<const f2*>(p); }
    static __device__ __forceinline__ void st(float* p, V v) { *reinterpret_cast<f2*>(p) = v; }
    static __device__ __forceinline__ V di(const float* p, V own)
    {
        const f2 l = ld(p - 2), r = ld(p + 2);
        return f2{ own.y - l.y, r.x - own.x };
    }
    static __device__ __forceinline__ V bc(float s) { return f2{ s, s }; }
    static __device__ __forceinline__ float get(V v, int e) { return e ? v.y : v.x; }
    static __device__ __forceinline__ void set(V& v, int e, float s) { if (e) v.y = s; else v.x = s; }
    static __device__ __forceinline__ V rcp(V d) { return f2{ __frcp_rn(d.x), __frcp_rn(d.y) }; }
};

}  // namespace mr
