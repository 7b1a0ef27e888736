// Element arithmetic of the scatter-march kernel.
//
// The kernel is written once against an 8-byte element type E:
//   E = double            fp64 build, one cell per element
//   E = f2                fp32 build, TWO cells per element (cell z and cell z + nz/2 of the same
//                         (x, y) column, see layout.cuh "packed pairs"), arithmetic in packed
//                         fma.rn.f32x2 / add.rn.f32x2 / mul.rn.f32x2 (SASS FFMA2 / FADD2 / FMUL2),
//                         each lane rounded exactly like the scalar fp32 instruction.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string.h>

namespace ac {

struct f2 {
    unsigned long long v;  // low 32 bits = lane 0 (cell z), high 32 bits = lane 1 (cell z + nz/2)
};

// ---- host + device construction ----------------------------------------------------------------
template <typename E>
struct Splat;
template <>
struct Splat<double> {
    __host__ __device__ static double of(double x) { return x; }
};
template <>
struct Splat<f2> {
    __host__ __device__ static f2 of(double x) {
        const float f = (float)x;
        uint32_t b;
#ifdef __CUDA_ARCH__
        b = __float_as_uint(f);
#else
        memcpy(&b, &f, 4);
#endif
        f2 r;
        r.v = ((unsigned long long)b << 32) | (unsigned long long)b;
        return r;
    }
};

template <typename T>
struct ElemOf;
template <>
struct ElemOf<double> {
    using E = double;
    static constexpr int LANES = 1;
};
template <>
struct ElemOf<float> {
    using E = f2;
    static constexpr int LANES = 2;
};

#ifdef __CUDACC__
// ---- double ------------------------------------------------------------------------------------
__device__ __forceinline__ double vadd(double a, double b) { return a + b; }
__device__ __forceinline__ double vsub(double a, double b) { return a - b; }
__device__ __forceinline__ double vmul(double a, double b) { return a * b; }
__device__ __forceinline__ double vfma(double a, double b, double c) { return fma(a, b, c); }
__device__ __forceinline__ double vneg(double a) { return -a; }
__device__ __forceinline__ double vabs(double a) { return fabs(a); }
__device__ __forceinline__ double vexpneg(double a) { return exp(-a); }
__device__ __forceinline__ double vswap(double a) { return a; }
__device__ __forceinline__ double vmake(double lo, double) { return lo; }

// ---- packed fp32 pair --------------------------------------------------------------------------
__device__ __forceinline__ f2 vadd(f2 a, f2 b) {
    f2 r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v));
    return r;
}
__device__ __forceinline__ f2 vsub(f2 a, f2 b) {
    f2 r;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v));
    return r;
}
__device__ __forceinline__ f2 vmul(f2 a, f2 b) {
    f2 r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v));
    return r;
}
__device__ __forceinline__ f2 vfma(f2 a, f2 b, f2 c) {
    f2 r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r.v) : "l"(a.v), "l"(b.v), "l"(c.v));
    return r;
}
__device__ __forceinline__ f2 vmake(float lo, float hi) {
    f2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r.v) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void vunpack(f2 a, float& lo, float& hi) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(a.v));
}
__device__ __forceinline__ f2 vneg(f2 a) {
    f2 r;
    r.v = a.v ^ 0x8000000080000000ull;
    return r;
}
__device__ __forceinline__ f2 vabs(f2 a) {
    f2 r;
    r.v = a.v & 0x7fffffff7fffffffull;
    return r;
}
__device__ __forceinline__ f2 vexpneg(f2 a) {
    float lo, hi;
    vunpack(a, lo, hi);
    return vmake(expf(-lo), expf(-hi));
}
__device__ __forceinline__ f2 vswap(f2 a) {
    float lo, hi;
    vunpack(a, lo, hi);
    return vmake(hi, lo);
}

// load through L2 only (data another thread of the CTA has just stored)
__device__ __forceinline__ double vldcg(const double* p) { return __ldcg(p); }
__device__ __forceinline__ f2 vldcg(const f2* p) {
    f2 r;
    r.v = __ldcg(reinterpret_cast<const unsigned long long*>(p));
    return r;
}

template <typename E>
__device__ __forceinline__ E vzero() {
    return Splat<E>::of(0.0);
}
#endif  // __CUDACC__

}  // namespace ac
