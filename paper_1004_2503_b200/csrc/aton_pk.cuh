// Packed fp32x2 arithmetic for sm_100a (Blackwell FFMA2 / FADD2 / FMUL2: one issue slot, two fp32 lanes
// per thread).  The fused step kernel is issue-bound, not HBM-bound (profiles/r01_a_step_tiled_512.md),
// so every straight-line fp32 expression of the step is evaluated on pairs of x-adjacent cells.
// Each half is an IEEE round-to-nearest fp32 operation: results are bit-identical to the scalar form.
#pragma once
#include <cuda_runtime.h>

namespace aton {

struct f2 {
    unsigned long long v;   // {lo = cell 2p, hi = cell 2p+1}
};

__device__ __forceinline__ f2 pk(float lo, float hi) {
    f2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r.v) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ f2 splat(float s) { return pk(s, s); }
__device__ __forceinline__ float lo(f2 a) {
    float x, y;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(x), "=f"(y) : "l"(a.v));
    (void)y;
    return x;
}
__device__ __forceinline__ float hi(f2 a) {
    float x, y;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(x), "=f"(y) : "l"(a.v));
    (void)x;
    return y;
}
__device__ __forceinline__ f2 operator+(f2 a, f2 b) {
    f2 r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v));
    return r;
}
__device__ __forceinline__ f2 operator-(f2 a, f2 b) {
    f2 r;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v));
    return r;
}
__device__ __forceinline__ f2 operator*(f2 a, f2 b) {
    f2 r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v));
    return r;
}
__device__ __forceinline__ f2 fma2(f2 a, f2 b, f2 c) {   // a*b + c
    f2 r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r.v) : "l"(a.v), "l"(b.v), "l"(c.v));
    return r;
}
// scalar (broadcast) operands
__device__ __forceinline__ f2 operator*(f2 a, float s) { return a * splat(s); }
__device__ __forceinline__ f2 operator*(float s, f2 a) { return a * splat(s); }
__device__ __forceinline__ f2 operator+(f2 a, float s) { return a + splat(s); }
__device__ __forceinline__ f2 operator+(float s, f2 a) { return a + splat(s); }
__device__ __forceinline__ f2 operator-(f2 a, float s) { return a - splat(s); }
__device__ __forceinline__ f2 operator-(float s, f2 a) { return splat(s) - a; }
__device__ __forceinline__ f2 fma2(float a, f2 b, f2 c) { return fma2(splat(a), b, c); }
__device__ __forceinline__ f2 fma2(f2 a, float b, f2 c) { return fma2(a, splat(b), c); }
__device__ __forceinline__ f2 fma2(f2 a, f2 b, float c) { return fma2(a, b, splat(c)); }
__device__ __forceinline__ f2 fma2(float a, f2 b, float c) { return fma2(splat(a), b, splat(c)); }
__device__ __forceinline__ f2 fma2(f2 a, float b, float c) { return fma2(a, splat(b), splat(c)); }

// per-half scalar operations (MUFU, min/max, select have no packed form)
#define ATON_PK_MAP1(name, expr)                                   \
    __device__ __forceinline__ f2 name(f2 a) {                     \
        float x = lo(a), y = hi(a);                                \
        float rx, ry;                                              \
        { float v = x; rx = (expr); }                              \
        { float v = y; ry = (expr); }                              \
        return pk(rx, ry);                                         \
    }
__device__ __forceinline__ float m_rcp(float x) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float m_sqrt(float x) { float r; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float m_ex2(float x) { float r; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float m_lg2(float x) { float r; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
ATON_PK_MAP1(rcp2, m_rcp(v))
ATON_PK_MAP1(sqrt2, m_sqrt(v))
ATON_PK_MAP1(ex22, m_ex2(v))
ATON_PK_MAP1(lg22, m_lg2(v))
ATON_PK_MAP1(abs2, fabsf(v))
#undef ATON_PK_MAP1
__device__ __forceinline__ f2 max2(f2 a, float m) { return pk(fmaxf(lo(a), m), fmaxf(hi(a), m)); }
__device__ __forceinline__ f2 min2(f2 a, float m) { return pk(fminf(lo(a), m), fminf(hi(a), m)); }

}  // namespace aton
