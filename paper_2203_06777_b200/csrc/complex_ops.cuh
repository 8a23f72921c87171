// complex_ops.cuh -- complex arithmetic on (re, im) register pairs for the Dhop kernels.
//
// fp32: the packed f32x2 PTX instructions of sm_100 (add/mul/fma.rn.f32x2 -> SASS FADD2 / FMUL2 /
// FFMA2) on 64-bit register pairs.  FFMA2 takes a 32-bit register broadcast to both halves and a
// HI/LO swap as free operand modifiers, FADD2 also a per-half negation.  The direct kernel
// (dhop.cu) keeps a complex number (re, im) in a pair; the staged kernel (dhop_staged.cu) keeps
// one real part of two spin components in a pair.  Each lane is an IEEE round-to-nearest
// operation, so the results are the ones scalar fmaf / + / * would give.
// fp64: plain DFMA / DADD on double2.
#pragma once
#include <cuda_runtime.h>

namespace dwf {

template <typename T> struct CxT;
template <> struct CxT<float>  { using type = float2;  };
template <> struct CxT<double> { using type = double2; };

// ---- packed fp32 primitives -------------------------------------------------------------------
__device__ __forceinline__ float2 f2_fma(float2 a, float2 b, float2 c)
{
    float2 d;
    asm("{\n\t.reg .b64 ra, rb, rc, rd;\n\t"
        "mov.b64 ra, {%2, %3};\n\tmov.b64 rb, {%4, %5};\n\tmov.b64 rc, {%6, %7};\n\t"
        "fma.rn.f32x2 rd, ra, rb, rc;\n\t"
        "mov.b64 {%0, %1}, rd;\n\t}"
        : "=f"(d.x), "=f"(d.y)
        : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y), "f"(c.x), "f"(c.y));
    return d;
}
__device__ __forceinline__ float2 f2_mul(float2 a, float2 b)
{
    float2 d;
    asm("{\n\t.reg .b64 ra, rb, rd;\n\t"
        "mov.b64 ra, {%2, %3};\n\tmov.b64 rb, {%4, %5};\n\t"
        "mul.rn.f32x2 rd, ra, rb;\n\t"
        "mov.b64 {%0, %1}, rd;\n\t}"
        : "=f"(d.x), "=f"(d.y)
        : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
    return d;
}
__device__ __forceinline__ float2 f2_add(float2 a, float2 b)
{
    float2 d;
    asm("{\n\t.reg .b64 ra, rb, rd;\n\t"
        "mov.b64 ra, {%2, %3};\n\tmov.b64 rb, {%4, %5};\n\t"
        "add.rn.f32x2 rd, ra, rb;\n\t"
        "mov.b64 {%0, %1}, rd;\n\t}"
        : "=f"(d.x), "=f"(d.y)
        : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
    return d;
}

// ---- complex ops, fp32 ------------------------------------------------------------------------
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return f2_add(a, b); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return f2_add(a, make_float2(-b.x, -b.y)); }
// a + i*b and a - i*b
__device__ __forceinline__ float2 caddi(float2 a, float2 b) { return f2_add(a, make_float2(-b.y, b.x)); }
__device__ __forceinline__ float2 csubi(float2 a, float2 b) { return f2_add(a, make_float2(b.y, -b.x)); }
__device__ __forceinline__ float2 cmul(float2 u, float2 h)
{
    float2 t = f2_mul(make_float2(u.x, u.x), h);
    return f2_fma(make_float2(u.y, u.y), make_float2(-h.y, h.x), t);
}
__device__ __forceinline__ float2 cmac(float2 acc, float2 u, float2 h)
{
    float2 t = f2_fma(make_float2(u.x, u.x), h, acc);
    return f2_fma(make_float2(u.y, u.y), make_float2(-h.y, h.x), t);
}

// ---- complex ops, fp64 ------------------------------------------------------------------------
__device__ __forceinline__ double2 cadd(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ double2 csub(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ double2 caddi(double2 a, double2 b) { return make_double2(a.x - b.y, a.y + b.x); }
__device__ __forceinline__ double2 csubi(double2 a, double2 b) { return make_double2(a.x + b.y, a.y - b.x); }
__device__ __forceinline__ double2 cmul(double2 u, double2 h)
{
    return make_double2(fma(-u.y, h.y, u.x * h.x), fma(u.y, h.x, u.x * h.y));
}
__device__ __forceinline__ double2 cmac(double2 acc, double2 u, double2 h)
{
    return make_double2(fma(-u.y, h.y, fma(u.x, h.x, acc.x)), fma(u.y, h.x, fma(u.x, h.y, acc.y)));
}

// i*x, -i*x, -x (register moves with sign flips; used once per site on the first leg)
template <typename C> __device__ __forceinline__ C cmuli(C x)  { C r; r.x = -x.y; r.y = x.x;  return r; }
template <typename C> __device__ __forceinline__ C cmulni(C x) { C r; r.x = x.y;  r.y = -x.x; return r; }
template <typename C> __device__ __forceinline__ C cneg(C x)   { C r; r.x = -x.x; r.y = -x.y; return r; }

// ---- 128-bit vector access to Sc consecutive complex numbers ------------------------------------
// default-cached read-only loads (input spinors are re-read by neighbouring sites: keep in L1/L2)
template <int SC> __device__ __forceinline__ void load_cx(const float2 *p, float2 (&v)[SC])
{
    if constexpr (SC == 1) {
        v[0] = __ldg(p);
    } else {
        static_assert(SC % 2 == 0, "SC must be 1 or even");
#pragma unroll
        for (int i = 0; i < SC / 2; i++) {
            float4 q = __ldg(reinterpret_cast<const float4 *>(p) + i);
            v[2 * i] = make_float2(q.x, q.y);
            v[2 * i + 1] = make_float2(q.z, q.w);
        }
    }
}
template <int SC> __device__ __forceinline__ void load_cx(const double2 *p, double2 (&v)[SC])
{
#pragma unroll
    for (int i = 0; i < SC; i++) v[i] = __ldg(p + i);
}
// streaming stores (the output is not re-read by this kernel: do not let it displace inputs)
template <int SC> __device__ __forceinline__ void store_cx(float2 *p, const float2 (&v)[SC])
{
    if constexpr (SC == 1) {
        __stcs(p, v[0]);
    } else {
#pragma unroll
        for (int i = 0; i < SC / 2; i++)
            __stcs(reinterpret_cast<float4 *>(p) + i,
                   make_float4(v[2 * i].x, v[2 * i].y, v[2 * i + 1].x, v[2 * i + 1].y));
    }
}
template <int SC> __device__ __forceinline__ void store_cx(double2 *p, const double2 (&v)[SC])
{
#pragma unroll
    for (int i = 0; i < SC; i++) __stcs(p + i, v[i]);
}

}  // namespace dwf
