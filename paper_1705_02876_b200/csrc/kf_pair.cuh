// kf_pair.cuh -- f2: two tracks per thread in one packed register pair (sm_100a FFMA2 / FMUL2 / FADD2).
//
// Blackwell issues one packed fp32x2 instruction for two fused multiply-adds.  The fit kernel is bound by
// instruction issue, not by the FMA pipes (profiles/r01_fit_kernel.md: issue 81 %, fma pipe 59 %), so the
// pair kernel gives each thread TWO tracks, component x = even track, y = odd track of a 64-track tile,
// and runs the same arithmetic (kf_math.cuh is written once, on a number type F = float or kf::f2).
//
// f2 carries the operators the math uses.  A product is a lazy `prod2` so that a*b + c contracts into one
// FFMA2 the way nvcc contracts the scalar expression into FFMA; a product used on its own is one FMUL2.
// mask2 is the per-component truth value of a comparison; status and other integer bookkeeping stay scalar
// per component (u2).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace kf {

struct f2 {
    float2 v;
    __device__ __forceinline__ f2() {}
    __device__ __forceinline__ f2(float2 a) : v(a) {}
    __device__ __forceinline__ f2(float a) : v(make_float2(a, a)) {}          // broadcast
    __device__ __forceinline__ f2(float a, float b) : v(make_float2(a, b)) {}
};

struct mask2 {
    bool x, y;
};
__device__ __forceinline__ mask2 operator&(mask2 a, mask2 b) { return {a.x && b.x, a.y && b.y}; }
__device__ __forceinline__ mask2 operator|(mask2 a, mask2 b) { return {a.x || b.x, a.y || b.y}; }
__device__ __forceinline__ mask2 operator!(mask2 a) { return {!a.x, !a.y}; }
__device__ __forceinline__ bool none_of(mask2 a) { return !a.x && !a.y; }
__device__ __forceinline__ bool all_of(mask2 a) { return a.x && a.y; }
__device__ __forceinline__ bool none_of(bool a) { return !a; }
__device__ __forceinline__ bool all_of(bool a) { return a; }

struct u2 {
    uint32_t x, y;
};

namespace pair_detail {
__device__ __forceinline__ float2 neg(float2 a) { return make_float2(-a.x, -a.y); }
}  // namespace pair_detail

// a * b, not yet rounded: becomes the multiplicand pair of an FFMA2 or, alone, an FMUL2.
struct prod2 {
    float2 a, b;
    __device__ __forceinline__ operator f2() const { return f2(__fmul2_rn(a, b)); }
};

// ---- products
__device__ __forceinline__ prod2 operator*(f2 a, f2 b) { return {a.v, b.v}; }
__device__ __forceinline__ prod2 operator*(float a, f2 b) { return {make_float2(a, a), b.v}; }
__device__ __forceinline__ prod2 operator*(f2 a, float b) { return {a.v, make_float2(b, b)}; }
__device__ __forceinline__ prod2 operator*(prod2 p, f2 b) { return {__fmul2_rn(p.a, p.b), b.v}; }
__device__ __forceinline__ prod2 operator*(f2 a, prod2 p) { return {a.v, __fmul2_rn(p.a, p.b)}; }
__device__ __forceinline__ prod2 operator*(prod2 p, float b) { return {__fmul2_rn(p.a, p.b), make_float2(b, b)}; }
__device__ __forceinline__ prod2 operator*(float a, prod2 p) { return {make_float2(a, a), __fmul2_rn(p.a, p.b)}; }
__device__ __forceinline__ prod2 operator*(prod2 p, prod2 q) { return {__fmul2_rn(p.a, p.b), __fmul2_rn(q.a, q.b)}; }
__device__ __forceinline__ prod2 operator-(prod2 p) { return {pair_detail::neg(p.a), p.b}; }
__device__ __forceinline__ f2 operator-(f2 a) { return f2(pair_detail::neg(a.v)); }

// ---- sums (every one is a single packed instruction; subtraction folds the sign into an operand)
__device__ __forceinline__ f2 operator+(f2 a, f2 b) { return f2(__fadd2_rn(a.v, b.v)); }
__device__ __forceinline__ f2 operator-(f2 a, f2 b) { return f2(__fadd2_rn(a.v, pair_detail::neg(b.v))); }
__device__ __forceinline__ f2 operator+(f2 a, float b) { return f2(__fadd2_rn(a.v, make_float2(b, b))); }
__device__ __forceinline__ f2 operator+(float a, f2 b) { return f2(__fadd2_rn(make_float2(a, a), b.v)); }
__device__ __forceinline__ f2 operator-(f2 a, float b) { return f2(__fadd2_rn(a.v, make_float2(-b, -b))); }
__device__ __forceinline__ f2 operator-(float a, f2 b) { return f2(__fadd2_rn(make_float2(a, a), pair_detail::neg(b.v))); }
__device__ __forceinline__ f2 operator+(prod2 p, f2 c) { return f2(__ffma2_rn(p.a, p.b, c.v)); }
__device__ __forceinline__ f2 operator+(f2 c, prod2 p) { return f2(__ffma2_rn(p.a, p.b, c.v)); }
__device__ __forceinline__ f2 operator-(prod2 p, f2 c) { return f2(__ffma2_rn(p.a, p.b, pair_detail::neg(c.v))); }
__device__ __forceinline__ f2 operator-(f2 c, prod2 p) { return f2(__ffma2_rn(pair_detail::neg(p.a), p.b, c.v)); }
__device__ __forceinline__ f2 operator+(prod2 p, float c) { return f2(__ffma2_rn(p.a, p.b, make_float2(c, c))); }
__device__ __forceinline__ f2 operator+(float c, prod2 p) { return f2(__ffma2_rn(p.a, p.b, make_float2(c, c))); }
__device__ __forceinline__ f2 operator-(prod2 p, float c) { return f2(__ffma2_rn(p.a, p.b, make_float2(-c, -c))); }
__device__ __forceinline__ f2 operator-(float c, prod2 p) { return f2(__ffma2_rn(pair_detail::neg(p.a), p.b, make_float2(c, c))); }
__device__ __forceinline__ f2 operator+(prod2 p, prod2 q) { return f2(__ffma2_rn(p.a, p.b, __fmul2_rn(q.a, q.b))); }
__device__ __forceinline__ f2 operator-(prod2 p, prod2 q) { return f2(__ffma2_rn(pair_detail::neg(q.a), q.b, __fmul2_rn(p.a, p.b))); }
__device__ __forceinline__ f2& operator+=(f2& a, f2 b) { a = a + b; return a; }
__device__ __forceinline__ f2& operator+=(f2& a, prod2 p) { a = a + p; return a; }
__device__ __forceinline__ f2& operator-=(f2& a, f2 b) { a = a - b; return a; }
__device__ __forceinline__ f2& operator-=(f2& a, prod2 p) { a = a - p; return a; }
__device__ __forceinline__ f2& operator*=(f2& a, f2 b) { a = a * b; return a; }
__device__ __forceinline__ f2& operator*=(f2& a, float b) { a = a * b; return a; }

// ---- comparisons against a scalar or component-wise
__device__ __forceinline__ mask2 operator>(f2 a, float b) { return {a.v.x > b, a.v.y > b}; }
__device__ __forceinline__ mask2 operator<(f2 a, float b) { return {a.v.x < b, a.v.y < b}; }
__device__ __forceinline__ mask2 operator>(f2 a, f2 b) { return {a.v.x > b.v.x, a.v.y > b.v.y}; }
__device__ __forceinline__ mask2 operator<(f2 a, f2 b) { return {a.v.x < b.v.x, a.v.y < b.v.y}; }
__device__ __forceinline__ mask2 operator>(prod2 p, float b) { return f2(p) > b; }
__device__ __forceinline__ mask2 operator>(float a, f2 b) { return {a > b.v.x, a > b.v.y}; }
__device__ __forceinline__ mask2 operator<(float a, f2 b) { return {a < b.v.x, a < b.v.y}; }

// ---- the few non-arithmetic functions the math needs, on both number types
__device__ __forceinline__ float fma_(float a, float b, float c) { return fmaf(a, b, c); }
__device__ __forceinline__ f2 fma_(f2 a, f2 b, f2 c) { return f2(__ffma2_rn(a.v, b.v, c.v)); }
__device__ __forceinline__ float abs_(float a) { return fabsf(a); }
__device__ __forceinline__ f2 abs_(f2 a) { return f2(fabsf(a.v.x), fabsf(a.v.y)); }
__device__ __forceinline__ float atan_(float a) { return atanf(a); }
// atan of a pair: while both arguments are below tan(pi/8) (a helix step that turns less than 45 degrees, i.e.
// every step of a track that is not about to loop) one packed odd polynomial, atan x = x + x z g(z), z = x^2,
// g of degree 3 fitted to (atan x / x - 1) / z over z in [0, tan^2(pi/8)] (weighted least squares on 4000
// Chebyshev nodes, Lawson-reweighted towards minimax); 7.9e-8 maximum relative error evaluated in fp32.
__device__ __forceinline__ f2 atan_(f2 a) {
    constexpr float kLim = 0.41421354f;
    if (fabsf(a.v.x) < kLim && fabsf(a.v.y) < kLim) {
        const f2 z = a * a;
        f2 g = fma_(f2(0.08053719252347946f), z, f2(-0.1387767791748047f));
        g = fma_(g, z, f2(0.19977709650993347f));
        g = fma_(g, z, f2(-0.3333294987678528f));
        return a + (a * z) * g;
    }
    return f2(atanf(a.v.x), atanf(a.v.y));
}
__device__ __forceinline__ float sqrt_(float a) { return sqrtf(a); }
__device__ __forceinline__ f2 sqrt_(f2 a) { return f2(sqrtf(a.v.x), sqrtf(a.v.y)); }
__device__ __forceinline__ float log_fast(float a) { return __logf(a); }
__device__ __forceinline__ f2 log_fast(f2 a) { return f2(__logf(a.v.x), __logf(a.v.y)); }
__device__ __forceinline__ float rsqrt_ieee(float a) { return rsqrtf(a); }
__device__ __forceinline__ f2 rsqrt_ieee(f2 a) { return f2(rsqrtf(a.v.x), rsqrtf(a.v.y)); }
__device__ __forceinline__ float select(bool m, float a, float b) { return m ? a : b; }
__device__ __forceinline__ f2 select(mask2 m, f2 a, f2 b) { return f2(m.x ? a.v.x : b.v.x, m.y ? a.v.y : b.v.y); }
__device__ __forceinline__ uint32_t select_u(bool m, uint32_t a, uint32_t b) { return m ? a : b; }
__device__ __forceinline__ u2 select_u(mask2 m, uint32_t a, uint32_t b) { return {m.x ? a : b, m.y ? a : b}; }
__device__ __forceinline__ u2 select_u(mask2 m, uint32_t a, u2 b) { return {m.x ? a : b.x, m.y ? a : b.y}; }

__device__ __forceinline__ bool is_zero(uint32_t a) { return a == 0u; }
__device__ __forceinline__ bool is_zero(u2 a) { return (a.x | a.y) == 0u; }

// number-type traits: the mask and status types that go with F
template <class F> struct num_traits;
template <> struct num_traits<float> { using mask = bool; using status = uint32_t; };
template <> struct num_traits<f2> { using mask = mask2; using status = u2; };

// a parameter of type F that takes no part in template argument deduction (so that a literal, a float or
// a lazy product can be passed where the track's number type is f2)
template <class T> struct same_as { using type = T; };
template <class T> using arg = typename same_as<T>::type;

}  // namespace kf
