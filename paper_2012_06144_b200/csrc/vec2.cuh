// vec2.cuh -- value types for kernels that update TWO x-adjacent cells per thread.
//
// The per-cell arithmetic of lb_math.cuh / lattice.cuh is written once, generically in the element type T.  With
// T = vec2<float> every operation acts on both cells of the pair, and maps onto Blackwell's PACKED fp32 pipe: sm_100
// executes fp32 add / mul / fma on register pairs (SASS FADD2 / FMUL2 / FFMA2, CUDA intrinsics __fadd2_rn, __fmul2_rn,
// __ffma2_rn; negation and scalar broadcast are operand modifiers), i.e. one instruction per pair of cells.  The
// compiler does not form them from scalar code, so the operators below emit them explicitly; a product is kept as a
// lazy `prod2` so that  a * b + c,  c - a * b,  a * b + c * d  become ONE fused multiply-add like their scalar twins.
// T = vec2<double> is the same pairing for fp64 (plain per-component arithmetic; there is no packed fp64 pipe): it
// exists for the 16-byte-access experiment of DESIGN.md section 5.7.
#pragma once
#include <cuda_runtime.h>
#include <type_traits>

namespace acm {

using ::sqrt;      // the overloads for pairs below must not hide the scalar ones

template <typename S> struct vec2;

// ---------------------------------------------------------------------------------------------------------
// fp32 pair on the packed pipe
// ---------------------------------------------------------------------------------------------------------
template <>
struct vec2<float> {
    float2 v;
    __host__ __device__ constexpr vec2() : v{0.f, 0.f} {}
    __host__ __device__ constexpr vec2(float s) : v{s, s} {}
    __host__ __device__ constexpr vec2(double s) : v{(float)s, (float)s} {}
    __host__ __device__ constexpr vec2(int s) : v{(float)s, (float)s} {}
    __host__ __device__ constexpr vec2(float a, float b) : v{a, b} {}
    __host__ __device__ constexpr explicit vec2(float2 p) : v{p.x, p.y} {}
};
using f32x2 = vec2<float>;

struct prod2 {      // a * b, not yet evaluated
    float2 a, b;
    __device__ __forceinline__ operator f32x2() const { return f32x2(__fmul2_rn(a, b)); }
};

__device__ __forceinline__ float2 neg2(float2 a) { return make_float2(-a.x, -a.y); }      // folds into an operand modifier

__device__ __forceinline__ f32x2 operator-(f32x2 a) { return f32x2(neg2(a.v)); }
__device__ __forceinline__ prod2 operator-(prod2 p) { return prod2{neg2(p.a), p.b}; }
__device__ __forceinline__ f32x2 operator+(f32x2 a, f32x2 b) { return f32x2(__fadd2_rn(a.v, b.v)); }
__device__ __forceinline__ f32x2 operator-(f32x2 a, f32x2 b) { return f32x2(__fadd2_rn(a.v, neg2(b.v))); }
__device__ __forceinline__ prod2 operator*(f32x2 a, f32x2 b) { return prod2{a.v, b.v}; }
__device__ __forceinline__ f32x2 operator/(f32x2 a, f32x2 b) { return f32x2(a.v.x / b.v.x, a.v.y / b.v.y); }
// fused forms
__device__ __forceinline__ f32x2 operator+(prod2 p, f32x2 c) { return f32x2(__ffma2_rn(p.a, p.b, c.v)); }
__device__ __forceinline__ f32x2 operator+(f32x2 c, prod2 p) { return f32x2(__ffma2_rn(p.a, p.b, c.v)); }
__device__ __forceinline__ f32x2 operator-(prod2 p, f32x2 c) { return f32x2(__ffma2_rn(p.a, p.b, neg2(c.v))); }
__device__ __forceinline__ f32x2 operator-(f32x2 c, prod2 p) { return f32x2(__ffma2_rn(neg2(p.a), p.b, c.v)); }
__device__ __forceinline__ f32x2 operator+(prod2 p, prod2 q) { return f32x2(__ffma2_rn(p.a, p.b, __fmul2_rn(q.a, q.b))); }
__device__ __forceinline__ f32x2 operator-(prod2 p, prod2 q) { return f32x2(__ffma2_rn(neg2(q.a), q.b, __fmul2_rn(p.a, p.b))); }
__device__ __forceinline__ f32x2& operator+=(f32x2& a, f32x2 b) { a = a + b; return a; }
__device__ __forceinline__ f32x2& operator-=(f32x2& a, f32x2 b) { a = a - b; return a; }
__device__ __forceinline__ f32x2& operator+=(f32x2& a, prod2 p) { a = a + p; return a; }
__device__ __forceinline__ f32x2& operator-=(f32x2& a, prod2 p) { a = a - p; return a; }
__device__ __forceinline__ f32x2 sqrt(f32x2 a) { return f32x2(sqrtf(a.v.x), sqrtf(a.v.y)); }

// ---------------------------------------------------------------------------------------------------------
// fp64 pair (component-wise)
// ---------------------------------------------------------------------------------------------------------
template <>
struct vec2<double> {
    double2 v;
    __host__ __device__ constexpr vec2() : v{0.0, 0.0} {}
    __host__ __device__ constexpr vec2(double s) : v{s, s} {}
    __host__ __device__ constexpr vec2(int s) : v{(double)s, (double)s} {}
    __host__ __device__ constexpr vec2(double a, double b) : v{a, b} {}
    __host__ __device__ constexpr explicit vec2(double2 p) : v{p.x, p.y} {}
};
using f64x2 = vec2<double>;

__device__ __forceinline__ f64x2 operator-(f64x2 a) { return f64x2(-a.v.x, -a.v.y); }
__device__ __forceinline__ f64x2 operator+(f64x2 a, f64x2 b) { return f64x2(a.v.x + b.v.x, a.v.y + b.v.y); }
__device__ __forceinline__ f64x2 operator-(f64x2 a, f64x2 b) { return f64x2(a.v.x - b.v.x, a.v.y - b.v.y); }
__device__ __forceinline__ f64x2 operator*(f64x2 a, f64x2 b) { return f64x2(a.v.x * b.v.x, a.v.y * b.v.y); }      // nvcc contracts a * b + c
__device__ __forceinline__ f64x2 operator/(f64x2 a, f64x2 b) { return f64x2(a.v.x / b.v.x, a.v.y / b.v.y); }
__device__ __forceinline__ f64x2& operator+=(f64x2& a, f64x2 b) { a = a + b; return a; }
__device__ __forceinline__ f64x2& operator-=(f64x2& a, f64x2 b) { a = a - b; return a; }
__device__ __forceinline__ f64x2 sqrt(f64x2 a) { return f64x2(::sqrt(a.v.x), ::sqrt(a.v.y)); }

// ---------------------------------------------------------------------------------------------------------
// traits and the few operations the generic arithmetic cannot spell with operators
// ---------------------------------------------------------------------------------------------------------
template <typename T> struct scalar_of { using type = T; };
template <typename S> struct scalar_of<vec2<S>> { using type = S; };
template <typename T> using scalar_of_t = typename scalar_of<T>::type;
// the fp32 instance (single cell or pair): deviation storage and rest population by subtraction, A22
template <typename T> inline constexpr bool is_f32 = std::is_same<scalar_of_t<T>, float>::value;

// 1 / sqrt(g2) where g2 > 0, else 0 (the interface normal vanishes where grad phi vanishes exactly, reading A7)
template <typename T> __device__ __forceinline__ T inv_norm_or_zero(T g2) { return (g2 > T(0)) ? T(1) / sqrt(g2) : T(0); }
template <typename S> __device__ __forceinline__ vec2<S> inv_norm_or_zero(vec2<S> g2)
{
    return vec2<S>(inv_norm_or_zero(g2.v.x), inv_norm_or_zero(g2.v.y));
}

}  // namespace acm
