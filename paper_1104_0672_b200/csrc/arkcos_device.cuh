// Device-side helpers shared by the kernels of libarkcos (complex arithmetic, exact-phase twiddles).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace arkcos {

template <class T> struct __align__(2 * sizeof(T)) cx { T x, y; };   // complex (re, im), naturally aligned: one 64/128-bit access

template <class T> __host__ __device__ __forceinline__ cx<T> mk(T a, T b) { cx<T> r; r.x = a; r.y = b; return r; }
template <class T> __device__ __forceinline__ cx<T> operator+(cx<T> a, cx<T> b) { return mk<T>(a.x + b.x, a.y + b.y); }
template <class T> __device__ __forceinline__ cx<T> operator-(cx<T> a, cx<T> b) { return mk<T>(a.x - b.x, a.y - b.y); }
template <class T> __device__ __forceinline__ cx<T> cmul(cx<T> a, cx<T> b)
{
    return mk<T>(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
template <class T> __device__ __forceinline__ cx<T> cmulc(cx<T> a, cx<T> b)   // a * conj(b)
{
    return mk<T>(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y);
}
template <class T> __device__ __forceinline__ cx<T> cconj(cx<T> a) { return mk<T>(a.x, -a.y); }
template <class T> __device__ __forceinline__ cx<T> cscale(cx<T> a, T s) { return mk<T>(a.x * s, a.y * s); }

__device__ __forceinline__ void sincospi_t(float x, float* s, float* c) { sincospif(x, s, c); }
__device__ __forceinline__ void sincospi_t(double x, double* s, double* c) { sincospi(x, s, c); }

// exp(i * pi * num / den) for integers 0 <= num < 2 den, den >= 1.  The argument is reduced to the first octant with
// integer arithmetic, so the result is accurate to about one ulp of T whatever the size of num and den.
template <class T> __device__ __forceinline__ cx<T> cispi_ratio(uint32_t num, uint32_t den)
{
    bool neg = num >= den;                  // e^{i (pi + a)} = -e^{i a}
    if (neg) num -= den;
    bool refl = 2u * num > den;             // a -> pi - a
    if (refl) num = den - num;
    bool swp = 4u * num > den;              // a -> pi/2 - a
    uint32_t rr = swp ? (den - 2u * num) : 2u * num;       // angle = pi * rr / (2 den), rr / (2 den) in [0, 1/4]
    T s, c;
    sincospi_t((T)rr / (T)(2u * den), &s, &c);
    if (swp) { T t = s; s = c; c = t; }
    if (refl) c = -c;
    if (neg) { c = -c; s = -s; }
    return mk<T>(c, s);
}

// Packed FP32 FMA of sm_100 (SASS FFMA2): two fused multiply-adds in one issue slot, d = a * b + c per component.
__device__ __forceinline__ float2 ffma2(float2 a, float2 b, float2 c)
{
    unsigned long long ra, rb, rc, rd;
    asm("mov.b64 %0, {%1, %2};" : "=l"(ra) : "f"(a.x), "f"(a.y));
    asm("mov.b64 %0, {%1, %2};" : "=l"(rb) : "f"(b.x), "f"(b.y));
    asm("mov.b64 %0, {%1, %2};" : "=l"(rc) : "f"(c.x), "f"(c.y));
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(rd) : "l"(ra), "l"(rb), "l"(rc));
    float2 d;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(d.x), "=f"(d.y) : "l"(rd));
    return d;
}

// cp.async (LDGSTS) of 8 bytes global -> shared, and its group bookkeeping
__device__ __forceinline__ void cp_async8(void* smem_dst, const void* gsrc)
{
    const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc)
{
    const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// gamma = 2 asin(sqrt(x) / 2) from the squared chord x = 2 - 2 cos(gamma) (Eq. 9).  Compact kernels only see small
// arguments: Maclaurin series of asin (10 terms, truncation < 1e-18 relative for sqrt(x)/2 < 1/8) instead of the library asin.
__device__ __forceinline__ double gamma_of_chord2(double x)
{
    double hx = 0.5 * sqrt(x);
    if (hx > 1.0) hx = 1.0;
    if (hx < 0.125) {
        const double q = hx * hx;
        double p = 34459425.0 / 3530096640.0;
        p = p * q + 2027025.0 / 175472640.0;
        p = p * q + 135135.0 / 9676800.0;
        p = p * q + 10395.0 / 599040.0;
        p = p * q + 945.0 / 42240.0;
        p = p * q + 105.0 / 3456.0;
        p = p * q + 15.0 / 336.0;
        p = p * q + 3.0 / 40.0;
        p = p * q + 1.0 / 6.0;
        return 2.0 * (hx + hx * q * p);
    }
    return 2.0 * asin(hx);
}

}  // namespace arkcos
