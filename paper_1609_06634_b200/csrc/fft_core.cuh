// fft_core.cuh -- register-resident radix-2 DIF FFT of N1 in {4, 8, 16, 32} points, templated on the scalar
// type (float for the hot path, double for the precompute / re-scoring path) and on the sign of the exponent.
// Building block of the "two-step" transform used everywhere in this library:
//     N = N1 * N2,   m = N2*j + t,   y[k] = sum_t w_N^{t k} Z_t[k mod N1],   Z_t[k1] = sum_j x[N2 j + t] w_N1^{j k1}
// step 1 (this file) runs per thread in registers; step 2 is a short direct sum that is naturally
// output-pruned (only the |k| <= D outputs of Eqs. 11-12, are ever formed).
#pragma once
#include <cuda_runtime.h>

namespace bioem {

// aligned to its own size, so that a complex number moves as ONE 64-bit (float) or 128-bit (double) access: without the
// attribute every complex load compiled to two scalar loads (the Q loads of the fused kernels, the FP64 transforms, a7)
template <typename T> struct alignas(2 * sizeof(T)) cx { T x, y; };

template <typename T> __device__ __forceinline__ cx<T> cmul(cx<T> a, cx<T> b) { return {a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x}; }
template <typename T> __device__ __forceinline__ cx<T> cmulc(cx<T> a, cx<T> b) { /* conj(a) * b */ return {a.x * b.x + a.y * b.y, a.x * b.y - a.y * b.x}; }
template <typename T> __device__ __forceinline__ cx<T> cadd(cx<T> a, cx<T> b) { return {a.x + b.x, a.y + b.y}; }
template <typename T> __device__ __forceinline__ cx<T> csub(cx<T> a, cx<T> b) { return {a.x - b.x, a.y - b.y}; }

// cos(2 pi k / 32), k = 0..8
__device__ __forceinline__ constexpr double cos32(int k)
{
    constexpr double t[9] = {1.0, 0.9807852804032304, 0.9238795325112867, 0.8314696123025452, 0.7071067811865476,
                             0.5555702330196023, 0.38268343236508984, 0.19509032201612833, 0.0};
    return t[k];
}

// a *= exp(SIGN * 2 pi i * K32 / 32), 0 <= K32 < 16, K32 a compile-time constant after unrolling.
template <typename T, int SIGN>
__device__ __forceinline__ void twiddle32(cx<T> &a, int K32)
{
    if (K32 == 0) return;
    if (K32 == 8) {                       // +-i
        T t = a.x;
        if (SIGN > 0) { a.x = -a.y; a.y = t; } else { a.x = a.y; a.y = -t; }
        return;
    }
    if (K32 == 4 || K32 == 12) {          // (+-1 +- i)/sqrt2
        const T c = (T)0.7071067811865476;
        T re, im;
        if (K32 == 4) { if (SIGN > 0) { re = a.x - a.y; im = a.x + a.y; } else { re = a.x + a.y; im = a.y - a.x; } }
        else          { if (SIGN > 0) { re = -a.x - a.y; im = a.x - a.y; } else { re = a.y - a.x; im = -a.x - a.y; } }
        a.x = re * c; a.y = im * c;
        return;
    }
    T c, s;
    if (K32 < 8) { c = (T)cos32(K32); s = (T)cos32(8 - K32); }
    else         { c = -(T)cos32(16 - K32); s = (T)cos32(K32 - 8); }
    if (SIGN < 0) s = -s;
    T re = a.x * c - a.y * s, im = a.x * s + a.y * c;
    a.x = re; a.y = im;
}

__host__ __device__ constexpr int ilog2(int n) { return n <= 1 ? 0 : 1 + ilog2(n / 2); }
__host__ __device__ constexpr int bitrev(int v, int bits) { int r = 0; for (int i = 0; i < bits; ++i) r |= ((v >> i) & 1) << (bits - 1 - i); return r; }

// In-place DIF FFT, y[k] = sum_j a[j] exp(SIGN 2 pi i j k / N1); on return a[r] holds y[bitrev(r)].
template <typename T, int N1, int SIGN>
__device__ __forceinline__ void fft_dif(cx<T> (&a)[N1])
{
#pragma unroll
    for (int half = N1 / 2; half >= 1; half /= 2) {
#pragma unroll
        for (int base = 0; base < N1; base += 2 * half) {
#pragma unroll
            for (int j = 0; j < half; ++j) {
                cx<T> u = a[base + j], v = a[base + j + half];
                a[base + j] = cadd(u, v);
                cx<T> d = csub(u, v);
                twiddle32<T, SIGN>(d, j * (16 / half));      // w_{2 half}^j = w_32^{j * 32/(2 half)}
                a[base + j + half] = d;
            }
        }
    }
}

}  // namespace bioem
