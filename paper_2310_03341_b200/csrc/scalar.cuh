// scalar.cuh -- one set of scalar helpers for the kernels that exist in a complex (c128) and a real (double) instance:
// the 1-stage solver of SURVEY.md 8(f)2 (tridiag_direct.cu).  For double, conjugation is the identity.
#pragma once
#include "common.cuh"

namespace eigh {

template <typename T> struct Sc;

template <> struct Sc<double> {
    static constexpr bool is_complex = false;
    __host__ __device__ static __forceinline__ double zero() { return 0.0; }
    __host__ __device__ static __forceinline__ double one() { return 1.0; }
    __host__ __device__ static __forceinline__ double from_real(double r) { return r; }
    __host__ __device__ static __forceinline__ double conj(double a) { return a; }
    __host__ __device__ static __forceinline__ double re(double a) { return a; }
    __host__ __device__ static __forceinline__ double im(double) { return 0.0; }
    __host__ __device__ static __forceinline__ double abs2(double a) { return a * a; }
    __host__ __device__ static __forceinline__ double add(double a, double b) { return a + b; }
    __host__ __device__ static __forceinline__ double sub(double a, double b) { return a - b; }
    __host__ __device__ static __forceinline__ double mul(double a, double b) { return a * b; }
    __host__ __device__ static __forceinline__ double scale(double s, double a) { return s * a; }
    // acc += a b ;  acc += conj(a) b
    __host__ __device__ static __forceinline__ void fma(double& acc, double a, double b) { acc = ::fma(a, b, acc); }
    __host__ __device__ static __forceinline__ void fmac(double& acc, double a, double b) { acc = ::fma(a, b, acc); }
    __host__ __device__ static __forceinline__ double neg(double a) { return -a; }
    __host__ __device__ static __forceinline__ double real_part_only(double a) { return a; }
};

template <> struct Sc<c128> {
    static constexpr bool is_complex = true;
    __host__ __device__ static __forceinline__ c128 zero() { return cmake(0.0, 0.0); }
    __host__ __device__ static __forceinline__ c128 one() { return cmake(1.0, 0.0); }
    __host__ __device__ static __forceinline__ c128 from_real(double r) { return cmake(r, 0.0); }
    __host__ __device__ static __forceinline__ c128 conj(c128 a) { return cconj(a); }
    __host__ __device__ static __forceinline__ double re(c128 a) { return a.x; }
    __host__ __device__ static __forceinline__ double im(c128 a) { return a.y; }
    __host__ __device__ static __forceinline__ double abs2(c128 a) { return cabs2(a); }
    __host__ __device__ static __forceinline__ c128 add(c128 a, c128 b) { return cadd(a, b); }
    __host__ __device__ static __forceinline__ c128 sub(c128 a, c128 b) { return csub(a, b); }
    __host__ __device__ static __forceinline__ c128 mul(c128 a, c128 b) { return cmul(a, b); }
    __host__ __device__ static __forceinline__ c128 scale(double s, c128 a) { return cscale(s, a); }
    __host__ __device__ static __forceinline__ void fma(c128& acc, c128 a, c128 b) { cfma(acc, a, b); }
    __host__ __device__ static __forceinline__ void fmac(c128& acc, c128 a, c128 b) { cfmac(acc, a, b); }
    __host__ __device__ static __forceinline__ c128 neg(c128 a) { return cmake(-a.x, -a.y); }
    __host__ __device__ static __forceinline__ c128 real_part_only(c128 a) { return cmake(a.x, 0.0); }
};

// LAPACK xLARFG scalars from alpha = x_0 and xnorm2 = sum_{i >= 1} |x_i|^2:  H = I - tau v v^H, v_0 = 1, v_i = s x_i,
// H x = beta e_1 with beta REAL.  (For double: tau = 0 iff xnorm2 = 0.)
template <typename T>
__host__ __device__ __forceinline__ void larfg_scalars(T alpha, double xnorm2, T& tau, T& s, double& beta) {
    using S = Sc<T>;
    tau = S::zero();
    s = S::zero();
    const double ar = S::re(alpha), ai = S::im(alpha);
    beta = ar;
    if (xnorm2 > 0.0 || ai != 0.0) {
        beta = -copysign(sqrt(ar * ar + ai * ai + xnorm2), ar);
        const double ib = 1.0 / beta;
        const double dr = ar - beta, di = ai;
        const double iden = 1.0 / (dr * dr + di * di);
        if constexpr (S::is_complex) {
            tau = cmake((beta - ar) * ib, -ai * ib);
            s = cmake(dr * iden, -di * iden);
        } else {
            tau = (beta - ar) * ib;
            s = dr * iden;
        }
    }
}

// 16-byte (c128) or 8-byte (double) asynchronous global -> shared copy of one element; bytes = 0 zero-fills
__device__ __forceinline__ void cp_async_elem(c128* dst, const c128* src, bool ok) { cp_async16(dst, src, ok ? 16 : 0); }
__device__ __forceinline__ void cp_async_elem(double* dst, const double* src, bool ok) { cp_async8(dst, src, ok ? 8 : 0); }

}  // namespace eigh
