// prs_arith.cuh -- per-site arithmetic of the PRS step and of the diagnostics, device side.
//
// PAPER.md Eq. 1 (:30) potential, Eq. 3 (:46) Laplacian, Eq. 4 (:49) velocity update, Eq. 5 (:51)
// field update, Eq. 8 (:64) kinetic/potential ratio.  Every operation goes through an explicit
// round-to-nearest intrinsic (__fadd_rn, __dmul_rn, ...): those are never contracted into an FMA,
// whatever -fmad says, so the result of one site does not depend on which kernel evaluated it
// (generic, tiled, temporally blocked) and is reproducible bit for bit on any IEEE machine that
// applies the same operations in the same order.
#pragma once

#include <cstdint>
#include <cuda_runtime.h>

namespace prs {

// Race hunting without a race checker (compute-sanitizer is closed on this pool's GPUs): a second build of the library
// with -DPRS_RACE_JITTER=1 puts random, warp-uniform delays of up to a few microseconds at the points below -- before
// and after every barrier, between a row's fetch and its publication, between the two halves of a stack push -- so that
// an ordering that holds only because the warps of a CTA happen to run in step shows up as a wrong bit in
// tests/sanitize_kernels.py (every result is compared with the one-thread-per-site kernel).  The delays change no value.
#ifdef PRS_RACE_JITTER
__device__ __forceinline__ void prs_jitter(unsigned salt) {
    unsigned h = (blockIdx.x * 73856093u) ^ (blockIdx.y * 19349663u) ^ ((threadIdx.y + (threadIdx.x >> 5)) * 83492791u) ^
                 (salt * 2654435761u) ^ (unsigned)clock();
    h ^= h >> 13; h *= 0x5bd1e995u; h ^= h >> 15;
    h = __shfl_sync(0xffffffffu, h, 0);                  // one decision per warp: the warp stays converged
    if ((h & 3u) == 0u) __nanosleep(h >> 20);            // one warp in four sleeps up to 4 us
}
#define PRS_JITTER(salt) ::prs::prs_jitter(salt)
#else
#define PRS_JITTER(salt) ((void)0)
#endif

template <typename T> struct Ar;

template <> struct Ar<float> {
    static __device__ __forceinline__ float add(float a, float b) { return __fadd_rn(a, b); }
    static __device__ __forceinline__ float sub(float a, float b) { return __fsub_rn(a, b); }
    static __device__ __forceinline__ float mul(float a, float b) { return __fmul_rn(a, b); }
    static __device__ __forceinline__ float div(float a, float b) { return __fdiv_rn(a, b); }
    static __device__ __forceinline__ float fma(float a, float b, float c) { return __fmaf_rn(a, b, c); }
    static __device__ __forceinline__ bool neg(float v) { return (__float_as_uint(v) >> 31) != 0u; }
};

template <> struct Ar<double> {
    static __device__ __forceinline__ double add(double a, double b) { return __dadd_rn(a, b); }
    static __device__ __forceinline__ double sub(double a, double b) { return __dsub_rn(a, b); }
    static __device__ __forceinline__ double mul(double a, double b) { return __dmul_rn(a, b); }
    static __device__ __forceinline__ double div(double a, double b) { return __ddiv_rn(a, b); }
    static __device__ __forceinline__ double fma(double a, double b, double c) { return __fma_rn(a, b, c); }
    static __device__ __forceinline__ bool neg(double v) { return __double2hiint(v) < 0; }
};

// Arithmetic forms (values of PRS_ARITH_* in prs.h).
constexpr int ARITH_LITERAL = 0, ARITH_COEF = 1, ARITH_FMA = 2;

// Per-step scalars in the field's precision; formed on the host in double (Eq. 6) and rounded once.
template <typename T>
struct StepCoef {
    T K;     // 4 V0 / phi0^2
    T I;     // 1 / phi0^2
    T deta;  // time step
    T omd;   // 1 - delta_n   (LITERAL form)
    T opd;   // 1 + delta_n   (LITERAL form)
    T A;     // (1 - delta_n) / (1 + delta_n)   (COEF form)
    T B;     // deta / (1 + delta_n)            (COEF form)
};

// f = lap(phi) - dV/dphi at one site from the axis-pair sums of its neighbours.
//   sxy = (phi[x+1] + phi[x-1]) + (phi[y+1] + phi[y-1]),  sz = phi[z+1] + phi[z-1] (3D only)
template <typename T, int DIMS>
__device__ __forceinline__ T force(const StepCoef<T>& k, T c, T sxy, T sz) {
    using A = Ar<T>;
    T sum = sxy;
    if (DIMS == 3) sum = A::add(sum, sz);
    const T lap = A::sub(sum, A::mul(T(2 * DIMS), c));            // Eq. 3
    const T q = A::mul(c, c);
    const T r = A::mul(q, k.I);
    const T t = A::sub(r, T(1));
    const T dV = A::mul(A::mul(k.K, c), t);                       // dV/dphi of Eq. 1
    return A::sub(lap, dV);
}

template <typename T, int ARITH>
__device__ __forceinline__ T velocity(const StepCoef<T>& k, T pd, T f) {
    using A = Ar<T>;
    if (ARITH == ARITH_LITERAL) {
        const T num = A::add(A::mul(k.omd, pd), A::mul(k.deta, f));
        return A::div(num, k.opd);                                // Eq. 4 as printed
    }
    return A::add(A::mul(k.A, pd), A::mul(k.B, f));               // Eq. 4, pre-divided coefficients
}

template <typename T>
__device__ __forceinline__ T advance(const StepCoef<T>& k, T c, T pd_new) {
    return Ar<T>::add(c, Ar<T>::mul(k.deta, pd_new));             // Eq. 5
}

template <typename T, int DIMS, int ARITH>
__device__ __forceinline__ void site_update(const StepCoef<T>& k, T c, T xm, T xp, T ym, T yp, T zm,
                                            T zp, T pd, T& phi_new, T& pd_new) {
    using A = Ar<T>;
    const T sxy = A::add(A::add(xp, xm), A::add(yp, ym));
    const T sz = (DIMS == 3) ? A::add(zp, zm) : T(0);
    if (ARITH == ARITH_FMA) {
        // Contracted form (R13): every product that feeds a sum is one fused multiply-add.
        const T sum = (DIMS == 3) ? A::add(sxy, sz) : sxy;
        const T lap = A::fma(T(-2 * DIMS), c, sum);               // Eq. 3
        const T t = A::fma(A::mul(c, c), k.I, T(-1));
        const T f = A::fma(A::mul(-k.K, c), t, lap);              // lap - dV/dphi
        pd_new = A::fma(k.A, pd, A::mul(k.B, f));                 // Eq. 4
        phi_new = A::fma(k.deta, pd_new, c);                      // Eq. 5
        return;
    }
    const T f = force<T, DIMS>(k, c, sxy, sz);
    pd_new = velocity<T, ARITH>(k, pd, f);
    phi_new = advance<T>(k, c, pd_new);
}

// Eq. 8 summand phidot^2 / V(phi) in double; 0 where V == 0 (phi = +-phi0 exactly).
template <typename T>
__device__ __forceinline__ double wall_ratio(T phi, T phidot, double V0, double I) {
    const double p = (double)phi, v = (double)phidot;
    const double w = __dsub_rn(__dmul_rn(__dmul_rn(p, p), I), 1.0);
    const double V = __dmul_rn(__dmul_rn(V0, w), w);
    return (V == 0.0) ? 0.0 : __ddiv_rn(__dmul_rn(v, v), V);
}

// 16-byte vectors of the field type.
template <typename T> struct Vec;
template <> struct Vec<float> {
    typedef float4 type;
    static constexpr int W = 4;
};
template <> struct Vec<double> {
    typedef double2 type;
    static constexpr int W = 2;
};

// Reduction record of the diagnostics pass.
struct DiagPartial {
    unsigned long long links;
    unsigned long long walls;
    double sum;
};

}  // namespace prs
