// prs_pack.cuh -- 16-byte site vectors as two "packs", and the PRS site update written on packs.
//
// FP32: a pack is two floats in one 64-bit register pair and the arithmetic is Blackwell's packed
// add.rn.f32x2 / mul.rn.f32x2 (SASS FADD2 / FMUL2): one instruction rounds two sites, each half
// exactly as the scalar __fadd_rn / __fmul_rn would (round-to-nearest-even, subnormals kept).
// Measured on B200: a packed instruction occupies its FP pipe for two cycles, so
// the flop rate equals the scalar one, but it takes one issue slot instead of two -- which is what an
// issue-bound temporally blocked kernel needs.  FP64: a pack is one double (__dadd_rn / __dmul_rn).
//
// The operation sequence per site is that of prs_arith.cuh (Eqs. 1, 3-5; R14), with
// two rewrites that do not change a bit: "a - b*c" is evaluated as "a + ((-b)*c)" and "r - 1" as
// "r + (-1)", because negation is exact in IEEE arithmetic.
#pragma once

#include "prs_arith.cuh"

namespace prs {

template <typename T> struct Pk;

template <> struct Pk<float> {
    typedef unsigned long long P;            // (lo, hi) = sites (x, x+1)
    typedef ulonglong2 V;                    // .x = sites 0,1   .y = sites 2,3
    static constexpr int W = 4;
    static __device__ __forceinline__ P add(P a, P b) { P r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
    static __device__ __forceinline__ P mul(P a, P b) { P r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
    static __device__ __forceinline__ P fma(P a, P b, P c) { P r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
    static __device__ __forceinline__ P pack(float lo, float hi) { P r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
    static __device__ __forceinline__ void unpack(P p, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(p)); }
    static __device__ __forceinline__ P dup(float s) { return pack(s, s); }
    // a + m where m is the result of a packed multiply.  ptxas 12.9 contracts mul.rn.f32x2 followed by
    // add.rn.f32x2 into one FFMA2 (a single rounding) whatever --fmad says, which would change the
    // bits; two scalar FADDs on the halves are left alone (checked in SASS by tests/test_library_cpu.py).
    static __device__ __forceinline__ P addm(P a, P m) {
        float a0, a1, m0, m1; unpack(a, a0, a1); unpack(m, m0, m1);
        return pack(__fadd_rn(a0, m0), __fadd_rn(a1, m1));
    }
    static __device__ __forceinline__ P div(P a, P b) {
        float a0, a1, b0, b1; unpack(a, a0, a1); unpack(b, b0, b1);
        return pack(__fdiv_rn(a0, b0), __fdiv_rn(a1, b1));
    }
    static __device__ __forceinline__ float first(V v) { float lo, hi; unpack(v.x, lo, hi); return lo; }
    static __device__ __forceinline__ float last(V v) { float lo, hi; unpack(v.y, lo, hi); return hi; }
    // phi[x+1] + phi[x-1] for the four sites of c; left / right are the scalars beside the vector
    static __device__ __forceinline__ V xsum(V c, float left, float right) {
        float c0, c1, c2, c3; unpack(c.x, c0, c1); unpack(c.y, c2, c3);
        V s;
        s.x = pack(__fadd_rn(c1, left), __fadd_rn(c2, c0));
        s.y = pack(__fadd_rn(c3, c1), __fadd_rn(right, c2));
        return s;
    }
    static __device__ __forceinline__ V ldg(const float* p) { return __ldg(reinterpret_cast<const ulonglong2*>(p)); }
    static __device__ __forceinline__ void stg(float* p, V v) { *reinterpret_cast<ulonglong2*>(p) = v; }
};

template <> struct Pk<double> {
    typedef double P;
    typedef double2 V;
    static constexpr int W = 2;
    static __device__ __forceinline__ P add(P a, P b) { return __dadd_rn(a, b); }
    static __device__ __forceinline__ P mul(P a, P b) { return __dmul_rn(a, b); }
    static __device__ __forceinline__ P fma(P a, P b, P c) { return __fma_rn(a, b, c); }
    static __device__ __forceinline__ P dup(double s) { return s; }
    static __device__ __forceinline__ P addm(P a, P m) { return __dadd_rn(a, m); }
    static __device__ __forceinline__ P div(P a, P b) { return __ddiv_rn(a, b); }
    static __device__ __forceinline__ double first(V v) { return v.x; }
    static __device__ __forceinline__ double last(V v) { return v.y; }
    static __device__ __forceinline__ V xsum(V c, double left, double right) {
        V s;
        s.x = __dadd_rn(c.y, left);
        s.y = __dadd_rn(right, c.x);
        return s;
    }
    static __device__ __forceinline__ V ldg(const double* p) { return __ldg(reinterpret_cast<const double2*>(p)); }
    static __device__ __forceinline__ void stg(double* p, V v) { *reinterpret_cast<double2*>(p) = v; }
};

// Per-step scalars as packs (both halves equal).  Built once per kernel from StepCoef<T>.
template <typename T>
struct PackCoef {
    typename Pk<T>::P nK, I, deta, omd, opd, A, B, n2d, m1;
    template <int DIMS>
    __device__ __forceinline__ void set(const StepCoef<T>& k) {
        using K = Pk<T>;
        nK = K::dup(-k.K); I = K::dup(k.I); deta = K::dup(k.deta); omd = K::dup(k.omd); opd = K::dup(k.opd);
        A = K::dup(k.A); B = K::dup(k.B); n2d = K::dup(T(-2 * DIMS)); m1 = K::dup(T(-1));
    }
};

// One pack of sites: c centre, sx = x+1 plus x-1 (already summed), (ym, yp), (zm, zp) neighbours,
// pd = phidot^{n-1/2}.  Same operations, same order as site_update() in prs_arith.cuh.
template <typename T, int DIMS, int ARITH>
__device__ __forceinline__ void pack_update(const PackCoef<T>& k, typename Pk<T>::P c, typename Pk<T>::P sx,
                                            typename Pk<T>::P ym, typename Pk<T>::P yp, typename Pk<T>::P zm,
                                            typename Pk<T>::P zp, typename Pk<T>::P pd, typename Pk<T>::P& phi_new,
                                            typename Pk<T>::P& pd_new) {
    using K = Pk<T>;
    typename K::P sum = K::add(sx, K::add(yp, ym));
    if (DIMS == 3) sum = K::add(sum, K::add(zp, zm));
    if (ARITH == ARITH_FMA) {
        // Contracted form (R13): FFMA2 / DFMA, one rounding per product-sum.
        const typename K::P lapf = K::fma(k.n2d, c, sum);                // Eq. 3
        const typename K::P tf = K::fma(K::mul(c, c), k.I, k.m1);
        const typename K::P ff = K::fma(K::mul(k.nK, c), tf, lapf);      // lap - dV/dphi
        pd_new = K::fma(k.A, pd, K::mul(k.B, ff));                       // Eq. 4
        phi_new = K::fma(k.deta, pd_new, c);                             // Eq. 5
        return;
    }
    const typename K::P lap = K::addm(sum, K::mul(k.n2d, c));             // Eq. 3:  sum - 2d*c
    const typename K::P q = K::mul(c, c);
    const typename K::P r = K::mul(q, k.I);
    const typename K::P t = K::addm(k.m1, r);                          // r - 1
    const typename K::P ndV = K::mul(K::mul(k.nK, c), t);                // -(K*c)*t = -dV/dphi (Eq. 1)
    const typename K::P f = K::addm(lap, ndV);                          // lap - dV
    if (ARITH == ARITH_LITERAL) pd_new = K::div(K::addm(K::mul(k.omd, pd), K::mul(k.deta, f)), k.opd);   // Eq. 4 as printed
    else pd_new = K::addm(K::mul(k.A, pd), K::mul(k.B, f));             // Eq. 4, pre-divided coefficients
    phi_new = K::addm(c, K::mul(k.deta, pd_new));                      // Eq. 5
}

// One 16-byte vector of sites (two packs).
template <typename T, int DIMS, int ARITH>
__device__ __forceinline__ void packed_vector_update(const PackCoef<T>& k, typename Pk<T>::V c, T left, T right,
                                                     typename Pk<T>::V ym, typename Pk<T>::V yp,
                                                     typename Pk<T>::V zm, typename Pk<T>::V zp,
                                                     typename Pk<T>::V pd, typename Pk<T>::V& phi_new,
                                                     typename Pk<T>::V& pd_new) {
    using K = Pk<T>;
    const typename K::V sx = K::xsum(c, left, right);
    pack_update<T, DIMS, ARITH>(k, c.x, sx.x, ym.x, yp.x, zm.x, zp.x, pd.x, phi_new.x, pd_new.x);
    pack_update<T, DIMS, ARITH>(k, c.y, sx.y, ym.y, yp.y, zm.y, zp.y, pd.y, phi_new.y, pd_new.y);
}

}  // namespace prs
