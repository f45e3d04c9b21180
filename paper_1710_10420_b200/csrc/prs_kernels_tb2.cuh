// prs_kernels_tb2.cuh -- temporally blocked kernels: TWO PRS steps (Eqs. 3-5 applied twice,
// with the two consecutive sets of Eq. 6 scalars) per pass over HBM.  The compulsory traffic per
// site-update halves to 8 B (FP32) / 16 B (FP64); the per-site arithmetic is the same sequence of
// individually rounded operations as two single steps, so the result is bit-identical to them.
//
// 3D scheme.  A CTA owns TY rows x 30 vectors of x (120 floats / 60 doubles) of output and marches a
// chunk of z planes.  It is 32 lanes wide and TY+4 warps tall: lane 0 / lane 31 and the two outer
// rows on each side are halo.  Per iteration j it
//   (0) has every thread issue one 16-byte cp.async for its own column of the phi^n plane two
//       ahead and of the phidot^{n-1/2} plane one ahead, straight into shared-memory rings (no
//       register staging, PF planes of prefetch);
//   (1) stage 1: rows 1..TY+2 compute phi^{n+1}, phidot^{n+1/2} on plane zi = z0-1+j from the
//       phi^n ring (z+-1 from the ring, y+-1 from the neighbouring rows of the ring, x+-1 by warp
//       shuffle) and publish phi^{n+1} to a two-slot shared plane;
//   (2) stage 2: rows 2..TY+1 compute phi^{n+2}, phidot^{n+3/2} on plane zi-1 from their own register
//       window of phi^{n+1} (three planes deep), the neighbouring rows of the published plane and
//       shuffles, and store lanes 1..30 to HBM.
// Values at the halo rim that lack a neighbour are computed from finite stand-ins and never used.
// Periodic wrap is plain index arithmetic on the cp.async source addresses.
//
// 2D scheme.  Same idea with the march along y and no shared memory at all: both register windows
// supply the y neighbours and shuffles supply the x neighbours; a warp outputs 30 vectors of x.
#pragma once

#include "prs_arith.cuh"
#include "prs_kernels_tiled.cuh"

namespace prs {

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src) {
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

__host__ __device__ __forceinline__ int wrap_mod(int i, int n) {
    i %= n;
    return i < 0 ? i + n : i;
}

constexpr int TB2_XOUT = 30;       // output vectors per warp row (lanes 1..30)
constexpr int TB2_PF = 2;          // planes of prefetch
constexpr int TB2_RA = 3 + TB2_PF; // phi^n ring slots
constexpr int TB2_RP = 1 + TB2_PF; // phidot^{n-1/2} ring slots

template <typename T, int TY>
constexpr size_t tb2_smem_bytes() {
    return (size_t)(TB2_RA + TB2_RP + 2) * (TY + 4) * 32 * 16;
}

template <typename T, bool LITERAL, int TY>
__global__ void __launch_bounds__(32 * (TY + 4))
step3d_tb2_kernel(const T* __restrict__ phi, const T* __restrict__ phidot, T* __restrict__ phi_out,
                  T* __restrict__ phidot_out, int N, int ZC, StepCoef<T> k1, StepCoef<T> k2) {
    using O = VecOps<T>;
    using V = typename O::V;
    constexpr int W = O::W;
    constexpr int ROWS = TY + 4;
    extern __shared__ __align__(16) unsigned char tb2_smem[];
    V* const ringA = reinterpret_cast<V*>(tb2_smem);                 // [RA][ROWS][32]
    V* const ringP = ringA + TB2_RA * ROWS * 32;                     // [RP][ROWS][32]
    V* const planeB = ringP + TB2_RP * ROWS * 32;                    // [2][ROWS][32]

    const int lane = threadIdx.x, row = threadIdx.y;
    const int NQ = N / W;
    const int qraw = TB2_XOUT * (int)blockIdx.x - 1 + lane;
    const int q = wrap_mod(qraw, NQ);
    const int yraw = TY * (int)blockIdx.y - 2 + row;
    const int y = wrap_mod(yraw, N);
    const int z0 = (int)blockIdx.z * ZC;
    const int zend = min(z0 + ZC, N);
    const int niter = (zend - z0) + 2;
    const size_t NN = (size_t)N * N;
    const size_t col = (size_t)y * N + (size_t)q * W;              // offset of this thread's column in a plane
    const bool stage1_row = (row >= 1) && (row <= TY + 2);
    const bool stage2_row = (row >= 2) && (row <= TY + 1);
    const bool store_ok = stage2_row && (yraw < N) && (lane >= 1) && (lane <= TB2_XOUT) && (qraw < NQ);
    const int me = row * 32 + lane;

    // ---- prologue: planes a = 0, 1 (z0-2, z0-1), then plane a = 2 with phidot plane p = 0, then PF-1 more
    cp_async16(&ringA[(0 * ROWS) * 32 + me], phi + (size_t)wrap_mod(z0 - 2, N) * NN + col);
    cp_async16(&ringA[(1 * ROWS) * 32 + me], phi + (size_t)wrap_mod(z0 - 1, N) * NN + col);
    cp_async_commit();
#pragma unroll
    for (int g = 0; g < TB2_PF; ++g) {          // group g carries A plane 2+g and P plane g
        if (g < niter) {
            cp_async16(&ringA[(((2 + g) % TB2_RA) * ROWS) * 32 + me], phi + (size_t)wrap_mod(z0 + g, N) * NN + col);
            if (stage1_row)
                cp_async16(&ringP[((g % TB2_RP) * ROWS) * 32 + me], phidot + (size_t)wrap_mod(z0 - 1 + g, N) * NN + col);
        }
        cp_async_commit();
    }

    V b_prev = {}, b_cur = {}, q_cur = {};
    for (int j = 0; j < niter; ++j) {
        // (0) prefetch group j+PF: A plane j+2+PF (z = z0+j+PF), P plane j+PF (z = z0-1+j+PF)
        if (j + TB2_PF < niter) {
            cp_async16(&ringA[(((j + 2 + TB2_PF) % TB2_RA) * ROWS) * 32 + me],
                       phi + (size_t)wrap_mod(z0 + j + TB2_PF, N) * NN + col);
            if (stage1_row)
                cp_async16(&ringP[(((j + TB2_PF) % TB2_RP) * ROWS) * 32 + me],
                           phidot + (size_t)wrap_mod(z0 - 1 + j + TB2_PF, N) * NN + col);
        }
        cp_async_commit();
        cp_async_wait<TB2_PF>();                // group j (A plane j+2, P plane j) has landed for this thread
        __syncthreads();                        // ... and for every thread; also fences last iteration's reads

        // (1) stage 1 on plane zi = z0-1+j
        V b_new = {}, q_new = {};
        if (stage1_row) {
            const V* A0 = ringA + ((j % TB2_RA) * ROWS) * 32;
            const V* A1 = ringA + (((j + 1) % TB2_RA) * ROWS) * 32;
            const V* A2 = ringA + (((j + 2) % TB2_RA) * ROWS) * 32;
            const V c = A1[me];
            const V zm = A0[me], zp = A2[me];
            const V ym = A1[me - 32], yp = A1[me + 32];
            const V pd = ringP[((j % TB2_RP) * ROWS) * 32 + me];
            const T left = __shfl_up_sync(0xffffffffu, O::last(c), 1);
            const T right = __shfl_down_sync(0xffffffffu, O::first(c), 1);
            vector_update<T, 3, LITERAL>(k1, c, left, right, ym, yp, zm, zp, pd, b_new, q_new);
            planeB[((j & 1) * ROWS) * 32 + me] = b_new;
        }
        // No barrier here: stage 2 below reads the plane published one iteration ago (slot (j-1)&1),
        // which the barrier at the top of this iteration already ordered; the slot written above is
        // read only after the next top-of-iteration barrier.

        // (2) stage 2 on plane zo = zi-1 = z0+j-2
        if (j >= 2 && stage2_row) {
            const V* B = planeB + (((j - 1) & 1) * ROWS) * 32;
            const V ym = B[me - 32], yp = B[me + 32];
            const T left = __shfl_up_sync(0xffffffffu, O::last(b_cur), 1);
            const T right = __shfl_down_sync(0xffffffffu, O::first(b_cur), 1);
            V pout, vout;
            vector_update<T, 3, LITERAL>(k2, b_cur, left, right, ym, yp, b_prev, b_new, q_cur, pout, vout);
            if (store_ok) {
                const size_t o = (size_t)(z0 + j - 2) * NN + col;
                O::st(phidot_out + o, vout);
                O::st(phi_out + o, pout);
            }
        }
        b_prev = b_cur; b_cur = b_new; q_cur = q_new;
    }
}

// ------------------------------------------------------------------------------------------------
// 2D: block = BX lanes (multiple of 32); every warp outputs 30 vectors of x and marches YC rows.
// ------------------------------------------------------------------------------------------------
template <typename T, bool LITERAL>
__global__ void __launch_bounds__(128)
step2d_tb2_kernel(const T* __restrict__ phi, const T* __restrict__ phidot, T* __restrict__ phi_out,
                  T* __restrict__ phidot_out, int N, int YC, StepCoef<T> k1, StepCoef<T> k2) {
    using O = VecOps<T>;
    using V = typename O::V;
    constexpr int W = O::W;
    const int lane = threadIdx.x & 31;
    const int warp_global = (int)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const int NQ = N / W;
    if (warp_global * TB2_XOUT >= NQ) return;                       // whole warp beyond the row
    const int qraw = TB2_XOUT * warp_global - 1 + lane;
    const int q = wrap_mod(qraw, NQ);
    const int y0 = (int)blockIdx.y * YC;
    const int yend = min(y0 + YC, N);
    const int niter = (yend - y0) + 2;
    const size_t colx = (size_t)q * W;
    const bool store_ok = (lane >= 1) && (lane <= TB2_XOUT) && (qraw < NQ);
    const V zero = {};

    // register windows: a* = phi^n rows, b* = phi^{n+1} rows
    V a_prev = O::ld(phi + (size_t)wrap_mod(y0 - 2, N) * N + colx);
    V a_cur = O::ld(phi + (size_t)wrap_mod(y0 - 1, N) * N + colx);
    V a_next = O::ld(phi + (size_t)wrap_mod(y0, N) * N + colx);
    V pd = O::ld(phidot + (size_t)wrap_mod(y0 - 1, N) * N + colx);
    V b_prev = zero, b_cur = zero, q_cur = zero;
    for (int j = 0; j < niter; ++j) {
        // loads of the next iteration first: phi^n row y0+j+1, phidot row y0+j
        V a_nn = a_next, pd_n = pd;
        if (j + 1 < niter) {
            a_nn = O::ld(phi + (size_t)wrap_mod(y0 + j + 1, N) * N + colx);
            pd_n = O::ld(phidot + (size_t)wrap_mod(y0 + j, N) * N + colx);
        }
        // stage 1 on row yi = y0-1+j
        V b_new, q_new;
        {
            const T left = __shfl_up_sync(0xffffffffu, O::last(a_cur), 1);
            const T right = __shfl_down_sync(0xffffffffu, O::first(a_cur), 1);
            vector_update<T, 2, LITERAL>(k1, a_cur, left, right, a_prev, a_next, zero, zero, pd, b_new, q_new);
        }
        // stage 2 on row yo = y0+j-2
        if (j >= 2) {
            const T left = __shfl_up_sync(0xffffffffu, O::last(b_cur), 1);
            const T right = __shfl_down_sync(0xffffffffu, O::first(b_cur), 1);
            V pout, vout;
            vector_update<T, 2, LITERAL>(k2, b_cur, left, right, b_prev, b_new, zero, zero, q_cur, pout, vout);
            if (store_ok) {
                const size_t o = (size_t)(y0 + j - 2) * N + colx;
                O::st(phidot_out + o, vout);
                O::st(phi_out + o, pout);
            }
        }
        a_prev = a_cur; a_cur = a_next; a_next = a_nn; pd = pd_n;
        b_prev = b_cur; b_cur = b_new; q_cur = q_new;
    }
}

}  // namespace prs
