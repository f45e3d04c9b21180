// prs_kernels_tb2.cuh -- temporally blocked kernels: TWO PRS steps (Eqs. 3-5 applied twice,
// with the two consecutive sets of Eq. 6 scalars) per pass over HBM.  The compulsory traffic per
// site-update halves to 8 B (FP32) / 16 B (FP64); the per-site arithmetic is the same sequence of
// individually rounded operations as two single steps, so the result is bit-identical to them.
//
// With half the HBM traffic the first version was bound by instruction issue, not by memory, so the
// design goal became instructions per site-update: packed FP32 arithmetic (prs_pack.cuh: FADD2 / FMUL2
// / FFMA2 round two sites per instruction), each thread's own column kept in a register window (only
// neighbour rows go through shared memory), no integer division and only 32-bit cursor arithmetic inside
// the march, one copy of the march per kind of row.  In that state it is HBM-bound again
// (profiles/r01b_*), which is why prs_kernels_tbs.cuh goes on to four steps per pass; this kernel now
// serves the leftovers of a prs_step call and the PRS_KERNEL_TB2 option.
//
// 3D scheme.  A CTA owns TY rows x 30 vectors of x (120 floats / 60 doubles) of output and marches a
// chunk of z planes.  It is 32 lanes wide and TY+4 warps tall: lane 0 / lane 31 and the two outer
// rows on each side are halo.  Plane index a = 0, 1, ... stands for z = z0-2+a (periodic).  In
// iteration j every thread
//   (0) waits for its cp.async group j (phi^n plane a = j+2 and the phidot plane of z = z0+j), then the
//       CTA barrier makes every thread's group j visible and retires all reads of iteration j-1;
//   (1) issues one 16-byte cp.async for its own column of phi^n plane a = j+4 and of the phidot plane
//       of the same z, straight into four-slot shared-memory rings (no register staging; the march is
//       unrolled four times, so every slot index is an immediate);
//   (2) stage 1 (rows 1..TY+2): phi^{n+1}, phidot^{n+1/2} on plane a = j+1 from its register window
//       (z-1, z), its own column of the ring (z+1), the neighbouring rows of the ring (y+-1) and warp
//       shuffles (x+-1); publishes phi^{n+1} to a two-slot shared plane;
//   (3) stage 2 (rows 2..TY+1, j >= 2): phi^{n+2}, phidot^{n+3/2} on plane a = j from its register
//       window of phi^{n+1}, the neighbouring rows of the plane published one iteration ago and
//       shuffles; lanes 1..30 store to HBM.
// Values at the halo rim that lack a neighbour are computed from stand-ins and never used.
//
// 2D scheme.  Same idea with the march along y and no shared memory at all: both register windows
// supply the y neighbours and shuffles supply the x neighbours; a warp outputs 30 vectors of x.
#pragma once

#include <type_traits>

#include "prs_arith.cuh"
#include "prs_pack.cuh"

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
constexpr int TB2_RA = 4;          // phi^n ring slots: planes a = j+1, j+2 being read, PF in flight
constexpr int TB2_RP = 4;          // phidot^{n-1/2} ring slots: 1 being read, PF in flight (power of two)

template <typename T, int TY>
constexpr size_t tb2_smem_bytes() {
    return (size_t)(TB2_RA + TB2_RP + 2) * (TY + 4) * 32 * 16;
}

template <typename T, int ARITH, int TY>
__global__ void __launch_bounds__(32 * (TY + 4), (32 * (TY + 4) > 512) ? 1 : 2)
step3d_tb2_kernel(const T* __restrict__ phi, const T* __restrict__ phidot, T* __restrict__ phi_out,
                  T* __restrict__ phidot_out, int N, int NZ, int ZC, StepCoef<T> k1, StepCoef<T> k2) {
    using K = Pk<T>;
    using V = typename K::V;
    constexpr int W = K::W;
    constexpr int ROWS = TY + 4;
    constexpr int PLANE = ROWS * 32;                                 // vectors per shared plane
    static_assert(TB2_RA == 4 && TB2_RP == 4 && TB2_PF == 2, "the slot arithmetic below assumes these");
    extern __shared__ __align__(16) unsigned char tb2_smem[];
    const int lane = threadIdx.x, row = threadIdx.y;
    const int me = row * 32 + lane;
    V* const sA = reinterpret_cast<V*>(tb2_smem) + me;               // ring A [4][PLANE], this thread's slot
    V* const sP = sA + TB2_RA * PLANE;                               // ring P [4][PLANE]
    V* const sB = sP + TB2_RP * PLANE;                               // plane B [2][PLANE]

    const int NQ = N / W;
    const int qraw = TB2_XOUT * (int)blockIdx.x - 1 + lane;
    const int q = wrap_mod(qraw, NQ);
    const int yraw = TY * (int)blockIdx.y - 2 + row;
    const int y = wrap_mod(yraw, N);
    const int z0 = (int)blockIdx.z * ZC;
    const int zend = min(z0 + ZC, NZ);                                // NZ planes: N, or a slab's (prs_create_slab)
    const int niter = (zend - z0) + 2;                               // >= 3
    const bool store_ok = (yraw < N) && (lane >= 1) && (lane <= TB2_XOUT) && (qraw < NQ);

    PackCoef<T> c1, c2;
    c1.template set<3>(k1);
    c2.template set<3>(k2);

    // All global addresses are unsigned 32-bit indices of 16-byte vectors (the host checks N^3 / W <= 2^31):
    // one IMAD.WIDE forms an address, one IADD advances a cursor.
    const V* const gA = reinterpret_cast<const V*>(phi);
    const V* const gP = reinterpret_cast<const V*>(phidot);
    V* const oA = reinterpret_cast<V*>(phi_out);
    V* const oP = reinterpret_cast<V*>(phidot_out);
    const unsigned NNv = (unsigned)N * (unsigned)NQ;                 // vectors per plane
    const unsigned colv = (unsigned)y * (unsigned)NQ + (unsigned)q;  // this thread's column within a plane
    // One load cursor serves both fields: issue i fetches phi^n plane a = i (z = z0-2+i, periodic)
    // and the phidot plane of the same z, which stage 1 needs one iteration later than phi^n.
    int zl = wrap_mod(z0 - 2, NZ);
    unsigned il = (unsigned)zl * NNv + colv;
    int left_to_wrap = NZ - zl;                                      // issues until z wraps to 0
    unsigned io = (unsigned)z0 * NNv + colv;                         // store cursor (plane a = j, from j = 2)

    // The three kinds of row run their own march, so that no per-iteration test of the row survives
    // and the register windows rotate by renaming in the unrolled code:
    //   role 0  rows 0, TY+3      load phi^n only (they are the y halo of stage 1)
    //   role 1  rows 1, TY+2      stage 1 only (they are the y halo of stage 2)
    //   role 2  rows 2 .. TY+1    stage 1 and stage 2, store
    auto march = [&](auto role_tag) {
        constexpr int ROLE = decltype(role_tag)::value;
        int ni = 0;                                                  // issues so far
        auto issue = [&](int slot_a, int slot_p) {
            if (ni < niter + 2) cp_async16(sA + slot_a * PLANE, gA + il);
            if (ROLE >= 1 && ni >= 1 && ni <= niter) cp_async16(sP + slot_p * PLANE, gP + il);
            ++ni; il += NNv;
            if (--left_to_wrap == 0) { il -= (unsigned)NZ * NNv; left_to_wrap = NZ; }   // modulo 2^32, exact
        };
        // prologue: group 0 = issues 0, 1, 2 (phi^n planes 0..2, phidot planes 0..1); group 1 = issue 3
        issue(0, 3); issue(1, 0); issue(2, 1);
        cp_async_commit();
        issue(3, 2);
        cp_async_commit();

        // Register window of the thread's own column: phi^n at planes a = j, j+1.  Plane 0 is needed
        // for nothing else, so it is read here, before its ring slot is reused (a thread's own
        // cp.async data is visible to it after wait_group; no barrier needed).
        cp_async_wait<TB2_PF - 1>();
        V a_zm = sA[0 * PLANE], a_c = sA[1 * PLANE];
        V b_prev = {}, b_cur = {}, q_cur = {};  // phi^{n+1} at planes a = j-1, j; phidot^{n+1/2} at plane j

        // One iteration; U = j mod 4 is a compile-time constant so that every ring slot is an immediate.
        auto iteration = [&](auto u_tag, auto s2_tag) {
            constexpr int U = decltype(u_tag)::value;
            constexpr bool STAGE2 = decltype(s2_tag)::value && ROLE == 2;
            cp_async_wait<TB2_PF - 1>();        // group j has landed for this thread
            PRS_JITTER(1u);
            __syncthreads();                    // ... and for every thread; retires iteration j-1's reads
            PRS_JITTER(2u);
            issue(U, (U + 3) & 3);              // issue j+4: phi^n plane j+4 takes the slot of plane j
            cp_async_commit();
            PRS_JITTER(3u);
            if (ROLE == 0) return;

            // stage 1 on plane a = j+1
            const V zp = sA[((U + 2) & 3) * PLANE];
            const V ym1 = sA[((U + 1) & 3) * PLANE - 32], yp1 = sA[((U + 1) & 3) * PLANE + 32];
            const V pd = sP[U * PLANE];
            const T left1 = __shfl_up_sync(0xffffffffu, K::last(a_c), 1);
            const T right1 = __shfl_down_sync(0xffffffffu, K::first(a_c), 1);
            V b_new, q_new;
            packed_vector_update<T, 3, ARITH>(c1, a_c, left1, right1, ym1, yp1, a_zm, zp, pd, b_new, q_new);
            sB[(U & 1) * PLANE] = b_new;
            a_zm = a_c; a_c = zp;
            // No barrier here: stage 2 reads the plane published one iteration ago (slot (j-1)&1),
            // which the barrier at the top of this iteration already ordered; the slot written above
            // is read only after the next top-of-iteration barrier.

            // stage 2 on plane a = j  (z = z0+j-2)
            if (STAGE2) {
                const V ym2 = sB[((U + 1) & 1) * PLANE - 32], yp2 = sB[((U + 1) & 1) * PLANE + 32];
                const T left2 = __shfl_up_sync(0xffffffffu, K::last(b_cur), 1);
                const T right2 = __shfl_down_sync(0xffffffffu, K::first(b_cur), 1);
                V pout, vout;
                packed_vector_update<T, 3, ARITH>(c2, b_cur, left2, right2, ym2, yp2, b_prev, b_new, q_cur, pout, vout);
                if (store_ok) {
                    oP[io] = vout;
                    oA[io] = pout;
                }
                io += NNv;
            }
            if (ROLE == 2) { b_prev = b_cur; b_cur = b_new; q_cur = q_new; }
        };
        using std::integral_constant;
        iteration(integral_constant<int, 0>{}, integral_constant<bool, false>{});
        iteration(integral_constant<int, 1>{}, integral_constant<bool, false>{});
        for (int j = 2; j < niter; j += 4) {
            iteration(integral_constant<int, 2>{}, integral_constant<bool, true>{});
            if (j + 1 >= niter) break;
            iteration(integral_constant<int, 3>{}, integral_constant<bool, true>{});
            if (j + 2 >= niter) break;
            iteration(integral_constant<int, 0>{}, integral_constant<bool, true>{});
            if (j + 3 >= niter) break;
            iteration(integral_constant<int, 1>{}, integral_constant<bool, true>{});
        }
        cp_async_wait<0>();
    };
    if (row == 0 || row == ROWS - 1) march(std::integral_constant<int, 0>{});
    else if (row == 1 || row == ROWS - 2) march(std::integral_constant<int, 1>{});
    else march(std::integral_constant<int, 2>{});
}

// ------------------------------------------------------------------------------------------------
// 2D: block = BX lanes (multiple of 32); every warp outputs 30 vectors of x and marches YC rows.
// ------------------------------------------------------------------------------------------------
template <typename T, int ARITH>
__global__ void __launch_bounds__(128)
step2d_tb2_kernel(const T* __restrict__ phi, const T* __restrict__ phidot, T* __restrict__ phi_out,
                  T* __restrict__ phidot_out, int N, int YC, StepCoef<T> k1, StepCoef<T> k2) {
    using K = Pk<T>;
    using V = typename K::V;
    constexpr int W = K::W;
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

    PackCoef<T> c1, c2;
    c1.template set<2>(k1);
    c2.template set<2>(k2);

    // load cursors (periodic rows): la = phi row two ahead of stage 1, lp = phidot row one ahead
    int yla = wrap_mod(y0 - 2, N), ylp = wrap_mod(y0 - 1, N);
    const T* la = phi + (size_t)yla * N + colx;
    const T* lp = phidot + (size_t)ylp * N + colx;
    const size_t wrap_back = (size_t)N * N;
#define TB2_NEXT_A(dst)                                         \
    do {                                                        \
        dst = K::ldg(la); la += N;                              \
        if (++yla == N) { yla = 0; la -= wrap_back; }           \
    } while (0)
#define TB2_NEXT_P(dst)                                         \
    do {                                                        \
        dst = K::ldg(lp); lp += N;                              \
        if (++ylp == N) { ylp = 0; lp -= wrap_back; }           \
    } while (0)

    // register windows: a* = phi^n rows, b* = phi^{n+1} rows
    V a_prev, a_cur, a_next, pd;
    TB2_NEXT_A(a_prev); TB2_NEXT_A(a_cur); TB2_NEXT_A(a_next); TB2_NEXT_P(pd);
    V b_prev = zero, b_cur = zero, q_cur = zero;
    T* po = phi_out + (size_t)y0 * N + colx;
    T* vo = phidot_out + (size_t)y0 * N + colx;
    for (int j = 0; j < niter; ++j) {
        // loads of the next iteration first: phi^n row y0+j+1, phidot row y0+j (unused past the end)
        V a_nn, pd_n;
        TB2_NEXT_A(a_nn); TB2_NEXT_P(pd_n);
        // stage 1 on row yi = y0-1+j
        V b_new, q_new;
        {
            const T left = __shfl_up_sync(0xffffffffu, K::last(a_cur), 1);
            const T right = __shfl_down_sync(0xffffffffu, K::first(a_cur), 1);
            packed_vector_update<T, 2, ARITH>(c1, a_cur, left, right, a_prev, a_next, zero, zero, pd, b_new, q_new);
        }
        // stage 2 on row yo = y0+j-2
        if (j >= 2) {
            const T left = __shfl_up_sync(0xffffffffu, K::last(b_cur), 1);
            const T right = __shfl_down_sync(0xffffffffu, K::first(b_cur), 1);
            V pout, vout;
            packed_vector_update<T, 2, ARITH>(c2, b_cur, left, right, b_prev, b_new, zero, zero, q_cur, pout, vout);
            if (store_ok) {
                K::stg(vo, vout);
                K::stg(po, pout);
            }
            po += N; vo += N;
        }
        a_prev = a_cur; a_cur = a_next; a_next = a_nn; pd = pd_n;
        b_prev = b_cur; b_cur = b_new; q_cur = q_new;
    }
#undef TB2_NEXT_A
#undef TB2_NEXT_P
}

}  // namespace prs
