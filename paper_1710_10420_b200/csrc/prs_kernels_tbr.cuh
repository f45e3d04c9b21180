// prs_kernels_tbr.cuh -- the 3D multi-step kernel with TWO adjacent rows per thread.
//
// Same scheme, same per-site operations and therefore the same bits as step3d_tbs_kernel
// (prs_kernels_tbs.cuh: S PRS steps of PAPER.md Eqs. 3-5 per pass over HBM as an S-stage pipeline along
// z), with one change of mapping: a warp owns rows 2w and 2w+1 of the tile.  Why: the four-step kernel
// is bound by the shared-memory pipe (profiles/r01f_*: l1tex 67 %, 54 wavefronts per warp and plane,
// most of them the y-neighbour rows every stage fetches).  With two adjacent rows in one thread the
// inner y neighbour of either row is a register of the same thread, so a stage fetches two rows from
// shared memory per TWO rows of output instead of four, and a CTA of 512 threads x 128 registers holds
// a taller tile (32 rows: 26 of output at S = 3) than 768 threads x 80 registers do (24 rows: 16 of
// output at S = 4), which cuts the redundant halo work from 1.5x to 1.23x.
//
// Measured on B200, 1024^3, ms per step: FP32 S = 4 1.22-1.24 against 1.27 with one
// row per thread, S = 3 1.26 against 1.33; FP64 S = 4 2.59-2.67 against 2.45 (slower: 16 warps hide the
// FP64 pipe's latency less well than 28).  The shared-memory wavefronts fall by 30 % as intended (ncu: l1tex
// 67 % -> 52 %), but the time barely moves: with every pipe at or below half load what bounds both kernels
// is the lock-step of the warps of the one CTA per SM.  Letting them drift (each pair synchronising with
// its two neighbours only, through 15 named barriers) is correct but slower (FP32 S = 3 1.40): planes apart
// in z are then in flight at once and DRAM locality suffers.  Opt-in: PRS_OPT_TBS_ROWS = 2.
//
// Rows near the tile edge: pair w runs min(S, 2 min(w, RP-1-w) + 1) stages on both of its rows; where
// that is more than a row is good for, the row computes values nobody uses (neighbour offsets are
// clamped to the tile, results are neither stored nor read by a row that is stored).
#pragma once

#include "prs_kernels_tbs.cuh"

namespace prs {

template <typename T, int S, int TY>
constexpr size_t tbr_smem_bytes() {
    return (size_t)(4 + 4 + 2 * (S - 1)) * (TY + 2 * S) * 32 * 16 + 64;       // + four mbarriers (bulk loader)
}

// BULK: the rings are filled by TMA bulk copies (see step3d_tbs_kernel): one elected lane per warp copies the
// warp's two rows of both rings, 512 bytes each (two runs where the row straddles the periodic seam in x); the
// first warp, which runs a single stage, waits on the slot's mbarrier before it joins the CTA barrier.
template <typename T, int ARITH, int S, int TY, bool BULK>
__global__ void __launch_bounds__(16 * (TY + 2 * S), (TY + 2 * S <= 16) ? 2 : 1)
step3d_tbr_kernel(const T* __restrict__ phi, const T* __restrict__ phidot, T* __restrict__ phi_out,
                  T* __restrict__ phidot_out, int N, int ZC, StepCoefs<T, S> coefs, ZRange zr) {
    using K = Pk<T>;
    using V = typename K::V;
    using std::integral_constant;
    constexpr int W = K::W;
    constexpr int XH = tbs_xhalo<T, S>(), XOUT = tbs_xout<T, S>();
    constexpr int ROWS = TY + 2 * S;
    static_assert(ROWS % 2 == 0, "two rows per thread");
    constexpr int RP = ROWS / 2;                                     // row pairs = warps
    constexpr int PLANE = ROWS * 32;                                 // vectors per shared plane
    extern __shared__ __align__(16) unsigned char tbr_smem[];
    const int lane = threadIdx.x, pr = threadIdx.y;
    const int row0 = 2 * pr;                                         // the lower row; the upper one is row0 + 1
    const int me = row0 * 32 + lane;
    V* const sA = reinterpret_cast<V*>(tbr_smem) + me;               // ring A [4][PLANE], slot of the lower row
    V* const sP = sA + 4 * PLANE;                                    // ring P [4][PLANE]
    V* const sB = sP + 4 * PLANE;                                    // published planes [S-1][2][PLANE]
    // neighbour rows outside the pair, as offsets from the lower row's slot, clamped to the tile
    const int dn = (row0 > 0) ? -32 : 0;
    const int up = (row0 + 2 < ROWS) ? 64 : 32;

    const int NQ = N / W;
    const int qraw = XOUT * (int)blockIdx.x - XH + lane;
    const int q = wrap_mod(qraw, NQ);
    const int yraw = TY * (int)blockIdx.y - S + row0;
    const int y0 = wrap_mod(yraw, N), y1 = wrap_mod(yraw + 1, N);
    const int z0 = zr.lo + (int)blockIdx.z * ZC;
    const int zend = min(z0 + ZC, zr.hi);
    const int niter = (zend - z0) + 2 * S - 2;                       // >= 2S-1
    const bool lanes_ok = (lane >= XH) && (lane < 32 - XH) && (qraw < NQ);
    const bool st0 = lanes_ok && (row0 >= S) && (row0 < S + TY) && (yraw < N);
    const bool st1 = lanes_ok && (row0 + 1 >= S) && (row0 + 1 < S + TY) && (yraw + 1 < N);

    PackCoef<T> pc[S];
#pragma unroll
    for (int s = 0; s < S; ++s) {
        pc[s].template set<3>(coefs.k[s]);
        // 1/phi0^2 and deta do not depend on the step (prs_host.cuh, coef_at): one register serves all stages
        pc[s].I = pc[0].I; pc[s].deta = pc[0].deta;
    }

    // unsigned 32-bit indices of 16-byte vectors, as in step3d_tbs_kernel
    const V* const gA = reinterpret_cast<const V*>(phi);
    const V* const gP = reinterpret_cast<const V*>(phidot);
    V* const oA = reinterpret_cast<V*>(phi_out);
    V* const oP = reinterpret_cast<V*>(phidot_out);
    const unsigned NNv = (unsigned)N * (unsigned)NQ;                 // vectors per plane
    const unsigned colv = (unsigned)y0 * (unsigned)NQ + (unsigned)q; // the lower row's column within a plane
    const unsigned dhi = ((unsigned)y1 - (unsigned)y0) * (unsigned)NQ;   // to the upper row's (modulo 2^32)
    int zl = wrap_mod(z0 - S, zr.nz);
    // bulk loader: mbarriers, and the pair's rows as warp-uniform values (a shuffle from lane 0: UBLKCP takes
    // uniform registers only)
    const unsigned bars = smem_u32(tbr_smem + (size_t)(4 + 4 + 2 * (S - 1)) * PLANE * 16);       // full[4], 8 bytes each
    if constexpr (BULK) {
        if (me == 0) {
#pragma unroll
            for (int u = 0; u < 4; ++u) mbar_init(bars + 8 * u, RP);                               // one arrival per warp
            mbar_init_fence();
        }
        __syncthreads();
    }
    const int pr_u = BULK ? __shfl_sync(0xffffffffu, pr, 0) : pr;
    const int q0 = wrap_mod(XOUT * (int)blockIdx.x - XH, NQ);       // first vector of the tile's rows (periodic)
    const unsigned len0 = (unsigned)min(32, NQ - q0) * 16u, len1 = 512u - len0;   // bytes before / after the x seam
    const unsigned rowA = smem_u32(tbr_smem) + (unsigned)pr_u * 1024u;             // the pair's lower row of ring A, slot 0
    const unsigned rowP = rowA + 4u * PLANE * 16u;
    const bool leader = BULK ? elect_one() : false;
    const int yu = TY * (int)blockIdx.y - S + 2 * pr_u;
    const unsigned rowv = (unsigned)wrap_mod(yu, N) * (unsigned)NQ + (unsigned)q0;                // lower row, first run
    const unsigned dhu = ((unsigned)wrap_mod(yu + 1, N) - (unsigned)wrap_mod(yu, N)) * (unsigned)NQ;
    // load cursor (issue i = plane a = i): of this thread's column (cp.async) or of the warp's lower row (bulk)
    unsigned il = (unsigned)zl * NNv + (BULK ? rowv : colv);
    int left_to_wrap = zr.nz - zl;                                   // issues until z wraps to 0
    unsigned io = (unsigned)z0 * NNv + colv;                         // store cursor

    auto march = [&](auto ns_tag) {
        constexpr int NS = decltype(ns_tag)::value;                  // stages this pair runs (>= 1)
        int ni = 0;
        auto issue = [&](int slot_a, int slot_p) {
            if constexpr (BULK) {
                if (leader) {          // unconditional, as in step3d_tbs_kernel: every issue is the same four copies
                    const unsigned bar = bars + 8u * (unsigned)slot_a;
                    mbar_arrive_expect_tx(bar, 2048u);
                    const unsigned d = rowA + (unsigned)slot_a * (PLANE * 16u), e = rowP + (unsigned)slot_p * (PLANE * 16u);
                    bulk_g2s(d, gA + il, len0, bar);
                    bulk_g2s(d + 512u, gA + (il + dhu), len0, bar);
                    bulk_g2s(e, gP + il, len0, bar);
                    bulk_g2s(e + 512u, gP + (il + dhu), len0, bar);
                    if (len1) {
                        bulk_g2s(d + len0, gA + (il - (unsigned)q0), len1, bar);
                        bulk_g2s(d + 512u + len0, gA + (il + dhu - (unsigned)q0), len1, bar);
                        bulk_g2s(e + len0, gP + (il - (unsigned)q0), len1, bar);
                        bulk_g2s(e + 512u + len0, gP + (il + dhu - (unsigned)q0), len1, bar);
                    }
                }
            } else {
                if (ni < niter + 2) {
                    cp_async16(sA + slot_a * PLANE, gA + il);
                    cp_async16(sA + slot_a * PLANE + 32, gA + (il + dhi));
                }
                if (ni >= 1 && ni <= niter) {
                    cp_async16(sP + slot_p * PLANE, gP + il);
                    cp_async16(sP + slot_p * PLANE + 32, gP + (il + dhi));
                }
            }
            ++ni; il += NNv;
            if (--left_to_wrap == 0) { il -= zr.wrap; left_to_wrap = zr.nz; }   // modulo 2^32, exact
        };
        issue(0, 3); issue(1, 0); issue(2, 1);
        unsigned ph[4] = {1u, 1u, 0u, 0u};      // parity of the next phase to wait for on each slot's mbarrier
        if constexpr (BULK) {
            issue(3, 2);
            if (pr_u == 0) { mbar_wait(bars + 0, 0u); mbar_wait(bars + 8, 0u); }       // planes 0 and 1 have landed
            __syncthreads();
        } else {
            cp_async_commit();
            issue(3, 2);
            cp_async_commit();
            cp_async_wait<1>();
        }
        // register windows per stage and row: input field at planes a_s-1, a_s; phidot input at a_s
        V wprev[S][2], wcur[S][2], qcur[S][2];
#pragma unroll
        for (int s = 0; s < S; ++s)
#pragma unroll
            for (int r = 0; r < 2; ++r) { wprev[s][r] = V{}; wcur[s][r] = V{}; qcur[s][r] = V{}; }
        wprev[0][0] = sA[0 * PLANE]; wprev[0][1] = sA[0 * PLANE + 32];
        wcur[0][0] = sA[1 * PLANE]; wcur[0][1] = sA[1 * PLANE + 32];

        auto iteration = [&](auto u_tag, auto act_tag) {
            constexpr int U = decltype(u_tag)::value, PAR = U & 1;
            constexpr int ACTRAW = decltype(act_tag)::value;
            constexpr int ACT = (NS > ACTRAW) ? ACTRAW : NS;
            if constexpr (BULK) {
                if constexpr (NS == 1) {        // the first warp runs one stage: it has the time to wait for issue j+2
                    if (pr_u == 0) mbar_wait(bars + 8u * (unsigned)((U + 2) & 3), ph[(U + 2) & 3]);
                    ph[(U + 2) & 3] ^= 1u;
                }
            } else {
                cp_async_wait<1>();             // group j has landed for this thread
            }
            PRS_JITTER(1u);
            __syncthreads();                    // ... and for every thread; retires iteration j-1's reads
            PRS_JITTER(2u);
            issue(U, (U + 3) & 3);              // issue j+4: plane j+4 takes the slot of plane j
            if constexpr (!BULK) cp_async_commit();
            PRS_JITTER(3u);
            V carry[2], qout[S][2];
            {   // stage 0 on plane a = j+1
                const V zp0 = sA[((U + 2) & 3) * PLANE], zp1 = sA[((U + 2) & 3) * PLANE + 32];
                const V ym = sA[((U + 1) & 3) * PLANE + dn], yp = sA[((U + 1) & 3) * PLANE + up];
                const V pd0 = sP[U * PLANE], pd1 = sP[U * PLANE + 32];
                const T l0 = __shfl_up_sync(0xffffffffu, K::last(wcur[0][0]), 1);
                const T r0 = __shfl_down_sync(0xffffffffu, K::first(wcur[0][0]), 1);
                const T l1 = __shfl_up_sync(0xffffffffu, K::last(wcur[0][1]), 1);
                const T r1 = __shfl_down_sync(0xffffffffu, K::first(wcur[0][1]), 1);
                V out0, out1;
                packed_vector_update<T, 3, ARITH>(pc[0], wcur[0][0], l0, r0, ym, wcur[0][1], wprev[0][0], zp0, pd0, out0, qout[0][0]);
                packed_vector_update<T, 3, ARITH>(pc[0], wcur[0][1], l1, r1, wcur[0][0], yp, wprev[0][1], zp1, pd1, out1, qout[0][1]);
                PRS_JITTER(4u);
                if (S > 1) { sB[(0 * 2 + PAR) * PLANE] = out0; sB[(0 * 2 + PAR) * PLANE + 32] = out1; }
                wprev[0][0] = wcur[0][0]; wprev[0][1] = wcur[0][1];
                wcur[0][0] = zp0; wcur[0][1] = zp1;
                carry[0] = out0; carry[1] = out1;
            }
            static_for<1, ACT>([&](auto s_tag) {                     // stage s on plane a = j+1-s
                constexpr int s = decltype(s_tag)::value;
                const V* Bs = sB + ((s - 1) * 2 + (PAR ^ 1)) * PLANE;          // published one iteration ago
                const V ym = Bs[dn], yp = Bs[up];
                const T l0 = __shfl_up_sync(0xffffffffu, K::last(wcur[s][0]), 1);
                const T r0 = __shfl_down_sync(0xffffffffu, K::first(wcur[s][0]), 1);
                const T l1 = __shfl_up_sync(0xffffffffu, K::last(wcur[s][1]), 1);
                const T r1 = __shfl_down_sync(0xffffffffu, K::first(wcur[s][1]), 1);
                V out0, out1;
                packed_vector_update<T, 3, ARITH>(pc[s], wcur[s][0], l0, r0, ym, wcur[s][1], wprev[s][0], carry[0], qcur[s][0], out0, qout[s][0]);
                packed_vector_update<T, 3, ARITH>(pc[s], wcur[s][1], l1, r1, wcur[s][0], yp, wprev[s][1], carry[1], qcur[s][1], out1, qout[s][1]);
                if constexpr (s < S - 1) {
                    PRS_JITTER(5u + s);
                    sB[(s * 2 + PAR) * PLANE] = out0; sB[(s * 2 + PAR) * PLANE + 32] = out1;
                } else {
                    if (st0) { oP[io] = qout[s][0]; oA[io] = out0; }
                    if (st1) { oP[io + dhi] = qout[s][1]; oA[io + dhi] = out1; }
                    io += NNv;
                }
                wprev[s][0] = wcur[s][0]; wprev[s][1] = wcur[s][1];
                wcur[s][0] = carry[0]; wcur[s][1] = carry[1];
                carry[0] = out0; carry[1] = out1;
            });
            if constexpr (ACT < NS) {           // feed the window of the stage that has not started yet
                wprev[ACT][0] = wcur[ACT][0]; wprev[ACT][1] = wcur[ACT][1];
                wcur[ACT][0] = carry[0]; wcur[ACT][1] = carry[1];
            }
            static_for<1, (ACT < NS ? ACT + 1 : NS)>([&](auto s_tag) {
                constexpr int s = decltype(s_tag)::value;
                qcur[s][0] = qout[s - 1][0]; qcur[s][1] = qout[s - 1][1];
            });
        };
        // start-up: iterations 0 .. 2S-3, stage s joins at j = 2s
        static_for<0, 2 * S - 2>([&](auto j_tag) {
            constexpr int j = decltype(j_tag)::value;
            iteration(integral_constant<int, j & 3>{}, integral_constant<int, j / 2 + 1>{});
        });
        // steady state from j = 2S-2, unrolled four times
        constexpr int J0 = 2 * S - 2;
        for (int j = J0; j < niter; j += 4) {
            iteration(integral_constant<int, (J0 + 0) & 3>{}, integral_constant<int, S>{});
            if (j + 1 >= niter) break;
            iteration(integral_constant<int, (J0 + 1) & 3>{}, integral_constant<int, S>{});
            if (j + 2 >= niter) break;
            iteration(integral_constant<int, (J0 + 2) & 3>{}, integral_constant<int, S>{});
            if (j + 3 >= niter) break;
            iteration(integral_constant<int, (J0 + 3) & 3>{}, integral_constant<int, S>{});
        }
        if constexpr (!BULK) cp_async_wait<0>();
    };
    const int nsp = 2 * min(pr, RP - 1 - pr) + 1;                    // stages the pair's better row is good for
    if (nsp >= S) march(integral_constant<int, S>{});
    else if (nsp == 1) march(integral_constant<int, 1>{});
    else if constexpr (S > 3) march(integral_constant<int, 3>{});
}

}  // namespace prs
