// prs_kernels_cluster.cuh -- the small-box regime (small boxes
// under-use a GPU and are dominated by per-step overheads).  A 256^2 lattice is 768 KB of state: every
// kernel launch of the streaming kernels is pure latency.  Here the whole state lives ON CHIP in ONE
// thread-block cluster for many steps: 8 CTAs (256^2: 16), each owning N/8 (N/16) rows.  A thread keeps the phi and phidot
// of its own sites in REGISTERS from the first step of a launch to the last; only phi is published, to
// a ping-pong pair of shared-memory buffers, for the neighbours: rows just across a CTA boundary are read
// from a halo row that the neighbouring CTA fills through distributed shared memory (st.async + mbarrier, below): a
// __syncthreads and a neighbour handshake per step replace a kernel launch.  HBM is touched once on entry and once
// on exit of a launch of up to CLUSTER_MAX_STEPS steps.
//
// The wall diagnostics (Eqs. 7-8) can run INSIDE the launch, at the cadence prs_run asks for:
// after a step's barrier the state is all on chip -- own sites in registers, neighbours in shared memory --
// so a pass costs a few hundred nanoseconds instead of a launch: sign masks, popcounts, Eq. 8's ratio at
// the wall sites in double, a warp reduction into a per-pass, per-warp slot of the CTA's shared memory -- no barrier; at
// the end of the launch each CTA adds up its warps' partials, and the warps of rank 0 fetch the CTAs' partials through
// distributed shared memory and add them, all in a fixed order (reproducible), into the records of the device ring.
//
// Per-site arithmetic: the packed update of prs_pack.cuh, so the fields are bit-identical to the other
// kernels in every arithmetic form; the diagnostics' integer counts are exact, its double sum differs from the
// stand-alone kernels' by the order of the additions only.  2D only, N in {64, 128, 256}.
#pragma once

#include <cooperative_groups.h>

#include "prs_arith.cuh"
#include "prs_pack.cuh"
#include "prs_kernels_tiled.cuh"     // VecOps, sign_mask, mask_links, block_reduce

namespace prs {

constexpr int CLUSTER_CTAS = 8;                  // portable cluster size; 256^2 takes 16 (opt-in, non-portable) where it fits
constexpr int CLUSTER_THREADS = 1024;
constexpr int CLUSTER_MAX_STEPS = 64;

// 16-byte vectors a thread owns (template argument VPT): N^2 / (8 CTAs x W x 1024 threads), at least 1 --
// with 8 CTAs 1 for N = 64, 128; 2 for 256^2 FP32; 4 for 256^2 FP64; with 16 CTAs 1 / 2 for 256^2 FP32 / FP64
template <typename T>
constexpr int cluster_vpt(int N, int ncta = CLUSTER_CTAS) {
    return (N / ncta) * (N / Pk<T>::W) <= CLUSTER_THREADS ? 1 : (N / ncta) * (N / Pk<T>::W) / CLUSTER_THREADS;
}

// The cluster barrier as its two halves: shared-memory writes before the arrive are visible to every CTA of the cluster
// after the wait.  Used at the start and the end of a launch only: its release compiles to a MEMBAR.ALL.GPU in every warp
// (as cooperative_groups' cluster.sync() does), 13 % `membar` stall in ncu when every step ended in one.
__device__ __forceinline__ void cluster_barrier() {
    asm volatile("barrier.cluster.arrive.release.aligned;\nbarrier.cluster.wait.acquire.aligned;\n" ::: "memory");
}

// Between steps a CTA depends on its TWO NEIGHBOURS only, and only through one row each: the row just below its rows and
// the row just above.  So the step loop takes no cluster barrier (measured at ~800 cycles a step: its release is a
// MEMBAR.ALL.GPU in every warp) and reads no remote shared memory (~215 cycles a load).  Instead the threads that own a
// CTA's first / last row PUSH the vectors they have just computed into a halo row in the neighbour's shared memory with
// st.async, whose bytes are counted on an mbarrier in that neighbour (complete_tx): data and signal travel together, no
// fence.  The neighbour's boundary-row threads wait on that mbarrier (acquire, cluster scope) right before they read the
// halo; everyone else needs the CTA's own __syncthreads only, so the inner rows of step s+1 run while the halo rows
// of phi^{s+1} are in flight.
//
// The halo rows are rows 0 and R + 1 of the two phi buffers, which alternate with the parity of the step.  Those of buffer
// (s+1)&1 receive phi^{s+1} during the neighbours' step s and are read in step s+1; they are written again in the
// neighbours' step s+2, which cannot start before this CTA's boundary rows of step s+1 have arrived there -- pushed by the
// very threads that read the halo rows, after they read them.  Each buffer and side has its own mbarrier (one arrival, by
// the thread that arms it with the row's byte count for the next use, plus the bytes); the arming thread is one of the
// row's pushers and arms before it pushes, so an arming always precedes the bytes it counts.
__device__ __forceinline__ unsigned cluster_smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ unsigned cluster_map(unsigned local, unsigned rank) {
    unsigned remote;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;\n" : "=r"(remote) : "r"(local), "r"(rank));
    return remote;
}
__device__ __forceinline__ void halo_bar_init(unsigned bar) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;\n" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void halo_arm(unsigned bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void halo_wait(unsigned bar, unsigned parity) {
    asm volatile(
        "{\n.reg .pred p;\nHALO_WAIT:\n"
        "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%0], %1;\n"
        "@p bra HALO_DONE;\nbra HALO_WAIT;\nHALO_DONE:\n}\n" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void halo_push(unsigned remote, unsigned remote_bar, unsigned long long a, unsigned long long b) {
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.b64 [%0], {%1, %2}, [%3];\n" ::"r"(remote), "l"(a),
                 "l"(b), "r"(remote_bar)
                 : "memory");
}
__device__ __forceinline__ void halo_push(unsigned remote, unsigned remote_bar, ulonglong2 v) { halo_push(remote, remote_bar, v.x, v.y); }
__device__ __forceinline__ void halo_push(unsigned remote, unsigned remote_bar, double2 v) {
    halo_push(remote, remote_bar, (unsigned long long)__double_as_longlong(v.x), (unsigned long long)__double_as_longlong(v.y));
}

// A packed vector (prs_pack.cuh) as the plain vector type of the diagnostics code, register to register.
__device__ __forceinline__ float4 plain_vec(ulonglong2 v) {
    float4 f;
    Pk<float>::unpack(v.x, f.x, f.y);
    Pk<float>::unpack(v.y, f.z, f.w);
    return f;
}
__device__ __forceinline__ double2 plain_vec(double2 v) { return v; }

template <typename T>
struct ClusterCoefs {
    StepCoef<T> k[CLUSTER_MAX_STEPS];
};

// When the diagnostics run inside a launch, and where their records go.
struct ClusterDiag {
    int every;                  // PRS steps between passes; 0 = no pass in this launch
    int until;                  // steps from the launch's first step to its first pass (1 <= until <= every)
    DiagPartial* records;       // DEVICE: the record of the launch's first pass; the following ones follow it
    double V0, I;               // Eq. 8's constants
};

constexpr size_t CLUSTER_SMEM_LIMIT = 176 * 1024;      // dynamic shared memory the kernels are configured for (most used: 168 KiB)

// What a warp keeps of a diagnostics pass until the end of the launch (its 32 vectors x VPT: the counts fit 16 bits).
struct ClusterWarpPart {
    unsigned links, walls;
    double sum;
};

template <typename T>
constexpr size_t cluster_smem_bytes(int N, int ncta = CLUSTER_CTAS) {
    return (size_t)2 * (size_t)(N / ncta + 2) * (size_t)N * sizeof(T)               // phi, ping and pong, each with its two halo rows
           + (size_t)CLUSTER_MAX_STEPS * (CLUSTER_THREADS / 32) * sizeof(ClusterWarpPart);      // the warps' partials, per pass
}

template <typename T, int ARITH, int VPT, int NCTA>
__global__ void __cluster_dims__(NCTA, 1, 1) __launch_bounds__(CLUSTER_THREADS, 1)
step2d_cluster_kernel(const T* __restrict__ phi, const T* __restrict__ phidot, T* __restrict__ phi_out,
                      T* __restrict__ phidot_out, int N, int nsteps, ClusterCoefs<T> coefs, ClusterDiag dg) {
    namespace cg = cooperative_groups;
    cg::cluster_group cluster = cg::this_cluster();
    extern __shared__ __align__(16) unsigned char cluster_smem[];
    __shared__ DiagPartial cta_part[CLUSTER_MAX_STEPS];              // this CTA's partials of the launch's diagnostics passes
    __shared__ __align__(8) unsigned long long halo_bar[2][2];       // [buffer][0: the row below arrives here, 1: the row above]
    using K = Pk<T>;
    using V = typename K::V;
    using O = VecOps<T>;
    constexpr int W = K::W;
    const int R = N / NCTA;                                          // rows held by this CTA
    const int RN = R * N;
    // Two phi buffers of R + 2 rows: row 0 is the halo row below the CTA's rows (the last row of the CTA below, pushed by
    // that CTA), rows 1 .. R its own, row R + 1 the halo row above.  A site's y neighbours are at -N and +N whatever the row.
    const int BUF = (R + 2) * N;
    T* const buf0 = reinterpret_cast<T*>(cluster_smem);
    T* const buf1 = buf0 + BUF;
    ClusterWarpPart* const warp_part = reinterpret_cast<ClusterWarpPart*>(buf1 + BUF);           // [pass][warp]
    const unsigned rank = cluster.block_rank();
    const unsigned below = (rank + NCTA - 1) % NCTA, above = (rank + 1) % NCTA;
    const unsigned row_bytes = (unsigned)N * (unsigned)sizeof(T), buf_bytes = (unsigned)BUF * (unsigned)sizeof(T);

    const int t = threadIdx.x;
    const int NQ = N / W, RNQ = R * NQ;                              // NQ is a power of two (N = 64, 128, 256)
    const int lgNQ = 31 - __clz(NQ);
    const size_t base = (size_t)rank * RN;                           // first site of this CTA's rows
    const unsigned bars = cluster_smem_u32(&halo_bar[0][0]);
    if (t == 0) {
        for (unsigned i = 0; i < 4; ++i) halo_bar_init(bars + 8u * i);
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
        for (unsigned i = 0; i < 4; ++i) halo_arm(bars + 8u * i, row_bytes);       // buffer 1: the pushes of step 0, buffer 0: of step 1
    }
    // where this CTA's first row goes: the halo row above the rows of the CTA below it (row R + 1 there); its last row: the
    // halo row below the rows of the CTA above (row 0 there) -- addresses in buffer 0, buffer 1 is buf_bytes further
    const unsigned push_down = cluster_map(cluster_smem_u32(buf0 + (R + 1) * N), below);
    const unsigned push_down_bar = cluster_map(bars + 8u, below);
    const unsigned push_up = cluster_map(cluster_smem_u32(buf0), above);
    const unsigned push_up_bar = cluster_map(bars, above);

    // A thread owns vectors v = t, t + 1024, ... of the CTA's R x NQ: phi and phidot stay in registers; what does not change
    // from step to step -- where the vector and its x neighbours sit in a buffer, whether it is in a boundary row -- is
    // worked out once.
    V creg[VPT], pdreg[VPT];
    int oc[VPT], ol[VPT], orr[VPT];
    bool first[VPT], last[VPT];
#pragma unroll
    for (int k = 0; k < VPT; ++k) {
        const int v = t + k * CLUSTER_THREADS;
        const int r = v >> lgNQ, x = (v & (NQ - 1)) * W;
        oc[k] = (r + 1) * N + x;
        ol[k] = (r + 1) * N + (x == 0 ? N - 1 : x - 1);
        orr[k] = (r + 1) * N + (x + W == N ? 0 : x + W);
        first[k] = (v < RNQ) && r == 0;
        last[k] = (v < RNQ) && r == R - 1;
        creg[k] = V{}; pdreg[k] = V{};
        if (v < RNQ) {
            creg[k] = K::ldg(phi + base + (size_t)v * W);
            pdreg[k] = K::ldg(phidot + base + (size_t)v * W);
            *reinterpret_cast<V*>(buf0 + oc[k]) = creg[k];
        }
    }
    if (t < 2 * NQ) {
        // the halo rows of buffer 0 for step 0: the rows around this CTA's rows straight from global memory (periodic in y)
        const int side = t >> lgNQ, q = t & (NQ - 1);
        const int grow = side == 0 ? ((int)rank * R + N - 1) % N : ((int)rank * R + R) % N;
        reinterpret_cast<V*>(buf0 + side * (R + 1) * N)[q] = K::ldg(phi + (size_t)grow * N + (size_t)q * W);
    }
    cluster_barrier();                                               // the state is on chip; every CTA's mbarriers are armed

    int next_diag = dg.every > 0 ? dg.until : -1;                    // the pass follows local step next_diag - 1
    int rec = 0;
    for (int s = 0; s < nsteps; ++s) {
        PackCoef<T> kc;
        kc.template set<2>(coefs.k[s]);
        const bool odd = (s & 1) != 0;
        const T* const src = odd ? buf1 : buf0;
        T* const dst = odd ? buf0 : buf1;
        const unsigned sbar = bars + (odd ? 16u : 0u);               // the barriers of the buffer read in this step
        const unsigned par = (unsigned)((s - 1) >> 1) & 1u;          // the buffer's use that holds phi^s (s >= 1)
        const unsigned dpush = odd ? 0u : buf_bytes, dbar = odd ? 0u : 16u;          // the buffer filled for the next step
#pragma unroll
        for (int k = 0; k < VPT; ++k) {
            if (t + k * CLUSTER_THREADS < RNQ) {
                if (s > 0 && first[k]) {                             // the neighbour's row of phi^s has landed?
                    halo_wait(sbar, par);
                    if (ol[k] != oc[k] - 1) halo_arm(sbar, row_bytes);               // (the thread at x = 0) for the next use, two steps on
                }
                if (s > 0 && last[k]) {
                    halo_wait(sbar + 8u, par);
                    if (ol[k] != oc[k] - 1) halo_arm(sbar + 8u, row_bytes);
                }
                const V ym = *reinterpret_cast<const V*>(src + oc[k] - N);
                const V yp = *reinterpret_cast<const V*>(src + oc[k] + N);
                const T left = src[ol[k]];
                const T right = src[orr[k]];
                V pn, vn;
                packed_vector_update<T, 2, ARITH>(kc, creg[k], left, right, ym, yp, V{}, V{}, pdreg[k], pn, vn);
                creg[k] = pn; pdreg[k] = vn;
                *reinterpret_cast<V*>(dst + oc[k]) = pn;
                // (x * sizeof(T): the vector's offset within its row = its offset in the buffer minus the row's)
                if (first[k]) halo_push(push_down + dpush + (unsigned)(oc[k] - N) * (unsigned)sizeof(T), push_down_bar + dbar, pn);
                if (last[k]) halo_push(push_up + dpush + (unsigned)(oc[k] - RN) * (unsigned)sizeof(T), push_up_bar + dbar, pn);
            }
        }
        // this CTA has published phi^{s+1} to itself and is done reading phi^s, whose buffer is overwritten next step
        PRS_JITTER(1u + s);
        __syncthreads();
        PRS_JITTER(80u + s);
        if (s + 1 == next_diag) {
            // ---- Eqs. 7-8 on the state just reached: own sites in registers, neighbours in dst, whose halo rows the
            // neighbours have just filled (or are filling)
            const T* const cur = dst;
            const unsigned cbar = bars + (odd ? 0u : 16u);
            const unsigned dpar = (unsigned)(s >> 1) & 1u;
            unsigned acc_links = 0u, acc_walls = 0u;
            double acc_sum = 0.0;
#pragma unroll
            for (int k = 0; k < VPT; ++k) {
                if (t + k * CLUSTER_THREADS < RNQ) {
                    if (first[k]) halo_wait(cbar, dpar);             // (armed again by the next step, not here)
                    if (last[k]) halo_wait(cbar + 8u, dpar);
                    const typename O::V c = plain_vec(creg[k]);
                    const typename O::V q = plain_vec(pdreg[k]);
                    const typename O::V ym = *reinterpret_cast<const typename O::V*>(cur + oc[k] - N);
                    const typename O::V yp = *reinterpret_cast<const typename O::V*>(cur + oc[k] + N);
                    const unsigned l = Ar<T>::neg(cur[ol[k]]) ? 1u : 0u;
                    const unsigned rr = Ar<T>::neg(cur[orr[k]]) ? 1u : 0u;
                    const unsigned mc = sign_mask<T>(c);
                    unsigned nlinks, wallmask;
                    mask_links<W, 2>(mc, l, rr, sign_mask<T>(ym), sign_mask<T>(yp), mc, mc, nlinks, wallmask);
                    acc_links += nlinks;
                    acc_walls += (unsigned)__popc(wallmask);
#pragma unroll
                    for (int i = 0; i < W; ++i)
                        if ((wallmask >> i) & 1u) acc_sum = __dadd_rn(acc_sum, wall_ratio<T>(O::get(c, i), O::get(q, i), dg.V0, dg.I));
                }
            }
            // The pass ends inside the WARP, without a barrier: one redux for both counts (16 bits each are plenty for a
            // warp's 32 x VPT vectors), a shuffle tree for the double, and the warp's partial waits in shared memory for
            // the end of the launch, where all passes are added up behind one __syncthreads and ONE cluster barrier (a block
            // reduction and a cluster barrier per pass cost 2.5 us a pass, 3.5 steps' worth).
            const unsigned counts = __reduce_add_sync(0xffffffffu, acc_links | (acc_walls << 16));
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) acc_sum = __dadd_rn(acc_sum, __shfl_down_sync(0xffffffffu, acc_sum, d));
            if ((t & 31) == 0) {
                ClusterWarpPart wp;
                wp.links = counts & 0xffffu; wp.walls = counts >> 16; wp.sum = acc_sum;
                warp_part[rec * (CLUSTER_THREADS / 32) + (t >> 5)] = wp;
            }
            PRS_JITTER(160u + s);
            ++rec;
            next_diag += dg.every;
        }
    }
    const unsigned fbar = bars + ((nsteps & 1) ? 16u : 0u), fpar = (unsigned)((nsteps - 1) >> 1) & 1u;
#pragma unroll
    for (int k = 0; k < VPT; ++k) {
        const int v = t + k * CLUSTER_THREADS;
        if (v < RNQ) {
            K::stg(phi_out + base + (size_t)v * W, creg[k]);
            K::stg(phidot_out + base + (size_t)v * W, pdreg[k]);
            // the neighbours' pushes of the last step land in this CTA's shared memory: it must outlive them
            if (nsteps > 0 && first[k]) halo_wait(fbar, fpar);
            if (nsteps > 0 && last[k]) halo_wait(fbar + 8u, fpar);
        }
    }
    if (rec > 0) {
        const int lane = t & 31;
        __syncthreads();                                             // the warps' partials of every pass are written
        // warp w adds up passes w, w + 32: lane l takes warp l's partial, then the shuffle tree -- a fixed order
        for (int w = t >> 5; w < rec; w += CLUSTER_THREADS / 32) {
            const ClusterWarpPart wp = warp_part[w * (CLUSTER_THREADS / 32) + lane];
            DiagPartial part = {(unsigned long long)wp.links, (unsigned long long)wp.walls, wp.sum};
            part = warp_reduce(part);
            if (lane == 0) cta_part[w] = part;
        }
        PRS_JITTER(200u);
        cluster_barrier();                                           // every CTA's partials are written
        if (rank == 0) {
            // warp w of rank 0 takes passes w, w + 32: lane l fetches CTA l's partial (the remote reads overlap instead of
            // queueing up), then the shuffle tree of warp_reduce adds them -- an order fixed by the lane numbers alone
            for (int w = t >> 5; w < rec; w += CLUSTER_THREADS / 32) {
                DiagPartial part = {0ull, 0ull, 0.0};
                if (lane < NCTA) {
                    const DiagPartial* rp = cluster.map_shared_rank(&cta_part[w], (unsigned)lane);
                    part.links = rp->links; part.walls = rp->walls; part.sum = rp->sum;
                }
                part = warp_reduce(part);
                if (lane == 0) dg.records[w] = part;
            }
        }
        PRS_JITTER(240u);
        cluster_barrier();                                           // no CTA exits while rank 0 reads its shared memory
    }
}

}  // namespace prs
