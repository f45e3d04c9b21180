// prs_kernels_cluster.cuh -- the small-box regime (small boxes
// under-use a GPU and are dominated by per-step overheads).  A 256^2 lattice is 768 KB of state: every
// kernel launch of the streaming kernels is pure latency.  Here the whole state lives ON CHIP in ONE
// thread-block cluster for many steps: 8 CTAs, each owning N/8 rows.  A thread keeps the phi and phidot
// of its own sites in REGISTERS from the first step of a launch to the last; only phi is published, to
// a ping-pong pair of shared-memory buffers, for the neighbours: rows just across a CTA boundary are read
// from the neighbouring CTA's shared memory (distributed shared memory), and one cluster barrier per step
// replaces a kernel launch.  HBM is touched once on entry and once on exit of a launch of up to
// CLUSTER_MAX_STEPS steps.
//
// The wall diagnostics (Eqs. 7-8) can run INSIDE the launch, at the cadence prs_run asks for:
// after a step's barrier the state is all on chip -- own sites in registers, neighbours in shared memory --
// so a pass costs a few hundred nanoseconds instead of a launch: sign masks, popcounts, Eq. 8's ratio at
// the wall sites in double, block reduction, and one warp of rank 0 fetches the CTAs' partials through distributed
// shared memory and adds them in a fixed order (reproducible) into the next record of the device ring.
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

// The cluster barrier as its two halves with exactly the ordering the kernel needs: shared-memory writes before the arrive
// are visible to every CTA of the cluster after the wait.  (cooperative_groups' cluster.sync() showed a `membar` stall of
// 13 % in ncu: it fences more than that.)
__device__ __forceinline__ void cluster_barrier() {
    asm volatile("barrier.cluster.arrive.release.aligned;\nbarrier.cluster.wait.acquire.aligned;\n" ::: "memory");
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

template <typename T>
constexpr size_t cluster_smem_bytes(int N, int ncta = CLUSTER_CTAS) {
    return (size_t)2 * (size_t)(N / ncta) * (size_t)N * sizeof(T);                  // phi, ping and pong
}

template <typename T, int ARITH, int VPT, int NCTA>
__global__ void __cluster_dims__(NCTA, 1, 1) __launch_bounds__(CLUSTER_THREADS, 1)
step2d_cluster_kernel(const T* __restrict__ phi, const T* __restrict__ phidot, T* __restrict__ phi_out,
                      T* __restrict__ phidot_out, int N, int nsteps, ClusterCoefs<T> coefs, ClusterDiag dg) {
    namespace cg = cooperative_groups;
    cg::cluster_group cluster = cg::this_cluster();
    extern __shared__ __align__(16) unsigned char cluster_smem[];
    __shared__ DiagPartial cta_part;                                 // this CTA's partial of a diagnostics pass
    using K = Pk<T>;
    using V = typename K::V;
    using O = VecOps<T>;
    constexpr int W = K::W;
    const int R = N / NCTA;                                          // rows held by this CTA
    const int RN = R * N;
    // (scalars picked by selects, not arrays indexed by the step's parity: those would live in local memory)
    T* const buf0 = reinterpret_cast<T*>(cluster_smem);
    T* const buf1 = buf0 + RN;
    const unsigned rank = cluster.block_rank();
    const unsigned below = (rank + NCTA - 1) % NCTA, above = (rank + 1) % NCTA;
    // the two phi buffers of the CTAs that hold the rows below / above this CTA's rows
    const T* const below0 = cluster.map_shared_rank(buf0, below);
    const T* const below1 = cluster.map_shared_rank(buf1, below);
    const T* const above0 = cluster.map_shared_rank(buf0, above);
    const T* const above1 = cluster.map_shared_rank(buf1, above);

    const int t = threadIdx.x;
    const int NQ = N / W, RNQ = R * NQ;                              // NQ is a power of two (N = 64, 128, 256)
    const int lgNQ = 31 - __clz(NQ);
    const size_t base = (size_t)rank * RN;                           // first site of this CTA's rows

    // A thread owns vectors v = t, t + 1024, ... of the CTA's R x NQ: phi and phidot stay in registers.
    V creg[VPT], pdreg[VPT];
#pragma unroll
    for (int k = 0; k < VPT; ++k) {
        const int v = t + k * CLUSTER_THREADS;
        creg[k] = V{}; pdreg[k] = V{};
        if (v < RNQ) {
            creg[k] = K::ldg(phi + base + (size_t)v * W);
            pdreg[k] = K::ldg(phidot + base + (size_t)v * W);
            reinterpret_cast<V*>(buf0)[v] = creg[k];
        }
    }
    cluster_barrier();

    int next_diag = dg.every > 0 ? dg.until : -1;                    // the pass follows local step next_diag - 1
    int rec = 0;
    bool tail_sync = false;
    for (int s = 0; s < nsteps; ++s) {
        PackCoef<T> kc;
        kc.template set<2>(coefs.k[s]);
        const bool odd = (s & 1) != 0;
        const T* const src = odd ? buf1 : buf0;
        T* const dst = odd ? buf0 : buf1;
        const T* const src_below = odd ? below1 : below0;
        const T* const src_above = odd ? above1 : above0;
#pragma unroll
        for (int k = 0; k < VPT; ++k) {
            const int v = t + k * CLUSTER_THREADS;
            if (v < RNQ) {
                const int r = v >> lgNQ, x = (v & (NQ - 1)) * W;
                const int o = r * N + x;
                const V ym = (r > 0) ? *reinterpret_cast<const V*>(src + o - N)
                                     : *reinterpret_cast<const V*>(src_below + (R - 1) * N + x);
                const V yp = (r < R - 1) ? *reinterpret_cast<const V*>(src + o + N)
                                         : *reinterpret_cast<const V*>(src_above + x);
                const T left = src[r * N + (x == 0 ? N - 1 : x - 1)];
                const T right = src[r * N + (x + W == N ? 0 : x + W)];
                V pn, vn;
                packed_vector_update<T, 2, ARITH>(kc, creg[k], left, right, ym, yp, V{}, V{}, pdreg[k], pn, vn);
                creg[k] = pn; pdreg[k] = vn;
                *reinterpret_cast<V*>(dst + o) = pn;
            }
        }
        // everyone has published phi^{n+1} and is done reading phi^n, whose buffer is overwritten next step
        PRS_JITTER(1u + s);
        cluster_barrier();
        PRS_JITTER(80u + s);
        if (s + 1 == next_diag) {
            // ---- Eqs. 7-8 on the state just reached: own sites in registers, neighbours in dst (and the CTAs beside)
            const T* const cur = dst;
            const T* const cur_below = odd ? below0 : below1;
            const T* const cur_above = odd ? above0 : above1;
            DiagPartial acc = {0ull, 0ull, 0.0};
#pragma unroll
            for (int k = 0; k < VPT; ++k) {
                const int v = t + k * CLUSTER_THREADS;
                if (v < RNQ) {
                    const int r = v >> lgNQ, x = (v & (NQ - 1)) * W;
                    const int o = r * N + x;
                    const typename O::V c = plain_vec(creg[k]);
                    const typename O::V q = plain_vec(pdreg[k]);
                    const typename O::V ym = (r > 0) ? *reinterpret_cast<const typename O::V*>(cur + o - N)
                                                     : *reinterpret_cast<const typename O::V*>(cur_below + (R - 1) * N + x);
                    const typename O::V yp = (r < R - 1) ? *reinterpret_cast<const typename O::V*>(cur + o + N)
                                                         : *reinterpret_cast<const typename O::V*>(cur_above + x);
                    const unsigned l = Ar<T>::neg(cur[r * N + (x == 0 ? N - 1 : x - 1)]) ? 1u : 0u;
                    const unsigned rr = Ar<T>::neg(cur[r * N + (x + W == N ? 0 : x + W)]) ? 1u : 0u;
                    const unsigned mc = sign_mask<T>(c);
                    unsigned nlinks, wallmask;
                    mask_links<W, 2>(mc, l, rr, sign_mask<T>(ym), sign_mask<T>(yp), mc, mc, nlinks, wallmask);
                    acc.links += nlinks;
                    acc.walls += __popc(wallmask);
#pragma unroll
                    for (int i = 0; i < W; ++i)
                        if ((wallmask >> i) & 1u) acc.sum = __dadd_rn(acc.sum, wall_ratio<T>(O::get(c, i), O::get(q, i), dg.V0, dg.I));
                }
            }
            acc = block_reduce(acc);
            if (t == 0) cta_part = acc;
            PRS_JITTER(160u + s);
            cluster_barrier();
            if (rank == 0 && t < 32) {
                // warp 0 of rank 0: lane l fetches CTA l's partial (the remote reads overlap instead of queueing up), then
                // the shuffle tree of warp_reduce adds them -- an order fixed by the lane numbers alone: reproducible
                DiagPartial part = {0ull, 0ull, 0.0};
                if (t < NCTA) {
                    const DiagPartial* rp = cluster.map_shared_rank(&cta_part, (unsigned)t);
                    part.links = rp->links; part.walls = rp->walls; part.sum = rp->sum;
                }
                part = warp_reduce(part);
                if (t == 0) dg.records[rec] = part;
            }
            // cta_part is written again only after a further cluster barrier, which rank 0's thread 0 joins after it has
            // read the partials; but no CTA may EXIT while rank 0 still reads its shared memory: see tail_sync
            tail_sync = (s + 1 == nsteps);
            ++rec;
            next_diag += dg.every;
        }
    }
#pragma unroll
    for (int k = 0; k < VPT; ++k) {
        const int v = t + k * CLUSTER_THREADS;
        if (v < RNQ) {
            K::stg(phi_out + base + (size_t)v * W, creg[k]);
            K::stg(phidot_out + base + (size_t)v * W, pdreg[k]);
        }
    }
    if (tail_sync) cluster_barrier();                                   // a pass after the last step: rank 0 is done reading
}

}  // namespace prs
