// prs_kernels_cluster.cuh -- the small-box regime (small boxes
// under-use a GPU and are dominated by per-step overheads).  A 256^2 lattice is 768 KB of state: every
// kernel launch of the streaming kernels is pure latency.  Here the whole state lives in the shared
// memory of ONE thread-block cluster for many steps: 8 CTAs, each holding N/8 rows of phi (two
// buffers, ping-pong) and phidot; the rows just across a CTA boundary are read from the neighbouring
// CTA's shared memory (distributed shared memory), and one cluster barrier per step replaces a kernel
// launch.  HBM is touched once on entry and once on exit of a launch of up to CLUSTER_MAX_STEPS steps.
//
// Per-site arithmetic: the packed update of prs_pack.cuh, so the result is bit-identical to the other
// kernels in every arithmetic form.  2D only, N in {64, 128, 256}; a thread owns whole 16-byte vectors.
#pragma once

#include <cooperative_groups.h>

#include "prs_arith.cuh"
#include "prs_pack.cuh"

namespace prs {

constexpr int CLUSTER_CTAS = 8;
constexpr int CLUSTER_THREADS = 1024;
constexpr int CLUSTER_MAX_STEPS = 32;

template <typename T>
struct ClusterCoefs {
    StepCoef<T> k[CLUSTER_MAX_STEPS];
};

template <typename T>
constexpr size_t cluster_smem_bytes(int N) {
    return (size_t)3 * (size_t)(N / CLUSTER_CTAS) * (size_t)N * sizeof(T);
}

template <typename T, int ARITH>
__global__ void __cluster_dims__(CLUSTER_CTAS, 1, 1) __launch_bounds__(CLUSTER_THREADS, 1)
step2d_cluster_kernel(const T* __restrict__ phi, const T* __restrict__ phidot, T* __restrict__ phi_out,
                      T* __restrict__ phidot_out, int N, int nsteps, ClusterCoefs<T> coefs) {
    namespace cg = cooperative_groups;
    cg::cluster_group cluster = cg::this_cluster();
    extern __shared__ __align__(16) unsigned char cluster_smem[];
    const int R = N / CLUSTER_CTAS;                                  // rows held by this CTA
    const int RN = R * N;
    T* const bufA = reinterpret_cast<T*>(cluster_smem);
    T* const bufB = bufA + RN;
    T* const pd = bufB + RN;
    const unsigned rank = cluster.block_rank();
    const unsigned below = (rank + CLUSTER_CTAS - 1) % CLUSTER_CTAS, above = (rank + 1) % CLUSTER_CTAS;
    // the two phi buffers of the CTAs that hold the rows below / above this CTA's rows
    const T* const belowA = cluster.map_shared_rank(bufA, below);
    const T* const belowB = cluster.map_shared_rank(bufB, below);
    const T* const aboveA = cluster.map_shared_rank(bufA, above);
    const T* const aboveB = cluster.map_shared_rank(bufB, above);

    // A thread owns whole 16-byte vectors (4 floats / 2 doubles): vector v = t, t+1024, ... of this CTA's
    // R x N/W vectors; the arithmetic is the packed form of prs_pack.cuh.
    using K = Pk<T>;
    using V = typename K::V;
    constexpr int W = K::W;
    const int t = threadIdx.x;
    const int NQ = N / W, RNQ = R * NQ;
    const int lgNQ = 31 - __clz(NQ);
    const size_t base = (size_t)rank * RN;                           // first site of this CTA's rows

    for (int i = t; i < RNQ; i += CLUSTER_THREADS) {
        reinterpret_cast<V*>(bufA)[i] = K::ldg(phi + base + (size_t)i * W);
        reinterpret_cast<V*>(pd)[i] = K::ldg(phidot + base + (size_t)i * W);
    }
    cluster.sync();

    for (int s = 0; s < nsteps; ++s) {
        PackCoef<T> k;
        k.template set<2>(coefs.k[s]);
        const T* const src = (s & 1) ? bufB : bufA;
        T* const dst = (s & 1) ? bufA : bufB;
        const T* const src_below = (s & 1) ? belowB : belowA;
        const T* const src_above = (s & 1) ? aboveB : aboveA;
        for (int v = t; v < RNQ; v += CLUSTER_THREADS) {
            const int r = v >> lgNQ, x = (v & (NQ - 1)) * W;          // NQ is a power of two (N = 64, 128, 256)
            const int o = r * N + x;
            const V c = *reinterpret_cast<const V*>(src + o);
            const V ym = (r > 0) ? *reinterpret_cast<const V*>(src + o - N)
                                 : *reinterpret_cast<const V*>(src_below + (R - 1) * N + x);
            const V yp = (r < R - 1) ? *reinterpret_cast<const V*>(src + o + N)
                                     : *reinterpret_cast<const V*>(src_above + x);
            const T left = src[r * N + (x == 0 ? N - 1 : x - 1)];
            const T right = src[r * N + (x + W == N ? 0 : x + W)];
            const V q = *reinterpret_cast<const V*>(pd + o);
            V pn, vn;
            packed_vector_update<T, 2, ARITH>(k, c, left, right, ym, yp, V{}, V{}, q, pn, vn);
            *reinterpret_cast<V*>(dst + o) = pn;
            *reinterpret_cast<V*>(pd + o) = vn;
        }
        // everyone has written phi^{n+1} and is done reading phi^n, which is overwritten next step
        PRS_JITTER(1u + s);
        cluster.sync();
        PRS_JITTER(40u + s);
    }
    const T* const fin = (nsteps & 1) ? bufB : bufA;
    for (int i = t; i < RNQ; i += CLUSTER_THREADS) {
        K::stg(phi_out + base + (size_t)i * W, reinterpret_cast<const V*>(fin)[i]);
        K::stg(phidot_out + base + (size_t)i * W, reinterpret_cast<const V*>(pd)[i]);
    }
}

}  // namespace prs
