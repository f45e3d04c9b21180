// prs_kernels_generic.cuh -- kernels that take any lattice size N >= 1: the seeded initial condition,
// a one-thread-per-site step, a grid-stride diagnostics pass and the final reduction.
#pragma once

#include "prs_arith.cuh"

namespace prs {

// ------------------------------------------------------------------------------------------------
// Initial condition.  Philox4x32-10 (Salmon et al., SC'11): ten rounds of
// two 32x32->64 multiplies and xors on a 128-bit counter, the 64-bit key bumped by Weyl constants
// between rounds.  One block of four words serves four consecutive sites.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint4 philox4x32_10(uint4 ctr, uint2 key) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const unsigned int hi0 = __umulhi(0xD2511F53u, ctr.x), lo0 = 0xD2511F53u * ctr.x;
        const unsigned int hi1 = __umulhi(0xCD9E8D57u, ctr.z), lo1 = 0xCD9E8D57u * ctr.z;
        ctr = make_uint4(hi1 ^ ctr.y ^ key.x, lo1, hi0 ^ ctr.w ^ key.y, lo0);
        key.x += 0x9E3779B9u;
        key.y += 0xBB67AE85u;
    }
    return ctr;
}

template <typename T>
__device__ __forceinline__ T init_value_from_word(unsigned int w, double phi0) {
    const int k = (int)(w >> 8);                                   // 24 random bits
    const double u = (double)(2 * k + 1 - 16777216) * (1.0 / 16777216.0);   // odd multiple of 2^-24
    return (T)__dmul_rn(phi0, u);
}

template <typename T>
__global__ void __launch_bounds__(256)
init_kernel(T* __restrict__ phi, T* __restrict__ phidot, long long S, unsigned long long seed,
            double phi0) {
    const long long nquads = (S + 3) >> 2;
    const uint2 key = make_uint2((unsigned int)(seed & 0xffffffffull), (unsigned int)(seed >> 32));
    for (long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x; q < nquads;
         q += (long long)gridDim.x * blockDim.x) {
        const uint4 w = philox4x32_10(
            make_uint4((unsigned int)(q & 0xffffffffll), (unsigned int)((unsigned long long)q >> 32), 0u, 0u), key);
        const long long s = q << 2;
        const T v0 = init_value_from_word<T>(w.x, phi0), v1 = init_value_from_word<T>(w.y, phi0);
        const T v2 = init_value_from_word<T>(w.z, phi0), v3 = init_value_from_word<T>(w.w, phi0);
        if (s + 3 < S) {           // S is a multiple of 4 whenever N is even: full, aligned quads
            if (sizeof(T) == 4) {
                reinterpret_cast<float4*>(phi)[q] = make_float4((float)v0, (float)v1, (float)v2, (float)v3);
                reinterpret_cast<float4*>(phidot)[q] = make_float4(0.f, 0.f, 0.f, 0.f);
            } else {
                reinterpret_cast<double2*>(phi)[2 * q] = make_double2((double)v0, (double)v1);
                reinterpret_cast<double2*>(phi)[2 * q + 1] = make_double2((double)v2, (double)v3);
                reinterpret_cast<double2*>(phidot)[2 * q] = make_double2(0.0, 0.0);
                reinterpret_cast<double2*>(phidot)[2 * q + 1] = make_double2(0.0, 0.0);
            }
        } else {
            const T v[4] = {v0, v1, v2, v3};
            for (int j = 0; j < 4 && s + j < S; ++j) {
                phi[s + j] = v[j];
                phidot[s + j] = T(0);
            }
        }
    }
}

// Initial condition of a z slab (prs_create_slab): local plane l holds global plane (zg0 + l) mod N,
// halo planes included, so a freshly initialised slab needs no halo exchange.  The Philox counter is
// the GLOBAL site index >> 2, as in init_kernel: the field does not depend on the decomposition.
// NN = N*N is a multiple of 4 (the host checks N % 4 == 0).
template <typename T>
__global__ void __launch_bounds__(256)
init_slab_kernel(T* __restrict__ phi, T* __restrict__ phidot, long long NN, long long nplanes, long long N,
                 long long zg0, unsigned long long seed, double phi0) {
    const long long qpp = NN >> 2;                                   // quads per plane
    const long long nquads = qpp * nplanes;
    const uint2 key = make_uint2((unsigned int)(seed & 0xffffffffull), (unsigned int)(seed >> 32));
    for (long long ql = blockIdx.x * (long long)blockDim.x + threadIdx.x; ql < nquads;
         ql += (long long)gridDim.x * blockDim.x) {
        const long long l = ql / qpp, r = ql - l * qpp;
        const long long zg = ((zg0 + l) % N + N) % N;
        const long long q = zg * qpp + r;                            // global quad
        const uint4 w = philox4x32_10(
            make_uint4((unsigned int)(q & 0xffffffffll), (unsigned int)((unsigned long long)q >> 32), 0u, 0u), key);
        const T v0 = init_value_from_word<T>(w.x, phi0), v1 = init_value_from_word<T>(w.y, phi0);
        const T v2 = init_value_from_word<T>(w.z, phi0), v3 = init_value_from_word<T>(w.w, phi0);
        if (sizeof(T) == 4) {
            reinterpret_cast<float4*>(phi)[ql] = make_float4((float)v0, (float)v1, (float)v2, (float)v3);
            reinterpret_cast<float4*>(phidot)[ql] = make_float4(0.f, 0.f, 0.f, 0.f);
        } else {
            reinterpret_cast<double2*>(phi)[2 * ql] = make_double2((double)v0, (double)v1);
            reinterpret_cast<double2*>(phi)[2 * ql + 1] = make_double2((double)v2, (double)v3);
            reinterpret_cast<double2*>(phidot)[2 * ql] = make_double2(0.0, 0.0);
            reinterpret_cast<double2*>(phidot)[2 * ql + 1] = make_double2(0.0, 0.0);
        }
    }
}

// ------------------------------------------------------------------------------------------------
// Generic step: one thread per site, neighbours by modulo wrap (Eqs. 3-5).  The lattice is
// N x N x NZ (NZ = N unless the handle is a z slab of a sharded lattice, prs_create_slab: there the
// wrap in z only ever feeds the outermost halo planes, which lose their validity with each step anyway).
// ------------------------------------------------------------------------------------------------
template <typename T, int DIMS, int ARITH>
__global__ void __launch_bounds__(256)
step_generic_kernel(const T* __restrict__ phi, const T* __restrict__ phidot, T* __restrict__ phi_next,
                    T* __restrict__ phidot_next, long long N, long long NZ, long long S, StepCoef<T> k) {
    const long long s = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (s >= S) return;
    const long long x = s % N;
    const long long yz = s / N;
    const long long y = (DIMS == 3) ? yz % N : yz;
    const long long z = (DIMS == 3) ? yz / N : 0;
    const long long row = s - x;
    const long long xm = row + (x == 0 ? N - 1 : x - 1), xp = row + (x == N - 1 ? 0 : x + 1);
    const long long col = s - y * N;
    const long long ym = col + (y == 0 ? N - 1 : y - 1) * N, yp = col + (y == N - 1 ? 0 : y + 1) * N;
    T zmv = T(0), zpv = T(0);
    if (DIMS == 3) {
        const long long NN = N * N;
        const long long pil = s - z * NN;
        zmv = phi[pil + (z == 0 ? NZ - 1 : z - 1) * NN];       // NZ planes: N on a cubic lattice, the slab's
        zpv = phi[pil + (z == NZ - 1 ? 0 : z + 1) * NN];       // planes (halo included) on a z slab
    }
    T pn, vn;
    site_update<T, DIMS, ARITH>(k, phi[s], phi[xm], phi[xp], phi[ym], phi[yp], zmv, zpv, phidot[s], pn, vn);
    phi_next[s] = pn;
    phidot_next[s] = vn;
}

// ------------------------------------------------------------------------------------------------
// Block reduction of a DiagPartial: warp shuffles, then one value per warp through shared memory.
// The order of the double additions is fixed by the launch configuration, so a given (grid, block)
// gives the same bits every run.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ DiagPartial warp_reduce(DiagPartial p) {
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        p.links += __shfl_down_sync(0xffffffffu, p.links, off);
        p.walls += __shfl_down_sync(0xffffffffu, p.walls, off);
        p.sum = __dadd_rn(p.sum, __shfl_down_sync(0xffffffffu, p.sum, off));
    }
    return p;
}

// All threads of the block must call; the result is valid in thread 0.
__device__ __forceinline__ DiagPartial block_reduce(DiagPartial p) {
    __shared__ DiagPartial warp_part[32];
    const int tid = threadIdx.x + blockDim.x * (threadIdx.y + blockDim.y * threadIdx.z);
    const int nthreads = blockDim.x * blockDim.y * blockDim.z;
    const int lane = tid & 31, warp = tid >> 5, nwarps = (nthreads + 31) >> 5;
    p = warp_reduce(p);
    __syncthreads();                       // protects warp_part when called twice in one kernel
    if (lane == 0) warp_part[warp] = p;
    __syncthreads();
    if (warp == 0) {
        DiagPartial q = {0ull, 0ull, 0.0};
        if (lane < nwarps) q = warp_part[lane];
        p = warp_reduce(q);
    }
    return p;
}

// Final reduction without a second launch.  Every block stores its partial and draws a ticket; the block that draws
// the last one adds all partials in index order -- thread-strided, then the block reduction: an order fixed by the
// launch configuration alone, whichever block happens to be last, so the double sum is reproducible -- writes the record
// and puts the ticket counter back to zero for the next pass.  (A launch costs 4-5 us of host time on this box: on a
// 256^2 lattice the separate one-block reduction kernel was a fifth of a 10-step cycle.)
struct DiagFinish {
    DiagPartial* partials;      // one per block
    DiagPartial* out;           // the reduced record
    unsigned* ticket;           // zero between passes
};

// All threads of the block must call; acc is the block's partial, valid in thread 0 (what block_reduce returns).
__device__ __forceinline__ void finish_partials(const DiagFinish& f, DiagPartial acc) {
    __shared__ bool is_last;
    const unsigned tid = threadIdx.x + blockDim.x * (threadIdx.y + blockDim.y * threadIdx.z);
    const unsigned nthreads = blockDim.x * blockDim.y * blockDim.z;
    const unsigned nblocks = gridDim.x * gridDim.y * gridDim.z;
    const unsigned block = blockIdx.x + gridDim.x * (blockIdx.y + gridDim.y * blockIdx.z);
    if (tid == 0) {
        f.partials[block] = acc;
        __threadfence();                                   // the partial is visible before the ticket is drawn
        is_last = (atomicAdd(f.ticket, 1u) == nblocks - 1u);
    }
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    DiagPartial sum = {0ull, 0ull, 0.0};
    for (unsigned i = tid; i < nblocks; i += nthreads) {
        const DiagPartial* q = f.partials + i;             // written by other SMs: read past L1
        sum.links += __ldcg(&q->links);
        sum.walls += __ldcg(&q->walls);
        sum.sum = __dadd_rn(sum.sum, __ldcg(&q->sum));
    }
    sum = block_reduce(sum);
    if (tid == 0) {
        *f.out = sum;
        *f.ticket = 0u;
    }
}

// Generic diagnostics: grid-stride over sites; each site owns its d forward links (Eq. 7) and tests
// all 2d links for the wall-site predicate (Eq. 8's N).
template <typename T, int DIMS>
__global__ void __launch_bounds__(256)
diag_generic_kernel(const T* __restrict__ phi, const T* __restrict__ phidot, long long N, long long NZ,
                    long long s0, long long S, double V0, double I, DiagFinish fin) {
    using A = Ar<T>;
    DiagPartial acc = {0ull, 0ull, 0.0};
    // sites s0 <= s < S of an N x N x NZ lattice (cubic: NZ = N, s0 = 0; z slab: the owned planes)
    for (long long s = s0 + blockIdx.x * (long long)blockDim.x + threadIdx.x; s < S;
         s += (long long)gridDim.x * blockDim.x) {
        const long long x = s % N;
        const long long yz = s / N;
        const long long y = (DIMS == 3) ? yz % N : yz;
        const long long z = (DIMS == 3) ? yz / N : 0;
        const long long row = s - x, col = s - y * N;
        const T c = phi[s];
        const bool me = A::neg(c);
        const bool xp = A::neg(phi[row + (x == N - 1 ? 0 : x + 1)]) != me;
        const bool xm = A::neg(phi[row + (x == 0 ? N - 1 : x - 1)]) != me;
        const bool yp = A::neg(phi[col + (y == N - 1 ? 0 : y + 1) * N]) != me;
        const bool ym = A::neg(phi[col + (y == 0 ? N - 1 : y - 1) * N]) != me;
        bool zp = false, zm = false;
        if (DIMS == 3) {
            const long long NN = N * N, pil = s - z * NN;
            zp = A::neg(phi[pil + (z == NZ - 1 ? 0 : z + 1) * NN]) != me;
            zm = A::neg(phi[pil + (z == 0 ? NZ - 1 : z - 1) * NN]) != me;
        }
        acc.links += (unsigned)xp + (unsigned)yp + (unsigned)zp;
        if (xp | xm | yp | ym | zp | zm) {
            acc.walls += 1;
            acc.sum = __dadd_rn(acc.sum, wall_ratio<T>(c, phidot[s], V0, I));
        }
    }
    acc = block_reduce(acc);
    finish_partials(fin, acc);
}

// ------------------------------------------------------------------------------------------------
// Orientation-weighted wall area, Eq. 7 as printed (:59-62; R15): sum over crossing
// forward links of |grad phi| / (|phi,x| + |phi,y| + |phi,z|), the gradient on the link s -> s+e_k
// being the forward difference along the link and, across it, the mean of the central differences
// at the two ends.  All arithmetic in double.
//
// Thread = one x; it marches L sites along the slowest axis, carrying the value one step ahead, and
// tests the d forward links of each site on the sign bits.  Crossing links are rare late in a run, so
// the gathers and the FP64 square root and division would run with a few lanes of a warp active: each
// warp instead pushes its crossing links (coordinates + direction, 8 bytes) on a small stack in shared
// memory (ballot + prefix count) and works them off 32 at a time with every lane busy.  The transverse
// neighbours are L1 / L2 hits: they lie within one site of what the warp streams anyway.  The
// crossing links are counted again on the way (partials[].links) as a cross-check against a6.
// ------------------------------------------------------------------------------------------------
constexpr int WAREA_THREADS = 256;
constexpr int WAREA_STACK = 64;                  // entries per warp: < 32 left over + up to 32 pushed at once

// Eq. 7's weight of one crossing link; entry = x | y << 20 | z << 40 | k << 60 (site and link axis).
// The axis is data, different from lane to lane: everything is selected arithmetically, nothing branches.
template <typename T, int DIMS>
__device__ __forceinline__ double link_weight(const T* __restrict__ phi, int N, int NM, unsigned long long entry) {
    const int k = (int)(entry >> 60);
    const int c0 = (int)(entry & 0xfffff), c1 = (int)((entry >> 20) & 0xfffff), c2 = (int)((entry >> 40) & 0xfffff);
    const long long NN = (long long)N * N;
    // offset to the periodic neighbour at distance d = -1, 0, +1 along axis a
    auto hop = [&](int a, int d) -> long long {
        const int ca = (a == 0) ? c0 : (a == 1 ? c1 : c2);
        const long long st = (a == 0) ? 1 : (a == 1 ? (long long)N : NN);
        const int ext = (a == DIMS - 1) ? NM : N;                    // the march axis holds NM sites (a slab: its planes)
        int w = ca + d;
        w = (w < 0) ? w + ext : (w >= ext ? w - ext : w);
        return (long long)(w - ca) * st;
    };
    const T* const site = phi + ((long long)c0 + (long long)c1 * N + (long long)c2 * NN);
    const long long ek = hop(k, 1);
    // along the link: forward difference; across it: mean of the central differences at the two ends
    const double gk = __dsub_rn((double)__ldg(site + ek), (double)__ldg(site));
    auto across = [&](int t) {
        const long long ep = hop(t, 1), em = hop(t, -1);
        const double dc = __dmul_rn(__dsub_rn((double)__ldg(site + ep), (double)__ldg(site + em)), 0.5);
        const double de = __dmul_rn(__dsub_rn((double)__ldg(site + ep + ek), (double)__ldg(site + em + ek)), 0.5);
        return __dmul_rn(__dadd_rn(dc, de), 0.5);
    };
    double g0, g1, g2 = 0.0;                                         // in x, y, z order whatever k is
    if (DIMS == 2) {
        const double gt = across(1 - k);
        g0 = (k == 0) ? gk : gt;
        g1 = (k == 0) ? gt : gk;
    } else {
        const int ta = (k == 0) ? 1 : 0, tb = (k == 2) ? 1 : 2;      // the other two axes, ta < tb
        const double ga = across(ta), gb = across(tb);
        g0 = (k == 0) ? gk : ga;
        g1 = (k == 1) ? gk : (k == 0 ? ga : gb);
        g2 = (k == 2) ? gk : gb;
    }
    const double num = __dsqrt_rn(__dadd_rn(__dadd_rn(__dmul_rn(g0, g0), __dmul_rn(g1, g1)), __dmul_rn(g2, g2)));
    const double den = __dadd_rn(__dadd_rn(fabs(g0), fabs(g1)), fabs(g2));
    return (den == 0.0) ? 1.0 : __ddiv_rn(num, den);
}

template <typename T, int DIMS>
__global__ void __launch_bounds__(WAREA_THREADS)
weighted_area_kernel(const T* __restrict__ phi, int N, int NM, int mlo, int mhi, int L, DiagFinish fin) {
    // the slowest (march) axis holds NM sites, of which mlo <= m < mhi are measured: N, 0, N on a whole lattice; on a
    // z slab (prs_create_slab) its NZ planes and the owned range, whose z neighbours are halo planes (never the wrap)
    using A = Ar<T>;
    __shared__ unsigned long long stack_all[WAREA_THREADS / 32][WAREA_STACK];
    unsigned long long* const stack = stack_all[threadIdx.x >> 5];
    const unsigned lane = threadIdx.x & 31, lt_mask = (1u << lane) - 1u;
    int held = 0;                                                    // entries on the warp's stack (uniform)
    DiagPartial acc = {0ull, 0ull, 0.0};
    // blockIdx.y = y (3D) or the chunk of rows (2D); blockIdx.z = the chunk of planes (3D)
    constexpr int M = DIMS - 1;                                      // march axis
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const bool live = x < N;
    const int xs = live ? x : 0;                                     // lanes past the row idle along on x = 0
    const long long stride[3] = {1, N, (long long)N * N};
    int c[3] = {xs, (DIMS == 3) ? (int)blockIdx.y : 0, 0};
    const int m0 = mlo + (int)((DIMS == 3) ? blockIdx.z : blockIdx.y) * L;
    const int m1 = min(m0 + L, mhi);
    c[M] = m0;
    // Linear offset o of the site, constant offsets to its x+1 (and y+1) neighbours, and the offset to
    // the next site of the march (negative at the periodic seam).
    long long o = 0;
#pragma unroll
    for (int m = 0; m < DIMS; ++m) o += c[m] * stride[m];
    const long long dx = (c[0] == N - 1) ? -(long long)(N - 1) : 1;
    const long long dy = (DIMS == 3) ? ((c[1] == N - 1) ? -(long long)(N - 1) * N : (long long)N) : 0;
    auto dm = [&](int m) { return (m == NM - 1) ? -(long long)(NM - 1) * stride[M] : stride[M]; };
    auto forward = [&](long long at, int m, T* out) {
        out[0] = __ldg(phi + at + dx);
        if (DIMS == 3) out[1] = __ldg(phi + at + dy);
        out[M] = __ldg(phi + at + dm(m));
    };
    auto work_off = [&](int n) {                                     // the top n <= 32 entries of the stack
        __syncwarp();
        if ((int)lane < n) acc.sum = __dadd_rn(acc.sum, link_weight<T, DIMS>(phi, N, NM, stack[held - n + (int)lane]));
        held -= n;
        __syncwarp();
    };
    T pc = __ldg(phi + o);
    T pe[DIMS], pn[DIMS];
    forward(o, m0, pe);
    const unsigned long long site_xy = (unsigned long long)c[0] | ((DIMS == 3) ? ((unsigned long long)c[1] << 20) : 0ull);
    for (int m = m0; m < m1; ++m) {
        // the forward neighbours of the next site of the march are requested before this site is
        // worked on (one iteration of latency hiding; past the end this re-reads harmlessly)
        const long long on = o + dm(m);
        forward(on, (m + 1 == NM) ? 0 : m + 1, pn);
        const bool me = A::neg(pc);
        const unsigned long long site = site_xy | ((unsigned long long)m << (20 * M));
#pragma unroll
        for (int k = 0; k < DIMS; ++k) {
            const bool cross = live && (A::neg(pe[k]) != me);
            const unsigned votes = __ballot_sync(0xffffffffu, cross);
            if (cross) {
                acc.links += 1;
                stack[held + __popc(votes & lt_mask)] = site | ((unsigned long long)k << 60);
            }
            held += __popc(votes);
            if (held >= 32) work_off(32);
        }
        pc = pe[M];                                                  // the forward neighbour along the march
#pragma unroll
        for (int k = 0; k < DIMS; ++k) pe[k] = pn[k];
        o = on;
    }
    work_off(held);
    acc = block_reduce(acc);
    finish_partials(fin, acc);
}

}  // namespace prs
