// prs_kernels_bits.cuh -- the wall diagnostics of large lattices on PACKED SIGN BITS (Eq. 7 link count,
// Eq. 8 wall-site velocity; readings R6-R10 of DESIGN.md).
//
// Why.  The one-pass kernel (prs_kernels_tiled.cuh, diag3d_tiled_kernel) is bound by instruction issue, not by HBM:
// 2.3-2.5 ms per pass at 1024^3 FP32 against 0.67 ms for one read of phi (profiles/r01f_*: issue slots 78 % busy, ALU
// pipe 62 % on sign-mask arithmetic; every thread re-loads its two y-neighbour vectors and rebuilds their masks).  The
// quantities of Eqs. 7-8 depend on phi only through its SIGN BIT except at wall sites, a few per cent of the lattice
// once the network has formed.  So the pass is split where the data volume changes by a factor of 32:
//
//   sign_bits_kernel    reads phi once (the only HBM-bound part) and writes one bit per site: a warp loads 32
//                       consecutive 16-byte vectors and one __ballot_sync per vector element packs their signs.
//                       1024^3: 4.3 GB read, 128 MiB written -- small enough to stay in the 126 MB L2.
//   bit_links_kernel    works on the bit words: XORs against the words of the x, y, z neighbours, popcounts for the
//                       link count and the wall-site count, and only for the set bits of the wall word fetches
//                       phi and phidot (4-byte gathers) and evaluates Eq. 8's ratio in double, the wall sites of a
//                       warp compacted through a shared-memory stack so that all lanes divide.
//
// Bit layout (no transposition needed, the ballots give it for free).  A lattice row (fixed y, z) of NQ = N / W
// vectors (W = 4 floats / 2 doubles) is NG = NQ / 32 GROUPS of W words: bit l of word i of group g is the sign of
// site x = W (32 g + l) + i.  Neighbours in x: within a group x+1 is the same bit of the next word (i < W-1) or bit
// l+1 of word 0 (i = W-1); across groups bit 0 of the next group's word 0 / bit 31 of the previous group's last
// word (periodic).  Neighbours in y and z: the same bits of the same group one row / one plane away.
// Requires NQ % 32 == 0 (N a multiple of 128 in FP32, 64 in FP64: every BASELINE.json size); other lattices keep the
// one-pass kernels.
#pragma once

#include "prs_arith.cuh"
#include "prs_kernels_generic.cuh"   // DiagPartial reduction
#include "prs_kernels_tiled.cuh"     // VecOps

namespace prs {

// Rows r0 <= r < r1 of the array (row r = y + N z holds N sites; a z slab passes the rows of the planes it needs).
// One warp per (row, group) and grid-stride over them.  bits: W words per group, groups in row-major order.
template <typename T>
__global__ void __launch_bounds__(256)
sign_bits_kernel(const T* __restrict__ phi, unsigned* __restrict__ bits, int N, long long r0, long long r1) {
    using O = VecOps<T>;
    using V = typename O::V;
    constexpr int W = O::W;
    const int lane = threadIdx.x & 31;
    const int NG = N / (32 * W);
    // A row is a whole number of groups, so group gi of the array (row-major, gi = r NG + g) starts at site 32 W gi and its
    // words at W gi: no row / group decomposition is needed here at all.  (The first version divided a 64-bit index by NG
    // per group: ncu showed 85 instructions per group, issue slots 73 % busy, DRAM at 61 % -- bound by that, not by HBM.)
    const long long gbeg = r0 * NG, gend = r1 * NG;
    const long long wstep = (long long)gridDim.x * (blockDim.x >> 5);
    constexpr int U = 4;                                             // four independent 16-byte loads per lane in flight
    for (long long g0 = gbeg + (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); g0 < gend; g0 += U * wstep) {
        V v[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const long long gi = g0 + u * wstep;
            if (gi < gend) v[u] = O::ld(phi + (gi * 32 + lane) * W);                  // warp-uniform condition
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const long long gi = g0 + u * wstep;
            if (gi >= gend) break;
            unsigned mine = 0u;
#pragma unroll
            for (int i = 0; i < W; ++i) {
                const unsigned w = __ballot_sync(0xffffffffu, Ar<T>::neg(O::get(v[u], i)));
                if (lane == i) mine = w;
            }
            if (lane < W) bits[gi * W + lane] = mine;
        }
    }
}

// W words of one group as one 8- or 16-byte load.
template <int W> struct BitWords;
template <> struct BitWords<4> {
    unsigned w[4];
    __device__ __forceinline__ void load(const unsigned* p) {
        const uint4 v = __ldg(reinterpret_cast<const uint4*>(p));
        w[0] = v.x; w[1] = v.y; w[2] = v.z; w[3] = v.w;
    }
};
template <> struct BitWords<2> {
    unsigned w[2];
    __device__ __forceinline__ void load(const unsigned* p) {
        const uint2 v = __ldg(reinterpret_cast<const uint2*>(p));
        w[0] = v.x; w[1] = v.y;
    }
};

constexpr int BITS_THREADS = 256;
constexpr int BITS_STACK = 64;                   // entries per warp: < 32 left over + up to 32 pushed per round

// Rows R0 <= r < R1 are measured (each site owns its DIMS forward links, Eq. 7; a wall site is one that touches a
// crossing link in any of its 2 DIMS directions, Eq. 8's N); the array holds N x N x NZ sites (2D: N x N), periodic
// in y over N and in z over NZ -- a z slab measures its owned planes, whose z neighbours are halo planes, never the
// wrap.  One thread per group; a warp takes 32 consecutive groups.
template <typename T, int DIMS>
__global__ void __launch_bounds__(BITS_THREADS)
bit_links_kernel(const T* __restrict__ phi, const T* __restrict__ phidot, const unsigned* __restrict__ bits, int N, int NZ,
                 long long R0, long long R1, double V0, double I, DiagFinish fin) {
    constexpr int W = VecOps<T>::W;
    __shared__ unsigned short stack_all[BITS_THREADS / 32][BITS_STACK];
    unsigned short* const stack = stack_all[threadIdx.x >> 5];
    const unsigned lane = threadIdx.x & 31, lt = (1u << lane) - 1u;
    const int NG = N / (32 * W);
    const long long ngroups = (R1 - R0) * NG;
    const long long wstep = (long long)gridDim.x * (BITS_THREADS / 32) * 32;
    DiagPartial acc = {0ull, 0ull, 0.0};
    int held = 0;                                                    // entries on the warp's stack (warp-uniform)
    for (long long g0 = ((long long)blockIdx.x * (BITS_THREADS / 32) + (threadIdx.x >> 5)) * 32; g0 < ngroups; g0 += wstep) {
        const long long gi = g0 + lane;
        const bool live = gi < ngroups;
        unsigned wall[W];
        long long site0 = 0;                                         // first site of this thread's group
#pragma unroll
        for (int i = 0; i < W; ++i) wall[i] = 0u;
        if (live) {
            // 32-bit arithmetic: an array has fewer than 2^31 groups and rows (the host checks), and 64-bit divisions
            // were most of this kernel's 360 instructions per thread
            const unsigned gu = (unsigned)gi, ru = gu / (unsigned)NG;
            const int g = (int)(gu - ru * (unsigned)NG);
            const long long r = R0 + (long long)ru;
            const unsigned rr = (unsigned)r, zu = rr / (unsigned)N;
            const int y = (int)(rr - zu * (unsigned)N);
            site0 = r * N + (long long)(32 * W) * g;
            const long long ryp = (y == N - 1) ? r - (N - 1) : r + 1, rym = (y == 0) ? r + (N - 1) : r - 1;
            const int gxp = (g == NG - 1) ? 0 : g + 1, gxm = (g == 0) ? NG - 1 : g - 1;
            BitWords<W> c, yp, ym, zp, zm;
            c.load(bits + (r * NG + g) * W);
            yp.load(bits + (ryp * NG + g) * W);
            ym.load(bits + (rym * NG + g) * W);
            if (DIMS == 3) {
                const long long z = (long long)zu, plane = (long long)N;
                const long long rzp = (z == NZ - 1) ? r - (long long)(NZ - 1) * plane : r + plane;
                const long long rzm = (z == 0) ? r + (long long)(NZ - 1) * plane : r - plane;
                zp.load(bits + (rzp * NG + g) * W);
                zm.load(bits + (rzm * NG + g) * W);
            }
            const unsigned next0 = __ldg(bits + (r * NG + gxp) * W);                 // word 0 of the group to the right
            const unsigned prevl = __ldg(bits + (r * NG + gxm) * W + (W - 1));       // last word of the group to the left
            unsigned nlinks = 0u;
#pragma unroll
            for (int i = 0; i < W; ++i) {
                // sign of x+1 / x-1 for the 32 sites of word i
                const unsigned right = (i < W - 1) ? c.w[i + 1] : ((c.w[0] >> 1) | (next0 << 31));
                const unsigned left = (i > 0) ? c.w[i - 1] : ((c.w[W - 1] << 1) | (prevl >> 31));
                const unsigned fx = c.w[i] ^ right, bx = c.w[i] ^ left;
                const unsigned fy = c.w[i] ^ yp.w[i], by = c.w[i] ^ ym.w[i];
                unsigned fz = 0u, bz = 0u;
                if (DIMS == 3) { fz = c.w[i] ^ zp.w[i]; bz = c.w[i] ^ zm.w[i]; }
                nlinks += __popc(fx) + __popc(fy) + __popc(fz);       // forward links owned by these sites
                wall[i] = fx | bx | fy | by | fz | bz;
                acc.walls += __popc(wall[i]);
            }
            acc.links += nlinks;
        }
        // ---- Eq. 8 at the wall sites: onto the warp's stack, worked off 32 at a time with every lane dividing
        const unsigned s0lo = (unsigned)(site0 & 0xffffffffll), s0hi = (unsigned)(site0 >> 32);
        auto work_off = [&](int n) {                                 // the top n <= 32 entries
            PRS_JITTER(1u);
            __syncwarp();
            const unsigned e = ((int)lane < n) ? stack[held - n + (int)lane] : 0u;
            const unsigned owner = e >> 7;
            const long long base = ((long long)__shfl_sync(0xffffffffu, s0hi, owner) << 32) |
                                   (long long)__shfl_sync(0xffffffffu, s0lo, owner);
            if ((int)lane < n) {
                const long long s = base + (long long)(W * (e & 31u) + ((e >> 5) & 3u));
                acc.sum = __dadd_rn(acc.sum, wall_ratio<T>(__ldg(phi + s), __ldg(phidot + s), V0, I));
            }
            held -= n;
            __syncwarp();
        };
        // Group by group and word by word (not one bit per lane and round): the 32 entries a pop works off are then
        // consecutive sites of one group, 16 bytes apart, so the gathers of phi and phidot touch 4 lines, not 32 --
        // on the white-noise start, where 72 % of the sites are wall sites, that is 9.0 -> 3 ms at 1024^3.  The wall
        // word of the owner IS the vote (bit l = lane l's site), so no ballot is needed.
        unsigned any = 0u;
#pragma unroll
        for (int i = 0; i < W; ++i) any |= wall[i];
        for (unsigned owners = __ballot_sync(0xffffffffu, any != 0u); owners; owners &= owners - 1u) {
            const unsigned owner = (unsigned)__ffs(owners) - 1u;
#pragma unroll
            for (int i = 0; i < W; ++i) {
                const unsigned m = __shfl_sync(0xffffffffu, wall[i], owner);
                if (m == 0u) continue;
                if ((m >> lane) & 1u) stack[held + __popc(m & lt)] = (unsigned short)((owner << 7) | ((unsigned)i << 5) | lane);
                held += __popc(m);
                if (held >= 32) work_off(32);
            }
        }
        if (held) work_off(held);                                    // the bases belong to this batch of groups
    }
    acc = block_reduce(acc);
    finish_partials(fin, acc);
}

// ------------------------------------------------------------------------------------------------------------------
// Eq. 7 with the PRS orientation weight (R15) on the same bit words: the crossing forward
// links ARE the set bits of c ^ right, c ^ up, c ^ above, so only they -- 2 % of the links of a formed network -- cost
// anything beyond the words: their entries (owner group, axis, word, bit) go onto the warp's stack group by group and
// are worked off 32 at a time by link_weight() (prs_kernels_generic.cuh: the gathers of the transverse neighbours, the
// square root and the division in double), every lane busy.  partials[].links counts the crossing links again as a
// cross-check against Eq. 7's unweighted count.  Rows and planes as in bit_links_kernel.
// ------------------------------------------------------------------------------------------------------------------
// One out-of-line copy of Eq. 7's link weight: inlined at the dozen places where the unrolled push loop may pop the stack
// it made the kernel so large that half its stall samples were instruction fetches (ncu: no_instructions 50 %).
template <typename T, int DIMS>
__device__ __noinline__ double link_weight_call(const T* __restrict__ phi, int N, int NM, unsigned long long entry) {
    return link_weight<T, DIMS>(phi, N, NM, entry);
}

template <typename T, int DIMS>
__global__ void __launch_bounds__(BITS_THREADS)
bit_area_kernel(const T* __restrict__ phi, const unsigned* __restrict__ bits, int N, int NZ, long long R0, long long R1,
                DiagFinish fin) {
    constexpr int W = VecOps<T>::W;
    __shared__ unsigned short stack_all[BITS_THREADS / 32][BITS_STACK];
    unsigned short* const stack = stack_all[threadIdx.x >> 5];
    const unsigned lane = threadIdx.x & 31, lt = (1u << lane) - 1u;
    const int NG = N / (32 * W);
    const int NM = (DIMS == 3) ? NZ : N;                             // extent of the slowest axis (a slab: its planes)
    const long long ngroups = (R1 - R0) * NG;
    const long long wstep = (long long)gridDim.x * (BITS_THREADS / 32) * 32;
    DiagPartial acc = {0ull, 0ull, 0.0};
    int held = 0;
    for (long long g0 = ((long long)blockIdx.x * (BITS_THREADS / 32) + (threadIdx.x >> 5)) * 32; g0 < ngroups; g0 += wstep) {
        const long long gi = g0 + lane;
        const bool live = gi < ngroups;
        unsigned f[DIMS][W];                                         // crossing forward links per axis and word
#pragma unroll
        for (int k = 0; k < DIMS; ++k)
#pragma unroll
            for (int i = 0; i < W; ++i) f[k][i] = 0u;
        int row = 0, grp = 0;                                        // this thread's row (y + N z) and group: < 2^31
        if (live) {
            const unsigned gu = (unsigned)gi, ru = gu / (unsigned)NG;                 // 32-bit: see bit_links_kernel
            const int g = (int)(gu - ru * (unsigned)NG);
            const long long r = R0 + (long long)ru;
            const unsigned rr = (unsigned)r, zu = rr / (unsigned)N;
            row = (int)r; grp = g;
            const int y = (int)(rr - zu * (unsigned)N);
            const long long ryp = (y == N - 1) ? r - (N - 1) : r + 1;
            const int gxp = (g == NG - 1) ? 0 : g + 1;
            BitWords<W> c, yp, zp;
            c.load(bits + (r * NG + g) * W);
            yp.load(bits + (ryp * NG + g) * W);
            if (DIMS == 3) {
                const long long z = (long long)zu;
                const long long rzp = (z == NZ - 1) ? r - (long long)(NZ - 1) * N : r + N;
                zp.load(bits + (rzp * NG + g) * W);
            }
            const unsigned next0 = __ldg(bits + (r * NG + gxp) * W);
#pragma unroll
            for (int i = 0; i < W; ++i) {
                const unsigned right = (i < W - 1) ? c.w[i + 1] : ((c.w[0] >> 1) | (next0 << 31));
                f[0][i] = c.w[i] ^ right;
                f[1][i] = c.w[i] ^ yp.w[i];
                if (DIMS == 3) f[2][i] = c.w[i] ^ zp.w[i];
#pragma unroll
                for (int k = 0; k < DIMS; ++k) acc.links += __popc(f[k][i]);
            }
        }
        auto work_off = [&](int n) {                                 // the top n <= 32 entries
            PRS_JITTER(1u);
            __syncwarp();
            const unsigned e = ((int)lane < n) ? stack[held - n + (int)lane] : 0u;
            const unsigned owner = e >> 9;
            const int orow = __shfl_sync(0xffffffffu, row, owner), ogrp = __shfl_sync(0xffffffffu, grp, owner);
            if ((int)lane < n) {
                const unsigned long long x = (unsigned long long)(W * (32 * ogrp + (int)(e & 31u)) + (int)((e >> 5) & 3u));
                const unsigned long long yy = (unsigned long long)(orow % N), zz = (unsigned long long)(orow / N);
                const unsigned long long k = (e >> 7) & 3u;
                // link_weight's entry: x | y << 20 | z << 40 | axis << 60 (2D: the row is y)
                const unsigned long long entry = x | (yy << 20) | (zz << 40) | (k << 60);
                acc.sum = __dadd_rn(acc.sum, link_weight_call<T, DIMS>(phi, N, NM, entry));
            }
            held -= n;
            __syncwarp();
        };
        unsigned any = 0u;
#pragma unroll
        for (int k = 0; k < DIMS; ++k)
#pragma unroll
            for (int i = 0; i < W; ++i) any |= f[k][i];
        for (unsigned owners = __ballot_sync(0xffffffffu, any != 0u); owners; owners &= owners - 1u) {
            const unsigned owner = (unsigned)__ffs(owners) - 1u;
#pragma unroll
            for (int k = 0; k < DIMS; ++k)
#pragma unroll
                for (int i = 0; i < W; ++i) {
                    const unsigned m = __shfl_sync(0xffffffffu, f[k][i], owner);
                    if (m == 0u) continue;
                    if ((m >> lane) & 1u)
                        stack[held + __popc(m & lt)] = (unsigned short)((owner << 9) | ((unsigned)k << 7) | ((unsigned)i << 5) | lane);
                    held += __popc(m);
                    if (held >= 32) work_off(32);
                }
        }
        if (held) work_off(held);
    }
    acc = block_reduce(acc);
    finish_partials(fin, acc);
}

}  // namespace prs
