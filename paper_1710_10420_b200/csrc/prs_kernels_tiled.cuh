// prs_kernels_tiled.cuh -- single-step kernels for HBM-bound lattices (N a multiple of the 16-byte
// vector width): one pass reads phi^n and phidot^{n-1/2} once and writes phidot^{n+1/2} and
// phi^{n+1} once (Eqs. 3-5 fused, ":101 concatenation of kernels").
//
// Layout of the work.  A thread owns one 16-byte vector of consecutive x (4 floats / 2 doubles) and
// marches along the slowest axis (z in 3D, y in 2D) keeping a three-deep register window of its own
// column, so the neighbours along the march axis cost no memory traffic at all.  In-row neighbours
// x-1 / x+VEC come from the adjacent lanes by warp shuffle; only the two edge lanes of a warp issue a
// scalar load (an L1/L2 hit: the line belongs to the neighbouring warp's tile).  In 3D the y-1 / y+1
// rows are 16-byte loads of lines that a neighbouring warp of the same CTA (or, at the tile edge, a
// neighbouring CTA marching the same planes) has just pulled in, i.e. L1 / L2 hits.  All loads of
// iteration z+1 are issued before the arithmetic of iteration z (one-deep software pipeline), so each
// thread keeps two 16-byte DRAM requests in flight.
#pragma once

#include "prs_arith.cuh"
#include "prs_kernels_generic.cuh"   // warp_reduce / block_reduce

namespace prs {

template <typename T> struct VecOps;

template <> struct VecOps<float> {
    typedef float4 V;
    static constexpr int W = 4;
    static __device__ __forceinline__ V ld(const float* p) { return __ldg(reinterpret_cast<const float4*>(p)); }
    static __device__ __forceinline__ void st(float* p, V v) { *reinterpret_cast<float4*>(p) = v; }
    static __device__ __forceinline__ float first(V v) { return v.x; }
    static __device__ __forceinline__ float last(V v) { return v.w; }
    static __device__ __forceinline__ float get(V v, int i) { return i == 0 ? v.x : i == 1 ? v.y : i == 2 ? v.z : v.w; }
    static __device__ __forceinline__ void set(V& v, int i, float a) {
        if (i == 0) v.x = a; else if (i == 1) v.y = a; else if (i == 2) v.z = a; else v.w = a;
    }
};

template <> struct VecOps<double> {
    typedef double2 V;
    static constexpr int W = 2;
    static __device__ __forceinline__ V ld(const double* p) { return __ldg(reinterpret_cast<const double2*>(p)); }
    static __device__ __forceinline__ void st(double* p, V v) { *reinterpret_cast<double2*>(p) = v; }
    static __device__ __forceinline__ double first(V v) { return v.x; }
    static __device__ __forceinline__ double last(V v) { return v.y; }
    static __device__ __forceinline__ double get(V v, int i) { return i == 0 ? v.x : v.y; }
    static __device__ __forceinline__ void set(V& v, int i, double a) {
        if (i == 0) v.x = a; else v.y = a;
    }
};

// One vector of sites: c = centre vector, left/right = the scalars beside it in x, (ym, yp) and
// (zm, zp) the vectors beside it along the other axes.
template <typename T, int DIMS, int ARITH>
__device__ __forceinline__ void vector_update(const StepCoef<T>& k, typename VecOps<T>::V c, T left, T right,
                                              typename VecOps<T>::V ym, typename VecOps<T>::V yp,
                                              typename VecOps<T>::V zm, typename VecOps<T>::V zp,
                                              typename VecOps<T>::V pd, typename VecOps<T>::V& phi_new,
                                              typename VecOps<T>::V& pd_new) {
    using O = VecOps<T>;
#pragma unroll
    for (int i = 0; i < O::W; ++i) {
        const T xm = (i == 0) ? left : O::get(c, i - 1);
        const T xp = (i == O::W - 1) ? right : O::get(c, i + 1);
        T pn, vn;
        site_update<T, DIMS, ARITH>(k, O::get(c, i), xm, xp, O::get(ym, i), O::get(yp, i), O::get(zm, i),
                                      O::get(zp, i), O::get(pd, i), pn, vn);
        O::set(phi_new, i, pn);
        O::set(pd_new, i, vn);
    }
}

// ------------------------------------------------------------------------------------------------
// 3D: block = 32 lanes in x  x  TYB rows in y; grid = (x tiles, y tiles, z chunks of ZC planes).
// ------------------------------------------------------------------------------------------------
template <typename T, int ARITH, int TYB>
__global__ void __launch_bounds__(32 * TYB)
step3d_tiled_kernel(const T* __restrict__ phi, const T* __restrict__ phidot, T* __restrict__ phi_next,
                    T* __restrict__ phidot_next, int N, int NZ, int ZC, StepCoef<T> k) {
    using O = VecOps<T>;
    using V = typename O::V;
    constexpr int W = O::W;
    const int lane = threadIdx.x;
    const int y = blockIdx.y * TYB + threadIdx.y;
    if (y >= N) return;                                   // whole warp leaves together
    const int xraw = (blockIdx.x * 32 + lane) * W;
    const bool live = xraw < N;
    const int x = live ? xraw : N - W;                    // dead lanes shadow a valid address
    const int z0 = blockIdx.z * ZC;
    const int z1 = min(z0 + ZC, NZ);                       // NZ planes: N, or a slab's (prs_create_slab)
    const size_t NN = (size_t)N * N;
    const int ym = (y == 0) ? N - 1 : y - 1, yp = (y == N - 1) ? 0 : y + 1;
    const size_t rc = (size_t)y * N + x, rm = (size_t)ym * N + x, rp = (size_t)yp * N + x;
    const bool edge_l = (lane == 0), edge_r = (lane == 31) || (x + W >= N);
    const size_t rl = (size_t)y * N + (x == 0 ? N - 1 : x - 1);
    const size_t rr = (size_t)y * N + (x + W >= N ? 0 : x + W);

    const int zprev = (z0 == 0) ? NZ - 1 : z0 - 1;
    const int znext0 = (z0 + 1 == NZ) ? 0 : z0 + 1;
    V prev = O::ld(phi + (size_t)zprev * NN + rc);
    V cur = O::ld(phi + (size_t)z0 * NN + rc);
    V nxt = O::ld(phi + (size_t)znext0 * NN + rc);
    V up = O::ld(phi + (size_t)z0 * NN + rp);
    V dn = O::ld(phi + (size_t)z0 * NN + rm);
    V pd = O::ld(phidot + (size_t)z0 * NN + rc);
    T el = T(0), er = T(0);
    if (edge_l) el = __ldg(phi + (size_t)z0 * NN + rl);
    if (edge_r) er = __ldg(phi + (size_t)z0 * NN + rr);

    for (int z = z0; z < z1; ++z) {
        // ---- issue the loads of iteration z+1 first
        V nn = nxt, up_n = up, dn_n = dn, pd_n = pd;
        T el_n = el, er_n = er;
        const int zn = (z + 1 == NZ) ? 0 : z + 1;
        if (z + 1 < z1) {
            const int znn = (zn + 1 == NZ) ? 0 : zn + 1;
            const size_t pn = (size_t)zn * NN;
            nn = O::ld(phi + (size_t)znn * NN + rc);
            pd_n = O::ld(phidot + pn + rc);
            up_n = O::ld(phi + pn + rp);
            dn_n = O::ld(phi + pn + rm);
            if (edge_l) el_n = __ldg(phi + pn + rl);
            if (edge_r) er_n = __ldg(phi + pn + rr);
        }
        // ---- arithmetic of plane z
        T left = __shfl_up_sync(0xffffffffu, O::last(cur), 1);
        T right = __shfl_down_sync(0xffffffffu, O::first(cur), 1);
        if (edge_l) left = el;
        if (edge_r) right = er;
        V pnew, vnew;
        vector_update<T, 3, ARITH>(k, cur, left, right, dn, up, prev, nxt, pd, pnew, vnew);
        if (live) {
            const size_t o = (size_t)z * NN + rc;
            O::st(phidot_next + o, vnew);
            O::st(phi_next + o, pnew);
        }
        prev = cur; cur = nxt; nxt = nn;
        up = up_n; dn = dn_n; pd = pd_n; el = el_n; er = er_n;
    }
}

// ------------------------------------------------------------------------------------------------
// 2D: block = BX lanes in x; grid = (x tiles, y chunks of YC rows).  The march axis is y, so the
// register window supplies both y neighbours and nothing but the two edge scalars is re-read.
// ------------------------------------------------------------------------------------------------
template <typename T, int ARITH>
__global__ void __launch_bounds__(128)
step2d_tiled_kernel(const T* __restrict__ phi, const T* __restrict__ phidot, T* __restrict__ phi_next,
                    T* __restrict__ phidot_next, int N, int YC, StepCoef<T> k) {
    using O = VecOps<T>;
    using V = typename O::V;
    constexpr int W = O::W;
    const int lane = threadIdx.x & 31;
    const long long xraw = ((long long)blockIdx.x * blockDim.x + threadIdx.x) * W;
    if (xraw - (long long)lane * W >= N) return;          // whole warp beyond the row
    const bool live = xraw < N;
    const int x = live ? (int)xraw : N - W;
    const int y0 = blockIdx.y * YC;
    const int y1 = min(y0 + YC, N);
    const bool edge_l = (lane == 0), edge_r = (lane == 31) || (x + W >= N);
    const int xl = (x == 0) ? N - 1 : x - 1, xr = (x + W >= N) ? 0 : x + W;

    const int yprev = (y0 == 0) ? N - 1 : y0 - 1;
    const int ynext0 = (y0 + 1 == N) ? 0 : y0 + 1;
    V prev = O::ld(phi + (size_t)yprev * N + x);
    V cur = O::ld(phi + (size_t)y0 * N + x);
    V nxt = O::ld(phi + (size_t)ynext0 * N + x);
    V pd = O::ld(phidot + (size_t)y0 * N + x);
    T el = T(0), er = T(0);
    if (edge_l) el = __ldg(phi + (size_t)y0 * N + xl);
    if (edge_r) er = __ldg(phi + (size_t)y0 * N + xr);
    const V zero = {};

    for (int y = y0; y < y1; ++y) {
        V nn = nxt, pd_n = pd;
        T el_n = el, er_n = er;
        const int yn = (y + 1 == N) ? 0 : y + 1;
        if (y + 1 < y1) {
            const int ynn = (yn + 1 == N) ? 0 : yn + 1;
            nn = O::ld(phi + (size_t)ynn * N + x);
            pd_n = O::ld(phidot + (size_t)yn * N + x);
            if (edge_l) el_n = __ldg(phi + (size_t)yn * N + xl);
            if (edge_r) er_n = __ldg(phi + (size_t)yn * N + xr);
        }
        T left = __shfl_up_sync(0xffffffffu, O::last(cur), 1);
        T right = __shfl_down_sync(0xffffffffu, O::first(cur), 1);
        if (edge_l) left = el;
        if (edge_r) right = er;
        V pnew, vnew;
        vector_update<T, 2, ARITH>(k, cur, left, right, prev, nxt, zero, zero, pd, pnew, vnew);
        if (live) {
            const size_t o = (size_t)y * N + x;
            O::st(phidot_next + o, vnew);
            O::st(phi_next + o, pnew);
        }
        prev = cur; cur = nxt; nxt = nn;
        pd = pd_n; el = el_n; er = er_n;
    }
}

}  // namespace prs

namespace prs {

// ------------------------------------------------------------------------------------------------
// Diagnostics (Eq. 7 link count, Eq. 8 wall velocity) with the same marching layout: one
// read of phi, phidot fetched only for vectors that contain a wall site (a few per cent of the
// lattice once the network has formed), the 16-byte phidot load of plane z issued as soon as its
// wall mask is known and consumed one iteration later.
// ------------------------------------------------------------------------------------------------
template <typename T>
__device__ __forceinline__ unsigned sign_mask(typename VecOps<T>::V v) {
    using O = VecOps<T>;
    unsigned m = 0;
#pragma unroll
    for (int i = 0; i < O::W; ++i) m |= (Ar<T>::neg(O::get(v, i)) ? 1u : 0u) << i;
    return m;
}

// Link / wall bookkeeping of one vector from sign masks.  c: this vector; l / r: sign of the scalar
// to the left / right (0 or 1); ym, yp, zm, zp: masks of the neighbouring vectors (zm = zp = c in 2D).
template <int W, int DIMS>
__device__ __forceinline__ void mask_links(unsigned c, unsigned l, unsigned r, unsigned ym, unsigned yp,
                                           unsigned zm, unsigned zp, unsigned& nlinks, unsigned& wallmask) {
    constexpr unsigned ALL = (1u << W) - 1u;
    const unsigned right_of = ((c >> 1) | (r << (W - 1))) & ALL;   // sign of x+1 for each site
    const unsigned left_of = ((c << 1) | l) & ALL;                 // sign of x-1 for each site
    const unsigned fx = c ^ right_of, bx = c ^ left_of;
    const unsigned fy = c ^ yp, by = c ^ ym;
    unsigned fz = 0, bz = 0;
    if (DIMS == 3) { fz = c ^ zp; bz = c ^ zm; }
    nlinks = __popc(fx) + __popc(fy) + __popc(fz);                 // forward links owned by these sites
    wallmask = (fx | bx | fy | by | fz | bz) & ALL;
}

// Wall sites are a few per cent of the lattice once the network has formed, so evaluating Eq. 8's
// FP64 ratio lane by lane under a predicate keeps 32 lanes busy for a handful of sites (ncu, r01b:
// 78 instructions per site, FP64 pipe 30 %).  Instead each warp compacts its wall sites into a small
// shared-memory stack (ballot + popcount give every site its slot) and pops 32 at a time, so the
// ratio is evaluated with all lanes active.  The order of the additions is fixed by the launch
// configuration and the data, hence reproducible.
template <typename T> struct Pair;
template <> struct Pair<float> { typedef float2 type; };
template <> struct Pair<double> { typedef double2 type; };

constexpr int WALLQ_CAP = 32 + 32 * 4;          // below 32 before a push, at most 4 sites per lane pushed

template <typename T>
struct WallQueue {
    typename Pair<T>::type* q;                  // this warp's stack
    int n;                                      // entries (warp-uniform)
    unsigned lt;                                // lanes below this one
    __device__ __forceinline__ void init(typename Pair<T>::type* base, int lane) {
        q = base; n = 0; lt = (1u << lane) - 1u;
    }
    // every lane of the warp must call (wallmask may be 0)
    __device__ __forceinline__ void push(unsigned wallmask, typename VecOps<T>::V c, typename VecOps<T>::V pd,
                                         double V0, double I, DiagPartial& acc) {
        using O = VecOps<T>;
        if (__ballot_sync(0xffffffffu, wallmask != 0u) == 0u) return;
        acc.walls += __popc(wallmask);
        PRS_JITTER(1u);
        __syncwarp();                           // pops of the previous call are done before slots are reused
#pragma unroll
        for (int i = 0; i < O::W; ++i) {
            const bool bit = (wallmask >> i) & 1u;
            const unsigned m = __ballot_sync(0xffffffffu, bit);
            if (bit) {
                typename Pair<T>::type e;
                e.x = O::get(c, i); e.y = O::get(pd, i);
                q[n + __popc(m & lt)] = e;
            }
            n += __popc(m);
        }
        __syncwarp();
        while (n >= 32) {
            n -= 32;
            const typename Pair<T>::type e = q[n + (int)__popc(lt)];
            acc.sum = __dadd_rn(acc.sum, wall_ratio<T>(e.x, e.y, V0, I));
        }
    }
    __device__ __forceinline__ void drain(double V0, double I, DiagPartial& acc) {
        __syncwarp();
        const int lane = (int)__popc(lt);
        if (lane < n) {
            const typename Pair<T>::type e = q[lane];
            acc.sum = __dadd_rn(acc.sum, wall_ratio<T>(e.x, e.y, V0, I));
        }
        n = 0;
    }
};

template <typename T, int TYB>
__global__ void __launch_bounds__(32 * TYB)
diag3d_tiled_kernel(const T* __restrict__ phi, const T* __restrict__ phidot, int N, int NZ, int zlo, int zhi, int ZC, double V0, double I,
                    DiagFinish fin) {
    using O = VecOps<T>;
    using V = typename O::V;
    constexpr int W = O::W;
    DiagPartial acc = {0ull, 0ull, 0.0};
    const int lane = threadIdx.x;
    const int y = blockIdx.y * TYB + threadIdx.y;
    const int xraw = (blockIdx.x * 32 + lane) * W;
    __shared__ typename Pair<T>::type wallq[TYB][WALLQ_CAP];
    WallQueue<T> wq;
    wq.init(wallq[threadIdx.y], lane);
    if (y < N) {                                           // warp-uniform
        const bool live = xraw < N;
        const int x = live ? xraw : N - W;
        const int z0 = zlo + blockIdx.z * ZC;             // planes zlo <= z < zhi of NZ (cubic: 0, N, N;
        const int z1 = min(z0 + ZC, zhi);                 // a slab: its owned planes)
        const size_t NN = (size_t)N * N;
        const int ym = (y == 0) ? N - 1 : y - 1, yp = (y == N - 1) ? 0 : y + 1;
        const size_t rc = (size_t)y * N + x, rm = (size_t)ym * N + x, rp = (size_t)yp * N + x;
        const bool edge_l = (lane == 0), edge_r = (lane == 31) || (x + W >= N);
        const size_t rl = (size_t)y * N + (x == 0 ? N - 1 : x - 1);
        const size_t rr = (size_t)y * N + (x + W >= N ? 0 : x + W);
        const int zprev = (z0 == 0) ? NZ - 1 : z0 - 1;
        // Plane offsets are kept incrementally (o_cur = z NN, o_n = (z+1) NN, periodic): no 64-bit
        // multiplications in the loop.  Everything loaded for plane z+1 (y neighbours, edge scalars) and
        // z+2 (own column) is turned into sign masks one iteration later, when it has long arrived.
        size_t o_cur = (size_t)z0 * NN;
        int zn = (z0 + 1 == NZ) ? 0 : z0 + 1;
        size_t o_n = (size_t)zn * NN;
        unsigned m_prev = sign_mask<T>(O::ld(phi + (size_t)zprev * NN + rc));
        V cur = O::ld(phi + o_cur + rc);
        V nxt = O::ld(phi + o_n + rc);
        V up = O::ld(phi + o_cur + rp), dn = O::ld(phi + o_cur + rm);
        T e_l = T(0), e_r = T(0);
        if (edge_l) e_l = __ldg(phi + o_cur + rl);
        if (edge_r) e_r = __ldg(phi + o_cur + rr);
        unsigned m_cur = sign_mask<T>(cur);
        // deferred wall work of the previous plane
        unsigned d_mask = 0;
        V d_c = cur, d_pd = cur;
        for (int z = z0; z < z1; ++z) {
            // requests for the next iteration (past the end of the chunk these re-read harmlessly)
            const bool seam = (zn + 1 == NZ);
            const size_t o_nn = seam ? 0 : o_n + NN;
            const V nn = O::ld(phi + o_nn + rc);
            const V up_n = O::ld(phi + o_n + rp), dn_n = O::ld(phi + o_n + rm);
            T e_l_n = T(0), e_r_n = T(0);
            if (edge_l) e_l_n = __ldg(phi + o_n + rl);
            if (edge_r) e_r_n = __ldg(phi + o_n + rr);
            const unsigned m_nxt = sign_mask<T>(nxt), m_up = sign_mask<T>(up), m_dn = sign_mask<T>(dn);
            unsigned l = __shfl_up_sync(0xffffffffu, (m_cur >> (W - 1)) & 1u, 1);
            unsigned r = __shfl_down_sync(0xffffffffu, m_cur & 1u, 1);
            if (edge_l) l = Ar<T>::neg(e_l);
            if (edge_r) r = Ar<T>::neg(e_r);
            unsigned nlinks, wallmask;
            mask_links<W, 3>(m_cur, l, r, m_dn, m_up, m_prev, m_nxt, nlinks, wallmask);
            if (!live) { nlinks = 0; wallmask = 0; }
            acc.links += nlinks;
            V pd_now = cur;
            if (wallmask) pd_now = O::ld(phidot + o_cur + rc);       // consumed next iteration
            wq.push(d_mask, d_c, d_pd, V0, I, acc);
            d_mask = wallmask; d_c = cur; d_pd = pd_now;
            m_prev = m_cur; m_cur = m_nxt; cur = nxt; nxt = nn;
            up = up_n; dn = dn_n; e_l = e_l_n; e_r = e_r_n;
            o_cur = o_n; o_n = o_nn; zn = seam ? 0 : zn + 1;
        }
        wq.push(d_mask, d_c, d_pd, V0, I, acc);
        wq.drain(V0, I, acc);
    }
    acc = block_reduce(acc);
    finish_partials(fin, acc);
}

template <typename T>
__global__ void __launch_bounds__(128)
diag2d_tiled_kernel(const T* __restrict__ phi, const T* __restrict__ phidot, int N, int YC, double V0, double I,
                    DiagFinish fin) {
    using O = VecOps<T>;
    using V = typename O::V;
    constexpr int W = O::W;
    DiagPartial acc = {0ull, 0ull, 0.0};
    const int lane = threadIdx.x & 31;
    const long long xraw = ((long long)blockIdx.x * blockDim.x + threadIdx.x) * W;
    __shared__ typename Pair<T>::type wallq[4][WALLQ_CAP];
    WallQueue<T> wq;
    wq.init(wallq[threadIdx.x >> 5], lane);
    if (xraw - (long long)lane * W < N) {                  // warp-uniform
        const bool live = xraw < N;
        const int x = live ? (int)xraw : N - W;
        const int y0 = blockIdx.y * YC;
        const int y1 = min(y0 + YC, N);
        const bool edge_l = (lane == 0), edge_r = (lane == 31) || (x + W >= N);
        const int xl = (x == 0) ? N - 1 : x - 1, xr = (x + W >= N) ? 0 : x + W;
        const int yprev = (y0 == 0) ? N - 1 : y0 - 1;
        // row offsets kept incrementally (o_cur = y N, o_n = (y+1) N, periodic), as in the 3D kernel
        size_t o_cur = (size_t)y0 * N;
        int yn = (y0 + 1 == N) ? 0 : y0 + 1;
        size_t o_n = (size_t)yn * N;
        unsigned m_prev = sign_mask<T>(O::ld(phi + (size_t)yprev * N + x));
        V cur = O::ld(phi + o_cur + x);
        V nxt = O::ld(phi + o_n + x);
        T e_l = T(0), e_r = T(0);
        if (edge_l) e_l = __ldg(phi + o_cur + xl);
        if (edge_r) e_r = __ldg(phi + o_cur + xr);
        unsigned m_cur = sign_mask<T>(cur);
        unsigned d_mask = 0;
        V d_c = cur, d_pd = cur;
        for (int y = y0; y < y1; ++y) {
            // requests for the next iteration (past the end of the chunk these re-read harmlessly)
            const bool seam = (yn + 1 == N);
            const size_t o_nn = seam ? 0 : o_n + N;
            const V nn = O::ld(phi + o_nn + x);
            T e_l_n = T(0), e_r_n = T(0);
            if (edge_l) e_l_n = __ldg(phi + o_n + xl);
            if (edge_r) e_r_n = __ldg(phi + o_n + xr);
            const unsigned m_nxt = sign_mask<T>(nxt);
            unsigned l = __shfl_up_sync(0xffffffffu, (m_cur >> (W - 1)) & 1u, 1);
            unsigned r = __shfl_down_sync(0xffffffffu, m_cur & 1u, 1);
            if (edge_l) l = Ar<T>::neg(e_l);
            if (edge_r) r = Ar<T>::neg(e_r);
            unsigned nlinks, wallmask;
            mask_links<W, 2>(m_cur, l, r, m_prev, m_nxt, m_cur, m_cur, nlinks, wallmask);
            if (!live) { nlinks = 0; wallmask = 0; }
            acc.links += nlinks;
            V pd_now = cur;
            if (wallmask) pd_now = O::ld(phidot + o_cur + x);
            wq.push(d_mask, d_c, d_pd, V0, I, acc);
            d_mask = wallmask; d_c = cur; d_pd = pd_now;
            m_prev = m_cur; m_cur = m_nxt; cur = nxt; nxt = nn;
            e_l = e_l_n; e_r = e_r_n;
            o_cur = o_n; o_n = o_nn; yn = seam ? 0 : yn + 1;
        }
        wq.push(d_mask, d_c, d_pd, V0, I, acc);
        wq.drain(V0, I, acc);
    }
    acc = block_reduce(acc);
    finish_partials(fin, acc);
}

}  // namespace prs
