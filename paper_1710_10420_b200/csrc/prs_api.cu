// prs_api.cu -- host side of libprs: context, workspace carving, per-step scalars, kernel selection
// and launch, and the C ABI declared in include/prs.h.  No device memory is allocated here: the
// caller's workspace holds everything (see prs.h, "Memory and ownership").
// The temporally blocked kernels are compiled in translation units of their own (prs_instances.cu);
// this one holds the single-step, cluster, diagnostics and initial-condition kernels.
#include "prs_host.cuh"

#include <algorithm>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

#include "prs_kernels_generic.cuh"
#include "prs_kernels_tiled.cuh"
#include "prs_kernels_cluster.cuh"
#include "prs_kernels_bits.cuh"

using namespace prs;

namespace {

constexpr size_t ALIGN = 256;
constexpr int MAX_PARTIALS = 1 << 16;        // upper bound on diagnostics blocks (1.5 MiB of scratch)
constexpr int RESULTS_CAP = 4096;            // diagnostics records prs_run keeps on the device between readbacks (96 KiB)

inline size_t align_up(size_t v) { return (v + ALIGN - 1) / ALIGN * ALIGN; }

inline bool args_ok(int dims, int64_t N, int precision) {
    if (dims != 2 && dims != 3) return false;
    if (N < 1 || N > (int64_t)1 << 20) return false;
    if (precision != PRS_F32 && precision != PRS_F64) return false;
    if (dims == 3 && N > 8192) return false;   // 8192^3 * 4 arrays would not fit anyway
    return true;
}

inline size_t sites_of(int dims, int64_t N) { return dims == 3 ? (size_t)N * N * N : (size_t)N * N; }

struct Layout {
    size_t field_bytes, off_phi[2], off_pd[2], off_partials, off_result, off_results, off_bits, total;
};

constexpr int SLAB_HALO = 4;                 // halo planes per side = the most steps one 3D launch takes

Layout layout_of_sites(size_t sites, int precision) {
    Layout L;
    L.field_bytes = align_up(sites * (precision == PRS_F32 ? 4 : 8));
    size_t o = 0;
    L.off_phi[0] = o; o += L.field_bytes;
    L.off_phi[1] = o; o += L.field_bytes;
    L.off_pd[0] = o; o += L.field_bytes;
    L.off_pd[1] = o; o += L.field_bytes;
    L.off_partials = o; o += align_up(sizeof(DiagPartial) * MAX_PARTIALS);
    L.off_result = o; o += align_up(sizeof(DiagPartial));
    L.off_results = o; o += align_up(sizeof(DiagPartial) * RESULTS_CAP);
    L.off_bits = o; o += align_up((sites + 7) / 8);             // one sign bit per site (prs_kernels_bits.cuh)
    L.total = o;
    return L;
}

Layout layout_of(int dims, int64_t N, int precision) { return layout_of_sites(sites_of(dims, N), precision); }

// A z slab: 3D, N a multiple of 4 (whole Philox quads and 16-byte vectors per row), at least SLAB_HALO
// owned planes (a neighbour's halo is filled from one rank only).
inline bool slab_args_ok(int64_t N, int64_t nz, int64_t z_begin, int precision) {
    if (!args_ok(3, N, precision)) return false;
    if (N % 4 != 0) return false;
    if (nz < SLAB_HALO || nz > N) return false;
    if (z_begin < 0 || z_begin >= N) return false;
    return true;
}
inline size_t slab_sites(int64_t N, int64_t nz) { return (size_t)N * N * (size_t)(nz + 2 * SLAB_HALO); }

}  // namespace

namespace {

int fail(prs_ctx* h, int code, const std::string& msg) {
    if (h) h->err = msg;
    return code;
}

int cuda_fail(prs_ctx* h, cudaError_t e, const char* where) {
    return fail(h, PRS_ERR_CUDA, std::string(where) + ": " + cudaGetErrorName(e) + " (" + cudaGetErrorString(e) + ")");
}

#define PRS_CUDA(h, call)                                        \
    do {                                                         \
        cudaError_t e_ = (call);                                 \
        if (e_ != cudaSuccess) return cuda_fail((h), e_, #call); \
    } while (0)

// Every exported call that touches CUDA runs with the handle's device current (the caller's is restored on return).
#define PRS_ON_DEVICE(h)                      \
    DeviceGuard guard_((h)->device);          \
    if (guard_.err != cudaSuccess) return cuda_fail((h), guard_.err, "cudaSetDevice")

inline int vec_width(int precision) { return precision == PRS_F32 ? 4 : 2; }

bool tiled_supported(const prs_ctx* h) {
    const int W = vec_width(h->precision);
    return h->N % W == 0 && h->N >= W && h->N <= (1 << 30);
}

// The temporally blocked kernels address 16-byte vectors with unsigned 32-bit indices whose load cursor
// overshoots by up to one lattice length before it wraps: N^d / W <= 2^31 (2048^3 FP32 just fits).
bool tb2_supported(const prs_ctx* h) {
    if (!tiled_supported(h)) return false;
    return h->dims == 2 || h->S / (size_t)vec_width(h->precision) <= ((size_t)1 << 31);
}
bool tbs_supported(const prs_ctx* h) {
    if (!tiled_supported(h)) return false;
    const size_t nv = h->S / (size_t)vec_width(h->precision);
    return h->dims == 3 ? nv <= ((size_t)1 << 31) : nv < ((size_t)1 << 30);     // the 2D kernel's cursors are signed
}

// The cluster-resident small-box kernel: 2D, whole rows per 1024-thread sweep, state in the registers and shared memory
// of 8 or 16 CTAs.
bool cluster_supported(const prs_ctx* h) {
    if (h->dims != 2 || (h->N != 64 && h->N != 128 && h->N != 256)) return false;
    const size_t smem = (h->precision == PRS_F32) ? cluster_smem_bytes<float>((int)h->N) : cluster_smem_bytes<double>((int)h->N);
    return smem <= 227 * 1024;
}

// Can this device co-schedule ONE cluster of 16 CTAs x 1024 threads (non-portable size)?  Asked once per device.
bool cluster16_fits(const prs_ctx* h) {
    static std::atomic<unsigned long long> asked{0}, yes{0};
    const unsigned long long bit = (h->device >= 0 && h->device < 64) ? (1ull << h->device) : 0ull;
    if (bit && (asked.load() & bit)) return (yes.load() & bit) != 0;
    auto kern = step2d_cluster_kernel<float, ARITH_FMA, 1, 16>;
    DeviceGuard guard(h->device);
    int n = 0;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)CLUSTER_SMEM_LIMIT);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
    if (e == cudaSuccess) {
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(16, 1, 1); cfg.blockDim = dim3(CLUSTER_THREADS, 1, 1); cfg.dynamicSmemBytes = cluster_smem_bytes<double>(256, 16);
        cudaLaunchAttribute at;
        at.id = cudaLaunchAttributeClusterDimension;
        at.val.clusterDim.x = 16; at.val.clusterDim.y = 1; at.val.clusterDim.z = 1;
        cfg.attrs = &at; cfg.numAttrs = 1;
        e = cudaOccupancyMaxActiveClusters(&n, kern, &cfg);
    }
    if (e != cudaSuccess) cudaGetLastError();
    const bool ok = (e == cudaSuccess && n >= 1);
    if (bit) { if (ok) yes.fetch_or(bit); asked.fetch_or(bit); }
    return ok;
}

int resolve_step_kernel(const prs_ctx* h) {
    int want = h->opt_step_kernel;
    if (want == PRS_KERNEL_AUTO) {
        // Measured on B200 (profiles/): the four-step kernel wins from 64^2 and
        // 128^3 up -- on small lattices because it needs a quarter of the launches, on large ones
        // because it moves a quarter of the bytes; below that the single-step march is quicker.
        if (!tiled_supported(h)) want = PRS_KERNEL_GENERIC;
        // the cluster-resident kernel against the streaming one, us per step (FP32 | FP64): 64^2 0.36 | 0.39 vs 1.03 | 1.03;
        // 128^2 0.43 | 0.61 vs 1.03 | 1.28; 256^2 on 16 CTAs 0.71 | 1.09 vs 1.05 | 1.37 (on 8 CTAs 1.09 | 2.2)
        else if ((h->N == 64 || h->N == 128) && cluster_supported(h)) want = PRS_KERNEL_CLUSTER;
        else if (h->N == 256 && h->opt_cluster_ctas != 8 && cluster_supported(h) && cluster16_fits(h)) want = PRS_KERNEL_CLUSTER;
        else if (tbs_supported(h) && ((h->dims == 2 && h->N >= 64) || (h->dims == 3 && h->N >= 128))) want = PRS_KERNEL_TBS;
        else if (h->S >= ((size_t)1 << 22) && tb2_supported(h)) want = PRS_KERNEL_TB2;
        else want = PRS_KERNEL_TILED;
    }
    return want;
}

// ---- launches -----------------------------------------------------------------------------------

template <typename T, int DIMS, int ARITH>
cudaError_t launch_generic(prs_ctx* h, const T* p, const T* v, T* pn, T* vn, const StepCoef<T>& k) {
    const unsigned blocks = (unsigned)((h->S + 255) / 256);
    step_generic_kernel<T, DIMS, ARITH><<<blocks, 256, 0, h->stream>>>(p, v, pn, vn, (long long)h->N,
                                                                         (long long)h->NZ, (long long)h->S, k);
    char name[96];
    snprintf(name, sizeof(name), "step_generic_kernel<%s,%d,%d>", type_name<T>(), DIMS, ARITH);
    note_launch(h, name, dim3(blocks, 1, 1), dim3(256, 1, 1), 0, 1);
    return cudaGetLastError();
}

int pick_chunk(const prs_ctx* h, long long tiles_per_slab, int threads_per_cta) {
    if (h->opt_chunk > 0) return (int)std::min<int64_t>(h->opt_chunk, h->N);
    // Short chunks win (measured, 1024^3: 8 planes 2.71 ms, 128 planes 2.74 ms, 1024 planes 2.87 ms):
    // the grid sweeps the march axis chunk by chunk in launch order, so the two halo planes of a
    // chunk are still in L2 from its predecessor, and many small CTAs balance the tail.  Keep at
    // least ~16 waves of CTAs and chunks between 8 and 32 long.
    const long long resident = (long long)h->sm_count * (1024 / threads_per_cta);
    const long long want_ctas = 16 * resident;
    long long chunks = (want_ctas + tiles_per_slab - 1) / tiles_per_slab;
    if (chunks < 1) chunks = 1;
    long long len = h->N / chunks;
    if (len > 32) len = 32;
    if (len < 8) len = 8;
    if (len > h->N) len = h->N;
    return (int)len;
}

template <typename T, int ARITH>
cudaError_t launch_tiled3d(prs_ctx* h, const T* p, const T* v, T* pn, T* vn, const StepCoef<T>& k) {
    constexpr int W = VecOps<T>::W;
    const int N = (int)h->N;
    const int ty = h->opt_tile_y;
    const unsigned gx = (unsigned)((N + 32 * W - 1) / (32 * W)), gy = (unsigned)((N + ty - 1) / ty);
    const int NZ = (int)h->NZ;                 // = N unless the handle is a z slab: then all its planes are advanced
    const int ZC = std::min(pick_chunk(h, (long long)gx * gy, 32 * ty), NZ);
    const dim3 grid(gx, gy, (unsigned)((NZ + ZC - 1) / ZC));
    const dim3 block(32, ty, 1);
    if (ty == 4) step3d_tiled_kernel<T, ARITH, 4><<<grid, block, 0, h->stream>>>(p, v, pn, vn, N, NZ, ZC, k);
    else if (ty == 16) step3d_tiled_kernel<T, ARITH, 16><<<grid, block, 0, h->stream>>>(p, v, pn, vn, N, NZ, ZC, k);
    else step3d_tiled_kernel<T, ARITH, 8><<<grid, block, 0, h->stream>>>(p, v, pn, vn, N, NZ, ZC, k);
    char name[96];
    snprintf(name, sizeof(name), "step3d_tiled_kernel<%s,%d,%d>", type_name<T>(), ARITH, (ty == 4 || ty == 16) ? ty : 8);
    note_launch(h, name, grid, block, 0, 1);
    return cudaGetLastError();
}

template <typename T, int ARITH>
cudaError_t launch_tiled2d(prs_ctx* h, const T* p, const T* v, T* pn, T* vn, const StepCoef<T>& k) {
    constexpr int W = VecOps<T>::W;
    const int N = (int)h->N;
    const int BX = 128;
    const unsigned gx = (unsigned)((N + BX * W - 1) / (BX * W));
    const int YC = pick_chunk(h, gx, BX);
    const dim3 grid(gx, (unsigned)((N + YC - 1) / YC), 1);
    step2d_tiled_kernel<T, ARITH><<<grid, BX, 0, h->stream>>>(p, v, pn, vn, N, YC, k);
    char name[96];
    snprintf(name, sizeof(name), "step2d_tiled_kernel<%s,%d>", type_name<T>(), ARITH);
    note_launch(h, name, grid, dim3(BX, 1, 1), 0, 1);
    return cudaGetLastError();
}

// Two steps in one pass (n -> n+2); the caller guarantees the lattice is supported.
template <typename T>
int step_twice(prs_ctx* h) {
    const StepCoef<T> k1 = coef_at<T>(h, h->step), k2 = coef_at<T>(h, h->step + 1);
    const T* p = (const T*)h->phi[h->cur];
    const T* v = (const T*)h->pd[h->cur];
    T* pn = (T*)h->phi[h->cur ^ 1];
    T* vn = (T*)h->pd[h->cur ^ 1];
    cudaError_t e;
#define PRS_TB2(AR) (h->dims == 3 ? launch_tb2_3d<T, AR>(h, p, v, pn, vn, k1, k2) : launch_tb2_2d<T, AR>(h, p, v, pn, vn, k1, k2))
    e = (h->opt_arith == PRS_ARITH_LITERAL) ? PRS_TB2(ARITH_LITERAL) : (h->opt_arith == PRS_ARITH_COEF) ? PRS_TB2(ARITH_COEF) : PRS_TB2(ARITH_FMA);
#undef PRS_TB2
    if (e != cudaSuccess) return cuda_fail(h, e, "two-step kernel launch");
    h->launches += 1;
    h->cur ^= 1;
    h->step += 2;
    return PRS_OK;
}

// S steps in one pass (n -> n+S); the caller guarantees tbs_supported(h).
template <typename T>
int step_many(prs_ctx* h, int S) {
    const T* p = (const T*)h->phi[h->cur];
    const T* v = (const T*)h->pd[h->cur];
    T* pn = (T*)h->phi[h->cur ^ 1];
    T* vn = (T*)h->pd[h->cur ^ 1];
    cudaError_t e;
#define PRS_TBS(AR)                                                                                                   \
    (h->dims == 3 ? (S == 3 ? launch_tbs_3d<T, AR, 3>(h, p, v, pn, vn) : launch_tbs_3d<T, AR, 4>(h, p, v, pn, vn)) \
                  : (S == 3 ? launch_tbs_2d<T, AR, 3>(h, p, v, pn, vn)                                                \
                     : S == 4 ? launch_tbs_2d<T, AR, 4>(h, p, v, pn, vn)                                              \
                     : S == 6 ? launch_tbs_2d<T, AR, 6>(h, p, v, pn, vn) : launch_tbs_2d<T, AR, 8>(h, p, v, pn, vn)))
    e = (h->opt_arith == PRS_ARITH_LITERAL) ? PRS_TBS(ARITH_LITERAL) : (h->opt_arith == PRS_ARITH_COEF) ? PRS_TBS(ARITH_COEF) : PRS_TBS(ARITH_FMA);
#undef PRS_TBS
    if (e != cudaSuccess) return cuda_fail(h, e, "multi-step kernel launch");
    h->launches += 1;
    h->cur ^= 1;
    h->step += S;
    return PRS_OK;
}

// Up to CLUSTER_MAX_STEPS steps inside one cluster-resident launch (2D small boxes), with the diagnostics passes `dg`
// schedules inside it (dg.every = 0: none).
template <typename T, int ARITH>
cudaError_t launch_cluster(prs_ctx* h, const T* p, const T* v, T* pn, T* vn, int nsteps, const ClusterDiag& dg) {
    ClusterCoefs<T> ks;
    for (int s = 0; s < nsteps; ++s) ks.k[s] = coef_at<T>(h, h->step + s);
    for (int s = nsteps; s < CLUSTER_MAX_STEPS; ++s) ks.k[s] = ks.k[0];
    // 256^2 runs as ONE cluster of 16 CTAs (non-portable size, opt-in) where the device can co-schedule one: a thread then
    // owns half as many vectors (FP32: one, like 128^2 with 8 CTAs).  Everything else, and the fall-back, is 8 CTAs.
    int ncta = (h->N == 256 && h->opt_cluster_ctas != 8) ? 16 : CLUSTER_CTAS;
    for (;;) {
        const size_t smem = cluster_smem_bytes<T>((int)h->N, ncta);
        const int vpt = cluster_vpt<T>((int)h->N, ncta);
        cudaError_t e = cudaSuccess;
        bool fits = true;
#define PRS_CLUSTER_LAUNCH(VPT, NCTA)                                                                                        \
    do {                                                                                                                     \
        auto kern = step2d_cluster_kernel<T, ARITH, VPT, NCTA>;                                                              \
        static std::atomic<unsigned long long> configured{0};  /* per instantiation: devices already set up */               \
        static std::atomic<unsigned long long> unfit{0};       /* devices that cannot hold a cluster of NCTA */              \
        const unsigned long long bit = (h->device >= 0 && h->device < 64) ? (1ull << h->device) : 0ull;                      \
        if (bit && (unfit.load() & bit)) { fits = false; break; }                                                            \
        const bool first = !(bit && (configured.load() & bit));                                                              \
        /* above the most any supported lattice needs (256^2 FP64 on 8 CTAs: 136 KiB); 227 KB would exceed the limit with   \
           the static part */                                                                                                \
        e = ensure_dynamic_smem(kern, CLUSTER_SMEM_LIMIT, h->device, configured);                                            \
        if (e != cudaSuccess) break;                                                                                         \
        if (NCTA > 8 && first) {                                                                                             \
            e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);                               \
            int nclusters = 0;                                                                                               \
            if (e == cudaSuccess) {                                                                                          \
                cudaLaunchConfig_t cfg = {};                                                                                 \
                cfg.gridDim = dim3(NCTA, 1, 1); cfg.blockDim = dim3(CLUSTER_THREADS, 1, 1); cfg.dynamicSmemBytes = smem;     \
                cudaLaunchAttribute at;                                                                                      \
                at.id = cudaLaunchAttributeClusterDimension;                                                                 \
                at.val.clusterDim.x = NCTA; at.val.clusterDim.y = 1; at.val.clusterDim.z = 1;                                \
                cfg.attrs = &at; cfg.numAttrs = 1;                                                                           \
                e = cudaOccupancyMaxActiveClusters(&nclusters, kern, &cfg);                                                  \
            }                                                                                                                \
            if (e != cudaSuccess || nclusters < 1) {                                                                         \
                cudaGetLastError();                                                                                          \
                e = cudaSuccess; fits = false;                                                                               \
                if (bit) unfit.fetch_or(bit);                                                                                \
                break;                                                                                                       \
            }                                                                                                                \
        }                                                                                                                    \
        kern<<<NCTA, CLUSTER_THREADS, smem, h->stream>>>(p, v, pn, vn, (int)h->N, nsteps, ks, dg);                           \
    } while (0)
        if (ncta == 16) { if (vpt == 1) PRS_CLUSTER_LAUNCH(1, 16); else PRS_CLUSTER_LAUNCH(2, 16); }
        else if (vpt == 1) PRS_CLUSTER_LAUNCH(1, 8);
        else if (vpt == 2) PRS_CLUSTER_LAUNCH(2, 8);
        else PRS_CLUSTER_LAUNCH(4, 8);
#undef PRS_CLUSTER_LAUNCH
        if (e != cudaSuccess) return e;
        if (!fits && ncta == 16) { ncta = CLUSTER_CTAS; continue; }       // no room for 16 CTAs in one cluster here
        char name[96];
        snprintf(name, sizeof(name), "step2d_cluster_kernel<%s,%d,%d,%d>", type_name<T>(), ARITH, vpt, ncta);
        note_launch(h, name, dim3(ncta, 1, 1), dim3(CLUSTER_THREADS, 1, 1), smem, nsteps);
        return cudaGetLastError();
    }
}

template <typename T>
int step_cluster(prs_ctx* h, int nsteps, const ClusterDiag& dg) {
    const T* p = (const T*)h->phi[h->cur];
    const T* v = (const T*)h->pd[h->cur];
    T* pn = (T*)h->phi[h->cur ^ 1];
    T* vn = (T*)h->pd[h->cur ^ 1];
    const cudaError_t e = (h->opt_arith == PRS_ARITH_LITERAL) ? launch_cluster<T, ARITH_LITERAL>(h, p, v, pn, vn, nsteps, dg)
                        : (h->opt_arith == PRS_ARITH_COEF)  ? launch_cluster<T, ARITH_COEF>(h, p, v, pn, vn, nsteps, dg)
                                                            : launch_cluster<T, ARITH_FMA>(h, p, v, pn, vn, nsteps, dg);
    if (e != cudaSuccess) return cuda_fail(h, e, "cluster kernel launch");
    h->launches += 1;
    h->cur ^= 1;
    h->step += nsteps;
    return PRS_OK;
}

template <typename T>
int step_once(prs_ctx* h, int kernel) {
    const StepCoef<T> k = coef_at<T>(h, h->step);
    const T* p = (const T*)h->phi[h->cur];
    const T* v = (const T*)h->pd[h->cur];
    T* pn = (T*)h->phi[h->cur ^ 1];
    T* vn = (T*)h->pd[h->cur ^ 1];
    cudaError_t e;
#define PRS_ONE(AR)                                                                                                      \
    (kernel == PRS_KERNEL_TILED                                                                                           \
         ? (h->dims == 3 ? launch_tiled3d<T, AR>(h, p, v, pn, vn, k) : launch_tiled2d<T, AR>(h, p, v, pn, vn, k))         \
         : (h->dims == 3 ? launch_generic<T, 3, AR>(h, p, v, pn, vn, k) : launch_generic<T, 2, AR>(h, p, v, pn, vn, k)))
    e = (h->opt_arith == PRS_ARITH_LITERAL) ? PRS_ONE(ARITH_LITERAL) : (h->opt_arith == PRS_ARITH_COEF) ? PRS_ONE(ARITH_COEF) : PRS_ONE(ARITH_FMA);
#undef PRS_ONE
    if (e != cudaSuccess) return cuda_fail(h, e, "step kernel launch");
    h->launches += 1;
    h->cur ^= 1;
    h->step += 1;
    return PRS_OK;
}

bool diag_tiled_supported(const prs_ctx* h) {
    if (!tiled_supported(h)) return false;
    const int W = vec_width(h->precision);
    const long long gx = (h->N + 32LL * W - 1) / (32LL * W);
    const long long tiles = (h->dims == 3) ? gx * ((h->N + 3) / 4) : (h->N + 128LL * W - 1) / (128LL * W);
    return tiles <= MAX_PARTIALS;
}

// The packed-sign-bit pass (prs_kernels_bits.cuh): whole groups of 32 vectors per row.
bool diag_bits_supported(const prs_ctx* h) {
    const int W = vec_width(h->precision);
    // whole groups of 32 vectors per row; the kernels index groups and rows with 32 bits
    return h->N % (32 * W) == 0 && h->N <= (1 << 30) && h->S / (size_t)(32 * W) < ((size_t)1 << 31) && h->S / (size_t)h->N < ((size_t)1 << 31);
}

int resolve_diag_kernel(const prs_ctx* h) {
    int want = h->opt_diag_kernel;
    if (want == PRS_KERNEL_AUTO) {
        // the three launches of the bit pass pay off once reading phi dominates (measured)
        if (diag_bits_supported(h) && h->S >= ((size_t)1 << 26)) want = PRS_KERNEL_BITS;
        else want = diag_tiled_supported(h) ? PRS_KERNEL_TILED : PRS_KERNEL_GENERIC;
    }
    return want;
}

// Chunk length of the diagnostics march (planes in 3D, rows in 2D; PRS_OPT_DIAG_CHUNK overrides).  Large lattices: as
// short as the partials scratch allows but no shorter than 16 (the first plane / row of a chunk costs three loads
// instead of one).  Small lattices are bound by the latency of the march, not by its loads: there the chunks are cut
// down (to no less than 2) until the grid holds about four CTAs per SM.
int diag_chunk(const prs_ctx* h, long long tiles_per_slab, int span) {
    if (h->opt_diag_chunk > 0) return std::max(1, std::min(h->opt_diag_chunk, span));
    long long max_chunks = MAX_PARTIALS / tiles_per_slab;
    if (max_chunks < 1) max_chunks = 1;
    long long len = (span + max_chunks - 1) / max_chunks;
    if (len < 16) len = 16;
    const long long want = 4LL * std::max(1, h->sm_count);
    while (len > 2 && tiles_per_slab * ((span + len - 1) / len) < want) len /= 2;
    if (len > span) len = span;
    return (int)len;
}

// The rows the sign-bit passes measure [m0, m1) and the rows whose signs they need [b0, b1) (a slab: its owned planes,
// and one halo plane on either side), in units of lattice rows (row = y + N z; 2D: y).
struct BitRows { long long m0, m1, b0, b1; };
BitRows bit_rows(const prs_ctx* h) {
    const long long rows_per_plane = (h->dims == 3) ? h->N : 1;
    const long long nplanes = (h->dims == 3) ? h->NZ : h->N;     // 2D: a "plane" is a row
    const long long p0 = h->slab ? h->halo : 0, p1 = h->slab ? h->halo + h->nz_own : nplanes;
    const long long b0 = h->slab ? p0 - 1 : 0, b1 = h->slab ? p1 + 1 : nplanes;
    return {p0 * rows_per_plane, p1 * rows_per_plane, b0 * rows_per_plane, b1 * rows_per_plane};
}

// Packs the sign bits of the current phi unless the bit array already holds them (prs_weighted_area right after
// prs_diagnostics: the state has not moved).  The tag is the step counter, the ping-pong index and a generation number
// that prs_init, prs_copy_in and prs_slab_halo_filled advance.
template <typename T>
int ensure_bits(prs_ctx* h) {
    if (h->bits_valid && h->bits_step == h->step && h->bits_cur == h->cur && h->bits_gen == h->state_gen) return PRS_OK;
    constexpr int W = VecOps<T>::W;
    const int N = (int)h->N, NG = N / (32 * W);
    const BitRows br = bit_rows(h);
    const long long sgroups = (br.b1 - br.b0) * NG;                  // one warp each
    const long long sblocks = std::min<long long>((sgroups + 7) / 8, (long long)h->sm_count * 16);
    sign_bits_kernel<T><<<(unsigned)sblocks, 256, 0, h->stream>>>((const T*)h->phi[h->cur], h->bits, N, br.b0, br.b1);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(h, e, "sign-bit kernel launch");
    h->launches += 1;
    h->bits_valid = true; h->bits_step = h->step; h->bits_cur = h->cur; h->bits_gen = h->state_gen;
    return PRS_OK;
}

// Launches the diagnostics pass on the current state; the reduced record goes to `dst` (device).
template <typename T>
int diag_launch(prs_ctx* h, DiagPartial* dst) {
    const double pi = 3.14159265358979323846;
    const double V0 = (pi * pi * h->phi0 * h->phi0) / (2.0 * h->W0 * h->W0);
    const double I = 1.0 / (h->phi0 * h->phi0);
    const T* p = (const T*)h->phi[h->cur];
    const T* v = (const T*)h->pd[h->cur];
    const int kernel = resolve_diag_kernel(h);
    const DiagFinish fin = {h->partials, dst, h->d_ticket};   // the last block to finish reduces the partials into dst
    long long blocks;
    if (kernel == PRS_KERNEL_BITS) {
        constexpr int W = VecOps<T>::W;
        const int N = (int)h->N, NG = N / (32 * W);
        const int rc = ensure_bits<T>(h);
        if (rc != PRS_OK) return rc;
        const BitRows br = bit_rows(h);
        const long long lgroups = (br.m1 - br.m0) * NG;                  // one thread each
        blocks = std::min<long long>((lgroups + BITS_THREADS - 1) / BITS_THREADS, std::min<long long>(MAX_PARTIALS, (long long)h->sm_count * 16));
        if (h->dims == 3)
            bit_links_kernel<T, 3><<<(unsigned)blocks, BITS_THREADS, 0, h->stream>>>(p, v, h->bits, N, (int)h->NZ, br.m0, br.m1, V0, I, fin);
        else
            bit_links_kernel<T, 2><<<(unsigned)blocks, BITS_THREADS, 0, h->stream>>>(p, v, h->bits, N, 1, br.m0, br.m1, V0, I, fin);
    } else if (kernel == PRS_KERNEL_TILED) {
        constexpr int W = VecOps<T>::W;
        const int N = (int)h->N;
        if (h->dims == 3) {
            constexpr int TY = 4;
            const unsigned gx = (unsigned)((N + 32 * W - 1) / (32 * W)), gy = (unsigned)((N + TY - 1) / TY);
            // a z slab measures its owned planes only (their z neighbours are halo planes, never the wrap)
            const int NZ = (int)h->NZ, zlo = h->slab ? (int)h->halo : 0, zhi = h->slab ? (int)(h->halo + h->nz_own) : N;
            const int ZC = diag_chunk(h, (long long)gx * gy, zhi - zlo);
            const dim3 grid(gx, gy, (unsigned)((zhi - zlo + ZC - 1) / ZC));
            blocks = (long long)grid.x * grid.y * grid.z;
            diag3d_tiled_kernel<T, TY><<<grid, dim3(32, TY, 1), 0, h->stream>>>(p, v, N, NZ, zlo, zhi, ZC, V0, I, fin);
        } else {
            const unsigned gx = (unsigned)((N + 128 * W - 1) / (128 * W));
            const int YC = diag_chunk(h, gx, N);
            const dim3 grid(gx, (unsigned)((N + YC - 1) / YC), 1);
            blocks = (long long)grid.x * grid.y;
            diag2d_tiled_kernel<T><<<grid, 128, 0, h->stream>>>(p, v, N, YC, V0, I, fin);
        }
    } else {
        // a z slab measures its owned planes only (their z neighbours are halo planes, never the wrap)
        const long long NN = (long long)h->N * h->N;
        const long long s0 = h->slab ? h->halo * NN : 0, s1 = h->slab ? (h->halo + h->nz_own) * NN : (long long)h->S;
        blocks = (s1 - s0 + 255) / 256;
        const long long cap = std::min<long long>(MAX_PARTIALS, (long long)h->sm_count * 8);
        if (blocks > cap) blocks = cap;
        if (h->dims == 3)
            diag_generic_kernel<T, 3><<<(unsigned)blocks, 256, 0, h->stream>>>(p, v, (long long)h->N, (long long)h->NZ, s0, s1, V0, I, fin);
        else
            diag_generic_kernel<T, 2><<<(unsigned)blocks, 256, 0, h->stream>>>(p, v, (long long)h->N, (long long)h->NZ, s0, s1, V0, I, fin);
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(h, e, "diagnostics kernel launch");
    (void)blocks;
    h->launches += 1;
    h->last_diag_kernel = kernel;
    return PRS_OK;
}

}  // namespace

extern "C" {

size_t prs_workspace_bytes(int dims, int64_t N, int precision) {
    if (!args_ok(dims, N, precision)) return 0;
    return layout_of(dims, N, precision).total;
}

// Shared by prs_create and prs_create_slab: checks the physics arguments and the workspace, builds the context
// over `sites` local sites.
static int create_common(prs_handle* out, int dims, int64_t N, size_t sites, int precision, double alpha, double era_m,
                         double deta, double W0, double phi0, uint64_t seed, void* workspace, size_t workspace_bytes,
                         void* cuda_stream) {
    if (!(deta > 0.0) || !(W0 > 0.0) || !(phi0 > 0.0) || !(alpha >= 0.0) || !(era_m >= 0.0))
        return PRS_ERR_INVALID_ARG;
    if (!std::isfinite(deta) || !std::isfinite(W0) || !std::isfinite(phi0) || !std::isfinite(alpha) ||
        !std::isfinite(era_m))
        return PRS_ERR_INVALID_ARG;
    const Layout L = layout_of_sites(sites, precision);
    if (!workspace || workspace_bytes < L.total || ((uintptr_t)workspace % ALIGN) != 0) return PRS_ERR_WORKSPACE;
    cudaPointerAttributes attr;
    if (cudaPointerGetAttributes(&attr, workspace) != cudaSuccess || attr.type != cudaMemoryTypeDevice) {
        cudaGetLastError();
        return PRS_ERR_WORKSPACE;
    }
    prs_ctx* h = new (std::nothrow) prs_ctx();
    if (!h) return PRS_ERR_NOMEM;
    h->dims = dims; h->precision = precision; h->N = N; h->S = sites;
    h->slab = false; h->NZ = N; h->nz_own = N; h->halo = 0; h->z_begin = 0; h->halo_valid = 0;
    h->alpha = alpha; h->era_m = era_m; h->deta = deta; h->W0 = W0; h->phi0 = phi0; h->seed = seed; h->beta = 0.0;
    h->stream = (cudaStream_t)cuda_stream;
    h->ws = (char*)workspace;
    h->phi[0] = h->ws + L.off_phi[0]; h->phi[1] = h->ws + L.off_phi[1];
    h->pd[0] = h->ws + L.off_pd[0]; h->pd[1] = h->ws + L.off_pd[1];
    h->partials = (DiagPartial*)(h->ws + L.off_partials);
    h->d_result = (DiagPartial*)(h->ws + L.off_result);
    h->d_ticket = (unsigned*)(h->ws + L.off_result + 64);         // in the record's 256-byte slot
    h->bits = (unsigned*)(h->ws + L.off_bits);
    h->d_results = (DiagPartial*)(h->ws + L.off_results);
    h->cur = 0; h->eta0 = 1.0; h->step = 0; h->inited = false;
    h->opt_step_kernel = PRS_KERNEL_AUTO; h->opt_arith = PRS_ARITH_FMA; h->opt_diag_kernel = PRS_KERNEL_AUTO;
    h->opt_chunk = 0; h->opt_tile_y = 4; h->opt_tb2_tile_y = 12;
    // measured, 16384^2, site-updates/s: FP32 1.29e12 (S = 4), 1.76e12 (6), 1.95e12 (8); FP64 6.8e11 (4), 9.5e11 (6), 8.9e11 (8)
    h->opt_tbs_steps = (dims == 3) ? 4 : (precision == PRS_F32 ? 8 : 6);
    h->opt_tbs_rows = 0;                          // auto (prs_launch_tbs.cuh)
    h->opt_tbs_loader = 0;
    h->opt_diag_chunk = 0;
    h->opt_cluster_ctas = 0;
    h->seen_valid = false; h->seen_links = 0; h->seen_step = 0; h->seen_cur = 0; h->seen_gen = 0;
    h->bits_valid = false; h->bits_step = 0; h->bits_cur = 0; h->bits_gen = 0; h->state_gen = 0;
    h->last_step_kernel = 0; h->last_diag_kernel = 0; h->launches = 0;
    memset(&h->main_launch, 0, sizeof(h->main_launch));
    h->h_result = nullptr;
    h->device = attr.device;                      // the device that owns the workspace: all launches go there
    DeviceGuard guard(h->device);
    if (guard.err != cudaSuccess) {
        cudaGetLastError();
        delete h;
        return PRS_ERR_CUDA;
    }
    if (cudaDeviceGetAttribute(&h->sm_count, cudaDevAttrMultiProcessorCount, h->device) != cudaSuccess) h->sm_count = 148;
    if (cudaMemsetAsync(h->d_ticket, 0, sizeof(unsigned), h->stream) != cudaSuccess) {     // the caller's workspace is uninitialised
        cudaGetLastError();
        delete h;
        return PRS_ERR_CUDA;
    }
    if (cudaHostAlloc((void**)&h->h_result, sizeof(DiagPartial), cudaHostAllocDefault) != cudaSuccess) {
        cudaGetLastError();
        delete h;
        return PRS_ERR_NOMEM;
    }
    *out = h;
    return PRS_OK;
}

int prs_create(prs_handle* out, int dims, int64_t N, int precision, double alpha, double era_m, double deta,
               double W0, double phi0, uint64_t seed, void* workspace, size_t workspace_bytes,
               void* cuda_stream) {
    if (!out) return PRS_ERR_INVALID_ARG;
    if (!args_ok(dims, N, precision)) return PRS_ERR_INVALID_ARG;
    return create_common(out, dims, N, sites_of(dims, N), precision, alpha, era_m, deta, W0, phi0, seed, workspace,
                         workspace_bytes, cuda_stream);
}

size_t prs_slab_workspace_bytes(int64_t N, int64_t nz, int precision) {
    if (!slab_args_ok(N, nz, 0, precision)) return 0;
    return layout_of_sites(slab_sites(N, nz), precision).total;
}

int prs_create_slab(prs_handle* out, int64_t N, int64_t z_begin, int64_t nz, int precision, double alpha, double era_m,
                    double deta, double W0, double phi0, uint64_t seed, void* workspace, size_t workspace_bytes,
                    void* cuda_stream) {
    if (!out) return PRS_ERR_INVALID_ARG;
    if (!slab_args_ok(N, nz, z_begin, precision)) return PRS_ERR_INVALID_ARG;
    const int rc = create_common(out, 3, N, slab_sites(N, nz), precision, alpha, era_m, deta, W0, phi0, seed, workspace,
                                 workspace_bytes, cuda_stream);
    if (rc != PRS_OK) return rc;
    prs_ctx* h = *out;
    h->slab = true; h->halo = SLAB_HALO; h->nz_own = nz; h->NZ = nz + 2 * SLAB_HALO; h->z_begin = z_begin;
    h->halo_valid = 0;
    return PRS_OK;
}

int prs_destroy(prs_handle h) {
    if (!h) return PRS_ERR_INVALID_ARG;
    DeviceGuard guard(h->device);
    if (h->h_result) cudaFreeHost(h->h_result);
    delete h;
    return PRS_OK;
}

int prs_init(prs_handle h, double eta0) {
    if (!h) return PRS_ERR_INVALID_ARG;
    PRS_ON_DEVICE(h);
    if (!(eta0 > 0.0) || !std::isfinite(eta0)) return fail(h, PRS_ERR_INVALID_ARG, "prs_init: eta0 must be > 0");
    const long long nquads = (long long)((h->S + 3) / 4);
    long long blocks = (nquads + 255) / 256;
    const long long cap = (long long)h->sm_count * 32;
    if (blocks > cap) blocks = cap;
    h->cur = 0;
    if (h->slab) {
        const long long NN = (long long)h->N * h->N, zg0 = (long long)h->z_begin - h->halo;
        if (h->precision == PRS_F32)
            init_slab_kernel<float><<<(unsigned)blocks, 256, 0, h->stream>>>((float*)h->phi[0], (float*)h->pd[0], NN, (long long)h->NZ, (long long)h->N, zg0, h->seed, h->phi0);
        else
            init_slab_kernel<double><<<(unsigned)blocks, 256, 0, h->stream>>>((double*)h->phi[0], (double*)h->pd[0], NN, (long long)h->NZ, (long long)h->N, zg0, h->seed, h->phi0);
        h->halo_valid = (int)h->halo;          // the halo planes were generated too: no exchange needed yet
    } else if (h->precision == PRS_F32)
        init_kernel<float><<<(unsigned)blocks, 256, 0, h->stream>>>((float*)h->phi[0], (float*)h->pd[0], (long long)h->S, h->seed, h->phi0);
    else
        init_kernel<double><<<(unsigned)blocks, 256, 0, h->stream>>>((double*)h->phi[0], (double*)h->pd[0], (long long)h->S, h->seed, h->phi0);
    PRS_CUDA(h, cudaGetLastError());
    h->launches += 1;
    h->eta0 = eta0; h->step = 0; h->inited = true;
    h->state_gen += 1;
    return PRS_OK;
}

static int step_impl(prs_handle h, int64_t nsteps);

int prs_step(prs_handle h, int64_t nsteps) {
    if (!h) return PRS_ERR_INVALID_ARG;
    PRS_ON_DEVICE(h);
    return step_impl(h, nsteps);
}

// the launches of prs_step; the handle's device is current
static int step_impl(prs_handle h, int64_t nsteps) {
    if (nsteps < 0) return fail(h, PRS_ERR_INVALID_ARG, "prs_step: nsteps must be >= 0");
    if (!h->inited) return fail(h, PRS_ERR_STATE, "prs_step: call prs_init or prs_copy_in first");
    if (nsteps > 0) h->main_launch.open = true;
    if (h->slab) {
        // Each step uses up one halo plane per side (the halo sites are advanced redundantly from the
        // planes beyond them).  nsteps = 4 or 3 is one pass of the multi-step kernel, which writes the
        // owned planes only (the halo is stale afterwards); 1 or 2 go through the single-step / two-step kernels
        // over all planes (PRS_KERNEL_GENERIC: generic single steps throughout).
        if (nsteps > h->halo_valid)
            return fail(h, PRS_ERR_STATE, "prs_step: a slab can advance at most as many steps as its halo is valid for; exchange the halo planes first (prs_slab_halo_regions / prs_slab_halo_filled)");
        const bool tbs_ok = h->opt_step_kernel != PRS_KERNEL_GENERIC && tbs_supported(h);
        if ((nsteps == SLAB_HALO || nsteps == 3) && tbs_ok) {
            const int rc = (h->precision == PRS_F32) ? step_many<float>(h, (int)nsteps) : step_many<double>(h, (int)nsteps);
            if (rc != PRS_OK) return rc;
            h->last_step_kernel = PRS_KERNEL_TBS;
            h->halo_valid = 0;                    // the multi-step kernel writes the owned planes only
        } else {
            // all NZ planes are advanced (the wrap in z feeds only the outermost halo planes, which lose
            // their validity anyway), so the halo stays good for halo_valid - nsteps more steps
            int64_t left = nsteps;
            if (tbs_ok && tb2_supported(h))
                for (; left >= 2; left -= 2) {
                    const int rc = (h->precision == PRS_F32) ? step_twice<float>(h) : step_twice<double>(h);
                    if (rc != PRS_OK) return rc;
                }
            const int single = tbs_ok ? PRS_KERNEL_TILED : PRS_KERNEL_GENERIC;
            for (; left > 0; --left) {
                const int rc = (h->precision == PRS_F32) ? step_once<float>(h, single) : step_once<double>(h, single);
                if (rc != PRS_OK) return rc;
            }
            if (nsteps > 0) h->last_step_kernel = tbs_ok ? (nsteps >= 2 ? PRS_KERNEL_TB2 : PRS_KERNEL_TILED) : PRS_KERNEL_GENERIC;
            h->halo_valid -= (int)nsteps;
        }
        return PRS_OK;
    }
    const int kernel = resolve_step_kernel(h);
    int64_t left = nsteps;
    if (kernel == PRS_KERNEL_CLUSTER) {
        while (left > 0) {
            const int n = (int)std::min<int64_t>(left, CLUSTER_MAX_STEPS);
            const ClusterDiag none = {0, 0, nullptr, 0.0, 0.0};
            const int rc = (h->precision == PRS_F32) ? step_cluster<float>(h, n, none) : step_cluster<double>(h, n, none);
            if (rc != PRS_OK) return rc;
            left -= n;
        }
    }
    if (kernel == PRS_KERNEL_TBS) {
        // S-step launches, then the remainder in as few launches as the instances allow (a launch costs a march whatever
        // its depth: measured at 4096^2 FP32, us per launch: 8 steps 89, 6: 71, 4: 58, 3: 61, two-step kernel 62, single
        // step 47; at 1024^3 FP32 4 steps 4.4 ms, two-step kernel 3.1, single 2.8): 3 -> one three-step launch (was 2 + 1),
        // 6 -> one six-step launch (was 4 + 2), 7 -> 4 + 3 (was 4 + 2 + 1); 2D FP32 only: a remainder of 2 after eight-step
        // launches trades the last 8 + 2 for 6 + 4 (150 -> 130 us at 4096^2; the 50-step cycle of BASELINE.json's 2D configs
        // ends that way).  What is left after this block is 0, 1 or 2 steps for the kernels below.
        const int S = h->opt_tbs_steps;
        int64_t mains = left / S;
        int rem = (int)(left % S);
        const bool trade = h->dims == 2 && h->precision == PRS_F32 && S == 8 && rem == 2 && mains >= 1;
        // ... and 2D FP64, whose pipeline is six deep: the last 6 + 2 become ONE eight-step launch (4096^2: 125 + 99 -> 184 us,
        // 16384^2: 1810 + 1505 -> 2769)
        const bool trade64 = h->dims == 2 && h->precision == PRS_F64 && S == 6 && rem == 2 && mains >= 1;
        // ... and 3D (four deep): the last 4 + 2 become 3 + 3 (1024^3 FP32, ms per launch: four steps 4.48, three 3.46, the
        // two-step kernel 3.38: 7.85 -> 6.91; the 50-step cycle of BASELINE.json's 3D configs ends that way)
        const bool trade3d = h->dims == 3 && S == 4 && rem == 2 && mains >= 1;
        if (trade || trade64 || trade3d) mains -= 1;
        for (int64_t i = 0; i < mains; ++i) {
            const int rc = (h->precision == PRS_F32) ? step_many<float>(h, S) : step_many<double>(h, S);
            if (rc != PRS_OK) return rc;
        }
        left -= mains * S;
        int parts[2] = {0, 0};
        if (trade) { parts[0] = 6; parts[1] = 4; }
        else if (trade64) parts[0] = 8;
        else if (trade3d) { parts[0] = 3; parts[1] = 3; }
        else if (rem == 7) { parts[0] = 4; parts[1] = 3; }
        else if (rem == 6 && h->dims == 2) parts[0] = 6;
        else if (rem >= 4) parts[0] = 4;                           // 4, 5 (-> 4 + 1), 6 in 3D never happens (S <= 4 there)
        else if (rem == 3) parts[0] = 3;
        for (int i = 0; i < 2 && parts[i] > 0; ++i) {
            const int rc = (h->precision == PRS_F32) ? step_many<float>(h, parts[i]) : step_many<double>(h, parts[i]);
            if (rc != PRS_OK) return rc;
            left -= parts[i];
        }
    }
    if ((kernel == PRS_KERNEL_TB2 || kernel == PRS_KERNEL_TBS) && tb2_supported(h)) {
        for (; left >= 2; left -= 2) {
            const int rc = (h->precision == PRS_F32) ? step_twice<float>(h) : step_twice<double>(h);
            if (rc != PRS_OK) return rc;
        }
    }
    const int single = (kernel == PRS_KERNEL_TB2 || kernel == PRS_KERNEL_TBS) ? PRS_KERNEL_TILED : kernel;   // odd remainder
    for (; left > 0; --left) {
        const int rc = (h->precision == PRS_F32) ? step_once<float>(h, single) : step_once<double>(h, single);
        if (rc != PRS_OK) return rc;
    }
    if (nsteps > 0) h->last_step_kernel = kernel;
    return PRS_OK;
}

int prs_diagnostics(prs_handle h, prs_diag* out) {
    if (!h) return PRS_ERR_INVALID_ARG;
    PRS_ON_DEVICE(h);
    if (!out) return fail(h, PRS_ERR_INVALID_ARG, "prs_diagnostics: out is NULL");
    if (!h->inited) return fail(h, PRS_ERR_STATE, "prs_diagnostics: call prs_init or prs_copy_in first");
    if (h->slab && h->halo_valid < 1)
        return fail(h, PRS_ERR_STATE, "prs_diagnostics: the slab's halo planes are stale; exchange them first");
    const int rc = (h->precision == PRS_F32) ? diag_launch<float>(h, h->d_result) : diag_launch<double>(h, h->d_result);
    if (rc != PRS_OK) return rc;
    PRS_CUDA(h, cudaMemcpyAsync(h->h_result, h->d_result, sizeof(DiagPartial), cudaMemcpyDeviceToHost, h->stream));
    PRS_CUDA(h, cudaStreamSynchronize(h->stream));
    prs_diag d;
    d.step = h->step;
    d.eta = h->eta0 + (double)h->step * h->deta;
    d.link_count = h->h_result->links;
    h->seen_valid = true; h->seen_links = d.link_count; h->seen_step = h->step; h->seen_cur = h->cur; h->seen_gen = h->state_gen;
    d.wall_sites = h->h_result->walls;
    d.sum_ratio = h->h_result->sum;
    // a slab reports its own partial sums; rho is its share of the global density (the shares add up)
    d.rho = (double)d.link_count / (h->slab ? (double)h->N * (double)h->N * (double)h->N : (double)h->S);
    d.gv2 = d.wall_sites ? d.sum_ratio / (2.0 * (double)d.wall_sites) : 0.0;
    *out = d;
    return PRS_OK;
}

static void fill_diag(const prs_ctx* h, const DiagPartial& r, int64_t step, prs_diag* d) {
    d->step = step;
    d->eta = h->eta0 + (double)step * h->deta;
    d->link_count = r.links;
    d->wall_sites = r.walls;
    d->sum_ratio = r.sum;
    d->rho = (double)r.links / (h->slab ? (double)h->N * (double)h->N * (double)h->N : (double)h->S);
    d->gv2 = r.walls ? r.sum / (2.0 * (double)r.walls) : 0.0;
}

int prs_run(prs_handle h, int64_t ncycles, int64_t steps_per_cycle, prs_diag* out) {
    if (!h) return PRS_ERR_INVALID_ARG;
    PRS_ON_DEVICE(h);
    if (ncycles < 0 || steps_per_cycle < 0) return fail(h, PRS_ERR_INVALID_ARG, "prs_run: ncycles and steps_per_cycle must be >= 0");
    if (ncycles > 0 && !out) return fail(h, PRS_ERR_INVALID_ARG, "prs_run: out is NULL");
    if (!h->inited) return fail(h, PRS_ERR_STATE, "prs_run: call prs_init or prs_copy_in first");
    if (h->slab) return fail(h, PRS_ERR_UNSUPPORTED, "prs_run: a slab needs its halo planes exchanged between passes; use prs_step / prs_diagnostics");
    std::vector<DiagPartial> host;
    std::vector<int64_t> steps;
    for (int64_t done = 0; done < ncycles;) {
        const int64_t batch = std::min<int64_t>(ncycles - done, RESULTS_CAP);
        host.resize((size_t)batch);
        steps.resize((size_t)batch);
        const bool run_on_cluster = resolve_step_kernel(h) == PRS_KERNEL_CLUSTER;
        if (run_on_cluster && steps_per_cycle > 0) {
            // small 2D boxes: the cluster-resident kernel runs the diagnostics passes inside its launches -- up to 64
            // steps and all their passes per launch, the state never leaving the chip in between
            const double pi = 3.14159265358979323846;
            const double V0 = (pi * pi * h->phi0 * h->phi0) / (2.0 * h->W0 * h->W0), I = 1.0 / (h->phi0 * h->phi0);
            h->main_launch.open = true;
            int64_t left = batch * steps_per_cycle, until = steps_per_cycle, rec = 0;
            const int64_t step0 = h->step;
            while (left > 0) {
                const int n = (int)std::min<int64_t>(left, CLUSTER_MAX_STEPS);
                const int64_t passes = (until <= n) ? 1 + (n - until) / steps_per_cycle : 0;
                const ClusterDiag dg = {passes ? (int)std::min<int64_t>(steps_per_cycle, 1 << 30) : 0, (int)std::min<int64_t>(until, 1 << 30),
                                        h->d_results + rec, V0, I};
                const int rc = (h->precision == PRS_F32) ? step_cluster<float>(h, n, dg) : step_cluster<double>(h, n, dg);
                if (rc != PRS_OK) return rc;
                // steps to the first pass of the next launch
                until = passes ? steps_per_cycle - (n - (until + (passes - 1) * steps_per_cycle)) : until - n;
                rec += passes;
                left -= n;
            }
            for (int64_t i = 0; i < batch; ++i) steps[(size_t)i] = step0 + (i + 1) * steps_per_cycle;
            h->last_step_kernel = PRS_KERNEL_CLUSTER;
            h->last_diag_kernel = PRS_KERNEL_CLUSTER;
        } else
        for (int64_t i = 0; i < batch; ++i) {                         // queued back to back: no sync, no transfer
            int rc = step_impl(h, steps_per_cycle);
            if (rc != PRS_OK) return rc;
            rc = (h->precision == PRS_F32) ? diag_launch<float>(h, h->d_results + i) : diag_launch<double>(h, h->d_results + i);
            if (rc != PRS_OK) return rc;
            steps[(size_t)i] = h->step;
        }
        PRS_CUDA(h, cudaMemcpyAsync(host.data(), h->d_results, sizeof(DiagPartial) * (size_t)batch, cudaMemcpyDeviceToHost, h->stream));
        PRS_CUDA(h, cudaStreamSynchronize(h->stream));
        for (int64_t i = 0; i < batch; ++i) fill_diag(h, host[(size_t)i], steps[(size_t)i], out + done + i);
        done += batch;
    }
    return PRS_OK;
}

int prs_weighted_area(prs_handle h, double* area, double* rho_weighted) {
    if (!h) return PRS_ERR_INVALID_ARG;
    PRS_ON_DEVICE(h);
    if (!area && !rho_weighted) return fail(h, PRS_ERR_INVALID_ARG, "prs_weighted_area: both outputs are NULL");
    if (!h->inited) return fail(h, PRS_ERR_STATE, "prs_weighted_area: call prs_init or prs_copy_in first");
    if (h->N > (1 << 30)) return fail(h, PRS_ERR_UNSUPPORTED, "prs_weighted_area: N too large");
    if (h->slab && h->halo_valid < 1)
        return fail(h, PRS_ERR_STATE, "prs_weighted_area: the slab's halo planes are stale; exchange them first");
    // x across the threads, y (3D) across blockIdx.y, the slowest axis marched in chunks of L sites,
    // L as short as the partials scratch allows (one partial per block).  A z slab measures its owned planes
    // (the transverse neighbours of their links lie at most one plane away: halo planes, valid for >= 1 more step).
    const int N = (int)h->N;
    const int NM = (h->dims == 3) ? (int)h->NZ : N;
    const int mlo = h->slab ? (int)h->halo : 0, mhi = h->slab ? (int)(h->halo + h->nz_own) : N, span = mhi - mlo;
    const unsigned gx = (unsigned)((N + 255) / 256);
    const long long per_chunk = (long long)gx * (h->dims == 3 ? N : 1);
    long long chunks = std::max<long long>(1, std::min<long long>(span, MAX_PARTIALS / per_chunk));
    int L = (int)((span + chunks - 1) / chunks);
    if (L < 8) L = std::min(8, span);
    const unsigned nch = (unsigned)((span + L - 1) / L);
    const dim3 grid = (h->dims == 3) ? dim3(gx, (unsigned)N, nch) : dim3(gx, nch, 1);
    const long long blocks = (long long)grid.x * grid.y * grid.z;
    // On the packed sign bits a crossing link costs ten scattered gathers, a non-crossing one nothing: it wins by 2-10x
    // on a formed network and loses on the white-noise start (1024^3: 22.8 against 16.6 ms), where more than one link
    // in four crosses.  If the last prs_diagnostics measured this very state, its link count decides.
    const bool dense = h->seen_valid && h->seen_step == h->step && h->seen_cur == h->cur && h->seen_gen == h->state_gen &&
                       (double)h->seen_links > 0.25 * (double)h->dims * (double)h->S;
    const bool on_bits = diag_bits_supported(h) && h->S >= ((size_t)1 << 22) && h->opt_diag_kernel != PRS_KERNEL_TILED &&
                         h->opt_diag_kernel != PRS_KERNEL_GENERIC && !dense;
    if (!on_bits && blocks > MAX_PARTIALS) return fail(h, PRS_ERR_UNSUPPORTED, "prs_weighted_area: lattice too large for the reduction scratch");
    const void* p = h->phi[h->cur];
    const DiagFinish fin = {h->partials, h->d_result, h->d_ticket};
    // from 2^22 sites up on lattices of whole 32-vector groups: on the packed sign bits (prs_kernels_bits.cuh), which
    // the preceding prs_diagnostics may have left behind
    if (on_bits) {
        const int rc = (h->precision == PRS_F32) ? ensure_bits<float>(h) : ensure_bits<double>(h);
        if (rc != PRS_OK) return rc;
        const int NG = N / (32 * vec_width(h->precision));
        const BitRows br = bit_rows(h);
        const long long lgroups = (br.m1 - br.m0) * NG;
        const unsigned bl = (unsigned)std::min<long long>((lgroups + BITS_THREADS - 1) / BITS_THREADS, std::min<long long>(MAX_PARTIALS, (long long)h->sm_count * 16));
        const int NZ = (int)h->NZ;
        if (h->precision == PRS_F32) {
            if (h->dims == 3) bit_area_kernel<float, 3><<<bl, BITS_THREADS, 0, h->stream>>>((const float*)p, h->bits, N, NZ, br.m0, br.m1, fin);
            else bit_area_kernel<float, 2><<<bl, BITS_THREADS, 0, h->stream>>>((const float*)p, h->bits, N, 1, br.m0, br.m1, fin);
        } else {
            if (h->dims == 3) bit_area_kernel<double, 3><<<bl, BITS_THREADS, 0, h->stream>>>((const double*)p, h->bits, N, NZ, br.m0, br.m1, fin);
            else bit_area_kernel<double, 2><<<bl, BITS_THREADS, 0, h->stream>>>((const double*)p, h->bits, N, 1, br.m0, br.m1, fin);
        }
    } else if (h->precision == PRS_F32) {
        if (h->dims == 3) weighted_area_kernel<float, 3><<<grid, 256, 0, h->stream>>>((const float*)p, N, NM, mlo, mhi, L, fin);
        else weighted_area_kernel<float, 2><<<grid, 256, 0, h->stream>>>((const float*)p, N, NM, mlo, mhi, L, fin);
    } else {
        if (h->dims == 3) weighted_area_kernel<double, 3><<<grid, 256, 0, h->stream>>>((const double*)p, N, NM, mlo, mhi, L, fin);
        else weighted_area_kernel<double, 2><<<grid, 256, 0, h->stream>>>((const double*)p, N, NM, mlo, mhi, L, fin);
    }
    PRS_CUDA(h, cudaGetLastError());
    h->launches += 1;
    PRS_CUDA(h, cudaMemcpyAsync(h->h_result, h->d_result, sizeof(DiagPartial), cudaMemcpyDeviceToHost, h->stream));
    PRS_CUDA(h, cudaStreamSynchronize(h->stream));
    if (area) *area = h->h_result->sum;
    // a slab reports its own partial sum; rho_weighted is its share of the lattice's density (the shares add up)
    if (rho_weighted) *rho_weighted = h->h_result->sum / (h->slab ? (double)h->N * (double)h->N * (double)h->N : (double)h->S);
    return PRS_OK;
}

int prs_diag_combine(const prs_diag* parts, int n, int dims, int64_t N, prs_diag* out) {
    if (!parts || !out || n < 1 || (dims != 2 && dims != 3) || N < 1) return PRS_ERR_INVALID_ARG;
    prs_diag d;
    d.step = parts[0].step;
    d.eta = parts[0].eta;
    d.link_count = 0;
    d.wall_sites = 0;
    d.sum_ratio = 0.0;
    for (int i = 0; i < n; ++i) {
        if (parts[i].step != d.step) return PRS_ERR_STATE;           // partial sums of different time levels
        d.link_count += parts[i].link_count;
        d.wall_sites += parts[i].wall_sites;
        d.sum_ratio += parts[i].sum_ratio;                           // in the order given: reproducible
    }
    const double sites = (dims == 3) ? (double)N * (double)N * (double)N : (double)N * (double)N;
    d.rho = (double)d.link_count / sites;                            // Eq. 7, Delta A = 1
    d.gv2 = d.wall_sites ? d.sum_ratio / (2.0 * (double)d.wall_sites) : 0.0;      // Eq. 8
    *out = d;
    return PRS_OK;
}

int prs_copy_out(prs_handle h, void* phi_dst, void* phidot_dst) {
    if (!h) return PRS_ERR_INVALID_ARG;
    PRS_ON_DEVICE(h);
    if (!h->inited) return fail(h, PRS_ERR_STATE, "prs_copy_out: no state yet");
    // a slab copies its owned planes (contiguous: z is the slowest axis)
    const size_t esz = (h->precision == PRS_F32 ? 4 : 8);
    const size_t bytes = (h->slab ? (size_t)h->N * h->N * h->nz_own : h->S) * esz;
    const size_t off = h->slab ? (size_t)h->N * h->N * h->halo * esz : 0;
    if (phi_dst) PRS_CUDA(h, cudaMemcpyAsync(phi_dst, (char*)h->phi[h->cur] + off, bytes, cudaMemcpyDefault, h->stream));
    if (phidot_dst) PRS_CUDA(h, cudaMemcpyAsync(phidot_dst, (char*)h->pd[h->cur] + off, bytes, cudaMemcpyDefault, h->stream));
    PRS_CUDA(h, cudaStreamSynchronize(h->stream));
    return PRS_OK;
}

int prs_copy_in(prs_handle h, const void* phi_src, const void* phidot_src, double eta0, int64_t step) {
    if (!h) return PRS_ERR_INVALID_ARG;
    PRS_ON_DEVICE(h);
    if (!phi_src || !phidot_src) return fail(h, PRS_ERR_INVALID_ARG, "prs_copy_in: both fields are required");
    if (!(eta0 > 0.0) || !std::isfinite(eta0) || step < 0)
        return fail(h, PRS_ERR_INVALID_ARG, "prs_copy_in: eta0 must be > 0 and step >= 0");
    const size_t esz = (h->precision == PRS_F32 ? 4 : 8);
    const size_t bytes = (h->slab ? (size_t)h->N * h->N * h->nz_own : h->S) * esz;
    const size_t off = h->slab ? (size_t)h->N * h->N * h->halo * esz : 0;
    PRS_CUDA(h, cudaMemcpyAsync((char*)h->phi[h->cur] + off, phi_src, bytes, cudaMemcpyDefault, h->stream));
    PRS_CUDA(h, cudaMemcpyAsync((char*)h->pd[h->cur] + off, phidot_src, bytes, cudaMemcpyDefault, h->stream));
    PRS_CUDA(h, cudaStreamSynchronize(h->stream));
    h->eta0 = eta0; h->step = step; h->inited = true;
    h->state_gen += 1;
    h->halo_valid = 0;                            // a slab's halo planes now belong to the old state
    return PRS_OK;
}

int prs_set_beta(prs_handle h, double beta) {
    if (!h) return PRS_ERR_INVALID_ARG;
    if (!std::isfinite(beta)) return fail(h, PRS_ERR_INVALID_ARG, "prs_set_beta: beta must be finite");
    h->beta = beta;
    return PRS_OK;
}

int prs_sync(prs_handle h) {
    if (!h) return PRS_ERR_INVALID_ARG;
    PRS_ON_DEVICE(h);
    PRS_CUDA(h, cudaStreamSynchronize(h->stream));
    return PRS_OK;
}

int prs_set_option(prs_handle h, int option, int64_t value) {
    if (!h) return PRS_ERR_INVALID_ARG;
    if (h->slab && option == PRS_OPT_STEP_KERNEL && value != PRS_KERNEL_AUTO && value != PRS_KERNEL_GENERIC && value != PRS_KERNEL_TBS)
        return fail(h, PRS_ERR_UNSUPPORTED, "a slab steps with the generic or the four-step kernel");
    if (h->slab && (option == PRS_OPT_DIAG_KERNEL || option == PRS_OPT_TBS_STEPS) && value != PRS_KERNEL_AUTO && !(option == PRS_OPT_TBS_STEPS && value == SLAB_HALO) &&
        !(option == PRS_OPT_DIAG_KERNEL && value == PRS_KERNEL_BITS))
        return fail(h, PRS_ERR_UNSUPPORTED, "not configurable on a slab");
    switch (option) {
        case PRS_OPT_STEP_KERNEL:
            if (value == PRS_KERNEL_AUTO || value == PRS_KERNEL_GENERIC) { h->opt_step_kernel = (int)value; return PRS_OK; }
            if (value == PRS_KERNEL_CLUSTER) {
                if (!cluster_supported(h)) return fail(h, PRS_ERR_UNSUPPORTED, "the cluster-resident kernel takes 2D lattices of 64, 128 or 256 sites per side");
                h->opt_step_kernel = (int)value;
                return PRS_OK;
            }
            if (value == PRS_KERNEL_TBS) {
                if (!tbs_supported(h)) return fail(h, PRS_ERR_UNSUPPORTED, "the multi-step kernel needs N a multiple of 16 bytes of T and at most 2^31 (3D) / fewer than 2^30 (2D) such vectors in the lattice");
                h->opt_step_kernel = (int)value;
                return PRS_OK;
            }
            if (value == PRS_KERNEL_TILED || value == PRS_KERNEL_TB2) {
                if (value == PRS_KERNEL_TB2 && !tb2_supported(h)) return fail(h, PRS_ERR_UNSUPPORTED, "the two-step kernel cannot take this lattice");
                if (!tiled_supported(h)) return fail(h, PRS_ERR_UNSUPPORTED, "tiled / two-step kernels need N to be a multiple of 16 bytes of T");
                h->opt_step_kernel = (int)value;
                return PRS_OK;
            }
            return fail(h, PRS_ERR_INVALID_ARG, "unknown step kernel");
        case PRS_OPT_ARITH:
            if (value != PRS_ARITH_LITERAL && value != PRS_ARITH_COEF && value != PRS_ARITH_FMA) return fail(h, PRS_ERR_INVALID_ARG, "unknown arithmetic");
            h->opt_arith = (int)value;
            return PRS_OK;
        case PRS_OPT_DIAG_KERNEL:
            if (value == PRS_KERNEL_AUTO || value == PRS_KERNEL_GENERIC) { h->opt_diag_kernel = (int)value; return PRS_OK; }
            if (value == PRS_KERNEL_BITS) {
                if (!diag_bits_supported(h)) return fail(h, PRS_ERR_UNSUPPORTED, "the sign-bit diagnostics pass needs N to be a multiple of 32 16-byte vectors");
                h->opt_diag_kernel = (int)value;
                return PRS_OK;
            }
            if (value == PRS_KERNEL_TILED) {
                if (!diag_tiled_supported(h)) return fail(h, PRS_ERR_UNSUPPORTED, "tiled diagnostics kernel cannot take this lattice");
                h->opt_diag_kernel = (int)value;
                return PRS_OK;
            }
            return fail(h, PRS_ERR_INVALID_ARG, "unknown diagnostics kernel");
        case PRS_OPT_CHUNK:
            if (value < 0 || value > (1 << 20)) return fail(h, PRS_ERR_INVALID_ARG, "chunk must be >= 0");
            h->opt_chunk = (int)value;
            return PRS_OK;
        case PRS_OPT_TILE_Y:
            if (value != 4 && value != 8 && value != 16) return fail(h, PRS_ERR_INVALID_ARG, "tile_y must be 4, 8 or 16");
            h->opt_tile_y = (int)value;
            return PRS_OK;
        case PRS_OPT_TBS_STEPS:
            if (value != 3 && value != 4 && !(h->dims == 2 && (value == 6 || value == 8)))
                return fail(h, PRS_ERR_INVALID_ARG, "tbs_steps must be 3 or 4 (2D: also 6 or 8)");
            h->opt_tbs_steps = (int)value;
            return PRS_OK;
        case PRS_OPT_TBS_ROWS:
            if (value != 0 && value != 1 && !(value == 2 && h->dims == 3))
                return fail(h, PRS_ERR_INVALID_ARG, "tbs_rows must be 0 (auto), 1 or, in 3D, 2");
            h->opt_tbs_rows = (int)value;
            return PRS_OK;
        case PRS_OPT_CLUSTER_CTAS:
            if (value != 0 && value != 8 && value != 16) return fail(h, PRS_ERR_INVALID_ARG, "cluster_ctas must be 0 (auto), 8 or 16");
            h->opt_cluster_ctas = (int)value;
            return PRS_OK;
        case PRS_OPT_DIAG_CHUNK:
            if (value < 0 || value > (1 << 20)) return fail(h, PRS_ERR_INVALID_ARG, "diag_chunk must be >= 0");
            h->opt_diag_chunk = (int)value;
            return PRS_OK;
        case PRS_OPT_TBS_LOADER:
            if (value != 0 && value != 1 && value != 2) return fail(h, PRS_ERR_INVALID_ARG, "tbs_loader must be 0 (auto), 1 (cp.async) or 2 (bulk)");
            h->opt_tbs_loader = (int)value;
            return PRS_OK;
        case PRS_OPT_TB2_TILE_Y:
            if (value != 4 && value != 8 && value != 12 && value != 28)
                return fail(h, PRS_ERR_INVALID_ARG, "tb2_tile_y must be 4, 8, 12 or 28");
            h->opt_tb2_tile_y = (int)value;
            return PRS_OK;
        default:
            return fail(h, PRS_ERR_INVALID_ARG, "unknown option");
    }
}

int prs_get_info(prs_handle h, int info, int64_t* value) {
    if (!h || !value) return PRS_ERR_INVALID_ARG;
    switch (info) {
        case PRS_INFO_KERNEL_LAUNCHES: *value = h->launches; return PRS_OK;
        case PRS_INFO_STEP_KERNEL: *value = h->last_step_kernel; return PRS_OK;
        case PRS_INFO_STEP: *value = h->step; return PRS_OK;
        case PRS_INFO_DIAG_KERNEL: *value = h->last_diag_kernel; return PRS_OK;
        case PRS_INFO_HALO_VALID: *value = h->slab ? h->halo_valid : 0; return PRS_OK;
        case PRS_INFO_HALO_PLANES: *value = h->slab ? h->halo : 0; return PRS_OK;
        case PRS_INFO_DEVICE: *value = h->device; return PRS_OK;
        default: return fail(h, PRS_ERR_INVALID_ARG, "unknown info key");
    }
}

int prs_step_launch_info(prs_handle h, char* name, size_t name_bytes, int64_t grid[3], int64_t block[3],
                         int64_t* smem_bytes, int64_t* steps_per_launch, int64_t* launches) {
    if (!h) return PRS_ERR_INVALID_ARG;
    const auto& m = h->main_launch;
    if (m.count == 0 || m.open) return fail(h, PRS_ERR_STATE, "prs_step_launch_info: no step kernel launched yet");
    if (name && name_bytes) snprintf(name, name_bytes, "%s", m.name);
    for (int i = 0; i < 3; ++i) {
        if (grid) grid[i] = m.grid[i];
        if (block) block[i] = m.block[i];
    }
    if (smem_bytes) *smem_bytes = (int64_t)m.smem;
    if (steps_per_launch) *steps_per_launch = m.steps;
    if (launches) *launches = m.count;
    return PRS_OK;
}

int prs_device_pointers(prs_handle h, void** phi, void** phidot) {
    if (!h) return PRS_ERR_INVALID_ARG;
    if (!h->inited) return fail(h, PRS_ERR_STATE, "prs_device_pointers: no state yet");
    if (phi) *phi = h->phi[h->cur];
    if (phidot) *phidot = h->pd[h->cur];
    return PRS_OK;
}

int prs_slab_halo_regions(prs_handle h, void* send[4], void* recv[4], size_t* bytes) {
    if (!h || !send || !recv || !bytes) return PRS_ERR_INVALID_ARG;
    if (!h->slab) return fail(h, PRS_ERR_STATE, "prs_slab_halo_regions: not a slab");
    if (!h->inited) return fail(h, PRS_ERR_STATE, "prs_slab_halo_regions: no state yet");
    const size_t plane = (size_t)h->N * h->N * (h->precision == PRS_F32 ? 4 : 8);
    const size_t H = (size_t)h->halo, nz = (size_t)h->nz_own;
    char* const f[2] = {(char*)h->phi[h->cur], (char*)h->pd[h->cur]};
    for (int i = 0; i < 2; ++i) {
        send[2 * i + 0] = f[i] + H * plane;              // lowest owned planes  -> the z-1 neighbour's upper halo
        send[2 * i + 1] = f[i] + nz * plane;             // highest owned planes -> the z+1 neighbour's lower halo
        recv[2 * i + 0] = f[i];                          // lower halo <- the z-1 neighbour's highest owned planes
        recv[2 * i + 1] = f[i] + (H + nz) * plane;       // upper halo <- the z+1 neighbour's lowest owned planes
    }
    *bytes = H * plane;
    return PRS_OK;
}

int prs_slab_halo_filled(prs_handle h) {
    if (!h) return PRS_ERR_INVALID_ARG;
    if (!h->slab) return fail(h, PRS_ERR_STATE, "prs_slab_halo_filled: not a slab");
    if (!h->inited) return fail(h, PRS_ERR_STATE, "prs_slab_halo_filled: no state yet");
    h->halo_valid = (int)h->halo;
    h->state_gen += 1;                            // the halo planes' signs changed
    return PRS_OK;
}

const char* prs_last_error(prs_handle h) {
    if (!h) return "null handle";
    return h->err.c_str();
}

}  // extern "C"
