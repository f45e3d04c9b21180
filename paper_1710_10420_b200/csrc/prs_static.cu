// prs_static.cu -- prs_diagnostics_static: the wall diagnostics (Eqs. 7-8, :57-66) for callers that must not
// allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  No handle, no
// workspace: the caller passes phi, phidot (inputs) and a 24-byte device record (output); the one piece of scratch the
// pass needs -- one partial per block and the ticket counter of the last-block reduction -- lives in a file-scope
// static __device__ array of fixed size, which every GPU that loads the library holds until the process exits.
//
// This file calls no cudaMalloc, cudaFree, cudaHostAlloc or any allocating library routine.
//
// The array's NAME is, in host code, a host-side stand-in, not a device address: a kernel given it would fault (or, where
// the GPU can reach host memory, silently use the wrong memory).  So the address is taken once per device, with that
// device current, by cudaGetSymbolAddress (scratch_of below), and that pointer is what the kernel gets.
//
// Sharing: every call on a device uses the same array, which keeps the last call's contents.  The ticket counter is
// cleared on the caller's stream before each launch; the partials are all written before they are read.  Calls that
// OVERLAP on one GPU (different streams, or threads) race on the array: serialise them.
#include "prs_host.cuh"

#include <atomic>
#include <cstdio>
#include <mutex>

#include "prs_kernels_generic.cuh"   // block_reduce, DiagFinish / finish_partials, wall_ratio (prs_arith.cuh)

using namespace prs;

namespace {

constexpr int STATIC_THREADS = 256;
constexpr int STATIC_SITES_PER_THREAD = 16;
constexpr long long STATIC_SITES_PER_BLOCK = (long long)STATIC_THREADS * STATIC_SITES_PER_THREAD;   // 4096
constexpr int STATIC_MAX_BLOCKS = 32768;                                     // one DiagPartial (24 bytes) each
constexpr long long STATIC_MAX_SITES = STATIC_SITES_PER_BLOCK * STATIC_MAX_BLOCKS;                    // 2^27
constexpr size_t STATIC_HEADER_BYTES = 256;                                  // the ticket counter, alone in its line
constexpr size_t STATIC_SCRATCH_BYTES = STATIC_HEADER_BYTES + sizeof(DiagPartial) * (size_t)STATIC_MAX_BLOCKS;   // 786 688

static_assert(sizeof(prs_diag_sums) == sizeof(DiagPartial) && sizeof(DiagPartial) == 24, "the output record is a DiagPartial");

// THE scratch: 768.25 KiB per GPU that loads the library, held until exit.  [0, 256): ticket; then the partials.
static __device__ __align__(256) unsigned char prs_static_scratch[STATIC_SCRATCH_BYTES];

// Device address of the scratch on `device` (which must be current): taken once per device, then cached.
constexpr int MAX_DEVICES = 64;
std::mutex scratch_mutex;
void* scratch_ptr[MAX_DEVICES] = {};

cudaError_t scratch_of(int device, unsigned char** out) {
    if (device < 0 || device >= MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(scratch_mutex);
    if (!scratch_ptr[device]) {
        void* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, prs_static_scratch);      // this device's copy of the array
        if (e != cudaSuccess) return e;
        scratch_ptr[device] = p;
    }
    *out = (unsigned char*)scratch_ptr[device];
    return cudaSuccess;
}

// One pass of Eqs. 7-8 over the lattice: block b takes sites [4096 b, 4096 (b+1)), thread t of it the sites
// 4096 b + t + 256 k (coalesced).  Each site owns its DIMS forward links (Eq. 7) and is a wall site if any of its
// 2 DIMS links crosses (Eq. 8's N); sign = IEEE sign bit; the ratio phidot^2 / V in double.  The same per-site
// operations as diag_generic_kernel; the block's partial goes to the scratch and the last block to finish adds all
// partials in index order into *fin.out (finish_partials).
template <typename T, int DIMS>
__global__ void __launch_bounds__(STATIC_THREADS)
diag_static_kernel(const T* __restrict__ phi, const T* __restrict__ phidot, long long N, long long S, double V0, double I,
                   DiagFinish fin) {
    using A = Ar<T>;
    DiagPartial acc = {0ull, 0ull, 0.0};
    const long long s0 = (long long)blockIdx.x * STATIC_SITES_PER_BLOCK + threadIdx.x;
#pragma unroll 4
    for (int k = 0; k < STATIC_SITES_PER_THREAD; ++k) {
        const long long s = s0 + (long long)k * STATIC_THREADS;
        if (s >= S) break;
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
            zp = A::neg(phi[pil + (z == N - 1 ? 0 : z + 1) * NN]) != me;
            zm = A::neg(phi[pil + (z == 0 ? N - 1 : z - 1) * NN]) != me;
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

int say(char* err, size_t err_bytes, int code, const char* fmt, long long a = 0, long long b = 0) {
    if (err && err_bytes) snprintf(err, err_bytes, fmt, a, b);
    return code;
}

}  // namespace

extern "C" {

size_t prs_diagnostics_static_scratch_bytes(void) { return STATIC_SCRATCH_BYTES; }
int64_t prs_diagnostics_static_max_sites(void) { return (int64_t)STATIC_MAX_SITES; }

int prs_diagnostics_static(int dims, int64_t N, int precision, double W0, double phi0, const void* phi, const void* phidot,
                           prs_diag_sums* sums_device, void* cuda_stream, char* err, size_t err_bytes) {
    if (err && err_bytes) err[0] = 0;
    if ((dims != 2 && dims != 3) || N < 1 || (precision != PRS_F32 && precision != PRS_F64) || !(W0 > 0.0) || !(phi0 > 0.0))
        return say(err, err_bytes, PRS_ERR_INVALID_ARG, "prs_diagnostics_static: dims in {2,3}, N >= 1, precision PRS_F32/PRS_F64, W0 > 0, phi0 > 0");
    if (!phi || !phidot || !sums_device)
        return say(err, err_bytes, PRS_ERR_INVALID_ARG, "prs_diagnostics_static: phi, phidot and sums_device are required");
    // sizes beyond the static scratch are refused, never truncated
    const long double sites_ld = (dims == 3) ? (long double)N * N * N : (long double)N * N;
    if (sites_ld > (long double)STATIC_MAX_SITES)
        return say(err, err_bytes, PRS_ERR_UNSUPPORTED,
                   "prs_diagnostics_static: N = %lld gives more sites than the static scratch's maximum of %lld (2^27: 512^3, "
                   "11585^2); use prs_diagnostics on a handle for larger lattices", (long long)N, STATIC_MAX_SITES);
    const long long S = (dims == 3) ? (long long)N * N * N : (long long)N * N;
    cudaPointerAttributes attr;
    if (cudaPointerGetAttributes(&attr, phi) != cudaSuccess || attr.type != cudaMemoryTypeDevice) {
        cudaGetLastError();
        return say(err, err_bytes, PRS_ERR_INVALID_ARG, "prs_diagnostics_static: phi is not a device pointer");
    }
    DeviceGuard guard(attr.device);                               // the fields' device is current from here on
    if (guard.err != cudaSuccess) return say(err, err_bytes, PRS_ERR_CUDA, "prs_diagnostics_static: cudaSetDevice failed");
    unsigned char* scratch = nullptr;
    const cudaError_t es = scratch_of(attr.device, &scratch);     // cudaGetSymbolAddress, once per device
    if (es != cudaSuccess) {
        if (err && err_bytes) snprintf(err, err_bytes, "prs_diagnostics_static: cudaGetSymbolAddress: %s", cudaGetErrorName(es));
        return PRS_ERR_CUDA;
    }
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    const unsigned blocks = (unsigned)((S + STATIC_SITES_PER_BLOCK - 1) / STATIC_SITES_PER_BLOCK);
    // the array keeps the last call's contents: the ticket must start at zero (the partials are written before read)
    cudaError_t e = cudaMemsetAsync(scratch, 0, STATIC_HEADER_BYTES, stream);
    if (e == cudaSuccess) {
        const double pi = 3.14159265358979323846;
        const double V0 = (pi * pi * phi0 * phi0) / (2.0 * W0 * W0), I = 1.0 / (phi0 * phi0);
        const DiagFinish fin = {reinterpret_cast<DiagPartial*>(scratch + STATIC_HEADER_BYTES),
                                reinterpret_cast<DiagPartial*>(sums_device), reinterpret_cast<unsigned*>(scratch)};
        if (precision == PRS_F32) {
            if (dims == 3) diag_static_kernel<float, 3><<<blocks, STATIC_THREADS, 0, stream>>>((const float*)phi, (const float*)phidot, N, S, V0, I, fin);
            else diag_static_kernel<float, 2><<<blocks, STATIC_THREADS, 0, stream>>>((const float*)phi, (const float*)phidot, N, S, V0, I, fin);
        } else {
            if (dims == 3) diag_static_kernel<double, 3><<<blocks, STATIC_THREADS, 0, stream>>>((const double*)phi, (const double*)phidot, N, S, V0, I, fin);
            else diag_static_kernel<double, 2><<<blocks, STATIC_THREADS, 0, stream>>>((const double*)phi, (const double*)phidot, N, S, V0, I, fin);
        }
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) {
        if (err && err_bytes) snprintf(err, err_bytes, "prs_diagnostics_static: %s (%s)", cudaGetErrorName(e), cudaGetErrorString(e));
        return PRS_ERR_CUDA;
    }
    return PRS_OK;
}

}  // extern "C"
