// prs_host.cuh -- what the translation units of libprs share on the host side: the context behind a
// prs_handle, the per-step scalars, and the declarations of the launchers whose kernels are compiled
// in translation units of their own (prs_instances.cu, one compiler run per precision and kernel
// family, so that the library builds in parallel).  prs_api.cu sees only these declarations.
#pragma once

#include "../../include/prs.h"

#include <atomic>
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <string>

#include <cuda_runtime.h>

#include "prs_arith.cuh"

struct prs_ctx {
    int dims, precision;
    int64_t N;
    size_t S;
    double alpha, era_m, deta, W0, phi0, beta;
    uint64_t seed;
    cudaStream_t stream;
    char* ws;
    void* phi[2];
    void* pd[2];
    int cur;                                  // index of the arrays holding phi^n, phidot^{n-1/2}
    prs::DiagPartial* partials;
    prs::DiagPartial* d_result;
    bool seen_valid;                          // link count of the last prs_diagnostics and the state it belongs to
    uint64_t seen_links, seen_gen;
    int64_t seen_step;
    int seen_cur;
    bool bits_valid;                          // the bit array holds the signs of the state (bits_step, bits_cur, bits_gen)
    int64_t bits_step;
    int bits_cur;
    uint64_t bits_gen, state_gen;             // state_gen: advanced by prs_init, prs_copy_in, prs_slab_halo_filled
    unsigned* d_ticket;                       // ticket counter of the diagnostics kernels' last-block reduction
    prs::DiagPartial* d_results;              // ring of reduced records for prs_run (RESULTS_CAP entries)
    unsigned* bits;                           // one sign bit per site: scratch of the sign-bit diagnostics pass
    prs::DiagPartial* h_result;               // pinned host, 24 bytes
    double eta0;
    int64_t step;
    bool inited;
    int opt_step_kernel, opt_arith, opt_diag_kernel, opt_chunk, opt_tile_y, opt_tb2_tile_y, opt_tbs_steps, opt_tbs_rows, opt_tbs_loader, opt_diag_chunk, opt_cluster_ctas;
    int last_step_kernel, last_diag_kernel;
    int64_t launches;
    int sm_count;
    int device;                               // ordinal of the device that owns the workspace; every exported call
                                              // makes it current for its duration (DeviceGuard)
    // z slab of a sharded 3D lattice (prs_create_slab): the arrays hold NZ = nz_own + 2*halo planes of
    // N x N sites, local plane l = global plane (z_begin - halo + l) mod N; S counts the local sites.
    // halo_valid = how many more steps the halo planes can feed before they must be exchanged again.
    // the first kernel launched by the most recent prs_step call (its main kernel: the schedule goes from the
    // deepest pipeline to single steps), as prs_step_launch_info reports it
    struct {
        char name[96];                        // e.g. "step3d_tbs_kernel<float,2,4,16,1>"
        unsigned grid[3], block[3];
        size_t smem;
        int steps;                            // PRS steps one launch advances
        int count;                            // launches of it in that prs_step call
        bool open;                            // no launch recorded yet in the current prs_step call
    } main_launch;
    bool slab;
    int64_t NZ, nz_own, halo, z_begin;
    int halo_valid;
    std::string err;
};

namespace prs {

// Makes the handle's device current for the lifetime of the guard and restores the caller's device afterwards,
// so that one process can drive handles on several devices (SlabGroup) whatever device is current.
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    cudaError_t err = cudaSuccess;
    explicit DeviceGuard(int device) {
        err = cudaGetDevice(&prev);
        if (err == cudaSuccess && prev != device) {
            err = cudaSetDevice(device);
            switched = (err == cudaSuccess);
        }
    }
    ~DeviceGuard() {
        if (switched) cudaSetDevice(prev);
    }
    DeviceGuard(const DeviceGuard&) = delete;
    DeviceGuard& operator=(const DeviceGuard&) = delete;
};

template <typename T> inline const char* type_name();
template <> inline const char* type_name<float>() { return "float"; }
template <> inline const char* type_name<double>() { return "double"; }

// Book-keeping for prs_step_launch_info: `name` is the kernel with its template arguments, written the way a
// profiler's demangled name reads once "(int)", "(bool)" and blanks are stripped.
inline void note_launch(prs_ctx* h, const char* name, dim3 grid, dim3 block, size_t smem, int steps) {
    auto& m = h->main_launch;
    if (m.open) {
        snprintf(m.name, sizeof(m.name), "%s", name);
        m.grid[0] = grid.x; m.grid[1] = grid.y; m.grid[2] = grid.z;
        m.block[0] = block.x; m.block[1] = block.y; m.block[2] = block.z;
        m.smem = smem; m.steps = steps; m.count = 1; m.open = false;
    } else if (strncmp(m.name, name, sizeof(m.name)) == 0 && m.grid[0] == grid.x && m.grid[1] == grid.y && m.grid[2] == grid.z) {
        m.count += 1;
    }
}

// cudaFuncAttributeMaxDynamicSharedMemorySize is a per-device attribute of a kernel: it is set once per
// (kernel instantiation, device).  `done` is the instantiation's own bit mask of devices already configured
// (devices >= 64 are configured on every launch); setting it twice from two threads is harmless.
template <typename F>
inline cudaError_t ensure_dynamic_smem(F* kernel, size_t bytes, int device, std::atomic<unsigned long long>& done) {
    const unsigned long long bit = (device >= 0 && device < 64) ? (1ull << device) : 0ull;
    if (bit && (done.load(std::memory_order_acquire) & bit)) return cudaSuccess;
    const cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    if (e == cudaSuccess && bit) done.fetch_or(bit, std::memory_order_release);
    return e;
}

// Per-step scalars, Eq. 6 (:55) and the constants of Eq. 1 (:30); all in double, rounded to
// the field type once.  eta_n = eta0 + n*deta is formed from n each time, never accumulated.
template <typename T>
StepCoef<T> coef_at(const prs_ctx* h, int64_t n) {
    const double pi = 3.14159265358979323846;
    const double V0 = (pi * pi * h->phi0 * h->phi0) / (2.0 * h->W0 * h->W0);
    double K = 4.0 * V0 / (h->phi0 * h->phi0);
    const double I = 1.0 / (h->phi0 * h->phi0);
    const double eta = h->eta0 + (double)n * h->deta;
    // Eq. 2 (:34) with beta != 0: dV/dphi times a^beta, a = (eta/eta0)^m (R16)
    if (h->beta != 0.0 && h->era_m != 0.0) K = K * std::pow(eta / h->eta0, h->era_m * h->beta);
    const double delta = ((0.5 * h->alpha) * (h->deta / eta)) * h->era_m;
    StepCoef<T> k;
    k.K = (T)K;
    k.I = (T)I;
    k.deta = (T)h->deta;
    const T dT = (T)delta;
    k.omd = T(1) - dT;
    k.opd = T(1) + dT;
    k.A = (T)((1.0 - delta) / (1.0 + delta));
    k.B = (T)(h->deta / (1.0 + delta));
    return k;
}

// Launchers defined in prs_launch_tb2.cuh / prs_launch_tbs.cuh and instantiated in prs_instances.cu.
// p, v: phi^n and phidot^{n-1/2}; pn, vn: where the advanced fields go; all device pointers in the
// context's workspace.  Each returns the launch error; the caller does the book-keeping.

// two steps per pass (n -> n+2) with the scalars of steps n and n+1
template <typename T, int ARITH>
cudaError_t launch_tb2_3d(prs_ctx* h, const T* p, const T* v, T* pn, T* vn, const StepCoef<T>& k1, const StepCoef<T>& k2);
template <typename T, int ARITH>
cudaError_t launch_tb2_2d(prs_ctx* h, const T* p, const T* v, T* pn, T* vn, const StepCoef<T>& k1, const StepCoef<T>& k2);

// S steps per pass (n -> n+S); the scalars are formed inside from h->step
template <typename T, int ARITH, int S>
cudaError_t launch_tbs_3d(prs_ctx* h, const T* p, const T* v, T* pn, T* vn);
template <typename T, int ARITH, int S>
cudaError_t launch_tbs_2d(prs_ctx* h, const T* p, const T* v, T* pn, T* vn);

}  // namespace prs
