// prs_launch_tb2.cuh -- grid sizing and launch of the two-step kernels (prs_kernels_tb2.cuh).
// Included only by the translation unit that instantiates them (prs_instances.cu).
#pragma once

#include <algorithm>

#include "prs_host.cuh"
#include "prs_kernels_tb2.cuh"

namespace prs {

template <typename T, int ARITH, int TY>
cudaError_t launch_tb2_3d_ty(prs_ctx* h, const T* p, const T* v, T* pn, T* vn, const StepCoef<T>& k1,
                             const StepCoef<T>& k2) {
    constexpr int W = Pk<T>::W;
    const int N = (int)h->N, NQ = N / W;
    const size_t smem = tb2_smem_bytes<T, TY>();
    static std::atomic<unsigned long long> configured{0};      // per instantiation: devices already set up
    {
        const cudaError_t e = ensure_dynamic_smem(step3d_tb2_kernel<T, ARITH, TY>, smem, h->device, configured);
        if (e != cudaSuccess) return e;
    }
    const unsigned gx = (unsigned)((NQ + TB2_XOUT - 1) / TB2_XOUT), gy = (unsigned)((N + TY - 1) / TY);
    const int NZ = (int)h->NZ;                 // = N unless the handle is a z slab: then all its planes are advanced
    int ZC = h->opt_chunk > 0 ? (int)std::min<int64_t>(h->opt_chunk, NZ) : (int)std::min<int64_t>(64, NZ);
    // small grids: shorter chunks (down to 8 planes) until there are about two CTAs per SM -- the march is serial
    if (h->opt_chunk <= 0)
        while (ZC > 8 && (long long)gx * gy * ((NZ + ZC - 1) / ZC) < 2LL * std::max(1, h->sm_count)) ZC /= 2;
    const dim3 grid(gx, gy, (unsigned)((NZ + ZC - 1) / ZC));
    const dim3 block(32, TY + 4, 1);
    step3d_tb2_kernel<T, ARITH, TY><<<grid, block, smem, h->stream>>>(p, v, pn, vn, N, NZ, ZC, k1, k2);
    char name[96];
    snprintf(name, sizeof(name), "step3d_tb2_kernel<%s,%d,%d>", type_name<T>(), ARITH, TY);
    note_launch(h, name, grid, block, smem, 2);
    return cudaGetLastError();
}

template <typename T, int ARITH>
cudaError_t launch_tb2_3d(prs_ctx* h, const T* p, const T* v, T* pn, T* vn, const StepCoef<T>& k1,
                          const StepCoef<T>& k2) {
    switch (h->opt_tb2_tile_y) {
        case 4: return launch_tb2_3d_ty<T, ARITH, 4>(h, p, v, pn, vn, k1, k2);
        case 8: return launch_tb2_3d_ty<T, ARITH, 8>(h, p, v, pn, vn, k1, k2);
        case 28: return launch_tb2_3d_ty<T, ARITH, 28>(h, p, v, pn, vn, k1, k2);
        default: return launch_tb2_3d_ty<T, ARITH, 12>(h, p, v, pn, vn, k1, k2);
    }
}

template <typename T, int ARITH>
cudaError_t launch_tb2_2d(prs_ctx* h, const T* p, const T* v, T* pn, T* vn, const StepCoef<T>& k1,
                          const StepCoef<T>& k2) {
    constexpr int W = Pk<T>::W;
    const int N = (int)h->N, NQ = N / W;
    const int BX = 128, warps = BX / 32;
    const unsigned nwarps = (unsigned)((NQ + TB2_XOUT - 1) / TB2_XOUT);
    const unsigned gx = (nwarps + warps - 1) / warps;
    // rows per march: the rule of launch_tbs_2d (N/64 between 8 and 128).  A fixed 64 left a 256^2 lattice with a grid
    // of 4 CTAs marching 66 rows each: 30 us for the two-step remainder of a 10-step cycle whose 8-step launch takes 8.
    int YC = h->opt_chunk > 0 ? (int)std::min<int64_t>(h->opt_chunk, N) : std::min<int>(N, std::max(8, std::min(128, N / 64)));
    const dim3 grid(gx, (unsigned)((N + YC - 1) / YC), 1);
    step2d_tb2_kernel<T, ARITH><<<grid, BX, 0, h->stream>>>(p, v, pn, vn, N, YC, k1, k2);
    char name[96];
    snprintf(name, sizeof(name), "step2d_tb2_kernel<%s,%d>", type_name<T>(), ARITH);
    note_launch(h, name, grid, dim3(BX, 1, 1), 0, 2);
    return cudaGetLastError();
}

}  // namespace prs
