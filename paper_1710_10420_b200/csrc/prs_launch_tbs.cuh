// prs_launch_tbs.cuh -- grid sizing and launch of the S-step kernels (prs_kernels_tbs.cuh).
// Included only by the translation unit that instantiates them (prs_instances.cu).
#pragma once

#include <algorithm>

#include "prs_host.cuh"
#include "prs_kernels_tbs.cuh"
#include "prs_kernels_tbr.cuh"

namespace prs {

template <typename T, int ARITH, int S>
cudaError_t launch_tbr_3d(prs_ctx* h, const T* p, const T* v, T* pn, T* vn);

// Planes per z chunk of the 3D multi-step kernels (one CTA per SM; `tiles` CTAs per chunk layer, nzo
// planes to write).  Large grids: 128 planes (measured 1024^3 FP32, S = 4: 64 planes 1.25 ms/step, 128 planes
// 1.21, 256 planes 1.24; each chunk re-reads 2S halo planes).  Grids of a few waves: the chunk count that
// minimises waves x (planes marched per CTA), because with one CTA per SM a last, nearly empty wave costs
// as much as a full one -- measured FP32: 256^3 36.6 -> 26.7 us per step (3 chunks of 86 planes = 144 CTAs,
// one wave, instead of 8 chunks = 384 CTAs, three waves), 512^3 184 -> 173 (8 chunks of 64 instead of 4 of
// 128: 9 waves of 74 planes instead of 5 of 138).
inline int tbs_pick_zc(const prs_ctx* h, long long tiles, int nzo, int S) {
    if (h->opt_chunk > 0) return (int)std::min<int64_t>(h->opt_chunk, nzo);
    const long long sms = std::max(1, h->sm_count);
    const int dflt = std::min(nzo, 128);
    const long long layers = (nzo + dflt - 1) / dflt;
    if ((tiles * layers + sms - 1) / sms > 12) return dflt;
    int best = dflt;
    long long best_cost = -1;
    for (int c = 1; c <= std::max(1, nzo / 16); ++c) {
        const int zc = (nzo + c - 1) / c;
        const long long cnt = (nzo + zc - 1) / zc;
        const long long waves = (tiles * cnt + sms - 1) / sms;
        const long long cost = waves * (zc + 2 * S + 2);
        if (best_cost < 0 || cost < best_cost) { best_cost = cost; best = zc; }
    }
    return best;
}

// S steps in one pass (n -> n+S); the caller guarantees tbs_supported(h).
template <typename T, int ARITH, int S>
cudaError_t launch_tbs_3d(prs_ctx* h, const T* p, const T* v, T* pn, T* vn) {
    // output rows per CTA: measured 1024^3, chunk 128: FP32 TY = 16 1.21 ms/step (20: 1.25, 12: 1.30);
    // FP64 TY = 20 2.41 ms/step (16: 2.52, 12: 2.60)
    constexpr int TY = (sizeof(T) == 8) ? 20 : 16;
    constexpr int W = Pk<T>::W;
    const int N = (int)h->N, NQ = N / W;
    // Rows of the tile per thread (PRS_OPT_TBS_ROWS; 0 = auto).  Measured on B200, 1024^3, us per step at S = 4
    // (cp.async | bulk loader): FP32 one row 1216 | 1157, two rows 1300 | 1034; FP64 one row 2556 | 2487, two rows
    // 2618 | 2737 -- the two-row kernel pays off once the bulk loader has taken the LDGSTS out of the l1tex pipe, and
    // only in FP32 (FP64 at two rows per thread runs 16 warps at the 128-register cap with spills).
    const bool bulk_ok = NQ >= 32 && h->opt_tbs_loader != 1;
    const int rows = h->opt_tbs_rows ? h->opt_tbs_rows : ((sizeof(T) == 4 && bulk_ok) ? 2 : 1);
    if (rows == 2) return launch_tbr_3d<T, ARITH, S>(h, p, v, pn, vn);
    StepCoefs<T, S> ks;
    for (int s = 0; s < S; ++s) ks.k[s] = coef_at<T>(h, h->step + s);
    constexpr int XOUT = tbs_xout<T, S>();
    const unsigned gx = (unsigned)((NQ + XOUT - 1) / XOUT), gy = (unsigned)((N + TY - 1) / TY);
    // z slab (prs_create_slab): the lattice is N x N x (owned + 2 halo) planes and only the owned planes
    // are written; the S halo planes on either side are what the S stages consume
    ZRange zr = {N, 0, N, 0u};
    if (h->slab) zr = {(int)h->NZ, (int)h->halo, (int)(h->halo + h->nz_own), 0u};
    zr.wrap = (unsigned)zr.nz * ((unsigned)N * (unsigned)NQ);
    const int nzo = zr.hi - zr.lo;
    const int ZC = tbs_pick_zc(h, (long long)gx * gy, nzo, S);
    const dim3 grid(gx, gy, (unsigned)((nzo + ZC - 1) / ZC));
    const dim3 block(32, TY + 2 * S, 1);
    const size_t smem = tbs_smem_bytes<T, S, TY>();
    // the rings are filled by TMA bulk copies of whole tile rows (at most two runs per row) when a row of the
    // lattice holds at least 32 vectors; smaller lattices, or PRS_OPT_TBS_LOADER = 1, keep the per-thread cp.async
    const bool bulk = NQ >= 32 && h->opt_tbs_loader != 1;
    if (bulk) {
        static std::atomic<unsigned long long> configured{0};      // per instantiation: devices already set up
        const cudaError_t e = ensure_dynamic_smem(step3d_tbs_kernel<T, ARITH, S, TY, true>, smem, h->device, configured);
        if (e != cudaSuccess) return e;
        step3d_tbs_kernel<T, ARITH, S, TY, true><<<grid, block, smem, h->stream>>>(p, v, pn, vn, N, ZC, ks, zr);
        char name[96];
        snprintf(name, sizeof(name), "step3d_tbs_kernel<%s,%d,%d,%d,1>", type_name<T>(), ARITH, S, TY);
        note_launch(h, name, grid, block, smem, S);
    } else {
        static std::atomic<unsigned long long> configured{0};
        const cudaError_t e = ensure_dynamic_smem(step3d_tbs_kernel<T, ARITH, S, TY, false>, smem, h->device, configured);
        if (e != cudaSuccess) return e;
        step3d_tbs_kernel<T, ARITH, S, TY, false><<<grid, block, smem, h->stream>>>(p, v, pn, vn, N, ZC, ks, zr);
        char name[96];
        snprintf(name, sizeof(name), "step3d_tbs_kernel<%s,%d,%d,%d,0>", type_name<T>(), ARITH, S, TY);
        note_launch(h, name, grid, block, smem, S);
    }
    return cudaGetLastError();
}

// The same S steps with two rows per thread (prs_kernels_tbr.cuh): 16 warps, tiles of 32 rows.
template <typename T, int ARITH, int S, int TY>
cudaError_t launch_tbr_3d_ty(prs_ctx* h, const T* p, const T* v, T* pn, T* vn) {
    constexpr int W = Pk<T>::W;
    const int N = (int)h->N, NQ = N / W;
    StepCoefs<T, S> ks;
    for (int s = 0; s < S; ++s) ks.k[s] = coef_at<T>(h, h->step + s);
    const size_t smem = tbr_smem_bytes<T, S, TY>();
    constexpr int XOUT = tbs_xout<T, S>();
    const unsigned gx = (unsigned)((NQ + XOUT - 1) / XOUT), gy = (unsigned)((N + TY - 1) / TY);
    ZRange zr = {N, 0, N, 0u};
    if (h->slab) zr = {(int)h->NZ, (int)h->halo, (int)(h->halo + h->nz_own), 0u};
    zr.wrap = (unsigned)zr.nz * ((unsigned)N * (unsigned)NQ);
    const int nzo = zr.hi - zr.lo;
    const int ZC = tbs_pick_zc(h, (long long)gx * gy, nzo, S);
    const dim3 grid(gx, gy, (unsigned)((nzo + ZC - 1) / ZC));
    const dim3 block(32, (TY + 2 * S) / 2, 1);
    const bool bulk = NQ >= 32 && h->opt_tbs_loader != 1;          // as in launch_tbs_3d
    char name[96];
    snprintf(name, sizeof(name), "step3d_tbr_kernel<%s,%d,%d,%d,%d>", type_name<T>(), ARITH, S, TY, bulk ? 1 : 0);
    if (bulk) {
        static std::atomic<unsigned long long> configured{0};      // per instantiation: devices already set up
        const cudaError_t e = ensure_dynamic_smem(step3d_tbr_kernel<T, ARITH, S, TY, true>, smem, h->device, configured);
        if (e != cudaSuccess) return e;
        step3d_tbr_kernel<T, ARITH, S, TY, true><<<grid, block, smem, h->stream>>>(p, v, pn, vn, N, ZC, ks, zr);
    } else {
        static std::atomic<unsigned long long> configured{0};
        const cudaError_t e = ensure_dynamic_smem(step3d_tbr_kernel<T, ARITH, S, TY, false>, smem, h->device, configured);
        if (e != cudaSuccess) return e;
        step3d_tbr_kernel<T, ARITH, S, TY, false><<<grid, block, smem, h->stream>>>(p, v, pn, vn, N, ZC, ks, zr);
    }
    note_launch(h, name, grid, block, smem, S);
    return cudaGetLastError();
}

template <typename T, int ARITH, int S>
cudaError_t launch_tbr_3d(prs_ctx* h, const T* p, const T* v, T* pn, T* vn) {
    // tiles of 32 rows, one CTA of 512 threads per SM (measured 1024^3 FP32 S = 3: 1.26 ms per step; tiles of
    // 16 rows, two CTAs of 256 threads per SM: 1.43 -- what the second CTA hides costs less than its halo)
    return launch_tbr_3d_ty<T, ARITH, S, 32 - 2 * S>(h, p, v, pn, vn);
}

template <typename T, int ARITH, int S>
cudaError_t launch_tbs_2d(prs_ctx* h, const T* p, const T* v, T* pn, T* vn) {
    constexpr int W = Pk<T>::W;
    const int N = (int)h->N, NQ = N / W;
    StepCoefs<T, S> ks;
    for (int s = 0; s < S; ++s) ks.k[s] = coef_at<T>(h, h->step + s);
    constexpr int XOUT = tbs_xout<T, S>();
    const int BX = 128, warps = BX / 32;
    const unsigned nwarps = (unsigned)((NQ + XOUT - 1) / XOUT);
    const unsigned gx = (nwarps + warps - 1) / warps;
    // Rows per march: long enough to amortise the 2S halo rows, short enough to fill 148 SMs.  Measured
    // (B200, us per step, FP32 S = 8 / FP64 S = 6, rows per march 16 | 32 | 64 | 128):
    //   1024^2   2.06 | 2.13 | 3.34 | 5.90      2.74 | 3.08 | 3.77 | 6.50
    //   2048^2   4.62 | 4.38 | 5.14 | 5.90      7.88 | 7.21 | 7.60 | 9.91
    //   4096^2  16.4  | 13.2 | 12.9 | 14.6      27.0 | 22.9 | 20.9 | 22.2
    // i.e. N/64, between 8 (launch-bound lattices: 256^2 1.6 us per step with 8-row marches, 2.6 with 32) and
    // 128 (16384^2).  (An earlier rule aimed at 8 CTAs per SM whatever the halo cost and marched 8 rows at
    // 2048^2: 6.15 us per step.)
    int YC;
    if (h->opt_chunk > 0) YC = (int)std::min<int64_t>(h->opt_chunk, N);
    else {
        YC = std::min<int>(N, std::max(8, std::min(128, N / 64)));
        // Grids of a few waves: the last wave costs a full march however few CTAs it holds, so pick the rows per march
        // that minimise waves x (rows marched per CTA) for the CTAs the device really holds at once (the FP32 eight-step
        // kernel: 214 registers, two blocks per SM).  Measured on B200, FP32, us per step, N/64 rule -> this rule:
        // 2048^2 5.25 -> 3.33 (320 CTAs on 296 slots -> 295), 4096^2 12.85 -> 10.99 (640 -> 290).
        static std::atomic<int> occupancy[64];                     // blocks per SM of this instantiation, per device
        const int dev = (h->device >= 0 && h->device < 64) ? h->device : 0;
        int per_sm = occupancy[dev].load();
        if (per_sm == 0) {
            if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, step2d_tbs_kernel<T, ARITH, S>, BX, 0) != cudaSuccess || per_sm < 1) {
                cudaGetLastError();
                per_sm = 1;
            }
            occupancy[dev].store(per_sm);
        }
        const long long slots = (long long)std::max(1, h->sm_count) * per_sm;
        if ((long long)gx * ((N + YC - 1) / YC) <= 6 * slots) {
            long long best_cost = -1;
            for (long long w = 1; w <= 8; ++w) {
                const long long gy_max = w * slots / gx;
                if (gy_max < 1) continue;
                const int yc = (int)std::max<long long>(8, (N + gy_max - 1) / gy_max);
                const long long gy = (N + yc - 1) / yc;
                const long long cost = (((long long)gx * gy + slots - 1) / slots) * (yc + 2 * S - 2);
                if (best_cost < 0 || cost < best_cost) { best_cost = cost; YC = yc; }
            }
        }
    }
    const dim3 grid(gx, (unsigned)((N + YC - 1) / YC), 1);
    // rows of L2 prefetch ahead of the load cursor: measured 16384^2 FP32 S = 6, ms per step:
    // none 0.180, 4 rows 0.154, 8 rows 0.153, 16 rows 0.163, 32 rows 0.215
    const int l2_ahead = std::min(TBS2D_L2_AHEAD, N);
    step2d_tbs_kernel<T, ARITH, S><<<grid, BX, 0, h->stream>>>(p, v, pn, vn, N, YC, l2_ahead, ks);
    char name[96];
    snprintf(name, sizeof(name), "step2d_tbs_kernel<%s,%d,%d>", type_name<T>(), ARITH, S);
    note_launch(h, name, grid, dim3(BX, 1, 1), 0, S);
    return cudaGetLastError();
}

}  // namespace prs
