// prs_instances.cu -- explicit instantiations of the temporally blocked launchers (and with them
// their kernels).  build.py compiles this file once per unit, in parallel:
//   -DPRS_UNIT=1  two-step kernels   (prs_launch_tb2.cuh)
//   -DPRS_UNIT=2  S-step kernels, 3D (prs_launch_tbs.cuh), S = 3, 4
//   -DPRS_UNIT=3  S-step kernels, 2D (prs_launch_tbs.cuh), S = 3, 4, 6, 8
// each with -DPRS_T=float|double and -DPRS_ARITH=0|1|2 (prs_arith.cuh: literal, coefficient, fused).
// prs_api.cu calls them through the declarations in prs_host.cuh.
#if !defined(PRS_UNIT) || !defined(PRS_T) || !defined(PRS_ARITH)
#error "compile with -DPRS_UNIT=1|2|3 -DPRS_T=float|double -DPRS_ARITH=0|1|2 (see build.py)"
#endif

#if PRS_UNIT == 1
#include "prs_launch_tb2.cuh"
namespace prs {
template cudaError_t launch_tb2_3d<PRS_T, PRS_ARITH>(prs_ctx*, const PRS_T*, const PRS_T*, PRS_T*, PRS_T*,
                                                     const StepCoef<PRS_T>&, const StepCoef<PRS_T>&);
template cudaError_t launch_tb2_2d<PRS_T, PRS_ARITH>(prs_ctx*, const PRS_T*, const PRS_T*, PRS_T*, PRS_T*,
                                                     const StepCoef<PRS_T>&, const StepCoef<PRS_T>&);
}  // namespace prs
#elif PRS_UNIT == 2
#include "prs_launch_tbs.cuh"
namespace prs {
template cudaError_t launch_tbs_3d<PRS_T, PRS_ARITH, 3>(prs_ctx*, const PRS_T*, const PRS_T*, PRS_T*, PRS_T*);
template cudaError_t launch_tbs_3d<PRS_T, PRS_ARITH, 4>(prs_ctx*, const PRS_T*, const PRS_T*, PRS_T*, PRS_T*);
}  // namespace prs
#elif PRS_UNIT == 3
#include "prs_launch_tbs.cuh"
namespace prs {
template cudaError_t launch_tbs_2d<PRS_T, PRS_ARITH, 3>(prs_ctx*, const PRS_T*, const PRS_T*, PRS_T*, PRS_T*);
template cudaError_t launch_tbs_2d<PRS_T, PRS_ARITH, 4>(prs_ctx*, const PRS_T*, const PRS_T*, PRS_T*, PRS_T*);
template cudaError_t launch_tbs_2d<PRS_T, PRS_ARITH, 6>(prs_ctx*, const PRS_T*, const PRS_T*, PRS_T*, PRS_T*);
template cudaError_t launch_tbs_2d<PRS_T, PRS_ARITH, 8>(prs_ctx*, const PRS_T*, const PRS_T*, PRS_T*, PRS_T*);
}  // namespace prs
#else
#error "unknown PRS_UNIT"
#endif
