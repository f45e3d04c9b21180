/*
 * prs.h -- C ABI of libprs: the Press-Ryden-Spergel (PRS) domain-wall step on one NVIDIA B200.
 *
 * The library advances a real scalar field phi on a periodic N^dims lattice (dims = 2 or 3, dx = 1)
 * with the damped staggered leapfrog of arxiv 1710.10420 (Eqs. 3-6, :46-55) for the quartic
 * potential of Eq. 1 (:30), and measures the two wall diagnostics of Eqs. 7-8 (:57-66).  Every step of
 * that path runs in hand-written sm_100a CUDA kernels; there is no CPU fallback.
 *
 * State held between calls: phi^n and phidot^{n-1/2} with step counter n, eta_n = eta0 + n*deta.
 *
 * Memory and ownership
 *   - The CALLER owns the device workspace (prs_workspace_bytes() bytes, 256-byte aligned DEVICE
 *     pointer, e.g. torch.empty(nbytes, dtype=uint8, device="cuda").data_ptr()) and the CUDA stream
 *     (a cudaStream_t passed as void*; NULL = the legacy default stream).  The library carves the
 *     workspace into its field arrays and reduction scratch, never allocates or frees device memory,
 *     and launches everything on that stream.
 *   - Fields are dense T[N^dims], linear index s = x + N*(y + N*z), x fastest; T = float
 *     (PRS_F32) or double (PRS_F64).
 *   - prs_destroy frees only host-side bookkeeping (and a few bytes of pinned host memory).
 *
 * Errors: every function returns PRS_OK (0) or a PRS_ERR_* code; nothing throws, aborts or prints.
 * On error out-parameters are untouched.  prs_last_error(h) gives a text for the last failure on h
 * (handle-owned, valid until the next call on h).  Asynchronous CUDA faults surface at the next
 * synchronising call (prs_diagnostics, prs_copy_out, prs_copy_in, prs_sync).
 * A handle is not thread-safe; distinct handles are independent.
 *
 * Devices: a handle belongs to the device that owns its workspace (taken from the pointer at prs_create).
 * Every call that touches CUDA makes that device current for its duration and restores the caller's current
 * device before it returns, so one process may drive handles on several devices in any order.  The stream
 * passed to prs_create must belong to that device.
 */
#ifndef PRS_H
#define PRS_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct prs_ctx* prs_handle;

enum { PRS_OK = 0, PRS_ERR_INVALID_ARG = 1, PRS_ERR_UNSUPPORTED = 2, PRS_ERR_WORKSPACE = 3,
       PRS_ERR_STATE = 4, PRS_ERR_CUDA = 5,
       PRS_ERR_NOMEM = 6 };   /* host-side allocation failed (context or the 24 bytes of pinned memory) */

enum { PRS_F32 = 0, PRS_F64 = 1 };

/* Diagnostics of the state in memory (phi^n, phidot^{n-1/2}); Eqs. 7-8 with the readings
 * of DESIGN.md section 3. */
typedef struct {
    int64_t  step;        /* n                                                                    */
    double   eta;         /* eta_n                                                                */
    uint64_t link_count;  /* C: forward nearest-neighbour links (d per site, periodic) whose two   *
                           * ends differ in IEEE sign bit (Eq. 7's sum of delta_pm) -- bit-exact   */
    uint64_t wall_sites;  /* N_w: sites touching at least one crossing link (Eq. 8's N)            */
    double   sum_ratio;   /* sum over wall sites of phidot^2 / V(phi), in double (0 where V == 0)  */
    double   rho;         /* C / N^dims   (Eq. 7 with Delta A = 1, unweighted)                     */
    double   gv2;         /* sum_ratio / (2 N_w), 0 if N_w == 0   (Eq. 8)                          */
} prs_diag;

/* Options for prs_set_option (all have defaults; tests use them to force one kernel). */
enum {
    PRS_OPT_STEP_KERNEL = 1,   /* PRS_KERNEL_*                                   default AUTO     */
    PRS_OPT_ARITH       = 2,   /* PRS_ARITH_*                                    default FMA      */
    PRS_OPT_DIAG_KERNEL = 3,   /* PRS_KERNEL_AUTO / GENERIC / TILED / BITS       default AUTO     */
    PRS_OPT_CHUNK       = 4,   /* tuning: planes (3D) / rows (2D) one CTA marches; 0 = auto        */
    PRS_OPT_TILE_Y      = 5,   /* tuning: rows per CTA of the 3D tiled kernel, 4 / 8 / 16          */
    PRS_OPT_TB2_TILE_Y  = 6,   /* tuning: output rows per CTA of the 3D two-step kernel, 4 / 8 / 12 / 28 */
    PRS_OPT_TBS_STEPS   = 7,   /* steps per pass of the multi-step kernel: 3 or 4, in 2D also 6 or 8;
                                * default 4 in 3D, in 2D 8 (FP32) or 6 (FP64)                       */
    PRS_OPT_TBS_ROWS    = 8,   /* tuning, 3D multi-step kernel: rows of the tile per thread: 1 (step3d_tbs_kernel),
                                * 2 (step3d_tbr_kernel: half the shared-memory traffic, taller tiles;
                                * bit-identical) or 0 = auto (default): 2 in FP32 where the bulk loader
                                * applies (1024^3: 17 % faster), else 1                                */
    PRS_OPT_DIAG_CHUNK  = 10,  /* tuning: planes (3D) / rows (2D) one CTA of the one-pass diagnostics kernel marches;
                                * 0 = auto                                                               */
    PRS_OPT_CLUSTER_CTAS = 11, /* tuning, cluster-resident kernel at N = 256: CTAs in the cluster, 16 (opt-in size; what 0 =
                                * auto takes where the device can co-schedule it) or 8                     */
    PRS_OPT_TBS_LOADER  = 9    /* tuning, 3D multi-step kernel: how the shared-memory rings are filled: 0 (default)
                                * = TMA bulk copies of whole tile rows completing on mbarriers where a lattice
                                * row holds >= 32 16-byte vectors, else per-thread cp.async; 1 = always cp.async;
                                * 2 = same as 0.  Bit-identical either way                              */
};
enum {
    PRS_KERNEL_AUTO    = 0,    /* fastest kernel that supports (dims, N, precision)                */
    PRS_KERNEL_GENERIC = 1,    /* one thread per site, any N >= 1                                  */
    PRS_KERNEL_TILED   = 2,    /* shared-memory tiled, one step per pass over HBM                  */
    PRS_KERNEL_TB2     = 3,    /* temporally blocked: two steps per pass over HBM (same per-site   *
                                * arithmetic, bit-identical to two single steps)                   */
    PRS_KERNEL_CLUSTER = 5,    /* small 2D boxes (N = 64, 128, 256): the state stays in the registers and shared *
                                * memory of one thread-block cluster of 8 (N = 256: 16) CTAs for up to 64 steps per  *
                                * launch; bit-identical to single steps; what AUTO takes at these sizes          */
    PRS_KERNEL_BITS    = 6,    /* PRS_OPT_DIAG_KERNEL only: diagnostics on packed sign bits -- one pass reads phi   *
                                * and packs a bit per site, a second counts links and wall sites on the bit words *
                                * and fetches phidot at wall sites only; N a multiple of 32 16-byte vectors; what *
                                * AUTO takes from 2^26 sites up                                                   */
    PRS_KERNEL_TBS     = 4     /* PRS_OPT_TBS_STEPS steps per pass over HBM (2D and 3D), bit-identical *
                                * to single steps; leftovers of a prs_step call go through the      *
                                * shorter pipelines (6, 4, 3 steps), TB2 and TILED                  */
};
/* Arithmetic form of Eqs. 3-5 (R13).  LITERAL: Eq. 4 (:49) as printed, one division per
 * site, ((1-d)*v + deta*f)/(1+d).  COEF: A = (1-d)/(1+d) and B = deta/(1+d) formed in double on the
 * host once per step, v' = A*v + B*f.  In both, every multiply and add is rounded on its own (never
 * contracted).  FMA (default): COEF with every product that feeds a sum contracted into one fused
 * multiply-add -- lap = fma(-2d, c, sum); t = fma(c*c, 1/phi0^2, -1); f = fma((-K)*c, t, lap);
 * v' = fma(A, v, B*f); phi' = fma(deta, v', c) -- what a compiler emits from the formulas by default,
 * and the fastest form.  Each form matches the oracle's form of the same name bit for bit; all three
 * agree within rounding (about 2e-7 FP32 / 4e-16 FP64 after 20 steps). */
enum { PRS_ARITH_LITERAL = 0, PRS_ARITH_COEF = 1, PRS_ARITH_FMA = 2 };

/* Read-only counters for prs_get_info. */
enum {
    PRS_INFO_KERNEL_LAUNCHES = 1,  /* kernels launched on behalf of this handle since creation     */
    PRS_INFO_STEP_KERNEL     = 2,  /* PRS_KERNEL_* actually used by the last prs_step              */
    PRS_INFO_STEP            = 3,  /* n                                                            */
    PRS_INFO_DIAG_KERNEL     = 4,  /* PRS_KERNEL_* actually used by the last prs_diagnostics       */
    PRS_INFO_HALO_VALID      = 5,  /* slab: steps the halo planes can still feed (0 = exchange)    */
    PRS_INFO_HALO_PLANES     = 6,  /* slab: halo planes per side (4); 0 on a whole lattice         */
    PRS_INFO_DEVICE          = 7   /* ordinal of the CUDA device that owns the workspace           */
};

/* Bytes of device workspace needed; 0 if the arguments are invalid. */
size_t prs_workspace_bytes(int dims, int64_t N, int precision);

/* Creates a simulation.  dims in {2,3}; N >= 1 sites per side; precision PRS_F32/PRS_F64;
 * alpha >= 0 (PRS: 3) multiplies the friction term of Eq. 2 (:34); era_m = dln a/dln eta >= 0
 * (1 radiation, 2 matter, 0 = no expansion); deta > 0 the conformal time step; W0 > 0 the wall
 * thickness, which sets V0 = pi^2 phi0^2 / (2 W0^2); phi0 > 0 the vacuum value; seed keys the
 * initial-condition generator.  workspace: DEVICE pointer (see above); cuda_stream: cudaStream_t. */
int prs_create(prs_handle* out, int dims, int64_t N, int precision,
               double alpha, double era_m, double deta, double W0, double phi0, uint64_t seed,
               void* workspace, size_t workspace_bytes, void* cuda_stream);

int prs_destroy(prs_handle h);

/* Seeded initial condition: phi_s = phi0 * u_s, u_s an odd multiple of 2^-24
 * in (-1,1) drawn from Philox4x32-10(counter = s>>2, key = seed), word s&3; phidot = +0; n = 0,
 * eta = eta0 > 0.  Asynchronous on the stream. */
int prs_init(prs_handle h, double eta0);

/* Advances nsteps >= 0 steps of Eqs. 3-6.  Asynchronous on the stream; no host sync, no transfer. */
int prs_step(prs_handle h, int64_t nsteps);

/* Measures Eqs. 7-8 on the current state; synchronises the stream; fills *out (HOST pointer). */
int prs_diagnostics(prs_handle h, prs_diag* out);

/* ncycles times: steps_per_cycle steps of Eqs. 3-6, then Eqs. 7-8 on the state reached -- the loop every config of
 * BASELINE.json runs ("diagnostics every 10 / 50 / 100 steps"), as ONE call: all launches are queued back to back, every
 * cycle's reduced record stays on the device (a ring of 4096 records in the workspace) and the records cross to the host
 * once per 4096 cycles, so a cycle costs its kernels and nothing else (the per-step transfer of the
 * partial sums is what hurts small boxes).  out: HOST array of ncycles records, out[i] = what prs_diagnostics would
 * have returned after (i + 1) * steps_per_cycle further steps: the fields and the integer counts identical, and
 * sum_ratio identical too (the same kernels in the same launch configuration) except where the cluster-resident
 * small-box kernel is the step kernel (2D, N = 64, 128 or 256 by default): there the diagnostics passes run INSIDE the step
 * launches, up to 64 steps and all their passes per launch with the state on chip throughout, and sum_ratio differs
 * from prs_diagnostics' by the order of its double additions (about 1e-15 relative).  Synchronises the stream before
 * it returns.  Not on a slab (PRS_ERR_UNSUPPORTED). */
int prs_run(prs_handle h, int64_t ncycles, int64_t steps_per_cycle, prs_diag* out);

/* Orientation-weighted wall area of the current phi^n: PAPER.md Eq. 7 as printed (:59-62), the sum over
 * crossing forward links of |grad phi| / (|phi,x| + |phi,y| + |phi,z|) with the gradient on a link taken as
 * in DESIGN.md R15 (forward difference along the link, mean of the two end-point central differences
 * across it), in double.  *area = that sum (between link_count/sqrt(dims) and link_count),
 * *rho_weighted = *area / N^dims; either pointer may be NULL (HOST pointers).  Synchronises the stream. */
int prs_weighted_area(prs_handle h, double* area, double* rho_weighted);

/* Snapshot: copies phi^n and/or phidot^{n-1/2} (T[N^dims]) to HOST or DEVICE memory (either pointer
 * may be NULL); synchronises the stream. */
int prs_copy_out(prs_handle h, void* phi_dst, void* phidot_dst);

/* Restores a state from HOST or DEVICE memory (both required) and sets eta0 > 0, n = step >= 0, so
 * that eta_n = eta0 + n*deta; synchronises the stream. */
int prs_copy_in(prs_handle h, const void* phi_src, const void* phidot_src, double eta0, int64_t step);

/* Exponent beta of the scale factor in front of dV/dphi in Eq. 2.  Default 0 (PRS, :42);
 * beta = 2 with alpha = 2 gives the exact equations of motion.  a(eta) = (eta/eta0)^era_m, a(eta0) = 1 with
 * eta0 the time given to prs_init / prs_copy_in (R16); takes effect from the next prs_step. */
int prs_set_beta(prs_handle h, double beta);

/* Blocks until everything queued for h has finished; reports a pending asynchronous CUDA fault. */
int prs_sync(prs_handle h);

int prs_set_option(prs_handle h, int option, int64_t value);   /* PRS_ERR_UNSUPPORTED if the kernel  *
                                                                * cannot take this (dims, N, T)      */
int prs_get_info(prs_handle h, int info, int64_t* value);

/* What the most recent prs_step call launched first -- its main kernel: the schedule goes from the deepest
 * pipeline to single steps, e.g. prs_step(50) = 12 four-step launches, then one two-step launch.  name: the kernel
 * with its template arguments as a profiler demangles it, minus "(int)", "(bool)" and blanks, e.g.
 * "step3d_tbs_kernel<float,2,4,16,1>" (truncated to name_bytes); grid, block: its launch configuration; smem_bytes:
 * dynamic shared memory; steps_per_launch: PRS steps one launch advances; launches: how many times that call launched
 * it.  Any pointer may be NULL (HOST pointers).  PRS_ERR_STATE before the first step.  Lets a benchmark tie a
 * profiler capture to the kernel that actually ran. */
int prs_step_launch_info(prs_handle h, char* name, size_t name_bytes, int64_t grid[3], int64_t block[3],
                         int64_t* smem_bytes, int64_t* steps_per_launch, int64_t* launches);

/* DEVICE pointers to the current phi^n and phidot^{n-1/2} arrays (valid until the next prs_step /
 * prs_copy_in / prs_init): lets a caller (e.g. a torch tensor view) read the state without a copy. */
int prs_device_pointers(prs_handle h, void** phi, void** phidot);

/* ---- z slabs: one 3D lattice sharded over several GPUs ("the
 * bottleneck at larger box sizes will be the amount of memory available") -------------------------------
 * A slab handle owns the nz planes z_begin <= z < z_begin + nz of a periodic N^3 lattice (N % 4 == 0,
 * 4 <= nz <= N, 0 <= z_begin < N) plus 4 halo planes below and above them, copies of the neighbouring slabs'
 * outermost owned planes of BOTH fields.  Eqs. 3-5 are applied to halo sites as well, from the planes
 * beyond them, so each step uses up one halo plane per side and every owned site sees exactly the
 * operations of the unsharded lattice: the owned planes stay bit-identical to it.  prs_step(h, k) needs
 * k <= PRS_INFO_HALO_VALID (else PRS_ERR_STATE); k = 4 or 3 is one pass of the multi-step kernel, which
 * writes the owned planes only and leaves PRS_INFO_HALO_VALID = 0; k = 1, 2 go through the single-step /
 * two-step kernels over all planes and leave PRS_INFO_HALO_VALID - k.  The caller
 * moves the halo planes between slabs -- any transport: NCCL send/recv, peer copies over NVLink -- :
 *   prs_slab_halo_regions  DEVICE pointers into the CURRENT arrays (they change with every prs_step), each
 *                          *bytes = 4*N*N*sizeof(T) long and contiguous: send[0], send[1] = phi's lowest / highest
 *                          four owned planes, for the z-1 / z+1 neighbour; recv[0], recv[1] = phi's lower / upper
 *                          halo, to be filled with the z-1 neighbour's send[1] / the z+1 neighbour's send[0];
 *                          [2], [3] the same for phidot.  Neighbours are periodic (one slab: itself).
 *   prs_slab_halo_filled   declares the halo planes current: PRS_INFO_HALO_VALID = 4.
 * prs_init fills the halo planes itself (the initial condition is a function of the global site), so a
 * fresh slab can take four steps at once.  prs_diagnostics needs PRS_INFO_HALO_VALID >= 1 and returns this
 * slab's partial sums (link_count, wall_sites, sum_ratio; rho = link_count / N^3, this slab's share): add
 * them over the slabs.  prs_copy_out / prs_copy_in move the owned planes, T[nz*N*N]; prs_copy_in leaves
 * the halo stale.  prs_weighted_area needs PRS_INFO_HALO_VALID >= 1 as well and returns the slab's partial sum
 * (*rho_weighted = *area / N^3, this slab's share): add them over the slabs.  Everything else as for prs_create. */
size_t prs_slab_workspace_bytes(int64_t N, int64_t nz, int precision);      /* 0 if args invalid */
int prs_create_slab(prs_handle* out, int64_t N, int64_t z_begin, int64_t nz, int precision,
                    double alpha, double era_m, double deta, double W0, double phi0, uint64_t seed,
                    void* workspace, size_t workspace_bytes, void* cuda_stream);
int prs_slab_halo_regions(prs_handle h, void* send[4], void* recv[4], size_t* bytes);
/* Adds the partial diagnostics of the n parts of one lattice (prs_diagnostics of each slab, all of the same step;
 * HOST pointers) and applies the normalisation of PAPER.md Eqs. 7-8 (:57-66): link_count, wall_sites and sum_ratio
 * are summed (sum_ratio in the order given), rho = link_count / N^dims, gv2 = sum_ratio / (2 wall_sites) or 0;
 * step and eta are parts[0]'s.  PRS_ERR_STATE if the parts are of different steps.  Touches no device. */
int prs_diag_combine(const prs_diag* parts, int n, int dims, int64_t N, prs_diag* out);
int prs_slab_halo_filled(prs_handle h);

/* ---- for callers that must not allocate ------------------------------------------------------------------------
 * (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).  prs_diagnostics_static
 * measures PAPER.md Eqs. 7-8 (:57-66; the readings of DESIGN.md section 3, as prs_diagnostics) on fields the CALLER
 * holds, with no handle and no workspace, and calls no cudaMalloc / cudaFree / cudaHostAlloc or any allocating routine:
 * the scratch of the pass (one partial sum per block of 4096 sites, and a ticket counter) is a file-scope
 * static __device__ array of prs_diagnostics_static_scratch_bytes() = 786 688 bytes, which every GPU that loads the
 * library holds until the process exits.
 *   phi, phidot   DEVICE pointers, inputs: dense T[N^dims], x fastest, T = float (PRS_F32) / double (PRS_F64);
 *                 the call runs on the device that owns phi (made current for the call, restored after)
 *   sums_device   DEVICE pointer, output: the three sums, written by the pass's last block; form rho and gv2 from them
 *                 with prs_diag_combine (a prs_diag with these three fields set is one "part")
 *   cuda_stream   cudaStream_t; the call queues one 256-byte memset and one kernel there and does NOT synchronise
 *   err           optional HOST buffer of err_bytes for the reason of a failure (there is no handle to ask)
 * Limit: N^dims <= prs_diagnostics_static_max_sites() = 2^27 = 134 217 728 sites (512^3, 11585^2): a larger lattice is
 * refused with PRS_ERR_UNSUPPORTED and a message, never truncated; use prs_diagnostics on a handle for those.
 * The array is shared by every call on a GPU and keeps the last call's contents; the ticket counter is cleared on the
 * stream before each pass.  Calls that OVERLAP on one GPU (two streams, two threads) race on it: serialise them.
 * The first call on a device looks the array's address up (cudaGetSymbolAddress, which may load the module): make
 * that first call outside any stream capture.  Counts are bit-exact; sum_ratio differs from prs_diagnostics' by the
 * order of its double additions only (about 1e-15 relative). */
typedef struct {
    uint64_t link_count;   /* C   (Eq. 7's sum of delta_pm)                   */
    uint64_t wall_sites;   /* N_w (Eq. 8's N)                                 */
    double   sum_ratio;    /* sum over wall sites of phidot^2 / V(phi)        */
} prs_diag_sums;
int prs_diagnostics_static(int dims, int64_t N, int precision, double W0, double phi0, const void* phi, const void* phidot,
                           prs_diag_sums* sums_device, void* cuda_stream, char* err, size_t err_bytes);
size_t  prs_diagnostics_static_scratch_bytes(void);
int64_t prs_diagnostics_static_max_sites(void);

const char* prs_last_error(prs_handle h);

#ifdef __cplusplus
}
#endif
#endif
