/*
 * prs_ref.h -- C ABI of the CPU ORACLE for the Press-Ryden-Spergel (PRS) domain-wall step.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load this library.  The product (paper_1710_10420_b200/) never does,
 * and the two share no source: this header is the oracle's own and is not included by the CUDA path.
 *
 * What it computes: PAPER.md Eqs. 1, 3-6 (step) and Eqs. 7-8 (diagnostics), written out site by
 * site; see prs_ref.cpp for the per-function citations and DESIGN.md section 3 for the readings
 * taken where the paper is silent.
 *
 * Layout: dense T[N^dims], linear index s = x + N*(y + N*z), x fastest.  T = float (precision 0)
 * or double (precision 1).  All functions return 0 on success, non-zero on bad arguments.
 */
#ifndef PRS_REF_H
#define PRS_REF_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct prs_ref_ctx* prs_ref_handle;

enum { PRS_REF_F32 = 0, PRS_REF_F64 = 1 };

/* Arithmetic of the velocity update (Eq. 4):
 *   LITERAL: phidot' = ((1-delta)*phidot + deta*f) / (1+delta), one division per site;
 *   COEF   : phidot' = A*phidot + B*f with A=(1-delta)/(1+delta), B=deta/(1+delta) formed in
 *            double once per step and rounded to T.  Algebraically identical; differs by rounding.
 *   FMA    : COEF with every product that feeds a sum contracted into one fused multiply-add
 *            (std::fma, one rounding): lap = fma(-2d, c, sum); t = fma(c*c, I, -1);
 *            f = fma((-K)*c, t, lap); phidot' = fma(A, phidot, B*f); phi' = fma(deta, phidot', c).
 *            IEEE-754 fixes fma exactly, so a GPU evaluating the same sequence matches bit for bit. */
enum { PRS_REF_ARITH_LITERAL = 0, PRS_REF_ARITH_COEF = 1, PRS_REF_ARITH_FMA = 2 };

typedef struct {
    int64_t  step;        /* n of the state measured                                  */
    double   eta;         /* eta_n = eta0 + n*deta                                    */
    uint64_t link_count;  /* C   = number of forward nearest-neighbour links crossing */
    uint64_t wall_sites;  /* N_w = number of sites with at least one crossing link    */
    double   sum_ratio;   /* sum over wall sites of phidot^2 / V(phi)                 */
    double   rho;         /* C / N^dims                                               */
    double   gv2;         /* sum_ratio / (2 N_w), 0 if N_w == 0                       */
} prs_ref_diag;

int prs_ref_create(prs_ref_handle* out, int dims, int64_t N, int precision,
                   double alpha, double era_m, double deta, double W0, double phi0, uint64_t seed);
int prs_ref_destroy(prs_ref_handle h);
int prs_ref_set_beta(prs_ref_handle h, double beta);    /* default 0 (PRS); a^beta multiplies dV/dphi,   *
                                                          * a = (eta/eta0)^m normalised at eta0          */
int prs_ref_set_arith(prs_ref_handle h, int arith);      /* default LITERAL                     */
int prs_ref_set_threads(prs_ref_handle h, int nthreads); /* default 1; >1 = OpenMP outer loop,  *
                                                          * results bit-identical (Jacobi step) */
int prs_ref_init(prs_ref_handle h, double eta0);         /* Philox field, phidot = 0, n = 0     */
int prs_ref_step(prs_ref_handle h, int64_t nsteps);
int prs_ref_diagnostics(prs_ref_handle h, prs_ref_diag* out);
int prs_ref_copy_out(prs_ref_handle h, void* phi_dst, void* phidot_dst);   /* either may be NULL */
int prs_ref_copy_in(prs_ref_handle h, const void* phi_src, const void* phidot_src,
                    double eta0, int64_t step);

/* Stateless helpers (used to pin the oracle and for sampled parity at sizes too big to step). */

/* Philox4x32-10 block function (Salmon et al. 2011): out = philox(ctr, key). */
void prs_ref_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);

/* Initial value of site s: phi0 * (2*(w>>8) + 1 - 2^24) * 2^-24 as double. */
double prs_ref_init_value(uint64_t seed, uint64_t s, double phi0);

/* Diagnostics (Eqs. 7-8) of a caller-held snapshot.  eta/step are only echoed into *out. */
int prs_ref_diagnostics_of(int dims, int64_t N, int precision, const void* phi, const void* phidot,
                           double W0, double phi0, prs_ref_diag* out);

/* Orientation-weighted wall area of a caller-held snapshot: PAPER.md Eq. 7 as printed, sum over crossing
 * links of |grad phi| / (|phi,x| + |phi,y| + |phi,z|); gradient on a link as in DESIGN.md R15.
 * rho_weighted = *area / N^dims. */
int prs_ref_weighted_area_of(int dims, int64_t N, int precision, const void* phi, double* area);

/* One PRS step (Eqs. 3-6) evaluated ONLY at the listed sites of a caller-held state at step n
 * (time eta0 + n*deta).  phi/phidot are full fields T[N^dims]; outputs are T[nsites]. */
int prs_ref_step_sites(int dims, int64_t N, int precision, int arith,
                       double alpha, double era_m, double deta, double W0, double phi0,
                       double eta0, int64_t n,
                       const void* phi, const void* phidot,
                       const int64_t* sites, int64_t nsites,
                       void* phi_next_out, void* phidot_next_out);

/* Per-step scalars (Eq. 6 and the derived coefficients), all in double: out[0]=eta_n,
 * out[1]=delta_n, out[2]=A, out[3]=B, out[4]=V0, out[5]=K=4V0/phi0^2, out[6]=I=1/phi0^2. */
/* The same with the scale-factor exponent beta of Eq. 2: K becomes K * (eta_n/eta0)^(m*beta). */
int prs_ref_scalars_beta(double alpha, double beta, double era_m, double deta, double W0, double phi0,
                         double eta0, int64_t n, double out[7]);
int prs_ref_scalars(double alpha, double era_m, double deta, double W0, double phi0,
                    double eta0, int64_t n, double out[7]);

#ifdef __cplusplus
}
#endif
#endif
