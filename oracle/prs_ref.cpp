/*
 * prs_ref.cpp -- CPU ORACLE for the Press-Ryden-Spergel domain-wall step and its diagnostics.
 *
 * TEST INFRASTRUCTURE ONLY (see prs_ref.h).  Plain nested loops with modulo wrap, every
 * floating-point operation individually rounded in precision T (build with -ffp-contract=off,
 * never -ffast-math), no blocking, no fusion, no reordering beyond what is written here.  It shares
 * no code with paper_1710_10420_b200/csrc.
 *
 * Passages followed (PAPER.md line : equation):
 *   :30  Eq. 1   V(phi) = V0 (phi^2/phi0^2 - 1)^2   ->  dV/dphi = (4 V0/phi0^2) phi (phi^2/phi0^2 - 1)
 *   :46  Eq. 3   5-point Laplacian, dx = 1, periodic; 3D = 7-point (":53 straightforward extension")
 *   :49  Eq. 4   phidot^{n+1/2} = ((1-delta) phidot^{n-1/2} + deta (lap phi^n - dV/dphi^n))/(1+delta)
 *   :51  Eq. 5   phi^{n+1} = phi^n + deta phidot^{n+1/2}
 *   :55  Eq. 6   delta = (1/2) alpha (deta/eta) (dln a/dln eta)
 *   :59-62 Eq. 7 links = nearest-neighbour pairs where phi changes sign; rho = (number of links)/V
 *                (the orientation weight of Eq. 7 is out of scope: north_star asks for the count)
 *   :64-66 Eq. 8 (gamma v)^2 = (1/2N) sum_walls E_k / V(phi), N = grid points containing walls
 *
 * Readings where the paper is silent: eta in Eq. 6 is eta_n (time level of
 * phi^n); "changes sign" is the IEEE sign bit; E_k = phidot^2; a wall site is a site touching at
 * least one crossing link; V == 0 contributes 0; V0 = pi^2 phi0^2 / (2 W0^2).
 *
 * Pins (tests/test_oracle_*.py, all -m "not gpu"): 4x4 hand-computed step (tests/golden), exact
 * fixed points, oddness / translation / reflection equivariance, uniform-field scalar recurrence,
 * exact discrete plane-wave dispersion (free and massive), damping envelope, planar kink pair,
 * boosted kink (Eq. 8), brute-force diagnostics on tiny fields, Philox published KAT vectors.
 */
#include "prs_ref.h"

#include <cmath>
#include <cstring>
#include <new>
#include <vector>

#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

/* ---------------------------------------------------------------- Philox4x32-10 (S8 / App. B) */

const uint32_t PHILOX_M0 = 0xD2511F53u, PHILOX_M1 = 0xCD9E8D57u;
const uint32_t PHILOX_W0 = 0x9E3779B9u, PHILOX_W1 = 0xBB67AE85u;

void philox_block(const uint32_t c_in[4], const uint32_t k_in[2], uint32_t out[4]) {
    uint32_t c0 = c_in[0], c1 = c_in[1], c2 = c_in[2], c3 = c_in[3];
    uint32_t k0 = k_in[0], k1 = k_in[1];
    for (int round = 0; round < 10; ++round) {
        if (round > 0) { k0 += PHILOX_W0; k1 += PHILOX_W1; }
        const uint64_t p0 = (uint64_t)PHILOX_M0 * c0;
        const uint64_t p1 = (uint64_t)PHILOX_M1 * c2;
        const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        const uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        const uint32_t n0 = hi1 ^ c1 ^ k0;
        const uint32_t n1 = lo1;
        const uint32_t n2 = hi0 ^ c3 ^ k1;
        const uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* Site s draws word (s & 3) of the block with counter (s >> 2) and key = seed.  The value
 * (2k + 1 - 2^24) 2^-24, k = word >> 8, is an odd multiple of 2^-24 in (-1, 1): exact in float. */
double init_value(uint64_t seed, uint64_t s, double phi0) {
    const uint64_t q = s >> 2;
    const uint32_t ctr[4] = {(uint32_t)(q & 0xffffffffu), (uint32_t)(q >> 32), 0u, 0u};
    const uint32_t key[2] = {(uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32)};
    uint32_t w[4];
    philox_block(ctr, key, w);
    const int64_t k = (int64_t)(w[s & 3] >> 8);
    const double u = (double)(2 * k + 1 - (int64_t)16777216) * (1.0 / 16777216.0);
    return phi0 * u;
}

/* ---------------------------------------------------------------- scalars (S1, S2) */

struct Scalars {
    double eta, delta, A, B, V0, K, I;
};

const double PI = 3.14159265358979323846;

/* beta: the exponent of the scale factor in front of dV/dphi in Eq. 2 (:34; printed "alpha^beta",
 * meant a^beta, R1).  PRS: beta = 0 (:42).  beta != 0 (e.g. the exact equations alpha = beta
 * = 2, :36) multiplies dV/dphi at step n by a(eta_n)^beta with a = (eta/eta0)^m, m = dln a/dln eta,
 * normalised to a(eta0) = 1 (R16); it enters only through the per-step constant K. */
Scalars scalars_at(double alpha, double era_m, double deta, double W0, double phi0,
                   double eta0, int64_t n, double beta = 0.0) {
    Scalars s;
    s.V0 = (PI * PI * phi0 * phi0) / (2.0 * W0 * W0);
    s.I = 1.0 / (phi0 * phi0);
    s.eta = eta0 + (double)n * deta;                       /* never accumulated step by step */
    s.K = 4.0 * s.V0 / (phi0 * phi0);
    if (beta != 0.0 && era_m != 0.0) s.K = s.K * std::pow(s.eta / eta0, era_m * beta);
    s.delta = ((0.5 * alpha) * (deta / s.eta)) * era_m;    /* Eq. 6 */
    s.A = (1.0 - s.delta) / (1.0 + s.delta);
    s.B = deta / (1.0 + s.delta);
    return s;
}

inline int64_t wrap(int64_t i, int64_t N) {
    i %= N;
    return i < 0 ? i + N : i;
}

/* ---------------------------------------------------------------- one site of one step (S3) */

template <typename T>
struct StepCoef {
    T K, I, deta, omd, opd, A, B;
    int dims;
    int arith;
};

template <typename T>
StepCoef<T> make_coef(const Scalars& sc, double deta, int dims, int arith) {
    StepCoef<T> c;
    c.K = (T)sc.K;
    c.I = (T)sc.I;
    c.deta = (T)deta;
    const T dT = (T)sc.delta;
    c.omd = T(1) - dT;
    c.opd = T(1) + dT;
    c.A = (T)sc.A;
    c.B = (T)sc.B;
    c.dims = dims;
    c.arith = arith;
    return c;
}

template <typename T>
inline void site_update(const StepCoef<T>& k, const T* phi, const T* phidot, int64_t N,
                        int64_t x, int64_t y, int64_t z, T* phi_next, T* phidot_next) {
    const int64_t xp = wrap(x + 1, N), xm = wrap(x - 1, N);
    const int64_t yp = wrap(y + 1, N), ym = wrap(y - 1, N);
    const int64_t plane = (k.dims == 3) ? z * N * N : 0;
    const int64_t s = x + N * y + plane;
    const T c = phi[s];
    const T sx = phi[xp + N * y + plane] + phi[xm + N * y + plane];
    const T sy = phi[x + N * yp + plane] + phi[x + N * ym + plane];
    T sum = sx + sy;
    if (k.dims == 3) {
        const int64_t zp = wrap(z + 1, N), zm = wrap(z - 1, N);
        const T sz = phi[x + N * y + zp * N * N] + phi[x + N * y + zm * N * N];
        sum = sum + sz;
    }
    if (k.arith == PRS_REF_ARITH_FMA) {
        /* Contracted form (R13): the same formulas with every product that feeds a sum
         * evaluated as one fused multiply-add (a single rounding), which is what an OpenCL / CUDA
         * compiler emits from Eqs. 3-5 by default.  Coefficients A, B as in the COEF form. */
        const T lapf = std::fma(-T(2 * k.dims), c, sum);  /* Eq. 3:  sum - 2d c            */
        const T tf = std::fma(c * c, k.I, T(-1));         /* phi^2/phi0^2 - 1               */
        const T ff = std::fma((-k.K) * c, tf, lapf);      /* lap - (K c) t = lap - dV/dphi  */
        const T vf = std::fma(k.A, phidot[s], k.B * ff);  /* Eq. 4                          */
        *phidot_next = vf;
        *phi_next = std::fma(k.deta, vf, c);              /* Eq. 5                          */
        return;
    }
    const T lap = sum - T(2 * k.dims) * c;               /* Eq. 3 */
    const T q = c * c;
    const T r = q * k.I;
    const T t = r - T(1);
    const T dV = (k.K * c) * t;                           /* dV/dphi from Eq. 1 */
    const T f = lap - dV;
    const T pd = phidot[s];
    T pd_new;
    if (k.arith == PRS_REF_ARITH_LITERAL) {
        const T num = k.omd * pd + k.deta * f;            /* Eq. 4 */
        pd_new = num / k.opd;
    } else {
        pd_new = k.A * pd + k.B * f;                      /* Eq. 4, coefficients pre-divided */
    }
    *phidot_next = pd_new;
    *phi_next = c + k.deta * pd_new;                      /* Eq. 5 */
}

/* ---------------------------------------------------------------- diagnostics (S5, S6) */

template <typename T>
inline bool neg(T v) { return std::signbit(v); }

template <typename T>
void diagnostics_of(int dims, int64_t N, const T* phi, const T* phidot, double W0, double phi0,
                    prs_ref_diag* out) {
    const double V0 = (PI * PI * phi0 * phi0) / (2.0 * W0 * W0);
    const double I = 1.0 / (phi0 * phi0);
    const int64_t Nz = (dims == 3) ? N : 1;
    uint64_t links = 0, walls = 0;
    double sum = 0.0, comp = 0.0;                         /* Kahan, index order */
    for (int64_t z = 0; z < Nz; ++z)
        for (int64_t y = 0; y < N; ++y)
            for (int64_t x = 0; x < N; ++x) {
                const int64_t s = x + N * (y + N * z);
                const bool me = neg(phi[s]);
                const bool xp = neg(phi[wrap(x + 1, N) + N * (y + N * z)]) != me;
                const bool xm = neg(phi[wrap(x - 1, N) + N * (y + N * z)]) != me;
                const bool yp = neg(phi[x + N * (wrap(y + 1, N) + N * z)]) != me;
                const bool ym = neg(phi[x + N * (wrap(y - 1, N) + N * z)]) != me;
                bool zp = false, zm = false;
                if (dims == 3) {
                    zp = neg(phi[x + N * (y + N * wrap(z + 1, N))]) != me;
                    zm = neg(phi[x + N * (y + N * wrap(z - 1, N))]) != me;
                }
                /* each site owns its forward links (Eq. 7: sum over links of delta_pm) */
                links += (uint64_t)xp + (uint64_t)yp + (uint64_t)zp;
                if (xp || xm || yp || ym || zp || zm) {   /* grid point containing a wall */
                    walls += 1;
                    const double p = (double)phi[s], v = (double)phidot[s];
                    const double w = p * p * I - 1.0;
                    const double V = V0 * w * w;          /* Eq. 1 */
                    const double term = (V == 0.0) ? 0.0 : (v * v) / V;   /* Eq. 8 summand */
                    const double yk = term - comp;
                    const double tk = sum + yk;
                    comp = (tk - sum) - yk;
                    sum = tk;
                }
            }
    const double S = (dims == 3) ? (double)N * (double)N * (double)N : (double)N * (double)N;
    out->link_count = links;
    out->wall_sites = walls;
    out->sum_ratio = sum;
    out->rho = (double)links / S;
    out->gv2 = walls ? sum / (2.0 * (double)walls) : 0.0;
}

/* ---------------------------------------------------------------- orientation-weighted area (Eq. 7) */

/* PAPER.md Eq. 7 (:59-62) as printed: A/V = (Delta A / V) * sum over links of delta_pm *
 * |grad phi| / (|phi,x| + |phi,y| + |phi,z|) -- the PRS weight that corrects plain link counting for the
 * orientation of the wall (1 for a wall normal to an axis, 1/sqrt(d) for a fully diagonal one).
 * The paper does not say where on a link the gradient is taken (R15); the reading here, for
 * the link from s to s+e_k: along the link the forward difference phi(s+e_k) - phi(s); across it, for
 * each other axis t, the mean of the central differences (phi(u+e_t) - phi(u-e_t))/2 at the two end
 * points u = s, s+e_k.  Everything in double; weight := 1 if all components vanish.  The sum runs over
 * sites in index order, axes x, y, z within a site, with Kahan compensation. */
template <typename T>
double weighted_area_of(int dims, int64_t N, const T* phi) {
    const int64_t Nz = (dims == 3) ? N : 1;
    const int64_t stride[3] = {1, N, N * N};
    double sum = 0.0, comp = 0.0;
    for (int64_t z = 0; z < Nz; ++z)
        for (int64_t y = 0; y < N; ++y)
            for (int64_t x = 0; x < N; ++x) {
                const int64_t c[3] = {x, y, z};
                auto at = [&](const int64_t q[3]) {
                    return (double)phi[wrap(q[0], N) * stride[0] + wrap(q[1], N) * stride[1] +
                                       (dims == 3 ? wrap(q[2], N) * stride[2] : 0)];
                };
                for (int k = 0; k < dims; ++k) {
                    int64_t e[3] = {c[0], c[1], c[2]};               /* other end of the forward link */
                    e[k] += 1;
                    if (neg((T)at(c)) == neg((T)at(e))) continue;    /* delta_pm = 0 */
                    double g[3] = {0.0, 0.0, 0.0};
                    g[k] = at(e) - at(c);
                    for (int t = 0; t < dims; ++t) {
                        if (t == k) continue;
                        int64_t cp[3] = {c[0], c[1], c[2]}, cm[3] = {c[0], c[1], c[2]};
                        int64_t ep[3] = {e[0], e[1], e[2]}, em[3] = {e[0], e[1], e[2]};
                        cp[t] += 1; cm[t] -= 1; ep[t] += 1; em[t] -= 1;
                        const double dc = (at(cp) - at(cm)) / 2.0;   /* central difference at s       */
                        const double de = (at(ep) - at(em)) / 2.0;   /* central difference at s + e_k */
                        g[t] = (dc + de) / 2.0;
                    }
                    const double num = std::sqrt(g[0] * g[0] + g[1] * g[1] + g[2] * g[2]);
                    const double den = std::fabs(g[0]) + std::fabs(g[1]) + std::fabs(g[2]);
                    const double w = (den == 0.0) ? 1.0 : num / den;
                    const double yk = w - comp;
                    const double tk = sum + yk;
                    comp = (tk - sum) - yk;
                    sum = tk;
                }
            }
    return sum;
}

}  // namespace

/* ---------------------------------------------------------------- context */

struct prs_ref_ctx {
    int dims, precision, arith, threads;
    int64_t N, S, step;
    double alpha, era_m, deta, W0, phi0, eta0, beta;
    uint64_t seed;
    bool inited;
    std::vector<float> f_phi, f_pd, f_phi2, f_pd2;
    std::vector<double> d_phi, d_pd, d_phi2, d_pd2;
};

namespace {

template <typename T>
void step_once(prs_ref_ctx* h, std::vector<T>& phi, std::vector<T>& pd, std::vector<T>& phi2,
               std::vector<T>& pd2) {
    const Scalars sc = scalars_at(h->alpha, h->era_m, h->deta, h->W0, h->phi0, h->eta0, h->step, h->beta);
    const StepCoef<T> k = make_coef<T>(sc, h->deta, h->dims, h->arith);
    const int64_t N = h->N, Nz = (h->dims == 3) ? N : 1;
    const T* p = phi.data();
    const T* v = pd.data();
    T* pn = phi2.data();
    T* vn = pd2.data();
    /* Jacobi: every site reads step-n arrays and writes step-(n+1) arrays, so the outer loop may
     * be split over threads without changing a single bit. */
    const int64_t outer = Nz * N;
#ifdef _OPENMP
#pragma omp parallel for schedule(static) num_threads(h->threads) if (h->threads > 1)
#endif
    for (int64_t zy = 0; zy < outer; ++zy) {
        const int64_t z = zy / N, y = zy % N;
        for (int64_t x = 0; x < N; ++x) {
            const int64_t s = x + N * (y + N * z);
            site_update<T>(k, p, v, N, x, y, z, &pn[s], &vn[s]);
        }
    }
    phi.swap(phi2);
    pd.swap(pd2);
    h->step += 1;
}

template <typename T>
void fill_init(prs_ref_ctx* h, std::vector<T>& phi, std::vector<T>& pd) {
    for (int64_t s = 0; s < h->S; ++s) {
        phi[s] = (T)init_value(h->seed, (uint64_t)s, h->phi0);
        pd[s] = T(0);
    }
}

bool args_ok(int dims, int64_t N, int precision, double alpha, double era_m, double deta,
             double W0, double phi0) {
    if (dims != 2 && dims != 3) return false;
    if (N < 1) return false;
    if (precision != PRS_REF_F32 && precision != PRS_REF_F64) return false;
    if (!(deta > 0.0) || !(W0 > 0.0) || !(phi0 > 0.0)) return false;
    if (!(alpha >= 0.0) || !(era_m >= 0.0)) return false;
    return true;
}

}  // namespace

extern "C" {

int prs_ref_create(prs_ref_handle* out, int dims, int64_t N, int precision, double alpha,
                   double era_m, double deta, double W0, double phi0, uint64_t seed) {
    if (!out || !args_ok(dims, N, precision, alpha, era_m, deta, W0, phi0)) return 1;
    prs_ref_ctx* h = new (std::nothrow) prs_ref_ctx();
    if (!h) return 3;
    h->dims = dims; h->N = N; h->precision = precision;
    h->S = (dims == 3) ? N * N * N : N * N;
    h->alpha = alpha; h->era_m = era_m; h->deta = deta; h->W0 = W0; h->phi0 = phi0; h->beta = 0.0;
    h->seed = seed; h->arith = PRS_REF_ARITH_LITERAL; h->threads = 1;
    h->eta0 = 1.0; h->step = 0; h->inited = false;
    try {
        if (precision == PRS_REF_F32) {
            h->f_phi.resize(h->S); h->f_pd.resize(h->S); h->f_phi2.resize(h->S); h->f_pd2.resize(h->S);
        } else {
            h->d_phi.resize(h->S); h->d_pd.resize(h->S); h->d_phi2.resize(h->S); h->d_pd2.resize(h->S);
        }
    } catch (...) {
        delete h;
        return 3;
    }
    *out = h;
    return 0;
}

int prs_ref_destroy(prs_ref_handle h) {
    if (!h) return 1;
    delete h;
    return 0;
}

int prs_ref_set_beta(prs_ref_handle h, double beta) {
    if (!h || !std::isfinite(beta)) return 1;
    h->beta = beta;
    return 0;
}

int prs_ref_set_arith(prs_ref_handle h, int arith) {
    if (!h || (arith != PRS_REF_ARITH_LITERAL && arith != PRS_REF_ARITH_COEF && arith != PRS_REF_ARITH_FMA)) return 1;
    h->arith = arith;
    return 0;
}

int prs_ref_set_threads(prs_ref_handle h, int nthreads) {
    if (!h || nthreads < 1) return 1;
    h->threads = nthreads;
    return 0;
}

int prs_ref_init(prs_ref_handle h, double eta0) {
    if (!h || !(eta0 > 0.0)) return 1;
    if (h->precision == PRS_REF_F32) fill_init<float>(h, h->f_phi, h->f_pd);
    else fill_init<double>(h, h->d_phi, h->d_pd);
    h->eta0 = eta0; h->step = 0; h->inited = true;
    return 0;
}

int prs_ref_step(prs_ref_handle h, int64_t nsteps) {
    if (!h || nsteps < 0) return 1;
    if (!h->inited) return 4;
    for (int64_t i = 0; i < nsteps; ++i) {
        if (h->precision == PRS_REF_F32) step_once<float>(h, h->f_phi, h->f_pd, h->f_phi2, h->f_pd2);
        else step_once<double>(h, h->d_phi, h->d_pd, h->d_phi2, h->d_pd2);
    }
    return 0;
}

int prs_ref_diagnostics(prs_ref_handle h, prs_ref_diag* out) {
    if (!h || !out) return 1;
    if (!h->inited) return 4;
    prs_ref_diag d;
    if (h->precision == PRS_REF_F32)
        diagnostics_of<float>(h->dims, h->N, h->f_phi.data(), h->f_pd.data(), h->W0, h->phi0, &d);
    else
        diagnostics_of<double>(h->dims, h->N, h->d_phi.data(), h->d_pd.data(), h->W0, h->phi0, &d);
    d.step = h->step;
    d.eta = h->eta0 + (double)h->step * h->deta;
    *out = d;
    return 0;
}

int prs_ref_copy_out(prs_ref_handle h, void* phi_dst, void* phidot_dst) {
    if (!h) return 1;
    if (!h->inited) return 4;
    const size_t bytes = (size_t)h->S * (h->precision == PRS_REF_F32 ? 4 : 8);
    const void* p = h->precision == PRS_REF_F32 ? (const void*)h->f_phi.data() : (const void*)h->d_phi.data();
    const void* v = h->precision == PRS_REF_F32 ? (const void*)h->f_pd.data() : (const void*)h->d_pd.data();
    if (phi_dst) std::memcpy(phi_dst, p, bytes);
    if (phidot_dst) std::memcpy(phidot_dst, v, bytes);
    return 0;
}

int prs_ref_copy_in(prs_ref_handle h, const void* phi_src, const void* phidot_src, double eta0,
                    int64_t step) {
    if (!h || !phi_src || !phidot_src || !(eta0 > 0.0) || step < 0) return 1;
    const size_t bytes = (size_t)h->S * (h->precision == PRS_REF_F32 ? 4 : 8);
    void* p = h->precision == PRS_REF_F32 ? (void*)h->f_phi.data() : (void*)h->d_phi.data();
    void* v = h->precision == PRS_REF_F32 ? (void*)h->f_pd.data() : (void*)h->d_pd.data();
    std::memcpy(p, phi_src, bytes);
    std::memcpy(v, phidot_src, bytes);
    h->eta0 = eta0; h->step = step; h->inited = true;
    return 0;
}

void prs_ref_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    philox_block(ctr, key, out);
}

double prs_ref_init_value(uint64_t seed, uint64_t s, double phi0) {
    return init_value(seed, s, phi0);
}

int prs_ref_diagnostics_of(int dims, int64_t N, int precision, const void* phi, const void* phidot,
                           double W0, double phi0, prs_ref_diag* out) {
    if (!phi || !phidot || !out || !args_ok(dims, N, precision, 0.0, 0.0, 1.0, W0, phi0)) return 1;
    prs_ref_diag d;
    if (precision == PRS_REF_F32)
        diagnostics_of<float>(dims, N, (const float*)phi, (const float*)phidot, W0, phi0, &d);
    else
        diagnostics_of<double>(dims, N, (const double*)phi, (const double*)phidot, W0, phi0, &d);
    d.step = 0;
    d.eta = 0.0;
    *out = d;
    return 0;
}

int prs_ref_weighted_area_of(int dims, int64_t N, int precision, const void* phi, double* area) {
    if ((dims != 2 && dims != 3) || N < 1 || !phi || !area) return 1;
    if (precision == PRS_REF_F32) *area = weighted_area_of<float>(dims, N, (const float*)phi);
    else if (precision == PRS_REF_F64) *area = weighted_area_of<double>(dims, N, (const double*)phi);
    else return 1;
    return 0;
}

int prs_ref_step_sites(int dims, int64_t N, int precision, int arith, double alpha, double era_m,
                       double deta, double W0, double phi0, double eta0, int64_t n,
                       const void* phi, const void* phidot, const int64_t* sites, int64_t nsites,
                       void* phi_next_out, void* phidot_next_out) {
    if (!phi || !phidot || !sites || !phi_next_out || !phidot_next_out || nsites < 0 || n < 0 ||
        !(eta0 > 0.0) || !args_ok(dims, N, precision, alpha, era_m, deta, W0, phi0))
        return 1;
    if (arith != PRS_REF_ARITH_LITERAL && arith != PRS_REF_ARITH_COEF && arith != PRS_REF_ARITH_FMA) return 1;
    const Scalars sc = scalars_at(alpha, era_m, deta, W0, phi0, eta0, n);
    const int64_t S = (dims == 3) ? N * N * N : N * N;
    for (int64_t i = 0; i < nsites; ++i) {
        const int64_t s = sites[i];
        if (s < 0 || s >= S) return 1;
        const int64_t x = s % N, y = (s / N) % N, z = (dims == 3) ? s / (N * N) : 0;
        if (precision == PRS_REF_F32) {
            const StepCoef<float> k = make_coef<float>(sc, deta, dims, arith);
            site_update<float>(k, (const float*)phi, (const float*)phidot, N, x, y, z,
                               &((float*)phi_next_out)[i], &((float*)phidot_next_out)[i]);
        } else {
            const StepCoef<double> k = make_coef<double>(sc, deta, dims, arith);
            site_update<double>(k, (const double*)phi, (const double*)phidot, N, x, y, z,
                                &((double*)phi_next_out)[i], &((double*)phidot_next_out)[i]);
        }
    }
    return 0;
}

int prs_ref_scalars_beta(double alpha, double beta, double era_m, double deta, double W0, double phi0,
                         double eta0, int64_t n, double out[7]) {
    if (!out) return 1;
    const Scalars s = scalars_at(alpha, era_m, deta, W0, phi0, eta0, n, beta);
    out[0] = s.eta; out[1] = s.delta; out[2] = s.A; out[3] = s.B;
    out[4] = s.V0; out[5] = s.K; out[6] = s.I;
    return 0;
}

int prs_ref_scalars(double alpha, double era_m, double deta, double W0, double phi0, double eta0,
                    int64_t n, double out[7]) {
    if (!out) return 1;
    const Scalars s = scalars_at(alpha, era_m, deta, W0, phi0, eta0, n);
    out[0] = s.eta; out[1] = s.delta; out[2] = s.A; out[3] = s.B;
    out[4] = s.V0; out[5] = s.K; out[6] = s.I;
    return 0;
}

}  // extern "C"
