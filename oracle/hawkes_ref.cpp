// ORACLE -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, obviously-correct CPU implementation of the phylogenetic-Hawkes log-likelihood, its
// gradient and its Hessian terms, written from PAPER.md (arXiv 2103.03348) as the plain definition:
// direct double loops over (n, n') with std::exp / std::erfc / std::log / std::expm1, every pair's
// derivative taken from the pair's own log-density, long-double accumulation.  It shares no code,
// header, table or constant with the CUDA path under paper_2103_03348_b200/csrc/ and only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it.
//
// What is computed (citations are PAPER.md lines; "DESIGN Rk" = reading k listed in DESIGN.md):
//
//   lambda_n = sum_{n'} [ B_{nn'} + theta_{n'} k_{nn'} ]                         (Eq. 1, l.78)
//   B_{nn'}  = mu0 tau_x^-D tau_t^-1 phi_D((x_n-x_n')/tau_x) phi_1((t_n-t_n')/tau_t) I[x_n != x_n']
//              (l.60 background, with the Gaussian-in-time factor BASELINE.json's north_star adds:
//               DESIGN R1; phi_D = D-dim standard normal pdf, l.62)
//   k_{nn'}  = xi0 omega h^-D exp(-omega (t_n-t_n')) phi_D((x_n-x_n')/h) I[t_n' < t_n]   (l.60, 78)
//   ell      = sum_n log lambda_n - Lambda(t_N)                                   (Eq. 1, l.76)
//   Lambda   = mu0 sum_n [Phi((t_N-t_n)/tau_t) - Phi(-t_n/tau_t)]                 (DESIGN R1/R2)
//            + xi0 sum_n theta_n (1 - exp(-omega (t_N-t_n)))                      (l.72; Eq. 7, l.253)
//   dell/dtheta_m     = sum_{t_m<t_n} k_{nm}/lambda_n - xi0 (1 - e^{-omega (t_N-t_m)})   (Eq. 4, l.137)
//   d2ell/dtheta_m^2  = - sum_{t_m<t_n} (k_{nm}/lambda_n)^2      (Eq. 5, l.143, strict '<': DESIGN R5)
//   hyperparameter gradient / Hessian / theta-hyper cross block: derivative of the sum = sum of the
//   per-pair derivatives, each pair's taken from d log(term)/dp (the paper has none: DESIGN R6).
//
// Hyperparameter order: (mu0, tau_x, tau_t, xi0, h, omega).
//
// Pins: tests/test_oracle_pins.py (closed forms N=1,2; worked examples; quadrature of Lambda and of
// the spatial normalisation; central finite differences of every derivative; invariances; leave-one-
// out KDE special case against scikit-learn).  No function here is "parity unpinned".
//
// Build: g++ -O2 -fopenmp -shared -fPIC (oracle/build.py).  `threads` > 1 only parallelises the
// outer loop over rows; every per-row sum is computed by one thread in index order, and all sums
// over n are done serially afterwards, so results do not depend on `threads`.

#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

typedef long double ld;

const double kPi = 3.14159265358979323846264338327950288;

// Background mode.  0 = "ST" (default): Gaussian-space x Gaussian-time background, the model above (DESIGN R1).
// 1 = "S": the paper's background exactly as printed -- space only,
//   mu(x) = mu0 tau_x^-D sum_n phi_D((x - x_n)/tau_x) I[x != x_n]
//   with the integral term printed beside it, Lambda_background = mu0 t_N     (DESIGN R2: the print
//   does not integrate the printed mu(x) -- N unit-mass kernels give mu0 N t_N -- and is followed as printed).
// tau_t is then unused: every derivative with respect to it is 0.
// The mode is an argument of every entry point (`bg_mode`), carried in P: no process-global state.
struct P {
    double mu0, tau_x, tau_t, xi0, h, omega;
    double norm_b, norm_k;   // (2 pi)^-(D+1)/2 tau_x^-D tau_t^-1  and  (2 pi)^-D/2 h^-D
    int bg_mode;
};

P make_params(const double* q, int dim, int bg_mode) {
    P p = {q[0], q[1], q[2], q[3], q[4], q[5], 0.0, 0.0, bg_mode == 1 ? 1 : 0};
    p.norm_b = p.bg_mode == 1 ? std::pow(2.0 * kPi, -0.5 * dim) * std::pow(p.tau_x, -dim)
                              : std::pow(2.0 * kPi, -0.5 * (dim + 1)) * std::pow(p.tau_x, -dim) / p.tau_t;
    p.norm_k = std::pow(2.0 * kPi, -0.5 * dim) * std::pow(p.h, -dim);
    return p;
}

inline double std_normal_pdf(double z) { return std::exp(-0.5 * z * z) / std::sqrt(2.0 * kPi); }
inline double std_normal_cdf(double z) { return 0.5 * std::erfc(-z / std::sqrt(2.0)); }

// One ordered pair (target n, source m): squared distance, time lag, and the two rate terms.
struct Pair {
    double r2, dt;
    bool same_place;   // all coordinates compare equal (DESIGN R3)
    bool causal;       // t_m < t_n strictly (DESIGN R4)
};

inline Pair make_pair(int dim, int64_t N, const double* x, const double* t, int64_t n, int64_t m) {
    Pair q;
    q.r2 = 0.0;
    q.same_place = true;
    for (int d = 0; d < dim; ++d) {
        const double a = x[(int64_t)d * N + n], b = x[(int64_t)d * N + m];
        if (a != b) q.same_place = false;
        const double dx = a - b;
        q.r2 += dx * dx;
    }
    q.dt = t[n] - t[m];
    q.causal = t[m] < t[n];
    return q;
}

// Background term B_{nm} (without the indicator) and excitation kernel k_{nm} (theta-free, without
// the causal indicator), exactly as the formulas above read.
inline double background(const P& p, double r2, double dt) {
    if (p.bg_mode == 1) return p.mu0 * p.norm_b * std::exp(-r2 / (2.0 * p.tau_x * p.tau_x));
    return p.mu0 * p.norm_b * std::exp(-r2 / (2.0 * p.tau_x * p.tau_x) - dt * dt / (2.0 * p.tau_t * p.tau_t));
}
inline double excitation(const P& p, double r2, double dt) {
    return p.xi0 * p.omega * p.norm_k * std::exp(-p.omega * dt - r2 / (2.0 * p.h * p.h));
}
// d log B / dp and d2 log B / dp dq for p,q in (mu0, tau_x, tau_t);  log B = log mu0 - D log tau_x
// - log tau_t - r2/(2 tau_x^2) - dt^2/(2 tau_t^2) + const.  Off-diagonal second derivatives vanish.
inline void dlog_background(const P& p, int dim, double r2, double dt, double g[3], double h[3]) {
    g[0] = 1.0 / p.mu0;
    g[1] = r2 / (p.tau_x * p.tau_x * p.tau_x) - dim / p.tau_x;
    g[2] = dt * dt / (p.tau_t * p.tau_t * p.tau_t) - 1.0 / p.tau_t;
    h[0] = -1.0 / (p.mu0 * p.mu0);
    h[1] = -3.0 * r2 / (p.tau_x * p.tau_x * p.tau_x * p.tau_x) + dim / (p.tau_x * p.tau_x);
    h[2] = -3.0 * dt * dt / (p.tau_t * p.tau_t * p.tau_t * p.tau_t) + 1.0 / (p.tau_t * p.tau_t);
    if (p.bg_mode == 1) g[2] = h[2] = 0.0;   // space-only background: no tau_t
}
// same for k with (xi0, h, omega);  log k = log xi0 + log omega - D log h - omega dt - r2/(2h^2) + c.
inline void dlog_excitation(const P& p, int dim, double r2, double dt, double g[3], double h[3]) {
    g[0] = 1.0 / p.xi0;
    g[1] = r2 / (p.h * p.h * p.h) - dim / p.h;
    g[2] = 1.0 / p.omega - dt;
    h[0] = -1.0 / (p.xi0 * p.xi0);
    h[1] = -3.0 * r2 / (p.h * p.h * p.h * p.h) + dim / (p.h * p.h);
    h[2] = -1.0 / (p.omega * p.omega);
}

// Row n of the double sum: lambda_n, d lambda_n / dp (6) and d2 lambda_n / dp dq (6x6).
struct Row {
    ld lam;
    ld d1[6];
    ld d2[6][6];
};

void compute_row(const P& p, int dim, int64_t N, const double* x, const double* t, const double* theta,
                 int64_t n, bool derivs, Row* out) {
    Row r;
    std::memset(&r, 0, sizeof(r));
    for (int64_t m = 0; m < N; ++m) {
        const Pair q = make_pair(dim, N, x, t, n, m);
        if (!q.same_place) {
            const double b = background(p, q.r2, q.dt);
            r.lam += b;
            if (derivs) {
                double g[3], h[3];
                dlog_background(p, dim, q.r2, q.dt, g, h);
                for (int a = 0; a < 3; ++a) {
                    r.d1[a] += (ld)b * g[a];
                    for (int c = 0; c < 3; ++c)
                        r.d2[a][c] += (ld)b * ((ld)g[a] * g[c] + (a == c ? h[a] : 0.0));
                }
            }
        }
        if (q.causal) {
            const double s = theta[m] * excitation(p, q.r2, q.dt);
            r.lam += s;
            if (derivs) {
                double g[3], h[3];
                dlog_excitation(p, dim, q.r2, q.dt, g, h);
                for (int a = 0; a < 3; ++a) {
                    r.d1[3 + a] += (ld)s * g[a];
                    for (int c = 0; c < 3; ++c)
                        r.d2[3 + a][3 + c] += (ld)s * ((ld)g[a] * g[c] + (a == c ? h[a] : 0.0));
                }
            }
        }
    }
    *out = r;
}

// Integral term Lambda(t_N) (Eq. 7, l.253; background part per DESIGN R1/R2) and its first and second
// derivatives in the six hyperparameters: an O(N) sum, written once and used by hawkes_ref_eval and hawkes_ref_integral.
void integral_terms(const P& p, int64_t N, const double* t, const double* theta, ld* Lam_out, ld L1[6], ld L2[6][6]) {
    const double tN = t[N - 1];
    ld Lam = 0;
    for (int a = 0; a < 6; ++a) L1[a] = 0;
    std::memset(L2, 0, sizeof(ld) * 36);
    {
        ld sPhi = 0, sAphi = 0, sAphi2 = 0, sTh = 0, sThTE = 0, sThT2E = 0;
        for (int64_t i = 0; i < N; ++i) {
            const double a = (tN - t[i]) / p.tau_t, b = -t[i] / p.tau_t;
            sPhi += (ld)std_normal_cdf(a) - (ld)std_normal_cdf(b);
            sAphi += (ld)a * std_normal_pdf(a) - (ld)b * std_normal_pdf(b);
            sAphi2 += (ld)a * std_normal_pdf(a) * (2.0 - a * a) - (ld)b * std_normal_pdf(b) * (2.0 - b * b);
            const double T = tN - t[i];
            const double E = std::exp(-p.omega * T);
            sTh += (ld)theta[i] * (-std::expm1(-p.omega * T));
            sThTE += (ld)theta[i] * T * E;
            sThT2E += (ld)theta[i] * T * T * E;
        }
        if (p.bg_mode == 1) { sPhi = (ld)tN; sAphi = 0; sAphi2 = 0; }   // Lambda_background = mu0 t_N
        Lam = (ld)p.mu0 * sPhi + (ld)p.xi0 * sTh;
        L1[0] = sPhi;
        L1[2] = -(ld)p.mu0 / p.tau_t * sAphi;
        L1[3] = sTh;
        L1[5] = (ld)p.xi0 * sThTE;
        L2[0][2] = L2[2][0] = -sAphi / p.tau_t;
        L2[2][2] = (ld)p.mu0 / (p.tau_t * p.tau_t) * sAphi2;
        L2[3][5] = L2[5][3] = sThTE;
        L2[5][5] = -(ld)p.xi0 * sThT2E;
    }
    *Lam_out = Lam;
}

}  // namespace

extern "C" {

// Status: 0 ok; 1 some lambda_n == 0 (ell = -inf, entries dividing by it are NaN); <0 bad argument.
// All pointers are HOST pointers; any output may be NULL (= not wanted).
//   x[dim*n] SoA (x[d*n+i]), t[n] non-decreasing, theta[n], params[6] = (mu0,tau_x,tau_t,xi0,h,omega)
//   ll[1], integral[1] (= Lambda(t_N)), lambda[n], grad_theta[n], grad_hyper[6],
//   hess_theta_diag[n], hess_hyper[36] row-major, hess_cross[n*6] row-major (m, p),
//   hess_theta_dense[n*n] row-major (small n only; O(n^3)),
//   row_d1[n*6] row-major: d lambda_n / dp (intermediate, for error scales in the parity tests).
//   bg_mode: 0 = ST (default model), 1 = S (paper-literal space-only background), see above.
int hawkes_ref_eval(int64_t n, int dim, const double* x, const double* t, const double* theta,
                    const double* params, double* ll, double* integral, double* lambda,
                    double* grad_theta, double* grad_hyper, double* hess_theta_diag,
                    double* hess_hyper, double* hess_cross, double* hess_theta_dense, double* row_d1,
                    int threads, int bg_mode) {
    if (n < 1 || dim < 1 || dim > 3 || !x || !t || !theta || !params) return -1;
    for (int i = 0; i < 6; ++i)
        if (!(params[i] > 0.0) || !std::isfinite(params[i])) return -2;
    for (int64_t i = 1; i < n; ++i)
        if (t[i] < t[i - 1]) return -3;
    const P p = make_params(params, dim, bg_mode);
    const int64_t N = n;
    const bool want_hyper = grad_hyper || hess_hyper || hess_cross || row_d1;
    const bool want_cols = grad_theta || hess_theta_diag || hess_cross || hess_theta_dense;
    (void)threads;
#ifdef _OPENMP
    const int nthreads = threads > 0 ? threads : 1;
#endif

    // ---- phase 1: every row of the double sum (Alg. 1/2 step 1, l.690/791: "compute rates") ----
    std::vector<Row> rows(want_hyper ? N : 0);
    std::vector<ld> lam(N);
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 16) num_threads(nthreads)
#endif
    for (int64_t i = 0; i < N; ++i) {
        Row r;
        compute_row(p, dim, N, x, t, theta, i, want_hyper, &r);
        lam[i] = r.lam;
        if (want_hyper) rows[i] = r;
    }
    int status = 0;
    for (int64_t i = 0; i < N; ++i) {
        if (lam[i] == 0) status = 1;
        if (lambda) lambda[i] = (double)lam[i];
        if (row_d1)
            for (int a = 0; a < 6; ++a) row_d1[i * 6 + a] = (double)rows[i].d1[a];
    }

    // ---- integral Lambda(t_N) and its derivatives ----
    const double tN = t[N - 1];
    ld Lam = 0, L1[6], L2[6][6];
    integral_terms(p, N, t, theta, &Lam, L1, L2);
    if (integral) *integral = (double)Lam;

    // ---- log-likelihood (Eq. 1) ----
    if (ll) {
        ld s = 0;
        bool zero = false;
        for (int64_t i = 0; i < N; ++i) {
            if (lam[i] == 0) zero = true;
            else s += std::log(lam[i]);   // long-double log
        }
        *ll = zero ? -std::numeric_limits<double>::infinity() : (double)(s - Lam);
    }

    // ---- hyperparameter gradient and Hessian ----
    if (grad_hyper) {
        for (int a = 0; a < 6; ++a) {
            ld s = 0;
            for (int64_t i = 0; i < N; ++i) s += rows[i].d1[a] / lam[i];
            grad_hyper[a] = (double)(s - L1[a]);
        }
    }
    if (hess_hyper) {
        for (int a = 0; a < 6; ++a)
            for (int c = 0; c < 6; ++c) {
                ld s = 0;
                for (int64_t i = 0; i < N; ++i)
                    s += rows[i].d2[a][c] / lam[i] - rows[i].d1[a] * rows[i].d1[c] / (lam[i] * lam[i]);
                hess_hyper[a * 6 + c] = (double)(s - L2[a][c]);
            }
    }

    // ---- phase 2: column sums over later targets (Alg. 1/2 step 2, l.737/825) ----
    if (want_cols) {
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 16) num_threads(nthreads)
#endif
        for (int64_t m = 0; m < N; ++m) {
            ld c = 0, d = 0, cr[6] = {0, 0, 0, 0, 0, 0};
            for (int64_t i = 0; i < N; ++i) {
                const Pair q = make_pair(dim, N, x, t, i, m);   // target i, source m
                if (!q.causal) continue;
                const double k = excitation(p, q.r2, q.dt);
                const ld a = (ld)k / lam[i];
                c += a;
                d += a * a;
                if (hess_cross) {
                    double g[3], h[3];
                    dlog_excitation(p, dim, q.r2, q.dt, g, h);
                    for (int b = 0; b < 6; ++b)
                        cr[b] += a * ((b >= 3 ? (ld)g[b - 3] : (ld)0) - rows[i].d1[b] / lam[i]);
                }
            }
            const double T = tN - t[m];
            const double E = std::exp(-p.omega * T);
            if (grad_theta) grad_theta[m] = (double)(c - (ld)p.xi0 * (-std::expm1(-p.omega * T)));
            if (hess_theta_diag) hess_theta_diag[m] = (double)(-d);
            if (hess_cross) {
                cr[3] -= (ld)(-std::expm1(-p.omega * T));   // d/dxi0  of xi0 (1 - E_m)
                cr[5] -= (ld)p.xi0 * T * E;                  // d/domega of xi0 (1 - E_m)
                for (int b = 0; b < 6; ++b) hess_cross[m * 6 + b] = (double)cr[b];
            }
        }
        if (hess_theta_dense) {
            // d2 ell / dtheta_m dtheta_m' = - sum_n k_nm k_nm' / lambda_n^2 (Lambda is linear in theta)
            std::vector<double> A((size_t)N * N, 0.0);   // A[i][m] = k_im / lambda_i, causal only
            for (int64_t i = 0; i < N; ++i)
                for (int64_t m = 0; m < N; ++m) {
                    const Pair q = make_pair(dim, N, x, t, i, m);
                    if (q.causal) A[(size_t)i * N + m] = (double)((ld)excitation(p, q.r2, q.dt) / lam[i]);
                }
            for (int64_t m = 0; m < N; ++m)
                for (int64_t m2 = 0; m2 < N; ++m2) {
                    ld s = 0;
                    for (int64_t i = 0; i < N; ++i) s += (ld)A[(size_t)i * N + m] * A[(size_t)i * N + m2];
                    hess_theta_dense[(size_t)m * N + m2] = (double)(-s);
                }
        }
    }
    return status;
}

// Sampled evaluation for parity at sizes where the full oracle is too slow: the listed rows'
// lambda_n, d lambda_n/dp (row_d1[k*6+p]) and d2 lambda_n/dp dq (row_d2[k*36+p*6+q]), and the listed columns' c_m = sum_{t_m<t_n} k_nm/lambda_n
// and d_m = sum (k_nm/lambda_n)^2 given a full lambda vector supplied by the caller.
int hawkes_ref_rows(int64_t n, int dim, const double* x, const double* t, const double* theta,
                    const double* params, int64_t n_rows, const int64_t* rows_idx, double* row_lambda,
                    double* row_d1, double* row_d2, int threads, int bg_mode) {
    if (n < 1 || dim < 1 || dim > 3) return -1;
    const P p = make_params(params, dim, bg_mode);
    (void)threads;
#ifdef _OPENMP
    const int nthreads = threads > 0 ? threads : 1;
#pragma omp parallel for schedule(dynamic, 4) num_threads(nthreads)
#endif
    for (int64_t k = 0; k < n_rows; ++k) {
        Row r;
        compute_row(p, dim, n, x, t, theta, rows_idx[k], row_d1 != nullptr || row_d2 != nullptr, &r);
        row_lambda[k] = (double)r.lam;
        if (row_d1)
            for (int a = 0; a < 6; ++a) row_d1[k * 6 + a] = (double)r.d1[a];
        if (row_d2)
            for (int a = 0; a < 6; ++a)
                for (int c = 0; c < 6; ++c) row_d2[k * 36 + a * 6 + c] = (double)r.d2[a][c];
    }
    return 0;
}

int hawkes_ref_cols(int64_t n, int dim, const double* x, const double* t, const double* params,
                    const double* lambda, int64_t n_cols, const int64_t* cols_idx, double* col_c,
                    double* col_d, int threads) {
    if (n < 1 || dim < 1 || dim > 3) return -1;
    const P p = make_params(params, dim, 0);   // the excitation kernel does not depend on the background mode
    (void)threads;
#ifdef _OPENMP
    const int nthreads = threads > 0 ? threads : 1;
#pragma omp parallel for schedule(dynamic, 4) num_threads(nthreads)
#endif
    for (int64_t k = 0; k < n_cols; ++k) {
        const int64_t m = cols_idx[k];
        ld c = 0, d = 0;
        for (int64_t i = 0; i < n; ++i) {
            const Pair q = make_pair(dim, n, x, t, i, m);
            if (!q.causal) continue;
            const ld a = (ld)excitation(p, q.r2, q.dt) / (ld)lambda[i];
            c += a;
            d += a * a;
        }
        col_c[k] = (double)c;
        col_d[k] = (double)d;
    }
    return 0;
}

// Error scale of the cross block d2 ell / d theta_m dp ("the sum of the magnitudes of the terms"),
// for the parity tests only -- it is not an output of the method.  Entry (m, p) of the block is
//   sum_{n: t_n > t_m} a_nm [ d log k_nm / dp - lambda_{n,p} / lambda_n ] - Lambda_{theta_m p},   a_nm = k_nm / lambda_n,
// and this routine sums, over the same pairs, a_nm times the magnitudes of what the bracket is made of:
//   abs[m*6 + p] = sum_n a_nm ( T_p(n, m) + |lambda_{n,p}| / lambda_n ),
//   T = (0, 0, 0, 1/xi0, r^2/h^3 + D/h, 1/omega + dt)    -- the terms of d log k / d(xi0, h, omega), taken positive.
// row_d1[n*6 + p] = lambda_{n,p} as returned by hawkes_ref_eval.  The integral part and the terms inside lambda_{n,p}
// are added by the test.
int hawkes_ref_cross_abs(int64_t n, int dim, const double* x, const double* t, const double* params,
                         const double* lambda, const double* row_d1, double* abs_out, int threads) {
    if (n < 1 || dim < 1 || dim > 3 || !lambda || !row_d1 || !abs_out) return -1;
    const P p = make_params(params, dim, 0);
    (void)threads;
#ifdef _OPENMP
    const int nthreads = threads > 0 ? threads : 1;
#pragma omp parallel for schedule(dynamic, 16) num_threads(nthreads)
#endif
    for (int64_t m = 0; m < n; ++m) {
        ld s[6] = {0, 0, 0, 0, 0, 0};
        for (int64_t i = 0; i < n; ++i) {
            const Pair q = make_pair(dim, n, x, t, i, m);   // target i, source m
            if (!q.causal) continue;
            const ld a = (ld)excitation(p, q.r2, q.dt) / (ld)lambda[i];
            const ld T[6] = {0, 0, 0, (ld)1 / p.xi0, (ld)q.r2 / ((ld)p.h * p.h * p.h) + (ld)dim / p.h, (ld)1 / p.omega + q.dt};
            for (int b = 0; b < 6; ++b) s[b] += a * (T[b] + std::fabs((ld)row_d1[i * 6 + b]) / (ld)lambda[i]);
        }
        for (int b = 0; b < 6; ++b) abs_out[m * 6 + b] = (double)s[b];
    }
    return 0;
}

// Lambda(t_N) and its hyperparameter derivatives alone (O(N)): integral[1], d1[6], d2[36] row-major.
int hawkes_ref_integral(int64_t n, int dim, const double* t, const double* theta, const double* params,
                        double* integral, double* d1, double* d2, int bg_mode) {
    if (n < 1 || dim < 1 || dim > 3 || !t || !theta || !params) return -1;
    const P p = make_params(params, dim, bg_mode);
    ld Lam, L1[6], L2[6][6];
    integral_terms(p, n, t, theta, &Lam, L1, L2);
    if (integral) *integral = (double)Lam;
    for (int a = 0; a < 6; ++a) {
        if (d1) d1[a] = (double)L1[a];
        for (int c = 0; c < 6; ++c)
            if (d2) d2[a * 6 + c] = (double)L2[a][c];
    }
    return 0;
}

int hawkes_ref_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

}  // extern "C"
