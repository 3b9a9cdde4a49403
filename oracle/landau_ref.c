/*
 * landau_ref.c -- CPU ORACLE.  TEST INFRASTRUCTURE ONLY (see landau_ref.h).
 *
 * A plain, slow, literal restatement of the multispecies particle Landau scheme of
 * arXiv:2212.00663 in three velocity dimensions.  Double loops, libm exp/log/sqrt, long double
 * accumulators, summation in ascending marker index, no tiling, no separable-exponential trick,
 * no symmetry exploitation.  OpenMP only splits the OUTER loop over target markers.
 *
 * It shares no code with the CUDA path.  Each function cites the passage it follows
 * (PAPER.md:<line>, equation) and the DESIGN.md reading where the paper is silent or garbled.
 *
 * Parity pins (tests/test_oracle_*.py, -m "not gpu"): Gauss-Hermite closed forms and moment
 * identities; Q identities; single-marker closed form of G and S_eps; 2-V reduction (v_z = 0
 * reproduces the paper's own 2-V Eq. 22 written out independently); translation / reflection /
 * scaling laws; conservation identities Eq. 27, 29; entropy production Eq. 49; stationary
 * two-marker and collinear systems; brute-force numpy re-evaluation; 1-D integral limit.
 * No function here is "parity unpinned".
 */
#include "landau_ref.h"

#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define REF_PI 3.14159265358979323846264338327950288L
#define REF_MAX_NQ 16

struct landau_ref_ctx {
    int S;
    double* mass;
    double* charge;
    double* eps;
    double* nu; /* S x S */
    int n_q;
    double knots[REF_MAX_NQ];
    double weights[REF_MAX_NQ];
    /* markers held for stepping */
    int64_t N;
    double* v;
    double* w;
    int32_t* sid;
};

static int g_threads = 0;

int landau_ref_num_threads(void) {
#ifdef _OPENMP
    return g_threads > 0 ? g_threads : omp_get_max_threads();
#else
    return 1;
#endif
}

void landau_ref_set_num_threads(int n) {
    g_threads = n;
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#endif
}

/* ------------------------------------------------------------------------------------------
 * O1  Gauss-Hermite rule for the weight exp(-k^2)   ("Gauss-Hermite
 * quadrature ... constructed as an outer product of ... one-dimensional" rules).
 *
 * Textbook construction with the ORTHONORMAL Hermite polynomials h_j:
 *     h_0 = pi^(-1/4),  h_{j+1}(x) = x sqrt(2/(j+1)) h_j(x) - sqrt(j/(j+1)) h_{j-1}(x).
 * The knots are the roots of h_n; they interlace the roots of h_{n-1}, so they are found by
 * bisection between consecutive roots of the previous degree (plus outer bounds), then polished
 * by Newton with h_n' = sqrt(2n) h_{n-1}.  Weights are the Christoffel numbers
 *     a_i = 1 / sum_{j<n} h_j(k_i)^2.
 * ------------------------------------------------------------------------------------------ */
static long double hermite_orthonormal(int n, long double x, long double* all /* n+1 values or NULL */) {
    long double hm = 0.0L;
    long double h = 1.0L / sqrtl(sqrtl(REF_PI));
    if (all) all[0] = h;
    for (int j = 0; j < n; ++j) {
        long double hn = x * sqrtl(2.0L / (j + 1)) * h - sqrtl((long double)j / (j + 1)) * hm;
        hm = h;
        h = hn;
        if (all) all[j + 1] = h;
    }
    return h;
}

int landau_ref_gauss_hermite(int n, double* knots, double* weights) {
    if (n < 1 || n > REF_MAX_NQ || !knots || !weights) return -1;
    long double prev[REF_MAX_NQ + 2], cur[REF_MAX_NQ + 2];
    int nprev = 0;
    for (int deg = 1; deg <= n; ++deg) {
        long double bound = sqrtl(2.0L * deg + 1.0L) + 1.0L; /* all roots lie inside (-bound, bound) */
        for (int i = 0; i < deg; ++i) {
            long double lo = (i == 0) ? -bound : prev[i - 1];
            long double hi = (i == deg - 1) ? bound : prev[i];
            long double flo = hermite_orthonormal(deg, lo, NULL);
            for (int it = 0; it < 200; ++it) {
                long double mid = 0.5L * (lo + hi);
                long double fm = hermite_orthonormal(deg, mid, NULL);
                if ((fm < 0) == (flo < 0)) { lo = mid; flo = fm; } else { hi = mid; }
            }
            long double x = 0.5L * (lo + hi);
            for (int it = 0; it < 4; ++it) { /* Newton polish */
                long double f = hermite_orthonormal(deg, x, NULL);
                long double fp = sqrtl(2.0L * deg) * hermite_orthonormal(deg - 1, x, NULL);
                x -= f / fp;
            }
            cur[i] = x;
        }
        if (deg % 2 == 1) cur[deg / 2] = 0.0L; /* odd degree: the middle root is exactly 0 */
        for (int i = 0; i < deg; ++i) prev[i] = cur[i];
        nprev = deg;
    }
    (void)nprev;
    for (int i = 0; i < n; ++i) {
        long double all[REF_MAX_NQ + 2];
        hermite_orthonormal(n, prev[i], all);
        long double s = 0.0L;
        for (int j = 0; j < n; ++j) s += all[j] * all[j];
        knots[i] = (double)prev[i];
        weights[i] = (double)(1.0L / s);
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------ */

static int check_markers(const landau_ref_ctx* c, int64_t N, const double* v, const double* w,
                         const int32_t* sid) {
    if (!c || N < 1 || !v || !w || !sid) return -1;
    for (int64_t p = 0; p < N; ++p) {
        if (sid[p] < 0 || sid[p] >= c->S) return -1;
        if (!isfinite(w[p]) || !isfinite(v[3 * p]) || !isfinite(v[3 * p + 1]) || !isfinite(v[3 * p + 2]))
            return -4;
        if (!(w[p] > 0.0)) return -1;
    }
    return 0;
}

int landau_ref_create(landau_ref_ctx** out, int S, const double* mass, const double* charge,
                      const double* eps, int n_q, double nu0, const double* nu) {
    if (!out || S < 1 || !mass || !charge || !eps || n_q < 1 || n_q > REF_MAX_NQ) return -1;
    for (int s = 0; s < S; ++s)
        if (!(mass[s] > 0.0) || !(eps[s] > 0.0) || !isfinite(charge[s])) return -1;
    landau_ref_ctx* c = (landau_ref_ctx*)calloc(1, sizeof(*c));
    if (!c) return -2;
    c->S = S;
    c->n_q = n_q;
    c->mass = (double*)malloc(sizeof(double) * S);
    c->charge = (double*)malloc(sizeof(double) * S);
    c->eps = (double*)malloc(sizeof(double) * S);
    c->nu = (double*)malloc(sizeof(double) * S * S);
    if (!c->mass || !c->charge || !c->eps || !c->nu) { landau_ref_destroy(c); return -2; }
    memcpy(c->mass, mass, sizeof(double) * S);
    memcpy(c->charge, charge, sizeof(double) * S);
    memcpy(c->eps, eps, sizeof(double) * S);
    for (int s = 0; s < S; ++s)
        for (int t = 0; t < S; ++t) {
            /* PAPER.md:37  nu_ss' = e_s^2 e_s'^2 lnLambda/(8 pi eps0^2); reading U1: normalised
             * units, nu_ss' = nu0 q_s^2 q_s'^2 unless an explicit symmetric matrix is given. */
            double val = nu ? nu[s * S + t] : nu0 * charge[s] * charge[s] * charge[t] * charge[t];
            c->nu[s * S + t] = val;
        }
    for (int s = 0; s < S; ++s)
        for (int t = 0; t < S; ++t)
            if (c->nu[s * S + t] != c->nu[t * S + s] || !isfinite(c->nu[s * S + t])) {
                landau_ref_destroy(c);
                return -1;
            }
    if (landau_ref_gauss_hermite(n_q, c->knots, c->weights) != 0) { landau_ref_destroy(c); return -1; }
    *out = c;
    return 0;
}

void landau_ref_destroy(landau_ref_ctx* c) {
    if (!c) return;
    free(c->mass); free(c->charge); free(c->eps); free(c->nu);
    free(c->v); free(c->w); free(c->sid);
    free(c);
}

/* ------------------------------------------------------------------------------------------
 * O2  Entropy gradient, 3-V restatement of Eq. (22).
 *
 * With the Gaussian mollifier of covariance eps_s I (Eq. 19 in d = 3:
 * psi_eps(v) = (2 pi eps)^(-3/2) exp(-|v|^2/(2 eps))) and the substitution
 * v = v_p + sqrt(2 eps_s) k in Eq. (21):
 *
 *   rho_p(k) = sum_{p' in s(p)} w_p' (2 pi eps_s)^(-3/2) exp(-| k + (v_p - v_p')/sqrt(2 eps_s) |^2)
 *   dS_eps/dv_p = - w_p sqrt(2/eps_s) pi^(-3/2) sum_{ijl} a_i a_j a_l k_ijl [1 + ln rho_p(k_ijl)]
 *   G_p = (1/w_p) dS_eps/dv_p                                              (Eq. 14)
 *   S_eps,s = - pi^(-3/2) sum_{p in s} w_p sum_{ijl} a_i a_j a_l ln rho_p(k_ijl)   (Eq. 20)
 *
 * (d = 2 gives the paper's prefactor w_p sqrt(2 eps_s)/(pi eps_s).)  Readings:
 * S1 the inner sum runs over the SAME species with eps_s; S2 a = weights, k = knots; S4 the
 * self term p' = p is included.
 * ------------------------------------------------------------------------------------------ */
static void entropy_grad_one(const landau_ref_ctx* c, int64_t N, const double* v, const double* w,
                             const int32_t* sid, int64_t p, double G[3], long double* s_node_sum) {
    const int s = sid[p];
    const int nq = c->n_q;
    const double eps = c->eps[s];
    const double sq = sqrt(2.0 * eps);
    const double norm = pow(2.0 * (double)REF_PI * eps, -1.5);
    long double gx = 0.0L, gy = 0.0L, gz = 0.0L, ssum = 0.0L;
    for (int i = 0; i < nq; ++i)
        for (int j = 0; j < nq; ++j)
            for (int l = 0; l < nq; ++l) {
                const double kx = c->knots[i], ky = c->knots[j], kz = c->knots[l];
                long double rho = 0.0L;
                for (int64_t q = 0; q < N; ++q) {
                    if (sid[q] != s) continue;
                    const double dx = kx + (v[3 * p] - v[3 * q]) / sq;
                    const double dy = ky + (v[3 * p + 1] - v[3 * q + 1]) / sq;
                    const double dz = kz + (v[3 * p + 2] - v[3 * q + 2]) / sq;
                    rho += (long double)(w[q] * norm * exp(-(dx * dx + dy * dy + dz * dz)));
                }
                const long double lnrho = logl(rho);
                const long double aaa = (long double)c->weights[i] * c->weights[j] * c->weights[l];
                gx += aaa * kx * (1.0L + lnrho);
                gy += aaa * ky * (1.0L + lnrho);
                gz += aaa * kz * (1.0L + lnrho);
                ssum += aaa * lnrho;
            }
    const long double pref = -sqrtl(2.0L / eps) / (REF_PI * sqrtl(REF_PI));
    G[0] = (double)(pref * gx);
    G[1] = (double)(pref * gy);
    G[2] = (double)(pref * gz);
    if (s_node_sum) *s_node_sum = ssum;
}

int landau_ref_entropy_grad(landau_ref_ctx* c, int64_t N, const double* v, const double* w,
                            const int32_t* sid, double* G_out, double* S_eps_out) {
    int rc = check_markers(c, N, v, w, sid);
    if (rc) return rc;
    if (!G_out) return -1;
    long double* node_sum = (long double*)malloc(sizeof(long double) * (size_t)N);
    if (!node_sum) return -2;
#pragma omp parallel for schedule(dynamic, 8)
    for (int64_t p = 0; p < N; ++p) entropy_grad_one(c, N, v, w, sid, p, &G_out[3 * p], &node_sum[p]);
    if (S_eps_out) {
        for (int s = 0; s < c->S; ++s) {
            long double acc = 0.0L;
            for (int64_t p = 0; p < N; ++p)
                if (sid[p] == s) acc += (long double)w[p] * node_sum[p];
            S_eps_out[s] = (double)(-acc / (REF_PI * sqrtl(REF_PI)));
        }
    }
    free(node_sum);
    for (int64_t i = 0; i < 3 * N; ++i)
        if (!isfinite(G_out[i])) return -4;
    return 0;
}

int landau_ref_entropy_grad_rows(landau_ref_ctx* c, int64_t N, const double* v, const double* w,
                                 const int32_t* sid, int64_t n_rows, const int64_t* rows, double* G_out) {
    int rc = check_markers(c, N, v, w, sid);
    if (rc) return rc;
    if (!G_out || !rows || n_rows < 0) return -1;
    for (int64_t r = 0; r < n_rows; ++r)
        if (rows[r] < 0 || rows[r] >= N) return -1;
#pragma omp parallel for schedule(dynamic, 8)
    for (int64_t r = 0; r < n_rows; ++r) entropy_grad_one(c, N, v, w, sid, rows[r], &G_out[3 * r], NULL);
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * O3  Field, Eq. (23) with Q of Eq. (4), Gamma^h of Eq. (16)
 * (reading S6: w_n, v_n are typos for w_p, v_p) and W^h of Eq. (17):
 *
 *   V_p = (1/m_s) sum_{s'} sum_{p' in s'} w_p' nu_ss' Q(v_p - v_p') . Gamma(p,p')
 *   Gamma(p,p') = G_p/m_s - G_p'/m_s'
 *   Q(xi) = (1/|xi|) (I - xi xi/|xi|^2)
 *
 * Reading S5: a pair with |v_p - v_p'|^2 == 0 (this includes p' = p) contributes 0; no softening.
 * ------------------------------------------------------------------------------------------ */
static void pair_field_one(const landau_ref_ctx* c, int64_t N, const double* v, const double* w,
                           const int32_t* sid, const double* G, int64_t p, double V[3]) {
    const int s = sid[p];
    const double ms = c->mass[s];
    long double ax = 0.0L, ay = 0.0L, az = 0.0L;
    for (int64_t q = 0; q < N; ++q) {
        const int sb = sid[q];
        const double xi0 = v[3 * p] - v[3 * q];
        const double xi1 = v[3 * p + 1] - v[3 * q + 1];
        const double xi2 = v[3 * p + 2] - v[3 * q + 2];
        const double r2 = xi0 * xi0 + xi1 * xi1 + xi2 * xi2;
        if (r2 == 0.0) continue;
        const double mb = c->mass[sb];
        const double g0 = G[3 * p] / ms - G[3 * q] / mb;
        const double g1 = G[3 * p + 1] / ms - G[3 * q + 1] / mb;
        const double g2 = G[3 * p + 2] / ms - G[3 * q + 2] / mb;
        const double r = sqrt(r2);
        const double xg = (xi0 * g0 + xi1 * g1 + xi2 * g2) / r2;
        /* Q . Gamma = (Gamma - xi (xi . Gamma)/|xi|^2) / |xi| */
        const double f = w[q] * c->nu[s * c->S + sb];
        ax += (long double)(f * (g0 - xi0 * xg) / r);
        ay += (long double)(f * (g1 - xi1 * xg) / r);
        az += (long double)(f * (g2 - xi2 * xg) / r);
    }
    V[0] = (double)(ax / ms);
    V[1] = (double)(ay / ms);
    V[2] = (double)(az / ms);
}

int landau_ref_pair_field(landau_ref_ctx* c, int64_t N, const double* v, const double* w,
                          const int32_t* sid, const double* G_in, double* out) {
    int rc = check_markers(c, N, v, w, sid);
    if (rc) return rc;
    if (!G_in || !out) return -1;
    for (int64_t i = 0; i < 3 * N; ++i)
        if (!isfinite(G_in[i])) return -4;
#pragma omp parallel for schedule(static)
    for (int64_t p = 0; p < N; ++p) pair_field_one(c, N, v, w, sid, G_in, p, &out[3 * p]);
    for (int64_t i = 0; i < 3 * N; ++i)
        if (!isfinite(out[i])) return -4;
    return 0;
}

int landau_ref_pair_field_rows(landau_ref_ctx* c, int64_t N, const double* v, const double* w,
                               const int32_t* sid, const double* G_in, int64_t n_rows,
                               const int64_t* rows, double* out) {
    int rc = check_markers(c, N, v, w, sid);
    if (rc) return rc;
    if (!G_in || !out || !rows || n_rows < 0) return -1;
    for (int64_t r = 0; r < n_rows; ++r)
        if (rows[r] < 0 || rows[r] >= N) return -1;
#pragma omp parallel for schedule(static)
    for (int64_t r = 0; r < n_rows; ++r) pair_field_one(c, N, v, w, sid, G_in, rows[r], &out[3 * r]);
    return 0;
}

int landau_ref_eval_field(landau_ref_ctx* c, int64_t N, const double* v, const double* w,
                          const int32_t* sid, double* out) {
    if (!out || N < 1) return -1;
    double* G = (double*)malloc(sizeof(double) * 3 * (size_t)N);
    if (!G) return -2;
    int rc = landau_ref_entropy_grad(c, N, v, w, sid, G, NULL);
    if (rc == 0) rc = landau_ref_pair_field(c, N, v, w, sid, G, out);
    free(G);
    return rc;
}

/* ------------------------------------------------------------------------------------------ */

int landau_ref_set_markers(landau_ref_ctx* c, int64_t N, const double* v, const double* w,
                           const int32_t* sid) {
    int rc = check_markers(c, N, v, w, sid);
    if (rc) return rc;
    double* nv = (double*)malloc(sizeof(double) * 3 * (size_t)N);
    double* nw = (double*)malloc(sizeof(double) * (size_t)N);
    int32_t* ns = (int32_t*)malloc(sizeof(int32_t) * (size_t)N);
    if (!nv || !nw || !ns) { free(nv); free(nw); free(ns); return -2; }
    memcpy(nv, v, sizeof(double) * 3 * (size_t)N);
    memcpy(nw, w, sizeof(double) * (size_t)N);
    memcpy(ns, sid, sizeof(int32_t) * (size_t)N);
    free(c->v); free(c->w); free(c->sid);
    c->v = nv; c->w = nw; c->sid = ns; c->N = N;
    return 0;
}

int landau_ref_get_markers(landau_ref_ctx* c, double* v_out) {
    if (!c || !c->v || !v_out) return -1;
    memcpy(v_out, c->v, sizeof(double) * 3 * (size_t)c->N);
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * O4  Step, Eq. (24)-(25)  (Algorithm 1).
 *
 *   G^n = O2(v^n)                       (entropy "with respect to time n")
 *   v^(0) = v^n
 *   repeat: u = (v^n + v^(k))/2         (Eq. 25)
 *           V = O3(u; G^n)              (Eq. 24 right-hand side)
 *           v^(k+1) = v^n + dt V        (Jacobi: every marker updated from the same iterate)
 *           r_k = sqrt( sum w m |v^(k+1)-v^(k)|^2 / sum w m |v^(k+1)|^2 )
 *   until r_k <= tol or k+1 == max_iter.
 * Reading S7 (Jacobi, start at v^n, energy-weighted relative increment), S8 (a non-converged
 * step is committed and reported with status 1).
 * ------------------------------------------------------------------------------------------ */
int landau_ref_step(landau_ref_ctx* c, double dt, double tol, int max_iter, landau_ref_step_info* info) {
    if (!c || !c->v || max_iter < 1 || !(dt > 0.0) || !(tol >= 0.0)) return -1;
    const int64_t N = c->N;
    double* G = (double*)malloc(sizeof(double) * 3 * (size_t)N);
    double* vk = (double*)malloc(sizeof(double) * 3 * (size_t)N);
    double* u = (double*)malloc(sizeof(double) * 3 * (size_t)N);
    double* V = (double*)malloc(sizeof(double) * 3 * (size_t)N);
    if (!G || !vk || !u || !V) { free(G); free(vk); free(u); free(V); return -2; }
    int rc = landau_ref_entropy_grad(c, N, c->v, c->w, c->sid, G, NULL);
    int iters = 0, converged = 0;
    double res = INFINITY;
    if (rc == 0) {
        memcpy(vk, c->v, sizeof(double) * 3 * (size_t)N);
        for (int k = 0; k < max_iter; ++k) {
            for (int64_t i = 0; i < 3 * N; ++i) u[i] = 0.5 * (c->v[i] + vk[i]);
            rc = landau_ref_pair_field(c, N, u, c->w, c->sid, G, V);
            if (rc) break;
            long double num = 0.0L, den = 0.0L;
            for (int64_t p = 0; p < N; ++p) {
                const long double wm = (long double)c->w[p] * c->mass[c->sid[p]];
                for (int d = 0; d < 3; ++d) {
                    const double vn = c->v[3 * p + d] + dt * V[3 * p + d];
                    const long double diff = (long double)vn - vk[3 * p + d];
                    num += wm * diff * diff;
                    den += wm * (long double)vn * vn;
                    vk[3 * p + d] = vn;
                }
            }
            res = (double)sqrtl(num / den);
            iters = k + 1;
            if (!isfinite(res)) { rc = -4; break; }
            if (res <= tol) { converged = 1; break; }
        }
    }
    if (rc == 0) memcpy(c->v, vk, sizeof(double) * 3 * (size_t)N);
    free(G); free(vk); free(u); free(V);
    if (info) { info->iterations = iters; info->residual = res; info->converged = converged; }
    if (rc) return rc;
    return converged ? 0 : 1;
}

/* ------------------------------------------------------------------------------------------
 * O4b  Discrete-gradient step, Eqs. (46)-(49), SURVEY.md NEXT-1.
 *   Gamma(K, p, q): the discrete gradient of the quadratic K is its midpoint gradient,
 *       (1/(m_s w_p)) dK/dv_p = (v_p^n + v_p^{n+1})/2 = u_p, so Q is evaluated at u_p - u_q as in Eq. (24).
 *   Gamma(S_eps, p, q): the paper leaves the discrete gradient open ("many existing options"); reading
 *   DG1 takes Gonzalez' midpoint discrete gradient (the paper's ref. [39]) in the Euclidean
 *   inner product of all 3N velocity components:
 *       dbar S/dv_p = w_p G_p(u) + lambda (v_p^{n+1} - v_p^n),
 *       lambda = [ S(v^{n+1}) - S(v^n) - sum_p w_p G_p(u).(v_p^{n+1} - v_p^n) ] / sum_p |v_p^{n+1} - v_p^n|^2
 *   (lambda = 0 when v^{n+1} = v^n), which satisfies Eq. (48) identically; S = sum_s S_eps,s.
 *   The step solves  v^{n+1} = v^n + dt * O3(u; Gbar),  Gbar_p = (1/w_p) dbar S/dv_p,  by the Jacobi
 *   fixed point of O4 with Gbar re-evaluated from (v^n, v^(k)) in every iteration.
 * ------------------------------------------------------------------------------------------ */
int landau_ref_step_dg(landau_ref_ctx* c, double dt, double tol, int max_iter, landau_ref_step_info* info) {
    if (!c || !c->v || max_iter < 1 || !(dt > 0.0) || !(tol >= 0.0)) return -1;
    const int64_t N = c->N;
    const size_t B3 = sizeof(double) * 3 * (size_t)N;
    double* G = (double*)malloc(B3);
    double* Gb = (double*)malloc(B3);
    double* vk = (double*)malloc(B3);
    double* u = (double*)malloc(B3);
    double* V = (double*)malloc(B3);
    double Ss[64];
    if (!G || !Gb || !vk || !u || !V || c->S > 64) { free(G); free(Gb); free(vk); free(u); free(V); return -2; }
    int rc = landau_ref_entropy_grad(c, N, c->v, c->w, c->sid, G, Ss);
    long double S0 = 0.0L;
    for (int s = 0; s < c->S; ++s) S0 += Ss[s];
    int iters = 0, converged = 0;
    double res = INFINITY;
    if (rc == 0) {
        memcpy(vk, c->v, B3);
        for (int k = 0; k < max_iter; ++k) {
            for (int64_t i = 0; i < 3 * N; ++i) u[i] = 0.5 * (c->v[i] + vk[i]);
            long double lambda = 0.0L;
            if (k > 0) {
                rc = landau_ref_entropy_grad(c, N, u, c->w, c->sid, G, NULL);          /* G(u)      */
                if (rc) break;
                rc = landau_ref_entropy_grad(c, N, vk, c->w, c->sid, Gb, Ss);           /* S(v^(k))  */
                if (rc) break;
                long double Sk = 0.0L, lin = 0.0L, dv2 = 0.0L;
                for (int s = 0; s < c->S; ++s) Sk += Ss[s];
                for (int64_t p = 0; p < N; ++p)
                    for (int d = 0; d < 3; ++d) {
                        const long double dv = (long double)vk[3 * p + d] - c->v[3 * p + d];
                        lin += (long double)c->w[p] * G[3 * p + d] * dv;
                        dv2 += dv * dv;
                    }
                if (dv2 > 0.0L) lambda = (Sk - S0 - lin) / dv2;
            }
            for (int64_t p = 0; p < N; ++p)
                for (int d = 0; d < 3; ++d)
                    Gb[3 * p + d] = (double)(G[3 * p + d]
                                             + lambda * ((long double)vk[3 * p + d] - c->v[3 * p + d]) / c->w[p]);
            rc = landau_ref_pair_field(c, N, u, c->w, c->sid, Gb, V);
            if (rc) break;
            long double num = 0.0L, den = 0.0L;
            for (int64_t p = 0; p < N; ++p) {
                const long double wm = (long double)c->w[p] * c->mass[c->sid[p]];
                for (int d = 0; d < 3; ++d) {
                    const double vn = c->v[3 * p + d] + dt * V[3 * p + d];
                    const long double diff = (long double)vn - vk[3 * p + d];
                    num += wm * diff * diff;
                    den += wm * (long double)vn * vn;
                    vk[3 * p + d] = vn;
                }
            }
            res = (double)sqrtl(num / den);
            iters = k + 1;
            if (!isfinite(res)) { rc = -4; break; }
            if (res <= tol) { converged = 1; break; }
        }
    }
    if (rc == 0) memcpy(c->v, vk, B3);
    free(G); free(Gb); free(vk); free(u); free(V);
    if (info) { info->iterations = iters; info->residual = res; info->converged = converged; }
    if (rc) return rc;
    return converged ? 0 : 1;
}

/* ------------------------------------------------------------------------------------------
 * O5  Moments (PAPER.md:151 Eq. 26, :162 Eq. 28, :191-193 Eq. 33, :118 Eq. 20):
 *   n_s = sum w_p,  P_s = m_s sum w_p v_p,  K_s = (m_s/2) sum w_p |v_p|^2,  S_eps,s as in O2.
 * ------------------------------------------------------------------------------------------ */
int landau_ref_moments(landau_ref_ctx* c, double* n, double* P, double* K, double* S_eps) {
    if (!c || !c->v) return -1;
    const int64_t N = c->N;
    for (int s = 0; s < c->S; ++s) {
        long double ns = 0, px = 0, py = 0, pz = 0, ks = 0;
        for (int64_t p = 0; p < N; ++p) {
            if (c->sid[p] != s) continue;
            const long double w = c->w[p];
            const long double x = c->v[3 * p], y = c->v[3 * p + 1], z = c->v[3 * p + 2];
            ns += w; px += w * x; py += w * y; pz += w * z;
            ks += w * (x * x + y * y + z * z);
        }
        if (n) n[s] = (double)ns;
        if (P) { P[3 * s] = (double)(c->mass[s] * px); P[3 * s + 1] = (double)(c->mass[s] * py); P[3 * s + 2] = (double)(c->mass[s] * pz); }
        if (K) K[s] = (double)(0.5L * c->mass[s] * ks);
    }
    if (S_eps) {
        double* G = (double*)malloc(sizeof(double) * 3 * (size_t)N);
        if (!G) return -2;
        int rc = landau_ref_entropy_grad(c, N, c->v, c->w, c->sid, G, S_eps);
        free(G);
        if (rc) return rc;
    }
    return 0;
}

int landau_ref_moments_ext(landau_ref_ctx* c, double* stress, double* m4) {
    if (!c || !c->v) return -1;
    const int64_t N = c->N;
    for (int s = 0; s < c->S; ++s) {
        long double ns = 0, ux = 0, uy = 0, uz = 0;
        long double t[6] = {0, 0, 0, 0, 0, 0};
        for (int64_t p = 0; p < N; ++p) {
            if (c->sid[p] != s) continue;
            const long double w = c->w[p];
            const long double x = c->v[3 * p], y = c->v[3 * p + 1], z = c->v[3 * p + 2];
            ns += w; ux += w * x; uy += w * y; uz += w * z;
            t[0] += w * x * x; t[1] += w * y * y; t[2] += w * z * z;
            t[3] += w * x * y; t[4] += w * x * z; t[5] += w * y * z;
        }
        if (stress) for (int i = 0; i < 6; ++i) stress[6 * s + i] = (double)(c->mass[s] * t[i]);
        if (m4) {
            long double q[3] = {0, 0, 0};
            if (ns > 0) { ux /= ns; uy /= ns; uz /= ns; }
            for (int64_t p = 0; p < N; ++p) {
                if (c->sid[p] != s) continue;
                const long double w = c->w[p];
                const long double dx = c->v[3 * p] - ux, dy = c->v[3 * p + 1] - uy, dz = c->v[3 * p + 2] - uz;
                q[0] += w * dx * dx * dx * dx; q[1] += w * dy * dy * dy * dy; q[2] += w * dz * dz * dz * dz;
            }
            for (int i = 0; i < 3; ++i) m4[3 * s + i] = (double)q[i];
        }
    }
    return 0;
}
