// stiff_pairs.cuh -- exact local treatment of stiff two-marker interactions inside the implicit step (SURVEY.md
// section 8(f) NEXT-4; "a local implicit treatment of the few stiff close ... pairs").
//
// Why the paper's fixed point "is unable to fully converge on occasion".  The pair term of
// Eq. (23), c Q(z) Gamma with Q(z) = (|z|^2 I - z z^T)/|z|^3, is not Lipschitz at z = 0: for two markers of one
// species that drift together (the smooth part of the field contracts velocity space) Gamma = g_p - g_q ~ H z, so
// the term stays O(c |H|) however small |z| is and its Jacobian grows like c |H| / |z|.  Once
//     L_pq = (dt/2) c_pq |Gamma_pq| / |z_pq|^2,     c_pq = nu_ss' (w_q/m_s + w_p/m_s'),
// exceeds 1 the Jacobi map of Eq. (24) expands in the relative coordinate of that ONE pair and the iteration ends in a
// two-cycle of amplitude ~|z| (residual ~1e-8 of the state, for ever); the oracle's literal Jacobi loop shows exactly the
// same (tests/golden/oracle_history_c1_*.csv).  Close unlike pairs (an electron inside the ion cloud) do the same with
// Gamma = O(1).  Anderson mixing and Newton-Krylov only partly cope, because the map is strongly non-linear on the
// scale |z| (profiles/r2_solvers.md).
//
// What is done here (same equation, no softening, no change of the scheme).  Pairs with L_pq > theta are found once per
// step, at v^n, by the first pass-2 evaluation itself (a comparison per pair against a per-species-pair bound, then
// the exact criterion for the rare candidates).  In every iteration, for each such pair, the mutual term is taken OUT
// of the explicit Jacobi update and solved implicitly and exactly, the field of all other markers being that of the
// current iterate ("nonlinear elimination" of two markers):
//     x_p = v_p^n + dt [ Vext_p + (nu/m_s ) w_q Q(z_m) Gamma ],      x_q = v_q^n + dt [ Vext_q - (nu/m_s') w_p Q(z_m) Gamma ],
//     z_m = (v_p^n + x_p)/2 - (v_q^n + x_q)/2        =>        z_m = a + beta Q(z_m) Gamma,
//     a = z^n + (dt/2)(Vext_p - Vext_q),   beta = (dt/2) c_pq,   Gamma = g_p - g_q  (G^n is frozen during the step).
// Q(z_m) Gamma is perpendicular to z_m, so z_m lies in the plane of a and Gamma; with z_m = r (cos phi e1 + sin phi e2),
// e1 = a/|a|, the equation reduces to r = |a| cos phi and ONE scalar equation
//     f(phi) = |a|^2 sin phi cos phi + beta (Gamma_1 sin phi - Gamma_2 cos phi) = 0,      Gamma_2 >= 0,
// whose root continuously connected to dt -> 0 is the first sign change of f from phi = 0 upwards (f(0) <= 0): inside
// [0, angle(a, Gamma)] when that angle is below pi/2, else found by a scan of [0, pi/2); then bisection.  The outer iteration then no longer sees the stiff term and contracts again; at its fixed point every marker,
// the eliminated ones included, satisfies Eq. (24) -- checked against the ORACLE's literal evaluation in the tests.
// If that branch has folded away (beta |Gamma| > ~|a|^2/2 with Gamma pointing away from a) the stiff branch of the
// implicit midpoint rule is taken, on which the pair passes through its midpoint (z^{n+1} ~ -z^n).  Markers with several
// stiff partners (three electrons that have drifted together) form a cluster -- a connected component of the stiff-pair
// graph, up to STIFF_KMAX markers -- whose mutual terms are all solved together by Newton's method with the analytic
// Jacobian of Q(z) Gamma.  Momentum: the two corrections are (nu/m_s) w_q T and -(nu/m_s') w_p T, so m_s w_p dx_p + m_s' w_q dx_q
// = 0 exactly as in Eq. (27).
#pragma once
#include "common.cuh"

namespace landau {

constexpr int STIFF_CAP = 4096;

struct StiffCtrl {
    int count;                 // candidates recorded by the detection pass of this step
    int overflow;              // 1 if more than STIFF_CAP pairs qualified (the rest are left to the plain update)
    int n_cluster;             // cluster solves (summed over the iterations of the step) that failed or were too large
    int n_noroot;              // pair solves (summed over the iterations of the step) that had to take the stiff branch
    double theta;              // stiffness threshold L_pq > theta
    double half_dt;
    double thr2[LD_MAX_SPECIES * LD_MAX_SPECIES];   // |z|^2 below which a pair of species (s, s') CAN be stiff
    int pairs[STIFF_CAP][2];   // slots (p, q)
};

// Start of a step: empty list and the per-species-pair candidate bound
//   |z|^2 < (dt/2) nu_ss' (wmax_s'/m_s + wmax_s/m_s') (gmax_s + gmax_s') / theta   (>= the exact criterion),
// g = G^n/m.  One block per species computes wmax_s, gmax_s; the last block to finish fills the table.
__global__ void __launch_bounds__(256)
stiff_begin_kernel(const DevTable* __restrict__ T, const DevLayout* __restrict__ L, StiffCtrl* __restrict__ sc,
                   int* __restrict__ mark, int npad_max, double dt, double theta, const double* __restrict__ w,
                   const double* __restrict__ Gx, const double* __restrict__ Gy, const double* __restrict__ Gz,
                   double* __restrict__ scratch /* 2 S doubles */, unsigned int* __restrict__ ticket) {
    const int s = blockIdx.x, S = T->S;
    const int p0 = L->off[s], p1 = L->off[s + 1];
    for (int p = p0 + threadIdx.x; p < p1; p += blockDim.x) mark[p] = 0;
    double wm = 0.0, gm = 0.0;
    const double im = T->inv_mass[s];
    for (int p = p0 + threadIdx.x; p < p1; p += blockDim.x) {
        if (w[p] > 0.0) {
            wm = fmax(wm, w[p]);
            gm = fmax(gm, im * sqrt(Gx[p] * Gx[p] + Gy[p] * Gy[p] + Gz[p] * Gz[p]));
        }
    }
    __shared__ double s_w[8], s_g[8];
    __shared__ int s_last;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        wm = fmax(wm, __shfl_xor_sync(0xffffffffu, wm, o));
        gm = fmax(gm, __shfl_xor_sync(0xffffffffu, gm, o));
    }
    if ((threadIdx.x & 31) == 0) { s_w[threadIdx.x >> 5] = wm; s_g[threadIdx.x >> 5] = gm; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int k = 1; k < 8; ++k) { wm = fmax(wm, s_w[k]); gm = fmax(gm, s_g[k]); }
        scratch[2 * s] = wm; scratch[2 * s + 1] = gm;
        __threadfence();
        const unsigned t = atomicInc(ticket, gridDim.x - 1);
        s_last = (t == gridDim.x - 1);
    }
    __syncthreads();
    if (!s_last || threadIdx.x != 0) return;
    __threadfence();
    sc->count = 0; sc->overflow = 0; sc->theta = theta; sc->half_dt = 0.5 * dt; sc->n_cluster = 0; sc->n_noroot = 0;
    for (int a = 0; a < S; ++a)
        for (int b = 0; b < S; ++b) {
            const double wa = __ldcg(scratch + 2 * a), ga = __ldcg(scratch + 2 * a + 1);
            const double wb = __ldcg(scratch + 2 * b), gb = __ldcg(scratch + 2 * b + 1);
            const double c = fabs(T->nu[a * S + b]) * (wb * T->inv_mass[a] + wa * T->inv_mass[b]);
            sc->thr2[a * S + b] = theta > 0.0 ? 0.5 * dt * c * (ga + gb) / theta : 0.0;
        }
}

// Called by the pass-2 kernels (first evaluation of a step) for a pair whose |z|^2 is below the bound of its species
// pair: the exact criterion, then the append.  wq_nu = nu w_q, wp_nu = nu w_p; (cx, cy, cz) = g_p - g_q.
__device__ __forceinline__ void stiff_candidate(StiffCtrl* __restrict__ sc, int* __restrict__ mark, int p, int q,
                                                double r2, double cx, double cy, double cz, double wq_nu,
                                                double wp_nu, double im_p, double im_q) {
    if (!(r2 > 0.0)) return;
    const double c = fabs(wq_nu) * im_p + fabs(wp_nu) * im_q;
    const double Lpq = sc->half_dt * c * sqrt(cx * cx + cy * cy + cz * cz) / r2;
    if (!(Lpq > sc->theta)) return;
    const int k = atomicAdd(&sc->count, 1);
    if (k >= STIFF_CAP) { sc->overflow = 1; return; }
    sc->pairs[k][0] = p; sc->pairs[k][1] = q;
    atomicAdd(mark + p, 1);
    atomicAdd(mark + q, 1);
}

constexpr int STIFF_KMAX = 6;          // markers in a cluster that is solved as one system
constexpr int STIFF_SCAN = 512;        // clusters are only assembled while the step has at most this many stiff pairs

// T = Q(z) gam = (gam - z (z.gam)/|z|^2)/|z|  (0 for z = 0, reading S5)
__device__ __forceinline__ void stiff_T(const double* z, const double* gam, double* T) {
    const double r2 = z[0] * z[0] + z[1] * z[1] + z[2] * z[2];
    if (!(r2 > 0.0)) { T[0] = T[1] = T[2] = 0.0; return; }
    const double ir = 1.0 / sqrt(r2), h = (z[0] * gam[0] + z[1] * gam[1] + z[2] * gam[2]) / r2;
    for (int d = 0; d < 3; ++d) T[d] = (gam[d] - z[d] * h) * ir;
}

// M = d[Q(z) gam]/dz = -(gam z^T + (z.gam) I + z gam^T)/r^3 + 3 (z.gam) z z^T / r^5
__device__ __forceinline__ void stiff_M(const double* z, const double* gam, double (*M)[3]) {
    const double r2 = z[0] * z[0] + z[1] * z[1] + z[2] * z[2];
    if (!(r2 > 0.0)) { for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b) M[a][b] = 0.0; return; }
    const double ir = 1.0 / sqrt(r2), ir3 = ir / r2, ir5 = ir3 / r2;
    const double zg = z[0] * gam[0] + z[1] * gam[1] + z[2] * gam[2];
    for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b)
            M[a][b] = -(gam[a] * z[b] + z[a] * gam[b] + (a == b ? zg : 0.0)) * ir3 + 3.0 * zg * z[a] * z[b] * ir5;
}

// A cluster of nn <= STIFF_KMAX markers whose mutual terms are ALL treated implicitly: Newton's method (analytic
// Jacobian, backtracking on |F|) on the midpoints m_i,
//     F_i(m) = m_i - v_i^n - (dt/2) [ Vext_i + sum_{j in C, j != i} c_ij Q(m_i - m_j) (g_i - g_j) ],   c_ij = nu_ij w_j / m_i,
// started from the midpoints of the current iterate.  The unknowns are carried as OFFSETS d_i = m_i - m_0(start): a
// stiff cluster has |z| ~ 1e-7 at coordinates ~1, so one ulp of an absolute coordinate moves F by L ulp ~ 1e-12 and
// Newton on absolute coordinates stalls at |F| ~ 2e-13 -- a position error that the stiffness turns into a 1e-9 defect
// of Eq. (24).  Differences of offsets are exact.  Returns false (nothing written) if it does not converge.
__device__ bool stiff_cluster_solve(const DevTable* __restrict__ T, const DevLayout* __restrict__ L, const int* nodes, int nn,
                                    int npad_max, int nparts, double dt, const double* __restrict__ xn,
                                    const double* __restrict__ yn, const double* __restrict__ zn,
                                    const double* __restrict__ rec, const double* __restrict__ soa,
                                    double* __restrict__ vpart) {
    const size_t np = (size_t)npad_max;
    const int S = T->S;
    double m[STIFF_KMAX][3], g[STIFF_KMAX][3], w[STIFF_KMAX], vn[STIFF_KMAX][3], Vext[STIFF_KMAX][3], im[STIFF_KMAX];
    double Told[STIFF_KMAX][STIFF_KMAX][3];
    int sp[STIFF_KMAX];
    for (int i = 0; i < nn; ++i) {
        const int p = nodes[i];
        if (soa) {
            for (int d = 0; d < 3; ++d) { m[i][d] = soa[d * np + p]; g[i][d] = soa[(4 + d) * np + p]; }
            w[i] = soa[3 * np + p];
        } else {
            const double* a = rec + (size_t)p * 8;
            for (int d = 0; d < 3; ++d) { m[i][d] = a[d]; g[i][d] = a[4 + d]; }
            w[i] = a[3];
        }
        vn[i][0] = xn[p]; vn[i][1] = yn[p]; vn[i][2] = zn[p];
        sp[i] = species_of_slot(L, S, p);
        im[i] = T->inv_mass[sp[i]];
        for (int d = 0; d < 3; ++d) {
            double v = 0.0;
            for (int c = 0; c < nparts; ++c) v += vpart[((size_t)c * 3 + d) * np + p];
            Vext[i][d] = v;
        }
    }
    for (int i = 0; i < nn; ++i) {
        for (int j = 0; j < nn; ++j) {
            if (j == i) { Told[i][j][0] = Told[i][j][1] = Told[i][j][2] = 0.0; continue; }
            double z[3], gam[3];
            for (int d = 0; d < 3; ++d) { z[d] = m[i][d] - m[j][d]; gam[d] = g[i][d] - g[j][d]; }
            stiff_T(z, gam, Told[i][j]);
            const double cij = T->nu[sp[i] * S + sp[j]] * w[j] * im[i];
            for (int d = 0; d < 3; ++d) Vext[i][d] -= cij * Told[i][j][d];
        }
    }
    // offsets from the first marker's midpoint; b_i = m_0 - v_i^n (both differences are exact or nearly so)
    double dd[STIFF_KMAX][3], bb[STIFF_KMAX][3], zmax = 0.0;
    for (int i = 0; i < nn; ++i)
        for (int d = 0; d < 3; ++d) {
            dd[i][d] = m[i][d] - m[0][d];
            bb[i][d] = m[0][d] - vn[i][d];
            zmax = fmax(zmax, fabs(dd[i][d]));
        }
    constexpr int NU = 3 * STIFF_KMAX;
    const int n3 = 3 * nn;
    double F[NU], A[NU][NU + 1];
    auto residual = [&](const double (*de)[3], double* Fo) -> double {
        double nrm = 0.0;
        for (int i = 0; i < nn; ++i) {
            double acc[3] = {Vext[i][0], Vext[i][1], Vext[i][2]};
            for (int j = 0; j < nn; ++j) {
                if (j == i) continue;
                double z[3], gam[3], Tn[3];
                for (int d = 0; d < 3; ++d) { z[d] = de[i][d] - de[j][d]; gam[d] = g[i][d] - g[j][d]; }
                stiff_T(z, gam, Tn);
                const double cij = T->nu[sp[i] * S + sp[j]] * w[j] * im[i];
                for (int d = 0; d < 3; ++d) acc[d] = fma(cij, Tn[d], acc[d]);
            }
            for (int d = 0; d < 3; ++d) {
                Fo[3 * i + d] = de[i][d] + fma(-0.5 * dt, acc[d], bb[i][d]);
                nrm = fmax(nrm, fabs(Fo[3 * i + d]));
            }
        }
        return nrm;
    };
    const double ftol = 1e-10 * fmax(zmax, 1e-300);             // position error << the cluster's own size
    double fn = residual(dd, F);
    for (int it = 0; it < 80; ++it) {
        for (int a = 0; a < n3; ++a) { for (int b = 0; b < n3; ++b) A[a][b] = a == b ? 1.0 : 0.0; A[a][n3] = -F[a]; }
        for (int i = 0; i < nn; ++i)
            for (int j = 0; j < nn; ++j) {
                if (j == i) continue;
                double z[3], gam[3], M[3][3];
                for (int d = 0; d < 3; ++d) { z[d] = dd[i][d] - dd[j][d]; gam[d] = g[i][d] - g[j][d]; }
                stiff_M(z, gam, M);
                const double cij = 0.5 * dt * T->nu[sp[i] * S + sp[j]] * w[j] * im[i];
                for (int a = 0; a < 3; ++a)
                    for (int b = 0; b < 3; ++b) { A[3 * i + a][3 * i + b] -= cij * M[a][b]; A[3 * i + a][3 * j + b] += cij * M[a][b]; }
            }
        bool singular = false;
        for (int c = 0; c < n3 && !singular; ++c) {               // Gaussian elimination, partial pivoting
            int piv = c;
            for (int r = c + 1; r < n3; ++r) if (fabs(A[r][c]) > fabs(A[piv][c])) piv = r;
            if (!(fabs(A[piv][c]) > 0.0) || !isfinite(A[piv][c])) { singular = true; break; }
            if (piv != c) for (int b = c; b <= n3; ++b) { const double t = A[c][b]; A[c][b] = A[piv][b]; A[piv][b] = t; }
            for (int r = c + 1; r < n3; ++r) {
                const double f = A[r][c] / A[c][c];
                if (f != 0.0) for (int b = c; b <= n3; ++b) A[r][b] -= f * A[c][b];
            }
        }
        if (singular) break;
        double dx[NU];
        for (int c = n3 - 1; c >= 0; --c) {
            double acc = A[c][n3];
            for (int b = c + 1; b < n3; ++b) acc -= A[c][b] * dx[b];
            dx[c] = acc / A[c][c];
        }
        double lam = 1.0, dt_[STIFF_KMAX][3], Ft[NU], ft = 0.0;
        bool accepted = false;
        for (int h = 0; h < 14; ++h) {                            // backtracking on |F|
            for (int i = 0; i < nn; ++i) for (int d = 0; d < 3; ++d) dt_[i][d] = dd[i][d] + lam * dx[3 * i + d];
            ft = residual(dt_, Ft);
            if (ft < fn) { accepted = true; break; }
            lam *= 0.5;
        }
        if (!accepted) break;                                      // no further decrease: round-off floor (or failure)
        for (int i = 0; i < nn; ++i) for (int d = 0; d < 3; ++d) dd[i][d] = dt_[i][d];
        for (int a = 0; a < n3; ++a) F[a] = Ft[a];
        fn = ft;
        if (fn <= 1e-3 * ftol) break;
    }
#ifdef LANDAU_STIFF_DEBUG
    printf("cluster nn=%d fn=%.3e ftol=%.3e zmax=%.3e\n", nn, fn, ftol, zmax);
#endif
    if (!(fn <= ftol)) return false;
    for (int i = 0; i < nn; ++i) for (int d = 0; d < 3; ++d) m[i][d] = dd[i][d];   // offsets: only differences are used below
    for (int i = 0; i < nn; ++i) {
        double dV[3] = {0.0, 0.0, 0.0};
        for (int j = 0; j < nn; ++j) {
            if (j == i) continue;
            double z[3], gam[3], Tn[3];
            for (int d = 0; d < 3; ++d) { z[d] = m[i][d] - m[j][d]; gam[d] = g[i][d] - g[j][d]; }
            stiff_T(z, gam, Tn);
            const double cij = T->nu[sp[i] * S + sp[j]] * w[j] * im[i];
            for (int d = 0; d < 3; ++d) dV[d] = fma(cij, Tn[d] - Told[i][j][d], dV[d]);
        }
        for (int d = 0; d < 3; ++d) vpart[(size_t)d * np + nodes[i]] += dV[d];
    }
    return true;
}

// One thread per stiff pair, after pass 2 and before the solver's update kernel: replaces, in the field slices, the
// explicit mutual term of the pair by its implicit solution (header comment).  u = midpoint sources of this
// evaluation (records of 8 doubles or the SoA copy), vpart = nparts field slices [3][npad_max].
__global__ void __launch_bounds__(128)
stiff_fix_kernel(const DevTable* __restrict__ T, const DevLayout* __restrict__ L, const StepCtrl* __restrict__ ctrl,
                 StiffCtrl* __restrict__ sc, const int* __restrict__ mark, int npad_max, int nparts, double dt,
                 const double* __restrict__ xn, const double* __restrict__ yn, const double* __restrict__ zn,
                 const double* __restrict__ rec, const double* __restrict__ soa, double* __restrict__ vpart) {
    if (ctrl->done) return;
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    const int n = min(sc->count, STIFF_CAP);
    if (k >= n) return;
    const int p = sc->pairs[k][0], q = sc->pairs[k][1];
    if (mark[p] != 1 || mark[q] != 1) {
        // a marker with several stiff partners: the connected component of the stiff-pair graph is solved as ONE system
        // by the thread of its lowest-numbered pair (Newton's method, stiff_cluster_solve)
        if (n > STIFF_SCAN) { atomicAdd(&sc->n_cluster, 1); return; }
        int nodes[STIFF_KMAX], nn = 2, minpair = k;
        nodes[0] = p; nodes[1] = q;
        bool grew = true, too_big = false;
        while (grew && !too_big) {
            grew = false;
            for (int j = 0; j < n && !too_big; ++j) {
                const int a = sc->pairs[j][0], b = sc->pairs[j][1];
                bool ina = false, inb = false;
                for (int t = 0; t < nn; ++t) { ina = ina || nodes[t] == a; inb = inb || nodes[t] == b; }
                if (!ina && !inb) continue;
                minpair = min(minpair, j);
                if (!ina || !inb) {
                    if (nn == STIFF_KMAX) { too_big = true; break; }
                    nodes[nn++] = ina ? b : a;
                    grew = true;
                }
            }
        }
        if (minpair != k) return;                                  // another thread owns this component
        if (too_big || !stiff_cluster_solve(T, L, nodes, nn, npad_max, nparts, dt, xn, yn, zn, rec, soa, vpart))
            atomicAdd(&sc->n_cluster, 1);
        return;
    }
    const size_t np = (size_t)npad_max;
    double up[3], uq[3], gp[3], gq[3], wp, wq;
    if (soa) {
        up[0] = soa[p]; up[1] = soa[np + p]; up[2] = soa[2 * np + p]; wp = soa[3 * np + p];
        gp[0] = soa[4 * np + p]; gp[1] = soa[5 * np + p]; gp[2] = soa[6 * np + p];
        uq[0] = soa[q]; uq[1] = soa[np + q]; uq[2] = soa[2 * np + q]; wq = soa[3 * np + q];
        gq[0] = soa[4 * np + q]; gq[1] = soa[5 * np + q]; gq[2] = soa[6 * np + q];
    } else {
        const double* a = rec + (size_t)p * 8;
        const double* b = rec + (size_t)q * 8;
        up[0] = a[0]; up[1] = a[1]; up[2] = a[2]; wp = a[3]; gp[0] = a[4]; gp[1] = a[5]; gp[2] = a[6];
        uq[0] = b[0]; uq[1] = b[1]; uq[2] = b[2]; wq = b[3]; gq[0] = b[4]; gq[1] = b[5]; gq[2] = b[6];
    }
    const int S = T->S;
    const int sp = species_of_slot(L, S, p), sq = species_of_slot(L, S, q);
    const double nu = T->nu[sp * S + sq], imp = T->inv_mass[sp], imq = T->inv_mass[sq];
    double Vp[3] = {0, 0, 0}, Vq[3] = {0, 0, 0};
    for (int c = 0; c < nparts; ++c)
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            Vp[d] += vpart[((size_t)c * 3 + d) * np + p];
            Vq[d] += vpart[((size_t)c * 3 + d) * np + q];
        }
    // mutual term of this evaluation, T_k = Q(z_k) Gamma at the current midpoint
    double z[3], gam[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) { z[d] = up[d] - uq[d]; gam[d] = gp[d] - gq[d]; }
    const double r2 = z[0] * z[0] + z[1] * z[1] + z[2] * z[2];
    double Tk[3] = {0, 0, 0};
    if (r2 > 0.0) {
        const double ir = 1.0 / sqrt(r2), h = (z[0] * gam[0] + z[1] * gam[1] + z[2] * gam[2]) / r2;
#pragma unroll
        for (int d = 0; d < 3; ++d) Tk[d] = (gam[d] - z[d] * h) * ir;
    }
    const double cp = nu * wq * imp, cq = nu * wp * imq;           // V_p contains +cp T, V_q contains -cq T
    const double xnp[3] = {xn[p], yn[p], zn[p]}, xnq[3] = {xn[q], yn[q], zn[q]};
    double a[3], Vep[3], Veq[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        Vep[d] = Vp[d] - cp * Tk[d];
        Veq[d] = Vq[d] + cq * Tk[d];
        a[d] = (xnp[d] - xnq[d]) + 0.5 * dt * (Vep[d] - Veq[d]);
    }
    const double beta = 0.5 * dt * (cp + cq);
    const double na2 = a[0] * a[0] + a[1] * a[1] + a[2] * a[2];
    if (!(na2 > 0.0) || !isfinite(na2)) return;
    const double na = sqrt(na2);
    double e1[3], e2[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) e1[d] = a[d] / na;
    const double g1 = gam[0] * e1[0] + gam[1] * e1[1] + gam[2] * e1[2];
#pragma unroll
    for (int d = 0; d < 3; ++d) e2[d] = gam[d] - g1 * e1[d];
    const double g2 = sqrt(e2[0] * e2[0] + e2[1] * e2[1] + e2[2] * e2[2]);
    double zm[3];
    if (!(g2 > 1e-14 * fabs(g1)) || g2 == 0.0) {
#pragma unroll
        for (int d = 0; d < 3; ++d) zm[d] = a[d];                  // Gamma parallel to a: Q(a) Gamma = 0
    } else {
#pragma unroll
        for (int d = 0; d < 3; ++d) e2[d] /= g2;
        const double HALF_PI = 1.5707963267948966;
        double lo = 0.0, hi = fmin(atan2(g2, g1), HALF_PI * (1.0 - 1e-12));
        double sh, ch;
        sincos(hi, &sh, &ch);
        if (!(na2 * sh * ch + beta * (g1 * sh - g2 * ch) >= 0.0)) {
            // Gamma points away from a (angle > pi/2): f(0) <= 0 and f(pi/2) < 0, but f may be positive in between
            // (it is when beta |Gamma| < ~|a|^2/2).  The physical root is the FIRST sign change from 0 upwards.
            bool found = false;
            double prev = 0.0;
            for (int k = 1; k <= 256 && !found; ++k) {
                const double ph = hi * (double)k / 256.0;
                sincos(ph, &sh, &ch);
                if (na2 * sh * ch + beta * (g1 * sh - g2 * ch) > 0.0) { lo = prev; hi = ph; found = true; }
                prev = ph;
            }
            if (!found) {
                // The branch connected to dt -> 0 has folded away (beta |Gamma| > ~|a|^2/2 with Gamma pointing away from
                // a).  What is left is the stiff branch of the implicit midpoint rule, on which the pair passes through
                // its midpoint (z^{n+1} ~ -z^n, amplification factor -> -1): f(-pi/2) = -beta Gamma_1 > 0 >= f(0), so it
                // always exists for Gamma_1 < 0; the root nearest to 0 is taken.
                atomicAdd(&sc->n_noroot, 1);
                prev = 0.0;
                const double end = -HALF_PI * (1.0 - 1e-12);
                for (int k = 1; k <= 256 && !found; ++k) {
                    const double ph = end * (double)k / 256.0;
                    sincos(ph, &sh, &ch);
                    if (na2 * sh * ch + beta * (g1 * sh - g2 * ch) > 0.0) { lo = prev; hi = ph; found = true; }
                    prev = ph;
                }
                if (!found) return;
            }
        }
        for (int it = 0; it < 64; ++it) {
            const double mid = 0.5 * (lo + hi);
            sincos(mid, &sh, &ch);
            const double f = na2 * sh * ch + beta * (g1 * sh - g2 * ch);
            if (f > 0.0) hi = mid; else lo = mid;
        }
        sincos(0.5 * (lo + hi), &sh, &ch);
        const double r = na * ch;
#pragma unroll
        for (int d = 0; d < 3; ++d) zm[d] = r * (ch * e1[d] + sh * e2[d]);
    }
    const double rm2 = zm[0] * zm[0] + zm[1] * zm[1] + zm[2] * zm[2];
    if (!(rm2 > 0.0)) return;
    const double irm = 1.0 / sqrt(rm2), hm = (zm[0] * gam[0] + zm[1] * gam[1] + zm[2] * gam[2]) / rm2;
    // new fields: V'_p = Vext_p + cp Q(z_m) Gamma, V'_q = Vext_q - cq Q(z_m) Gamma; slice 0 carries the difference
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const double Tm = (gam[d] - zm[d] * hm) * irm;
        vpart[(size_t)d * np + p] += cp * (Tm - Tk[d]);
        vpart[(size_t)d * np + q] -= cq * (Tm - Tk[d]);
    }
}

}  // namespace landau
