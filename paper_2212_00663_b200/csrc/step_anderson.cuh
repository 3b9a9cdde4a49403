// step_anderson.cuh -- SURVEY.md section 8(f) NEXT-4: Anderson acceleration of the fixed point of Eq. (24).
//
// The paper solves Eq. (24) by plain fixed-point iteration and reports steps that fail to
// converge; profiles/r1_histories.md shows the same on configs 1 and 3.  The equation
// itself is unchanged here: with  g(x) = v^n + dt V[(v^n + x)/2 ; G^n]  the step is the fixed point x = g(x).
// Anderson mixing of depth m (type II, no damping) keeps the last m differences
//     dF_j = f_{j+1} - f_j,   dG_j = g_{j+1} - g_j,      f_j = g(x_j) - x_j,
// solves the m x m least-squares problem  gamma = argmin || f_k - dF gamma ||  in the energy inner product
// <a,b> = sum_p w_p m_s a_p.b_p  (the norm of the residual r_k, reading S7), and continues from
//     x_{k+1} = g(x_k) - dG gamma.
// Every g(x_j) has exactly the momentum of v^n (Eq. 27), dG_j has none, so every iterate conserves momentum as
// the Jacobi iterates do.  The committed state is g(x_k) of the last evaluation, with the same
// stopping rule as the Jacobi loop (r_k = |g(x_k) - x_k| / |g(x_k)| <= tol), so a converged step solves Eq. (24)
// to the same tolerance and energy is conserved to the same accuracy.  Depth 0 columns = the Jacobi step.
// Device driven like step.cuh: the Gram matrix is updated and the small system solved by the last block of the
// update kernel (fixed-order sums: deterministic), no host synchronisation inside a step.
#pragma once
#include "common.cuh"
#include "step.cuh"

namespace landau {

constexpr int AA_MAXM = 10;
constexpr int AA_NRED = 2 + 2 * AA_MAXM;    // num, den, b_j, a_j

struct AndersonCtrl {
    int m;                       // depth (1..AA_MAXM)
    int _r;
    double gram[AA_MAXM][AA_MAXM];
    double gamma[AA_MAXM];
};

// Solve the nc x nc normal equations after scaling the columns to unit norm (Gaussian elimination with partial
// pivoting); returns false when the scaled Gram matrix is numerically singular (nearly dependent columns).
__device__ inline bool aa_solve(int nc, const double (*G)[AA_MAXM], const double* b, double* x) {
    double A[AA_MAXM][AA_MAXM + 1], sc[AA_MAXM];
    for (int i = 0; i < nc; ++i) {
        if (!(G[i][i] > 0.0) || !isfinite(G[i][i])) return false;
        sc[i] = 1.0 / sqrt(G[i][i]);
    }
    for (int i = 0; i < nc; ++i) {
        for (int j = 0; j < nc; ++j) A[i][j] = G[i][j] * sc[i] * sc[j];
        A[i][nc] = b[i] * sc[i];
    }
    for (int c = 0; c < nc; ++c) {
        int piv = c;
        for (int r = c + 1; r < nc; ++r) if (fabs(A[r][c]) > fabs(A[piv][c])) piv = r;
        if (!(fabs(A[piv][c]) > 1e-10)) return false;
        if (piv != c) for (int j = c; j <= nc; ++j) { const double t = A[c][j]; A[c][j] = A[piv][j]; A[piv][j] = t; }
        for (int r = c + 1; r < nc; ++r) {
            const double f = A[r][c] / A[c][c];
            for (int j = c; j <= nc; ++j) A[r][j] -= f * A[c][j];
        }
    }
    for (int c = nc - 1; c >= 0; --c) {
        double s = A[c][nc];
        for (int j = c + 1; j < nc; ++j) s -= A[c][j] * x[j];
        x[c] = s / A[c][c];
    }
    for (int c = 0; c < nc; ++c) {
        x[c] *= sc[c];
        if (!isfinite(x[c])) return false;
    }
    return true;
}

// Start of a step: empty history (a kernel, so that the reset is part of a captured step graph).
__global__ void anderson_begin_kernel(AndersonCtrl* __restrict__ aa, int m) {
    if (threadIdx.x == 0 && blockIdx.x == 0) { aa->m = m; aa->_r = 0; }
}

// g_k = v^n + dt V(u_k), f_k = g_k - x_k; new difference columns; residual; Gram update and solve.
// hist layout: dF[slot][3][npad_max], dG[slot][3][npad_max], fprev[3][npad_max], gcur[3][npad_max].
__global__ void __launch_bounds__(UPD_THREADS)
anderson_update_kernel(const DevTable* __restrict__ T, const DevLayout* __restrict__ L, StepCtrl* __restrict__ ctrl,
                       AndersonCtrl* __restrict__ aa, int npad_max, int nparts, double dt, double tol, int max_iter,
                       const double* __restrict__ vpart, const double* __restrict__ xn,
                       const double* __restrict__ yn, const double* __restrict__ zn, const double* __restrict__ w,
                       const double* __restrict__ xk, const double* __restrict__ yk, const double* __restrict__ zk,
                       double* __restrict__ dF, double* __restrict__ dG, double* __restrict__ fprev,
                       double* __restrict__ gcur, double* __restrict__ blockpart, cudaGraphConditionalHandle cond) {
    if (ctrl->done) return;
    __shared__ double s_red[UPD_THREADS / 32][AA_NRED];
    __shared__ int s_last;
    const int k = ctrl->iterations;                 // completed iterations before this one
    const int m = aa->m;
    const int nc = min(k, m);                       // active columns once this iteration's column is stored
    const int slot_new = k > 0 ? (k - 1) % m : -1;
    const size_t np = (size_t)npad_max, col = 3 * np;
    const int p = blockIdx.x * UPD_THREADS + threadIdx.x;
    double red[AA_NRED];
#pragma unroll
    for (int i = 0; i < AA_NRED; ++i) red[i] = 0.0;
    if (p < npad_max && p < L->npad) {
        double a = 0.0, b = 0.0, c = 0.0;
        for (int q = 0; q < nparts; ++q) {
            const double* o = vpart + (size_t)q * 3 * np + p;
            a += o[0]; b += o[np]; c += o[2 * np];
        }
        const double wp = w[p];
        if (wp == 0.0) { a = 0.0; b = 0.0; c = 0.0; }
        const double g0 = fma(dt, a, xn[p]), g1 = fma(dt, b, yn[p]), g2 = fma(dt, c, zn[p]);
        const double f0 = g0 - xk[p], f1 = g1 - yk[p], f2 = g2 - zk[p];
        const double wm = wp * T->mass[species_of_slot(L, T->S, p)];
        red[0] = wm * (f0 * f0 + f1 * f1 + f2 * f2);
        red[1] = wm * (g0 * g0 + g1 * g1 + g2 * g2);
        double c0 = 0.0, c1 = 0.0, c2 = 0.0;
        if (k > 0) {
            c0 = f0 - fprev[p]; c1 = f1 - fprev[np + p]; c2 = f2 - fprev[2 * np + p];
            double* cf = dF + (size_t)slot_new * col + p;
            double* cg = dG + (size_t)slot_new * col + p;
            cf[0] = c0; cf[np] = c1; cf[2 * np] = c2;
            cg[0] = g0 - gcur[p]; cg[np] = g1 - gcur[np + p]; cg[2 * np] = g2 - gcur[2 * np + p];
        }
        fprev[p] = f0; fprev[np + p] = f1; fprev[2 * np + p] = f2;
        gcur[p] = g0; gcur[np + p] = g1; gcur[2 * np + p] = g2;
#pragma unroll
        for (int j = 0; j < AA_MAXM; ++j) {
            if (j < nc) {
                double e0 = c0, e1 = c1, e2 = c2;
                if (j != slot_new) {
                    const double* cf = dF + (size_t)j * col + p;
                    e0 = cf[0]; e1 = cf[np]; e2 = cf[2 * np];
                }
                red[2 + j] = wm * (e0 * f0 + e1 * f1 + e2 * f2);
                red[2 + AA_MAXM + j] = wm * (e0 * c0 + e1 * c1 + e2 * c2);
            }
        }
    }
    const int lane = threadIdx.x & 31, wv = threadIdx.x >> 5;
#pragma unroll
    for (int i = 0; i < AA_NRED; ++i) {
        const double v = warp_sum(red[i]);
        if (lane == 0) s_red[wv][i] = v;
    }
    __syncthreads();
    if (threadIdx.x < AA_NRED) {
        double a = 0.0;
        for (int q = 0; q < UPD_THREADS / 32; ++q) a += s_red[q][threadIdx.x];
        blockpart[(size_t)blockIdx.x * AA_NRED + threadIdx.x] = a;
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) {
        const unsigned t = atomicInc(&ctrl->ticket, gridDim.x - 1);
        s_last = (t == gridDim.x - 1);
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    // fixed-order totals: warp i sums quantity i over the blocks in index order (strided, then a shuffle tree)
    __shared__ double s_tot[AA_NRED];
    for (int i = wv; i < AA_NRED; i += UPD_THREADS / 32) {
        double a = 0.0;
        for (int q = lane; q < (int)gridDim.x; q += 32) a += __ldcg(blockpart + (size_t)q * AA_NRED + i);
        a = warp_sum(a);
        if (lane == 0) s_tot[i] = a;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        const double res = sqrt(s_tot[0] / s_tot[1]);
        const int it = k + 1;
        ctrl->iterations = it;
        ctrl->residual = res;
        if (!isfinite(res)) { ctrl->err = -4; ctrl->done = 1; }
        else if (res <= tol) { ctrl->converged = 1; ctrl->done = 1; }
        else if (it >= max_iter) ctrl->done = 1;
        double gam[AA_MAXM];
        for (int j = 0; j < AA_MAXM; ++j) gam[j] = 0.0;
        if (nc > 0) {
            for (int j = 0; j < nc; ++j) { aa->gram[slot_new][j] = s_tot[2 + AA_MAXM + j]; aa->gram[j][slot_new] = s_tot[2 + AA_MAXM + j]; }
            // least squares over the nu most recent columns, nu = nc, nc-1, ..., 1: the first window whose
            // Gram matrix is numerically regular wins (old, nearly dependent columns are dropped first)
            for (int nu = nc; nu >= 1; --nu) {
                int slots[AA_MAXM];
                double Gs[AA_MAXM][AA_MAXM], rhs[AA_MAXM], sol[AA_MAXM];
                for (int a = 0; a < nu; ++a) slots[a] = ((slot_new - a) % m + m) % m;
                for (int a = 0; a < nu; ++a) {
                    rhs[a] = s_tot[2 + slots[a]];
                    for (int b2 = 0; b2 < nu; ++b2) Gs[a][b2] = aa->gram[slots[a]][slots[b2]];
                }
                if (aa_solve(nu, Gs, rhs, sol)) {
                    for (int a = 0; a < nu; ++a) gam[slots[a]] = sol[a];
                    break;
                }
            }
        }
        for (int j = 0; j < AA_MAXM; ++j) aa->gamma[j] = gam[j];
        // CUDA-graph mode: keep the WHILE node that holds this iteration alive until the step is done
        if (cond) cudaGraphSetConditional(cond, ctrl->done ? 0u : 1u);
    }
}

// x_{k+1} = g_k - dG gamma; next midpoint sources (Eq. 25).
__global__ void anderson_mix_kernel(const DevLayout* __restrict__ L, const StepCtrl* __restrict__ ctrl,
                                    const AndersonCtrl* __restrict__ aa, int npad_max,
                                    const double* __restrict__ xn, const double* __restrict__ yn,
                                    const double* __restrict__ zn, const double* __restrict__ gcur,
                                    const double* __restrict__ dG, double* __restrict__ xk,
                                    double* __restrict__ yk, double* __restrict__ zk, double* __restrict__ rec,
                                    double* __restrict__ soa) {
    if (ctrl->done) return;
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= npad_max || p >= L->npad) return;
    const size_t np = (size_t)npad_max, col = 3 * np;
    const int nc = min(ctrl->iterations - 1, aa->m);
    double x0 = gcur[p], x1 = gcur[np + p], x2 = gcur[2 * np + p];
    for (int j = 0; j < nc; ++j) {
        const double gj = aa->gamma[j];
        const double* cg = dG + (size_t)j * col + p;
        x0 = fma(-gj, cg[0], x0); x1 = fma(-gj, cg[np], x1); x2 = fma(-gj, cg[2 * np], x2);
    }
    xk[p] = x0; yk[p] = x1; zk[p] = x2;
    const double ux = 0.5 * (xn[p] + x0), uy = 0.5 * (yn[p] + x1), uz = 0.5 * (zn[p] + x2);
    if (rec) {
        double2* o = reinterpret_cast<double2*>(rec + (size_t)p * 8);
        o[0] = make_double2(ux, uy);
        reinterpret_cast<double*>(o + 1)[0] = uz;
    }
    if (soa) { soa[p] = ux; soa[np + p] = uy; soa[2 * np + p] = uz; }
}

}  // namespace landau
