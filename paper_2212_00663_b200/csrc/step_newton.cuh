// step_newton.cuh -- SURVEY.md section 8(f) NEXT-4, first half: a Jacobian-free Newton-Krylov solver for the
// implicit step, for the steps the paper's fixed-point iteration cannot converge ("the
// solver is unable to fully converge on occasion").
//
// Same equation, same residual, same stopping rule as step.cuh / step_anderson.cuh.  With
//     g(x) = v^n + dt V[(v^n + x)/2 ; G^n]            (Eqs. 24-25)
// the step is the root of  F(x) = x - g(x).  The Jacobi iteration is Richardson's method for it and diverges as soon
// as one eigenvalue of g'(x) leaves the unit disk -- which a single close pair of unlike markers can cause
// (d(Q Gamma)/dz ~ Gamma/|z|^2, SURVEY.md reading S8).  Newton's method solves  (I - g'(x)) d = g(x) - x  and
// sets x <- x + d; the linear systems are solved by GMRES(m) in the energy inner product <a,b> = sum_p w_p m_s a_p.b_p
// (the norm of the residual r_k, reading S7) with Jacobian-vector products by one-sided differences of the FIELD,
//     (I - g'(x)) q  ~  q - dt (V[u(x) + e q/2] - V[u(x)])/e,       e = 1e-11 |x| / |q|,
// i.e. ONE more pass 2 (the same kernel, markers moved by e q / 2) per Krylov vector.  The difference quotient has
// two errors: round-off of the moved positions, eps_mach |u| / e ~ 1e-5, and e q_p against the separation of the
// closest pairs -- a Krylov vector concentrated on two nearly coincident markers (|z| ~ 1e-6 of the thermal speed
// occurs) moves them by e / sqrt(w m) ~ 1e-9, which a larger step would not resolve.  A linear
// solve is therefore never asked for more than 1e-4, and Newton's outer iteration -- whose residual is a TRUE
// evaluation of g(x) - x -- supplies the rest (measured: profiles/r2_solvers.md).  GMRES minimises the linear residual over the Krylov space, so it needs no more products than Jacobi needs
// sweeps when Jacobi converges, and a few more per outlying eigenvalue when it does not.  Inexact Newton: the first
// system is solved to 1e-3, later ones to what the tolerance still asks for (clamped to [1e-4, 1e-3]).
// Globalisation: if a Newton update does not reduce the residual, it is halved (up to 6 times) before the next
// linearisation (backtracking on |g(x) - x|).
//
// Device driven like the other solvers: one "iteration" = one pass 2 + three small kernels whose behaviour is decided
// by a state block in device memory (phase 0: evaluate g(x), residual, start a Krylov space; phase 1: one Arnoldi
// step, Givens update of the least-squares problem, and -- when the linear solve is good enough or the space is
// full -- the Newton update).  `iterations` therefore counts pass-2 evaluations, as for Jacobi and Anderson.  All
// reductions are block partials summed in index order by the last block (deterministic).  The committed state is
// g(x) of the last phase-0 evaluation and `residual` is r = |g(x) - x| / |g(x)| of that evaluation, exactly the
// quantities the Jacobi loop reports; every g(x) has the momentum of v^n (Eq. 27), so momentum is conserved whether
// or not the step converged, and energy to the accuracy of the residual.
#pragma once
#include "common.cuh"
#include "step.cuh"

namespace landau {

#ifndef NK_EPS_REL      // tuning knobs of the difference quotient (see the header comment)
#define NK_EPS_REL 1e-11
#endif
#ifndef NK_ETA_MIN
#define NK_ETA_MIN 1e-4
#endif
constexpr int NK_MAXM = 30;
constexpr int NK_NRED = NK_MAXM + 2;

struct NewtonCtrl {
    int m;              // restart length (1..NK_MAXM)
    int phase;          // 0: next evaluation is g(x); 1: next evaluation is a Jacobian-vector product
    int j;              // Krylov vectors q_0..q_j exist (phase 1)
    int k4_mode;        // what nk_update_kernel has to do after this post kernel: 0 nothing, 1 q_0 = f/beta,
                        // 2 orthonormalise the new vector, 3 Newton update x += Q y, 4 backtrack x -= lam_back Q y
    int napply;         // number of Krylov vectors in the Newton update (k4_mode 3)
    int newton_its;     // phase-0 evaluations so far
    int backtracks;     // halvings of the current Newton update so far
    int have_update;    // 1 if x is the result of a Newton update whose vectors are still in Q
    double lam;         // current length of the last update in units of the full Newton step
    double lam_back;    // amount to take back (k4_mode 4)
    double beta;        // |f| of the current Newton iterate (energy norm)
    double eps_fd;      // finite-difference step of the current Newton iterate
    double eta;         // forcing term of the current linear solve
    double res_prev;
    double hnorm;       // h_{j+1,j}
    double hcol[NK_MAXM + 1];
    double y[NK_MAXM];
    double cs[NK_MAXM], sn[NK_MAXM], grhs[NK_MAXM + 1];
    double R[NK_MAXM][NK_MAXM];
};

// Start of a step: phase 0, no Krylov space (a kernel, so that the reset is part of a captured step graph).
__global__ void nk_begin_kernel(NewtonCtrl* __restrict__ nk, int m) {
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        nk->m = m; nk->phase = 0; nk->j = 0; nk->k4_mode = 0; nk->napply = 0; nk->newton_its = 0;
        nk->beta = 0.0; nk->eps_fd = 0.0; nk->eta = 1e-3; nk->res_prev = 0.0; nk->hnorm = 0.0;
        nk->backtracks = 0; nk->have_update = 0; nk->lam = 1.0; nk->lam_back = 0.0;
    }
}

// Sources of the next evaluation: the midpoint of Eq. (25) at x (phase 0) or at x + e q_j (phase 1).
__global__ void nk_sources_kernel(const DevLayout* __restrict__ L, const StepCtrl* __restrict__ ctrl,
                                  const NewtonCtrl* __restrict__ nk, int npad_max, const double* __restrict__ xn,
                                  const double* __restrict__ yn, const double* __restrict__ zn,
                                  const double* __restrict__ xk, const double* __restrict__ yk,
                                  const double* __restrict__ zk, const double* __restrict__ Q,
                                  double* __restrict__ rec, double* __restrict__ soa) {
    if (ctrl->done) return;
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= npad_max || p >= L->npad) return;
    const size_t np = (size_t)npad_max;
    double ux = 0.5 * (xn[p] + xk[p]), uy = 0.5 * (yn[p] + yk[p]), uz = 0.5 * (zn[p] + zk[p]);
    if (nk->phase == 1) {
        const double* q = Q + (size_t)nk->j * 3 * np + p;
        const double he = 0.5 * nk->eps_fd;
        ux = fma(he, q[0], ux); uy = fma(he, q[np], uy); uz = fma(he, q[2 * np], uz);
    }
    if (rec) {
        double2* o = reinterpret_cast<double2*>(rec + (size_t)p * 8);
        o[0] = make_double2(ux, uy);
        reinterpret_cast<double*>(o + 1)[0] = uz;
    }
    if (soa) { soa[p] = ux; soa[np + p] = uy; soa[2 * np + p] = uz; }
}

// After pass 2.  Phase 0: g = v^n + dt V, f = g - x, residual, start of the Krylov space.  Phase 1: the new Krylov
// direction w = q_j - (g(x + e q_j) - g(x))/e, its projections on q_0..q_j, the Givens update and the decision.
// hist layout: Q[(m+1)][3][npad_max], then gcur, Vcur (the field at x) and fvec (g(x) - x), [3][npad_max] each.
__global__ void __launch_bounds__(UPD_THREADS)
nk_post_kernel(const DevTable* __restrict__ T, const DevLayout* __restrict__ L, StepCtrl* __restrict__ ctrl,
               NewtonCtrl* __restrict__ nk, int npad_max, int nparts, double dt, double tol, int max_iter,
               const double* __restrict__ vpart, const double* __restrict__ xn, const double* __restrict__ yn,
               const double* __restrict__ zn, const double* __restrict__ w, const double* __restrict__ xk,
               const double* __restrict__ yk, const double* __restrict__ zk, double* __restrict__ Q,
               double* __restrict__ gcur, double* __restrict__ Vcur, double* __restrict__ fvec,
               double* __restrict__ blockpart, cudaGraphConditionalHandle cond) {
    if (ctrl->done) return;
    __shared__ double s_red[UPD_THREADS / 32][NK_NRED];
    __shared__ double s_tot[NK_NRED];
    __shared__ int s_last;
    const int phase = nk->phase, j = nk->j;
    const int nred = phase == 0 ? 3 : j + 2;
    const size_t np = (size_t)npad_max, col = 3 * np;
    const int p = blockIdx.x * UPD_THREADS + threadIdx.x;
    double red[NK_NRED];
#pragma unroll
    for (int i = 0; i < NK_NRED; ++i) red[i] = 0.0;
    if (p < npad_max && p < L->npad) {
        double a = 0.0, b = 0.0, c = 0.0;
        for (int q = 0; q < nparts; ++q) {
            const double* o = vpart + (size_t)q * 3 * np + p;
            a += o[0]; b += o[np]; c += o[2 * np];
        }
        const double wp = w[p];
        if (wp == 0.0) { a = 0.0; b = 0.0; c = 0.0; }
        const double g0 = fma(dt, a, xn[p]), g1 = fma(dt, b, yn[p]), g2 = fma(dt, c, zn[p]);
        const double wm = wp * T->mass[species_of_slot(L, T->S, p)];
        if (phase == 0) {
            const double x0 = xk[p], x1 = yk[p], x2 = zk[p];
            const double f0 = g0 - x0, f1 = g1 - x1, f2 = g2 - x2;
            gcur[p] = g0; gcur[np + p] = g1; gcur[2 * np + p] = g2;
            Vcur[p] = a; Vcur[np + p] = b; Vcur[2 * np + p] = c;
            fvec[p] = f0; fvec[np + p] = f1; fvec[2 * np + p] = f2;   // becomes q_0 = f/beta if a Krylov space is started
            red[0] = wm * (f0 * f0 + f1 * f1 + f2 * f2);
            red[1] = wm * (g0 * g0 + g1 * g1 + g2 * g2);
            red[2] = wm * (x0 * x0 + x1 * x1 + x2 * x2);
        } else {
            const double ie = dt / nk->eps_fd;
            const double* qj = Q + (size_t)j * col + p;
            const double w0 = qj[0] - (a - Vcur[p]) * ie, w1 = qj[np] - (b - Vcur[np + p]) * ie,
                         w2 = qj[2 * np] - (c - Vcur[2 * np + p]) * ie;
            double* qn = Q + (size_t)(j + 1) * col + p;
            qn[0] = w0; qn[np] = w1; qn[2 * np] = w2;                 // q_{j+1} before orthonormalisation
            red[0] = wm * (w0 * w0 + w1 * w1 + w2 * w2);
#pragma unroll
            for (int i = 0; i < NK_MAXM; ++i) {
                if (i <= j) {
                    const double* qi = Q + (size_t)i * col + p;
                    red[1 + i] = wm * (w0 * qi[0] + w1 * qi[np] + w2 * qi[2 * np]);
                }
            }
        }
    }
    const int lane = threadIdx.x & 31, wv = threadIdx.x >> 5;
#pragma unroll
    for (int i = 0; i < NK_NRED; ++i) {
        if (i < nred) {
            const double v = warp_sum(red[i]);
            if (lane == 0) s_red[wv][i] = v;
        }
    }
    __syncthreads();
    if (threadIdx.x < nred) {
        double a = 0.0;
        for (int q = 0; q < UPD_THREADS / 32; ++q) a += s_red[q][threadIdx.x];
        blockpart[(size_t)blockIdx.x * NK_NRED + threadIdx.x] = a;
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
    for (int i = wv; i < nred; i += UPD_THREADS / 32) {
        double a = 0.0;
        for (int q = lane; q < (int)gridDim.x; q += 32) a += __ldcg(blockpart + (size_t)q * NK_NRED + i);
        a = warp_sum(a);
        if (lane == 0) s_tot[i] = a;
    }
    __syncthreads();
    if (threadIdx.x != 0) return;
    const int it = ctrl->iterations + 1;
    ctrl->iterations = it;
    nk->k4_mode = 0;
    if (phase == 0) {
        const double res = sqrt(s_tot[0] / s_tot[1]);
        ctrl->residual = res;
        nk->newton_its += 1;
        if (!isfinite(res)) { ctrl->err = -4; ctrl->done = 1; }
        else if (res <= tol) { ctrl->converged = 1; ctrl->done = 1; }
        else if (it >= max_iter) ctrl->done = 1;
        else if (nk->have_update && !(res < nk->res_prev) && nk->backtracks < 6) {
            // the Newton update made things worse: take half of it back and evaluate again (Q is still intact)
            nk->backtracks += 1;
            nk->lam_back = 0.5 * nk->lam;
            nk->lam *= 0.5;
            nk->k4_mode = 4;
        } else {
            const double beta = sqrt(s_tot[0]);
            nk->beta = beta;
            nk->eps_fd = NK_EPS_REL * fmax(sqrt(s_tot[2]), 1e-300);   // |q| = 1 in the same norm
            // inexact Newton: first system to 1e-3, later ones to what the tolerance still asks for, never beyond
            // the accuracy of the difference quotient
            double eta = nk->newton_its <= 1 ? 1e-3 : 0.3 * tol / res;
            eta = fmin(1e-3, fmax(eta, NK_ETA_MIN));
            nk->eta = eta;
            nk->res_prev = res;
            nk->backtracks = 0; nk->have_update = 0; nk->lam = 1.0;
            nk->phase = 1; nk->j = 0;
            nk->grhs[0] = beta;
            nk->k4_mode = 1;
        }
    } else {
        double h[NK_MAXM + 2];
        double ss = 0.0;
        for (int i = 0; i <= j; ++i) { h[i] = s_tot[1 + i]; nk->hcol[i] = h[i]; ss += h[i] * h[i]; }
        const double ww = s_tot[0];
        const double hn = sqrt(fmax(ww - ss, 0.0));                   // classical Gram-Schmidt, Pythagoras
        nk->hnorm = hn;
        h[j + 1] = hn;
        for (int i = 0; i < j; ++i) {
            const double t = nk->cs[i] * h[i] + nk->sn[i] * h[i + 1];
            h[i + 1] = -nk->sn[i] * h[i] + nk->cs[i] * h[i + 1];
            h[i] = t;
        }
        const double dn = hypot(h[j], h[j + 1]);
        const double c = dn > 0.0 ? h[j] / dn : 1.0, s = dn > 0.0 ? h[j + 1] / dn : 0.0;
        nk->cs[j] = c; nk->sn[j] = s;
        for (int i = 0; i < j; ++i) nk->R[i][j] = h[i];
        nk->R[j][j] = dn;
        nk->grhs[j + 1] = -s * nk->grhs[j];
        nk->grhs[j] = c * nk->grhs[j];
        const double lin = fabs(nk->grhs[j + 1]);
        const int j1 = j + 1;
        const bool breakdown = !(hn > 1e-13 * sqrt(ww)) || !isfinite(dn);
        if (!isfinite(ww)) { ctrl->err = -4; ctrl->done = 1; }
        else if (it >= max_iter) ctrl->done = 1;                      // commits g(x) of the last phase-0 evaluation
        else if (lin <= nk->eta * nk->beta || j1 >= nk->m || breakdown || it + 1 >= max_iter) {
            for (int r = j1 - 1; r >= 0; --r) {                       // R y = grhs
                double acc = nk->grhs[r];
                for (int cidx = r + 1; cidx < j1; ++cidx) acc -= nk->R[r][cidx] * nk->y[cidx];
                nk->y[r] = nk->R[r][r] != 0.0 ? acc / nk->R[r][r] : 0.0;
            }
            nk->napply = j1;
            nk->k4_mode = 3;
            nk->phase = 0;
            nk->have_update = 1; nk->lam = 1.0; nk->backtracks = 0;
        } else {
            nk->j = j1;
            nk->k4_mode = 2;
        }
    }
    if (cond) cudaGraphSetConditional(cond, ctrl->done ? 0u : 1u);
}

// The vector work that needs the reduced coefficients: q_0 = f/beta; q_{j+1} = (w - sum_i h_i q_i)/h_{j+1,j}; the
// Newton update x += sum_i y_i q_i; or taking part of it back.
__global__ void nk_update_kernel(const DevLayout* __restrict__ L, const StepCtrl* __restrict__ ctrl,
                                 const NewtonCtrl* __restrict__ nk, int npad_max, double* __restrict__ Q,
                                 const double* __restrict__ fvec, double* __restrict__ xk, double* __restrict__ yk,
                                 double* __restrict__ zk) {
    if (ctrl->done) return;
    const int mode = nk->k4_mode;
    if (mode == 0) return;
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= npad_max || p >= L->npad) return;
    const size_t np = (size_t)npad_max, col = 3 * np;
    if (mode == 1) {
        const double ib = 1.0 / nk->beta;
        Q[p] = fvec[p] * ib; Q[np + p] = fvec[np + p] * ib; Q[2 * np + p] = fvec[2 * np + p] * ib;
    } else if (mode == 2) {
        const int jn = nk->j;                                        // index of the new vector
        double* qn = Q + (size_t)jn * col + p;
        double a = qn[0], b = qn[np], c = qn[2 * np];
        for (int i = 0; i < jn; ++i) {
            const double hi = nk->hcol[i];
            const double* qi = Q + (size_t)i * col + p;
            a = fma(-hi, qi[0], a); b = fma(-hi, qi[np], b); c = fma(-hi, qi[2 * np], c);
        }
        const double ih = 1.0 / nk->hnorm;
        qn[0] = a * ih; qn[np] = b * ih; qn[2 * np] = c * ih;
    } else {
        const double sc = mode == 3 ? 1.0 : -nk->lam_back;
        double a = xk[p], b = yk[p], c = zk[p];
        for (int i = 0; i < nk->napply; ++i) {
            const double yi = sc * nk->y[i];
            const double* qi = Q + (size_t)i * col + p;
            a = fma(yi, qi[0], a); b = fma(yi, qi[np], b); c = fma(yi, qi[2 * np], c);
        }
        xk[p] = a; yk[p] = b; zk[p] = c;
    }
}

}  // namespace landau
