// step_dg.cuh -- SURVEY.md section 8(f) NEXT-1: the discrete-gradient step, Eqs. (46)-(49).
//
//   (v^{n+1} - v^n)/dt = (1/m_s) sum_s' sum_q w_q nu_ss' Q(Gamma(K,p,q)) Gamma(S_eps,p,q)          Eq. (46)
//   Gamma(A,p,q) = (1/(m_s w_p)) dbar A/dv_p - (1/(m_s' w_q)) dbar A/dv_q                           Eq. (47)
//
// The discrete gradient of the quadratic K is its midpoint gradient, so Q is evaluated at the midpoint
// difference u_p - u_q exactly as in Eq. (24).  For S_eps the paper leaves the choice open; reading DG1
// takes Gonzalez' midpoint discrete gradient (the paper's ref. [39]) in the Euclidean inner product
// of all 3N velocity components:
//   dbar S/dv_p = w_p G_p(u) + lambda (v_p^{n+1} - v_p^n),
//   lambda = [S(v^{n+1}) - S(v^n) - sum_p w_p G_p(u).(v_p^{n+1} - v_p^n)] / sum_p |v_p^{n+1} - v_p^n|^2,
// which satisfies Eq. (48) identically and therefore Eq. (49): S_eps^{n+1} >= S_eps^n.
// Every fixed-point iteration costs two pass-1 evaluations (G at the midpoint, S at the iterate) and one
// pass 2; the kernels below are the O(N) glue around the existing all-pairs kernels.  The loop is device driven:
// the entropies, lambda's two sums and the convergence decision are reduced on the device (block partials, last
// block in index order) into DgCtrl / StepCtrl, every kernel of an iteration exits at once when the step is done,
// and the host only looks at the done flag once per chunk of enqueued iterations.
#pragma once
#include "common.cuh"

namespace landau {

constexpr int DG_THREADS = 256;

struct DgCtrl {
    double S0;           // S_eps(v^n), all species
    double Sk;           // S_eps(v^(k))
    double lin, dv2;     // sum_p w_p G_p(u).dv_p,  sum_p |dv_p|^2
    double lambda;
    unsigned int ticket;
    int _r;
};

__global__ void dg_begin_kernel(DgCtrl* __restrict__ dg) {
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        dg->S0 = 0.0; dg->Sk = 0.0; dg->lin = 0.0; dg->dv2 = 0.0; dg->lambda = 0.0; dg->ticket = 0u;
    }
}

// Total regularised entropy  S = -pi^(-3/2) sum_p w_p s_p  (Eq. 20; s_p from entropy_finalize_kernel) into
// dg->S0 (which = 0) or dg->Sk (which = 1).
__global__ void __launch_bounds__(DG_THREADS)
dg_entropy_total_kernel(const DevLayout* __restrict__ L, const StepCtrl* __restrict__ ctrl, int npad_max,
                        const double* __restrict__ w, const double* __restrict__ snode,
                        double* __restrict__ part, DgCtrl* __restrict__ dg, int which) {
    if (ctrl->done) return;
    __shared__ double s_a[DG_THREADS / 32];
    __shared__ int s_last;
    const int p = blockIdx.x * DG_THREADS + threadIdx.x;
    double a = 0.0;
    if (p < npad_max && p < L->npad && w[p] > 0.0) a = w[p] * snode[p];
    a = warp_sum(a);
    const int lane = threadIdx.x & 31, wv = threadIdx.x >> 5;
    if (lane == 0) s_a[wv] = a;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int k = 0; k < DG_THREADS / 32; ++k) t += s_a[k];
        part[blockIdx.x] = t;
        __threadfence();
        const unsigned tk = atomicInc(&dg->ticket, gridDim.x - 1);
        s_last = (tk == gridDim.x - 1);
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    double t = 0.0;
    for (int k = threadIdx.x; k < (int)gridDim.x; k += DG_THREADS) t += __ldcg(part + k);
    t = warp_sum(t);
    __syncthreads();
    if (lane == 0) s_a[wv] = t;
    __syncthreads();
    if (threadIdx.x == 0) {
        double tot = 0.0;
        for (int k = 0; k < DG_THREADS / 32; ++k) tot += s_a[k];
        const double PI = 3.14159265358979323846;
        const double S = -tot / (PI * sqrt(PI));
        if (which == 0) dg->S0 = S; else dg->Sk = S;
    }
}

// u = (v^n + v^(k))/2 into a cloud-shaped buffer {x,y,z,w}[npad_max] (dummies: 0, w = 0).
__global__ void dg_midpoint_kernel(const DevLayout* __restrict__ L, const StepCtrl* __restrict__ ctrl, int npad_max,
                                   const double* __restrict__ xn,
                                   const double* __restrict__ yn, const double* __restrict__ zn,
                                   const double* __restrict__ w, const double* __restrict__ xk,
                                   const double* __restrict__ yk, const double* __restrict__ zk,
                                   double* __restrict__ u) {
    if (ctrl->done) return;
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= npad_max) return;
    double a = 0.0, b = 0.0, c = 0.0, ww = 0.0;
    if (p < L->npad) {
        a = 0.5 * (xn[p] + xk[p]); b = 0.5 * (yn[p] + yk[p]); c = 0.5 * (zn[p] + zk[p]); ww = w[p];
    }
    u[p] = a; u[(size_t)npad_max + p] = b; u[2 * (size_t)npad_max + p] = c; u[3 * (size_t)npad_max + p] = ww;
}

// lin = sum_p w_p G_p(u).dv_p  and  dv2 = sum_p |dv_p|^2,  dv = v^(k) - v^n  (block partials, then the last block
// adds them in index order), and Gonzalez' lambda = (S_k - S_0 - lin)/dv2 (0 if dv = 0).
__global__ void __launch_bounds__(DG_THREADS)
dg_lambda_kernel(const DevLayout* __restrict__ L, const StepCtrl* __restrict__ ctrl, DgCtrl* __restrict__ dg,
                 int npad_max, const double* __restrict__ xn,
                         const double* __restrict__ yn, const double* __restrict__ zn,
                         const double* __restrict__ w, const double* __restrict__ xk,
                         const double* __restrict__ yk, const double* __restrict__ zk,
                         const double* __restrict__ Gx, const double* __restrict__ Gy,
                         const double* __restrict__ Gz, double* __restrict__ part) {
    if (ctrl->done) return;
    __shared__ double s_a[DG_THREADS / 32], s_b[DG_THREADS / 32];
    __shared__ int s_last;
    const int p = blockIdx.x * DG_THREADS + threadIdx.x;
    double lin = 0.0, dv2 = 0.0;
    if (p < npad_max && p < L->npad && w[p] > 0.0) {
        const double dx = xk[p] - xn[p], dy = yk[p] - yn[p], dz = zk[p] - zn[p];
        lin = w[p] * fma(Gz[p], dz, fma(Gy[p], dy, Gx[p] * dx));
        dv2 = fma(dz, dz, fma(dy, dy, dx * dx));
    }
    lin = warp_sum(lin); dv2 = warp_sum(dv2);
    const int lane = threadIdx.x & 31, wv = threadIdx.x >> 5;
    if (lane == 0) { s_a[wv] = lin; s_b[wv] = dv2; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double a = 0.0, b = 0.0;
        for (int k = 0; k < DG_THREADS / 32; ++k) { a += s_a[k]; b += s_b[k]; }
        part[2 * blockIdx.x] = a; part[2 * blockIdx.x + 1] = b;
        __threadfence();
        const unsigned tk = atomicInc(&dg->ticket, gridDim.x - 1);
        s_last = (tk == gridDim.x - 1);
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    if (threadIdx.x == 0) {
        double a = 0.0, b = 0.0;
        for (int k = 0; k < (int)gridDim.x; ++k) { a += __ldcg(part + 2 * k); b += __ldcg(part + 2 * k + 1); }
        dg->lin = a; dg->dv2 = b;
        dg->lambda = b > 0.0 ? (dg->Sk - dg->S0 - a) / b : 0.0;
    }
}

// Sources of pass 2 at the midpoint u with  g_p = (G_p(u) + lambda dv_p / w_p)/m_s  (records or SoA copy).
__global__ void dg_build_kernel(const DevTable* __restrict__ T, const DevLayout* __restrict__ L,
                                const StepCtrl* __restrict__ ctrl, const DgCtrl* __restrict__ dg, int npad_max,
                                const double* __restrict__ u, const double* __restrict__ xn,
                                const double* __restrict__ yn, const double* __restrict__ zn,
                                const double* __restrict__ xk, const double* __restrict__ yk,
                                const double* __restrict__ zk, const double* __restrict__ Gx,
                                const double* __restrict__ Gy, const double* __restrict__ Gz,
                                double* __restrict__ rec, double* __restrict__ soa) {
    if (ctrl->done) return;
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= npad_max) return;
    const double lambda = dg->lambda;
    double v[7] = {0, 0, 0, 0, 0, 0, 0};
    if (p < L->npad) {
        const double ww = u[3 * (size_t)npad_max + p];
        v[0] = u[p]; v[1] = u[(size_t)npad_max + p]; v[2] = u[2 * (size_t)npad_max + p]; v[3] = ww;
        if (ww > 0.0) {
            const double im = T->inv_mass[species_of_slot(L, T->S, p)];
            const double s = lambda / ww;
            v[4] = fma(s, xk[p] - xn[p], Gx[p]) * im;
            v[5] = fma(s, yk[p] - yn[p], Gy[p]) * im;
            v[6] = fma(s, zk[p] - zn[p], Gz[p]) * im;
        }
    }
    if (rec && p < L->npad) {
        double2* o = reinterpret_cast<double2*>(rec + (size_t)p * 8);
        o[0] = make_double2(v[0], v[1]); o[1] = make_double2(v[2], v[3]);
        o[2] = make_double2(v[4], v[5]); o[3] = make_double2(v[6], 0.0);
    }
    if (soa)
#pragma unroll
        for (int c = 0; c < 7; ++c) soa[(size_t)c * npad_max + p] = v[c];
}

}  // namespace landau
