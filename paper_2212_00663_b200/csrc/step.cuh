// step.cuh -- steps a4/a5 of the hot path: the implicit midpoint-Q step, Eq. (24)-(25)
// (Algorithm 1), solved by Jacobi fixed-point iteration with
// the entropy gradient frozen at t_n:
//
//   v^(0) = v^n;  u = (v^n + v^(k))/2;  V = pass2(u; G^n);  v^(k+1) = v^n + dt V
//   r_k = sqrt( sum w m |v^(k+1) - v^(k)|^2 / sum w m |v^(k+1)|^2 ),  stop at r_k <= tol or k+1 = max_iter
//
// The loop is driven from the device.  Large clouds: every iteration's kernels are enqueued up front and exit
// at once when StepCtrl::done is set.  Small clouds (launch-latency bound): the whole step is one CUDA graph whose
// iteration body sits in a conditional WHILE node that step_update_kernel keeps alive through
// cudaGraphSetConditional until the step is done (landau_api.cu, build_step_graph).  Either way the host never
// waits inside a step.  The residual is reduced in a fixed order (block partials, then the last block to finish
// sums them in index order), so iteration counts are reproducible run to run.
#pragma once
#include "common.cuh"

namespace landau {

constexpr int UPD_THREADS = 256;

// Start of a step: reset the control block, v^(0) = v^n, source records at u = v^n with g = G^n/m.
__global__ void step_begin_kernel(const DevTable* __restrict__ T, const DevLayout* __restrict__ L,
                                  StepCtrl* __restrict__ ctrl, int npad_max,
                                  const double* __restrict__ xn, const double* __restrict__ yn,
                                  const double* __restrict__ zn, const double* __restrict__ w,
                                  const double* __restrict__ Gx, const double* __restrict__ Gy,
                                  const double* __restrict__ Gz, double* __restrict__ xk,
                                  double* __restrict__ yk, double* __restrict__ zk,
                                  double* __restrict__ rec, double* __restrict__ soa, int start_f32 = 0) {
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p == 0) {
        ctrl->done = 0; ctrl->iterations = 0; ctrl->converged = 0; ctrl->ticket = 0u; ctrl->use_f32 = start_f32;
        ctrl->residual = __longlong_as_double(0x7ff0000000000000LL);
    }
    if (p >= npad_max) return;
    if (p >= L->npad) {
        if (soa)
            for (int c = 0; c < 7; ++c) soa[(size_t)c * npad_max + p] = 0.0;
        return;
    }
    const double im = T->inv_mass[species_of_slot(L, T->S, p)];
    const double a = xn[p], b = yn[p], c = zn[p];
    xk[p] = a; yk[p] = b; zk[p] = c;
    const double g0 = Gx[p] * im, g1 = Gy[p] * im, g2 = Gz[p] * im, ww = w[p];
    if (rec) {
        double2* o = reinterpret_cast<double2*>(rec + (size_t)p * 8);
        o[0] = make_double2(a, b);
        o[1] = make_double2(c, ww);
        o[2] = make_double2(g0, g1);
        o[3] = make_double2(g2, 0.0);
    }
    if (soa) {
        soa[p] = a; soa[(size_t)npad_max + p] = b; soa[2 * (size_t)npad_max + p] = c;
        soa[3 * (size_t)npad_max + p] = ww;
        soa[4 * (size_t)npad_max + p] = g0; soa[5 * (size_t)npad_max + p] = g1; soa[6 * (size_t)npad_max + p] = g2;
    }
}

// Slot p of the Jacobi update: v^(k+1) = v^n + dt * (fixed-order sum of the partial fields), its share of the residual
// sums, the next midpoint into the source records.  COH: the partial fields and the iterate were written by other CTAs
// of the same launch (step_small.cuh) and are read past L1.
template <bool COH>
__device__ __forceinline__ void step_update_slot(const DevTable* __restrict__ T, const DevLayout* __restrict__ L,
                                                 int p, int npad_max, int nparts, double dt, const double* vpart,
                                                 const double* __restrict__ xn, const double* __restrict__ yn,
                                                 const double* __restrict__ zn, const double* __restrict__ w, double* xk,
                                                 double* yk, double* zk, double* rec, double* soa, double& num,
                                                 double& den) {
    double a = 0.0, b = 0.0, c = 0.0;
    for (int k = 0; k < nparts; ++k) {
        const double* o = vpart + (size_t)k * 3 * (size_t)npad_max + p;
        if (COH) { a += __ldcg(o); b += __ldcg(o + (size_t)npad_max); c += __ldcg(o + 2 * (size_t)npad_max); }
        else { a += o[0]; b += o[(size_t)npad_max]; c += o[2 * (size_t)npad_max]; }
    }
    const double wp = w[p];
    if (wp == 0.0) { a = 0.0; b = 0.0; c = 0.0; }          // dummies stay at the origin
    const double x0 = xn[p], y0 = yn[p], z0 = zn[p];
    const double x1 = fma(dt, a, x0), y1 = fma(dt, b, y0), z1 = fma(dt, c, z0);
    const double dx = x1 - xk[p], dy = y1 - yk[p], dz = z1 - zk[p];      // xk[p] is only ever touched by p's own thread
    const double wm = wp * T->mass[species_of_slot(L, T->S, p)];
    num = wm * (dx * dx + dy * dy + dz * dz);
    den = wm * (x1 * x1 + y1 * y1 + z1 * z1);
    xk[p] = x1; yk[p] = y1; zk[p] = z1;
    const double ux = 0.5 * (x0 + x1), uy = 0.5 * (y0 + y1), uz = 0.5 * (z0 + z1);   // Eq. (25)
    if (rec) {
        double2* o = reinterpret_cast<double2*>(rec + (size_t)p * 8);
        o[0] = make_double2(ux, uy);
        reinterpret_cast<double*>(o + 1)[0] = uz;
    }
    if (soa) { soa[p] = ux; soa[(size_t)npad_max + p] = uy; soa[2 * (size_t)npad_max + p] = uz; }
}

// v^(k+1) = v^n + dt * (fixed-order sum of the partial fields); residual; next midpoint records.
__global__ void __launch_bounds__(UPD_THREADS)
step_update_kernel(const DevTable* __restrict__ T, const DevLayout* __restrict__ L,
                   StepCtrl* __restrict__ ctrl, int npad_max, int nparts, double dt, double tol,
                   int max_iter, const double* __restrict__ vpart, const double* __restrict__ xn,
                   const double* __restrict__ yn, const double* __restrict__ zn,
                   const double* __restrict__ w, double* __restrict__ xk, double* __restrict__ yk,
                   double* __restrict__ zk, double* __restrict__ rec, double* __restrict__ soa,
                   double* __restrict__ blockpart, cudaGraphConditionalHandle cond, double f32_until = 0.0) {
    if (ctrl->done) return;
    __shared__ double s_num[UPD_THREADS / 32], s_den[UPD_THREADS / 32];
    __shared__ int s_last;
    const int p = blockIdx.x * UPD_THREADS + threadIdx.x;
    double num = 0.0, den = 0.0;
    if (p < npad_max && p < L->npad)
        step_update_slot<false>(T, L, p, npad_max, nparts, dt, vpart, xn, yn, zn, w, xk, yk, zk, rec, soa, num, den);
    num = warp_sum(num); den = warp_sum(den);
    const int lane = threadIdx.x & 31, wv = threadIdx.x >> 5;
    if (lane == 0) { s_num[wv] = num; s_den[wv] = den; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double a = 0.0, b = 0.0;
        for (int k = 0; k < UPD_THREADS / 32; ++k) { a += s_num[k]; b += s_den[k]; }
        blockpart[2 * blockIdx.x] = a; blockpart[2 * blockIdx.x + 1] = b;
        __threadfence();
        const unsigned t = atomicInc(&ctrl->ticket, gridDim.x - 1);
        s_last = (t == gridDim.x - 1);
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    double a = 0.0, b = 0.0;
    for (int k = threadIdx.x; k < (int)gridDim.x; k += UPD_THREADS) {
        a += __ldcg(blockpart + 2 * k); b += __ldcg(blockpart + 2 * k + 1);
    }
    a = warp_sum(a); b = warp_sum(b);
    __syncthreads();
    if (lane == 0) { s_num[wv] = a; s_den[wv] = b; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double n = 0.0, d = 0.0;
        for (int k = 0; k < UPD_THREADS / 32; ++k) { n += s_num[k]; d += s_den[k]; }
        const double res = sqrt(n / d);
        const int it = ctrl->iterations + 1;
        ctrl->iterations = it;
        ctrl->residual = res;
        // mixed-precision step: pass 2 runs in FP32 while the iterates still move by more than f32_until; an iterate
        // that came from an FP32 evaluation never ends the step as converged (the next evaluation is FP64)
        const int was_f32 = ctrl->use_f32;
        // ... and the last iteration the caller allows is always FP64, so that a step that ends at max_iter commits
        // an FP64 iterate as well
        ctrl->use_f32 = (f32_until > 0.0 && res > f32_until && it + 1 < max_iter) ? 1 : 0;
        if (!isfinite(res)) { ctrl->err = -4; ctrl->done = 1; }
        else if (res <= tol && !was_f32) { ctrl->converged = 1; ctrl->done = 1; }
        else if (it >= max_iter) ctrl->done = 1;
        // CUDA-graph mode: this kernel is the last node of a WHILE body; keep looping until the step is done
        if (cond) cudaGraphSetConditional(cond, ctrl->done ? 0u : 1u);
    }
}

// End of a step: v^n <- last iterate (committed whether or not it converged, reading S8).
__global__ void step_commit_kernel(const DevLayout* __restrict__ L, StepCtrl* __restrict__ ctrl,
                                   int npad_max, double* __restrict__ xn, double* __restrict__ yn,
                                   double* __restrict__ zn, const double* __restrict__ xk,
                                   const double* __restrict__ yk, const double* __restrict__ zk,
                                   StepRecord* __restrict__ records, int* __restrict__ record_cursor) {
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p == 0) {
        const int i = (*record_cursor)++;
        records[i].iterations = ctrl->iterations;
        records[i].residual = ctrl->residual;
        records[i].converged = ctrl->converged;
    }
    if (p >= npad_max || p >= L->npad) return;
    if (ctrl->err) return;
    if (ctrl->hold && !ctrl->converged) return;      // adaptive sub-stepping: the caller retries with a shorter step
    xn[p] = xk[p]; yn[p] = yk[p]; zn[p] = zk[p];
}

}  // namespace landau
