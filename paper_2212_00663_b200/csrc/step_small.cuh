// step_small.cuh -- steps a3-a5 of a launch-bound cloud (a few thousand markers: the paper's own tests, BASELINE
// configs 0-1) as ONE persistent kernel: every Jacobi iteration of Eq. (24) (Algorithm 1
// PAPER.md:289-303) inside a single launch, with a grid-wide barrier where the launch sequence has a kernel boundary.
//
// The launch sequence (and the CUDA-graph WHILE node that replays it, landau_api.cu) spends ~25 us per iteration on a
// 2048-marker cloud whose pass 2 is ~4 us of work: two kernel nodes and the re-evaluation of the conditional node per
// iteration.  Here the grid of pair_onesided_kernel (target tiles x source chunks, all CTAs resident: cooperative
// launch) loops over
//     pass 2 (pair_onesided_body, the kernel's own body)  ->  barrier  ->  update + residual partials
//     (step_update_slot, in the 256-slot units and the summation order of step_update_kernel)  ->  barrier  ->
//     every CTA adds the unit partials in index order and takes the same decision,
// so the arithmetic, the order of every sum and therefore the results are bit-identical to the launch sequence
// (tests/test_gpu_parity.py).  Data written by other CTAs inside the launch (source records, partial fields, unit
// partials) is read past L1 (ld.global.cg).  The barrier is a monotone counter zeroed by step_begin_kernel; a wait that
// does not end (a CTA that never became resident: cannot happen under a cooperative launch) raises the error flag
// instead of hanging the GPU.
#pragma once
#include "common.cuh"
#include "pair.cuh"
#include "pair_sym.cuh"   // ld_acquire_gpu
#include "step.cuh"

namespace landau {

__device__ __forceinline__ bool small_grid_barrier(unsigned int* bar, unsigned int target, int* errflag) {
    __shared__ int s_ok;
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        atomicAdd(bar, 1u);
        unsigned spins = 0;
        int ok = 1;
        while ((unsigned)ld_acquire_gpu(reinterpret_cast<const int*>(bar)) < target) {
            if (++spins > (1u << 28)) { atomicExch(errflag, -3); ok = 0; break; }
        }
        __threadfence();
        s_ok = ok;
    }
    __syncthreads();
    return s_ok != 0;
}

// grid = ttiles * nchunks CTAs of PAIR_THREADS threads (1-D: tile = blockIdx.x % ttiles, chunk = blockIdx.x / ttiles);
// needs ceil(npad_max / UPD_THREADS) <= PAIR_THREADS unit partials (npad_max <= 32768).
template <int R, int DIM>
__global__ void __launch_bounds__(PAIR_THREADS)
step_small_kernel(const DevTable* __restrict__ T, DevLayout* __restrict__ L, StepCtrl* ctrl, int npad_max, int ttiles,
                  int nchunks, double dt, double tol, int max_iter, double* rec, double* vpart,
                  const double* __restrict__ xn, const double* __restrict__ yn, const double* __restrict__ zn,
                  const double* __restrict__ w, double* xk, double* yk, double* zk, double* blockpart,
                  unsigned int* bar) {
    __shared__ __align__(16) double sm[PAIR_SRC_TILE * 8];
    __shared__ double s_nu[LD_MAX_SPECIES * LD_MAX_SPECIES];
    __shared__ double s_num[UPD_THREADS / 32], s_den[UPD_THREADS / 32];
    for (int i = threadIdx.x; i < T->S * T->S; i += PAIR_THREADS) s_nu[i] = T->nu[i];
    const int bx = blockIdx.x % ttiles, by = blockIdx.x / ttiles;
    const int G = (int)gridDim.x;
    const int npad = L->npad;
    const int nub = ceil_div(npad_max, UPD_THREADS);
    const int lane = threadIdx.x & 31, wv = threadIdx.x >> 5;
    unsigned int nbar = 0;
    int it = 0;
    for (;;) {
        // ---- pass 2 at the current midpoint records
        pair_onesided_body<R, DIM, false, true>(T, L, npad_max, nchunks, rec, vpart, nullptr, nullptr, bx, by, sm, s_nu);
        if (!small_grid_barrier(bar, ++nbar * (unsigned)G, &L->err)) return;
        // ---- update, in the units of step_update_kernel (256 slots = two halves of this CTA's 128 threads)
        for (int u = blockIdx.x; u < nub; u += G) {
#pragma unroll
            for (int h = 0; h < UPD_THREADS / PAIR_THREADS; ++h) {
                const int p = u * UPD_THREADS + h * PAIR_THREADS + threadIdx.x;
                double num = 0.0, den = 0.0;
                if (p < npad_max && p < npad)
                    step_update_slot<true>(T, L, p, npad_max, nchunks, dt, vpart, xn, yn, zn, w, xk, yk, zk, rec, nullptr,
                                           num, den);
                num = warp_sum(num); den = warp_sum(den);
                if (lane == 0) { s_num[h * (PAIR_THREADS / 32) + wv] = num; s_den[h * (PAIR_THREADS / 32) + wv] = den; }
            }
            __syncthreads();
            if (threadIdx.x == 0) {
                double a = 0.0, b = 0.0;
                for (int k = 0; k < UPD_THREADS / 32; ++k) { a += s_num[k]; b += s_den[k]; }
                blockpart[2 * u] = a; blockpart[2 * u + 1] = b;
            }
            __syncthreads();
        }
        if (!small_grid_barrier(bar, ++nbar * (unsigned)G, &L->err)) return;
        // ---- residual: the last block of step_update_kernel, done by every CTA (same data, same order, same decision)
        double a = 0.0, b = 0.0;
        if ((int)threadIdx.x < nub) { a = __ldcg(blockpart + 2 * threadIdx.x); b = __ldcg(blockpart + 2 * threadIdx.x + 1); }
        a = warp_sum(a); b = warp_sum(b);
        __syncthreads();
        if (lane == 0) { s_num[wv] = a; s_den[wv] = b; }
        __syncthreads();
        double n = 0.0, d = 0.0;
        for (int k = 0; k < PAIR_THREADS / 32; ++k) { n += s_num[k]; d += s_den[k]; }
        // (the other four warps of step_update_kernel's 256-thread block hold zeros when nub <= 128: same sum)
        const double res = sqrt(n / d);
        ++it;
        int done = 0, conv = 0, err = 0;
        if (!isfinite(res)) { err = -4; done = 1; }
        else if (res <= tol) { conv = 1; done = 1; }
        else if (it >= max_iter) done = 1;
        if (blockIdx.x == 0 && threadIdx.x == 0) {
            ctrl->iterations = it; ctrl->residual = res;
            if (err) ctrl->err = err;
            if (conv) ctrl->converged = 1;
            if (done) ctrl->done = 1;
        }
        if (done) return;
        __syncthreads();                                  // s_num is rewritten by the next update phase
    }
}

}  // namespace landau
