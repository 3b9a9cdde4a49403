// moments.cuh -- step a6 of the hot path: per-species diagnostics as device reductions.
//   n_s = sum w (Eq. 33), P_s = m_s sum w v (Eq. 26),
//   K_s = (m_s/2) sum w |v|^2 (Eq. 28), stress m_s sum w v_i v_j (Eqs. 30-31),
//   S_eps,s = -pi^(-3/2) sum_p w_p s_p (Eq. 20; s_p from entropy.cuh),
//   m4_i = sum w (v_i - u_i)^4.
// Pairwise (tree) FP64 sums in a fixed order: 128-slot blocks (species-uniform, pad % 128 == 0),
// then one block per species over that species' block partials.
#pragma once
#include "common.cuh"

namespace landau {

constexpr int MOM_THREADS = 128;
constexpr int MOM_NQ = 12;   // w, wx, wy, wz, w|v|^2, wxx, wyy, wzz, wxy, wxz, wyz, w*s_p
constexpr int MOM_OUT = 16;  // per species: the 12 sums + m4 x,y,z + spare

template <int NV>
__device__ __forceinline__ void block_sum_store(double (&v)[NV], double* __restrict__ out) {
    __shared__ double sm[MOM_THREADS / 32][NV];
    const int lane = threadIdx.x & 31, wv = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < NV; ++k) {
        const double s = warp_sum(v[k]);
        if (lane == 0) sm[wv][k] = s;
    }
    __syncthreads();
    if (threadIdx.x < NV) {
        double s = 0.0;
#pragma unroll
        for (int k = 0; k < MOM_THREADS / 32; ++k) s += sm[k][threadIdx.x];
        out[threadIdx.x] = s;
    }
    __syncthreads();
}

__global__ void __launch_bounds__(MOM_THREADS)
moments_block_kernel(const DevLayout* __restrict__ L, int npad_max, const double* __restrict__ x,
                     const double* __restrict__ y, const double* __restrict__ z,
                     const double* __restrict__ w, const double* __restrict__ snode,
                     double* __restrict__ blockpart) {
    const int p = blockIdx.x * MOM_THREADS + threadIdx.x;
    double v[MOM_NQ];
#pragma unroll
    for (int k = 0; k < MOM_NQ; ++k) v[k] = 0.0;
    if (p < npad_max && p < L->npad) {
        const double a = x[p], b = y[p], c = z[p], ww = w[p];
        v[0] = ww; v[1] = ww * a; v[2] = ww * b; v[3] = ww * c;
        v[4] = ww * (a * a + b * b + c * c);
        v[5] = ww * a * a; v[6] = ww * b * b; v[7] = ww * c * c;
        v[8] = ww * a * b; v[9] = ww * a * c; v[10] = ww * b * c;
        v[11] = snode ? ww * snode[p] : 0.0;
    }
    block_sum_store<MOM_NQ>(v, blockpart + (size_t)blockIdx.x * MOM_NQ);
}

// One block per species: fixed-order sum of its block partials.  which = 0: the 12 sums into
// out[s*MOM_OUT + 0..11]; which = 1: three m4 partials into out[s*MOM_OUT + 12..14].
__global__ void __launch_bounds__(MOM_THREADS)
moments_species_kernel(const DevLayout* __restrict__ L, const double* __restrict__ blockpart, int nv,
                       int dst, double* __restrict__ out) {
    const int s = blockIdx.x;
    const int b0 = L->off[s] / MOM_THREADS, b1 = L->off[s + 1] / MOM_THREADS;
    double v[MOM_NQ];
#pragma unroll
    for (int k = 0; k < MOM_NQ; ++k) v[k] = 0.0;
    for (int b = b0 + threadIdx.x; b < b1; b += MOM_THREADS)
#pragma unroll
        for (int k = 0; k < MOM_NQ; ++k)
            if (k < nv) v[k] += blockpart[(size_t)b * nv + k];
    __shared__ double res[MOM_NQ];
    block_sum_store<MOM_NQ>(v, res);
    if (threadIdx.x < nv) out[s * MOM_OUT + dst + threadIdx.x] = res[threadIdx.x];
}

// Central fourth moments about u = (sum w v)/(sum w) taken from the species sums.
__global__ void __launch_bounds__(MOM_THREADS)
moments_m4_block_kernel(const DevTable* __restrict__ T, const DevLayout* __restrict__ L, int npad_max,
                        const double* __restrict__ x, const double* __restrict__ y,
                        const double* __restrict__ z, const double* __restrict__ w,
                        const double* __restrict__ sums, double* __restrict__ blockpart) {
    const int p = blockIdx.x * MOM_THREADS + threadIdx.x;
    double v[3] = {0.0, 0.0, 0.0};
    if (p < npad_max && p < L->npad) {
        const int s = species_of_slot(L, T->S, p);
        const double n = sums[s * MOM_OUT];
        const double ux = n > 0.0 ? sums[s * MOM_OUT + 1] / n : 0.0;
        const double uy = n > 0.0 ? sums[s * MOM_OUT + 2] / n : 0.0;
        const double uz = n > 0.0 ? sums[s * MOM_OUT + 3] / n : 0.0;
        const double a = x[p] - ux, b = y[p] - uy, c = z[p] - uz, ww = w[p];
        v[0] = ww * a * a * a * a; v[1] = ww * b * b * b * b; v[2] = ww * c * c * c * c;
    }
    block_sum_store<3>(v, blockpart + (size_t)blockIdx.x * 3);
}

}  // namespace landau
