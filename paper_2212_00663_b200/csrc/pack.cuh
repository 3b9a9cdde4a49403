// pack.cuh -- step a0 of the hot path: validate, bucket markers by species with a stable counting
// sort, AoS [N x 3] -> padded SoA (common.cuh), permutation back to caller order.
// The paper initialises its markers per species (Algorithm 1); the C ABI accepts
// any order, so the bucketing is ours.  Everything runs on the device; the layout (counts, padded
// offsets) stays in device memory so no host round trip is needed before the passes are launched.
#pragma once
#include "common.cuh"

namespace landau {

constexpr int PACK_THREADS = 256;

// Per-block species histogram + input validation.
__global__ void __launch_bounds__(PACK_THREADS)
pack_count_kernel(int N, const double* __restrict__ v, const double* __restrict__ w,
                  const int32_t* __restrict__ sid, int S, int* __restrict__ blockcnt,
                  DevLayout* __restrict__ L) {
    __shared__ int cnt[PACK_THREADS / 32][LD_MAX_SPECIES];
    const int i = blockIdx.x * PACK_THREADS + threadIdx.x;
    const int lane = threadIdx.x & 31, wv = threadIdx.x >> 5;
    int s = -1;
    if (i < N) {
        s = sid[i];
        int bad = 0;
        if (s < 0 || s >= S) { bad = -1; s = -1; }
        const double wi = w[i];
        const double a = v[3 * (size_t)i], b = v[3 * (size_t)i + 1], c = v[3 * (size_t)i + 2];
        if (!(isfinite(wi) && isfinite(a) && isfinite(b) && isfinite(c))) bad = -4;
        else if (!(wi > 0.0)) bad = -1;
        if (bad) atomicMin(&L->err, bad);
    }
    for (int t = 0; t < S; ++t) {
        const unsigned m = __ballot_sync(0xffffffffu, s == t);
        if (lane == 0) cnt[wv][t] = __popc(m);
    }
    __syncthreads();
    if (threadIdx.x < S) {
        int c = 0;
        for (int k = 0; k < PACK_THREADS / 32; ++k) c += cnt[k][threadIdx.x];
        blockcnt[blockIdx.x * S + threadIdx.x] = c;
    }
}

// Exclusive scan of the block histograms per species; padded species offsets.
__global__ void pack_scan_kernel(int nblocks, int S, int pad, const int* __restrict__ blockcnt,
                                 int* __restrict__ blockoff, DevLayout* __restrict__ L) {
    __shared__ int total[LD_MAX_SPECIES];
    const int s = threadIdx.x;
    if (s < S) {
        int run = 0;
        for (int b = 0; b < nblocks; ++b) {
            const int c = blockcnt[b * S + s];
            blockoff[b * S + s] = run;
            run += c;
        }
        total[s] = run;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        int off = 0;
        for (int t = 0; t < S; ++t) {
            L->count[t] = total[t];
            L->off[t] = off;
            off += ceil_div(total[t], pad) * pad;
        }
        for (int t = S; t <= LD_MAX_SPECIES; ++t) L->off[t] = off;
        L->npad = off;
    }
}

// Stable scatter into the padded SoA.  Dummy slots keep the zeros / -1 the arrays were cleared to.
__global__ void __launch_bounds__(PACK_THREADS)
pack_scatter_kernel(int N, const double* __restrict__ v, const double* __restrict__ w,
                    const int32_t* __restrict__ sid, int S, const int* __restrict__ blockoff,
                    const DevLayout* __restrict__ L, double* __restrict__ x, double* __restrict__ y,
                    double* __restrict__ z, double* __restrict__ wo, int* __restrict__ perm) {
    __shared__ int cnt[PACK_THREADS / 32][LD_MAX_SPECIES];
    const int i = blockIdx.x * PACK_THREADS + threadIdx.x;
    const int lane = threadIdx.x & 31, wv = threadIdx.x >> 5;
    int s = -1;
    if (i < N) {
        s = sid[i];
        if (s < 0 || s >= S) s = -1;
    }
    int rank = 0;
    for (int t = 0; t < S; ++t) {
        const unsigned m = __ballot_sync(0xffffffffu, s == t);
        if (lane == 0) cnt[wv][t] = __popc(m);
        if (s == t) rank = __popc(m & ((1u << lane) - 1u));
    }
    __syncthreads();
    if (s >= 0) {
        for (int k = 0; k < wv; ++k) rank += cnt[k][s];
        const int slot = L->off[s] + blockoff[blockIdx.x * S + s] + rank;
        x[slot] = v[3 * (size_t)i];
        y[slot] = v[3 * (size_t)i + 1];
        z[slot] = v[3 * (size_t)i + 2];
        wo[slot] = w[i];
        perm[slot] = i;
    }
}

// Gather a caller-order [N x 3] array into packed SoA (used for a supplied entropy gradient).
__global__ void gather3_kernel(int npad_max, const DevLayout* __restrict__ L, const int* __restrict__ perm,
                               const double* __restrict__ a, double* __restrict__ ox,
                               double* __restrict__ oy, double* __restrict__ oz) {
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= npad_max || p >= L->npad) return;
    const int i = perm[p];
    double ax = 0.0, ay = 0.0, az = 0.0;
    if (i >= 0) {
        ax = a[3 * (size_t)i]; ay = a[3 * (size_t)i + 1]; az = a[3 * (size_t)i + 2];
        if (!(isfinite(ax) && isfinite(ay) && isfinite(az))) atomicMin(const_cast<int*>(&L->err), -4);
    }
    ox[p] = ax; oy[p] = ay; oz[p] = az;
}

// Scatter packed SoA back to a caller-order [N x 3] array.
__global__ void scatter3_kernel(int npad_max, DevLayout* __restrict__ L, const int* __restrict__ perm,
                                const double* __restrict__ ax, const double* __restrict__ ay,
                                const double* __restrict__ az, double* __restrict__ out) {
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= npad_max || p >= L->npad) return;
    const int i = perm[p];
    if (i < 0) return;
    const double a = ax[p], b = ay[p], c = az[p];
    if (!(isfinite(a) && isfinite(b) && isfinite(c))) atomicMin(&L->err, -4);
    out[3 * (size_t)i] = a; out[3 * (size_t)i + 1] = b; out[3 * (size_t)i + 2] = c;
}

}  // namespace landau
