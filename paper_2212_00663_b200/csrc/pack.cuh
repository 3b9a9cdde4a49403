// pack.cuh -- step a0 of the hot path: validate, bucket markers by species with a stable counting
// sort (clouds of >= 4096 markers: by species and Morton cell, see below), AoS [N x 3] -> padded SoA
// (common.cuh), permutation back to caller order.
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

// ---- Morton bucketing inside a species ------------------------------------------------------------------------
// Markers of one species are ordered by the Morton (Z-order) index of the cell of a 2^LC x 2^LC x 2^LC mesh over
// the species' bounding box that holds them, markers of one cell in caller order (stable): consecutive slots are
// neighbours in velocity space, so the 64-slot tiles of pass 1 are compact boxes and its Gaussian cutoff
// (entropy.cuh) can skip whole tiles.  Any order is a valid packing (outputs go back through perm), the sums of both
// passes are merely taken in another order.  A stable counting sort on the key (species, cell): per-chunk histograms
// and in-chunk ranks, a scan over chunks and bins, and the scatter.
constexpr int CELL_CHUNK = 2048;            // markers per block of the counting sort
constexpr int CELL_MAX_BINS = 32768;        // species x cells (shared-memory histogram of the count kernel)
constexpr size_t CELL_SCRATCH_MAX_BYTES = (size_t)32 << 20;   // per-chunk histograms of the counting sort, at most

struct SpeciesBox { unsigned long long lo[LD_MAX_SPECIES][3], hi[LD_MAX_SPECIES][3]; };

// order-preserving map double -> unsigned (for atomicMin / atomicMax on coordinates)
__device__ __forceinline__ unsigned long long ordered_bits(double v) {
    const unsigned long long b = (unsigned long long)__double_as_longlong(v);
    return (b >> 63) ? ~b : (b | 0x8000000000000000ull);
}
__device__ __forceinline__ double ordered_value(unsigned long long u) {
    const unsigned long long b = (u >> 63) ? (u & 0x7fffffffffffffffull) : ~u;
    return __longlong_as_double((long long)b);
}

__global__ void pack_box_init_kernel(SpeciesBox* __restrict__ box) {
    const int t = threadIdx.x;
    if (t < LD_MAX_SPECIES * 3) {
        box->lo[t / 3][t % 3] = ~0ull;
        box->hi[t / 3][t % 3] = 0ull;
    }
}

// Bounding box of every species over the caller-order arrays: one atomic set per warp and species present.
__global__ void __launch_bounds__(PACK_THREADS)
pack_box_kernel(int N, const double* __restrict__ v, const int32_t* __restrict__ sid, int S,
                SpeciesBox* __restrict__ box) {
    const int i = blockIdx.x * PACK_THREADS + threadIdx.x;
    const int lane = threadIdx.x & 31;
    int s = -1;
    unsigned long long c[3] = {0ull, 0ull, 0ull};
    if (i < N) {
        s = sid[i];
        if (s < 0 || s >= S) s = -1;
        const double a = v[3 * (size_t)i], b = v[3 * (size_t)i + 1], d = v[3 * (size_t)i + 2];
        if (!(isfinite(a) && isfinite(b) && isfinite(d))) s = -1;
        c[0] = ordered_bits(a); c[1] = ordered_bits(b); c[2] = ordered_bits(d);
    }
    for (int t = 0; t < S; ++t) {
        const unsigned m = __ballot_sync(0xffffffffu, s == t);
        if (!m) continue;
        const int leader = __ffs(m) - 1;
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            unsigned long long lo = s == t ? c[k] : ~0ull, hi = s == t ? c[k] : 0ull;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                const unsigned long long l2 = __shfl_xor_sync(0xffffffffu, lo, o), h2 = __shfl_xor_sync(0xffffffffu, hi, o);
                lo = l2 < lo ? l2 : lo; hi = h2 > hi ? h2 : hi;
            }
            if (lane == leader) { atomicMin(&box->lo[t][k], lo); atomicMax(&box->hi[t][k], hi); }
        }
    }
}

__device__ __forceinline__ int morton_cell(const SpeciesBox* __restrict__ box, int s, int LC, double a, double b,
                                           double c) {
    const double p[3] = {a, b, c};
    int q[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const double lo = ordered_value(box->lo[s][k]), hi = ordered_value(box->hi[s][k]);
        const double ext = hi - lo;
        int t = ext > 0.0 ? (int)((p[k] - lo) / ext * (double)(1 << LC)) : 0;
        q[k] = min(max(t, 0), (1 << LC) - 1);
    }
    int code = 0;
    for (int bit = 0; bit < LC; ++bit)
        code |= (((q[0] >> bit) & 1) << (3 * bit)) | (((q[1] >> bit) & 1) << (3 * bit + 1)) | (((q[2] >> bit) & 1) << (3 * bit + 2));
    return code;
}

// Per chunk of CELL_CHUNK consecutive markers: key and stable in-chunk rank of every marker, chunk histogram.
__global__ void __launch_bounds__(PACK_THREADS)
pack_cell_count_kernel(int N, const double* __restrict__ v, const int32_t* __restrict__ sid, int S, int LC, int nbins,
                       const SpeciesBox* __restrict__ box, int* __restrict__ key, int* __restrict__ rank,
                       int* __restrict__ chunkcnt) {
    extern __shared__ int s_hist[];
    for (int b = threadIdx.x; b < nbins; b += PACK_THREADS) s_hist[b] = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31, wv = threadIdx.x >> 5;
    const int cells = 1 << (3 * LC);
    for (int r = 0; r < CELL_CHUNK / PACK_THREADS; ++r) {
        const int i = blockIdx.x * CELL_CHUNK + r * PACK_THREADS + threadIdx.x;
        int kb = -1;
        if (i < N) {
            int s = sid[i];
            const double a = v[3 * (size_t)i], b = v[3 * (size_t)i + 1], c = v[3 * (size_t)i + 2];
            if (s >= 0 && s < S && isfinite(a) && isfinite(b) && isfinite(c)) kb = s * cells + morton_cell(box, s, LC, a, b, c);
            key[i] = kb;
        }
        for (int q = 0; q < PACK_THREADS / 32; ++q) {          // warps in index order: the ranks are stable
            if (wv == q) {
                const unsigned m = __match_any_sync(0xffffffffu, kb);
                const int leader = __ffs(m) - 1;
                int base = 0;
                if (kb >= 0 && lane == leader) { base = s_hist[kb]; s_hist[kb] = base + __popc(m); }
                base = __shfl_sync(0xffffffffu, base, leader);
                if (kb >= 0) rank[i] = base + __popc(m & ((1u << lane) - 1u));
            }
            __syncthreads();
        }
    }
    for (int b = threadIdx.x; b < nbins; b += PACK_THREADS) chunkcnt[(size_t)blockIdx.x * nbins + b] = s_hist[b];
}

// chunkcnt[chunk][bin] -> exclusive offsets over the chunks of each bin; bintot[bin] = markers of the bin.
__global__ void pack_cell_scan_chunks_kernel(int nchunks, int nbins, int* __restrict__ chunkcnt,
                                             int* __restrict__ bintot) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= nbins) return;
    int run = 0;
    for (int k = 0; k < nchunks; ++k) {
        const int c = chunkcnt[(size_t)k * nbins + b];
        chunkcnt[(size_t)k * nbins + b] = run;
        run += c;
    }
    bintot[b] = run;
}

// Exclusive scan of bintot over the bins (one block); binoff[nbins] = total.
__global__ void __launch_bounds__(1024)
pack_cell_scan_bins_kernel(int nbins, const int* __restrict__ bintot, int* __restrict__ binoff) {
    __shared__ int s_part[1024];
    const int per = ceil_div(nbins, 1024);
    const int b0 = threadIdx.x * per, b1 = min(nbins, b0 + per);
    int sum = 0;
    for (int b = b0; b < b1; ++b) sum += bintot[b];
    s_part[threadIdx.x] = sum;
    __syncthreads();
    if (threadIdx.x == 0) {
        int run = 0;
        for (int k = 0; k < 1024; ++k) { const int c = s_part[k]; s_part[k] = run; run += c; }
        binoff[nbins] = run;
    }
    __syncthreads();
    int run = s_part[threadIdx.x];
    for (int b = b0; b < b1; ++b) { binoff[b] = run; run += bintot[b]; }
}

// Scatter into the padded SoA in (species, Morton cell, caller index) order.
__global__ void __launch_bounds__(PACK_THREADS)
pack_cell_scatter_kernel(int N, const double* __restrict__ v, const double* __restrict__ w, int S, int LC, int nbins,
                         const int* __restrict__ key, const int* __restrict__ rank,
                         const int* __restrict__ chunkoff, const int* __restrict__ binoff,
                         const DevLayout* __restrict__ L, double* __restrict__ x, double* __restrict__ y,
                         double* __restrict__ z, double* __restrict__ wo, int* __restrict__ perm) {
    const int i = blockIdx.x * PACK_THREADS + threadIdx.x;
    if (i >= N) return;
    const int kb = key[i];
    if (kb < 0) return;
    const int cells = 1 << (3 * LC);
    const int s = kb / cells;
    const int pos = binoff[kb] + chunkoff[(size_t)(i / CELL_CHUNK) * nbins + kb] + rank[i];
    const int slot = L->off[s] + (pos - binoff[s * cells]);
    x[slot] = v[3 * (size_t)i];
    y[slot] = v[3 * (size_t)i + 1];
    z[slot] = v[3 * (size_t)i + 2];
    wo[slot] = w[i];
    perm[slot] = i;
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
