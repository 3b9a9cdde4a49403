// entropy.cuh -- steps a1/a2 of the hot path: mollified density at the Gauss-Hermite nodes and the
// entropy gradient, 3-V restatement of Eq. (22) (Eqs. 19-21).
//
//   rho_p(k) = sum_{q in s(p)} w_q (2 pi eps_s)^(-3/2) exp(-|k + (v_p - v_q)/sqrt(2 eps_s)|^2)
//   G_p      = -sqrt(2/eps_s) pi^(-3/2) sum_{ijl} a_i a_j a_l (k_i,k_j,k_l) [1 + ln rho_p(k_ijl)]
//   s_p      = sum_{ijl} a_i a_j a_l ln rho_p(k_ijl)        (S_eps,s = -pi^(-3/2) sum_p w_p s_p)
//
// Two all-pairs kernels produce the node sums  A_p(k) = sum_q w_q exp(...)  :
//   * literal-separable:  exp(-|k+d|^2) = prod_axis exp(-(k_i + d_axis)^2): 3 n_q exponentials per
//     pair, every factor <= 1, no overflow anywhere; valid for any marker cloud.
//   * factorised (entropy_fact.cuh): one exponential per pair, per-marker tables.
// entropy_finalize_kernel turns node sums into G_p and s_p (n_q^3 logarithms per marker).
#pragma once
#include "common.cuh"

namespace landau {

constexpr double FACT_EXP_LIMIT = 500.0;

// Can the factorised kernel be used for this cloud?  (Same answer in every kernel of one pass: the
// layout's half-widths are written once per pass by entropy_bounds_kernel.)
__device__ __forceinline__ bool fact_usable(const DevTable* __restrict__ T, const DevLayout* __restrict__ L) {
    const double kmax = fabs(T->knot[T->n_q - 1]);
    bool ok = true;
    for (int s = 0; s < T->S; ++s) ok = ok && (6.0 * kmax * L->halfwidth[s] <= FACT_EXP_LIMIT);
    return ok;
}

// ---- Gaussian cutoff of pass 1 (second half; the paper's own rule
// eps_s = 1.2 (L_s/N)^1.98, shrinks the mollifier like the marker spacing squared, so that almost every
// same-species pair contributes an exact or numerical zero to Eq. (22)).
// Criterion.  The node sum A_p(k) = sum_q w_q exp(-|k + d_pq|^2) contains the target's own term w_p exp(-|k|^2).
// For a source at distance |d| >= D > |k|_max = sqrt(3) k_max from the target,
//     w_q exp(-|k + d|^2) / (w_p exp(-|k|^2)) <= (w_max/w_min) exp(-(D^2 - 2 D |k|_max)),
// so if  D^2 - 2 D |k|_max >= cut_T = 60 ln 2 + ln(w_max/w_min) + ln N_s  then ALL sources beyond D together change
// A_p(k) by less than 2^-60 relative, i.e. ln A_p(k) by < 1e-18: far below the round-off of the sum itself.  D is the
// distance between the bounding boxes of a target tile and a source tile (64 consecutive slots, mollifier units);
// whole source tiles are skipped.  Tiles are compact when the caller's marker order is (the paper's mesh order is),
// and after the Morton bucketing of pack.cuh for any order.
struct TileBox { double lo[3], hi[3]; };

__device__ __forceinline__ bool tile_is_far(const TileBox& a, const TileBox& b, double cut_T, double kmax3) {
    double d2 = 0.0;
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        const double g = fmax(fmax(a.lo[i] - b.hi[i], b.lo[i] - a.hi[i]), 0.0);
        d2 = fma(g, g, d2);
    }
    const double d = sqrt(d2);
    return !(a.lo[0] <= a.hi[0]) || !(b.lo[0] <= b.hi[0]) || (d > kmax3 && d2 - 2.0 * d * kmax3 >= cut_T);
}

// Bounding box (mollifier units) of the real markers of every tile of 64 slots; an empty tile gets lo > hi.
__global__ void __launch_bounds__(64)
entropy_tilebox_kernel(const DevTable* __restrict__ T, const DevLayout* __restrict__ L, int npad_max,
                       const double* __restrict__ x, const double* __restrict__ y, const double* __restrict__ z,
                       const double* __restrict__ w, TileBox* __restrict__ box, const StepCtrl* __restrict__ stop) {
    if (stop && stop->done) return;      // a device-driven loop (step_dg) has finished: the rest of its launches exit
    const int p = blockIdx.x * 64 + threadIdx.x;
    const double BIG = 1.7976931348623157e308;
    double lo[3] = {BIG, BIG, BIG}, hi[3] = {-BIG, -BIG, -BIG};
    if (p < L->npad && w[p] > 0.0) {
        const double inv = T->inv_sqrt_2eps[species_of_slot(L, T->S, p)];
        lo[0] = hi[0] = x[p] * inv; lo[1] = hi[1] = y[p] * inv; lo[2] = hi[2] = z[p] * inv;
    }
    __shared__ double s[2][6];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            lo[d] = fmin(lo[d], __shfl_xor_sync(0xffffffffu, lo[d], o));
            hi[d] = fmax(hi[d], __shfl_xor_sync(0xffffffffu, hi[d], o));
        }
        if ((threadIdx.x & 31) == 0) { s[threadIdx.x >> 5][d] = lo[d]; s[threadIdx.x >> 5][3 + d] = hi[d]; }
    }
    __syncthreads();
    if (threadIdx.x < 3) {
        box[blockIdx.x].lo[threadIdx.x] = fmin(s[0][threadIdx.x], s[1][threadIdx.x]);
        box[blockIdx.x].hi[threadIdx.x] = fmax(s[0][3 + threadIdx.x], s[1][3 + threadIdx.x]);
    }
}

__device__ __forceinline__ TileBox box_union(const TileBox& a, const TileBox& b) {
    TileBox r;
#pragma unroll
    for (int i = 0; i < 3; ++i) { r.lo[i] = fmin(a.lo[i], b.lo[i]); r.hi[i] = fmax(a.hi[i], b.hi[i]); }
    return r;
}

constexpr int ENT_THREADS = 128;   // targets per block (one target per thread)
constexpr int ENT_SRC_TILE = 64;   // sources staged in shared memory per tile

// Node sums are stored node-major: part[((chunk * M + node) * npad_max) + slot].
//
// NQ knots per axis; each thread owns NI consecutive x-node indices i (i0 = blockIdx.z * NI) and all
// (j,l): NI*NQ*NQ accumulators in registers.
template <int NQ, int NI>
__global__ void __launch_bounds__(ENT_THREADS)
entropy_literal_kernel(const DevTable* __restrict__ T, const DevLayout* __restrict__ L, int npad_max,
                       int nchunks, int skip_if_fact, const double* __restrict__ x,
                       const double* __restrict__ y, const double* __restrict__ z,
                       const double* __restrict__ w, const TileBox* __restrict__ box,
                       unsigned long long* __restrict__ cutstats, double* __restrict__ part,
                       const StepCtrl* __restrict__ stop) {
    if (stop && stop->done) return;
    const int slot0 = blockIdx.x * ENT_THREADS;
    if (slot0 >= L->npad) return;
    if (skip_if_fact && fact_usable(T, L)) return;   // the factorised kernel does this pass
    const int S = T->S;
    const int s = species_of_slot(L, S, slot0);
    const double inv = T->inv_sqrt_2eps[s];
    const int src0 = L->off[s], src1 = L->off[s + 1];
    const int ntiles = (src1 - src0) / ENT_SRC_TILE;
    const int tpc = ceil_div(ntiles, nchunks);
    const int t0 = blockIdx.y * tpc, t1 = min(ntiles, t0 + tpc);
    const int i0 = (NI == NQ) ? 0 : blockIdx.z * NI;
    static_assert(ENT_THREADS == 2 * ENT_SRC_TILE, "a target tile is two boxes");
    const TileBox tbox = box_union(box[slot0 / ENT_SRC_TILE], box[slot0 / ENT_SRC_TILE + 1]);
    const double cutT = L->cut_T[s], kmax3 = 1.7320508075688772 * fabs(T->knot[NQ - 1]);
    int nskip = 0;

    __shared__ double sx[ENT_SRC_TILE], sy[ENT_SRC_TILE], sz[ENT_SRC_TILE], sw[ENT_SRC_TILE];
    double kn[NQ];
#pragma unroll
    for (int i = 0; i < NQ; ++i) kn[i] = T->knot[i];

    const int p = slot0 + threadIdx.x;
    const double px = x[p] * inv, py = y[p] * inv, pz = z[p] * inv;
    double acc[NI][NQ][NQ];
#pragma unroll
    for (int i = 0; i < NI; ++i)
#pragma unroll
        for (int j = 0; j < NQ; ++j)
#pragma unroll
            for (int l = 0; l < NQ; ++l) acc[i][j][l] = 0.0;

    for (int t = t0; t < t1; ++t) {
        if (tile_is_far(tbox, box[src0 / ENT_SRC_TILE + t], cutT, kmax3)) { ++nskip; continue; }   // block-uniform
        __syncthreads();
        if (threadIdx.x < ENT_SRC_TILE) {
            const int q = src0 + t * ENT_SRC_TILE + threadIdx.x;
            sx[threadIdx.x] = x[q] * inv;
            sy[threadIdx.x] = y[q] * inv;
            sz[threadIdx.x] = z[q] * inv;
            sw[threadIdx.x] = w[q];
        }
        __syncthreads();
#pragma unroll 1
        for (int j0 = 0; j0 < ENT_SRC_TILE; ++j0) {
            const double dx = px - sx[j0], dy = py - sy[j0], dz = pz - sz[j0];
            const double wq = sw[j0];
            double ex[NI], ey[NQ], ez[NQ];
#pragma unroll
            for (int i = 0; i < NI; ++i) { const double a = kn[i0 + i] + dx; ex[i] = wq * exp(-a * a); }
#pragma unroll
            for (int i = 0; i < NQ; ++i) { const double a = kn[i] + dy; ey[i] = exp(-a * a); }
#pragma unroll
            for (int i = 0; i < NQ; ++i) { const double a = kn[i] + dz; ez[i] = exp(-a * a); }
#pragma unroll
            for (int i = 0; i < NI; ++i)
#pragma unroll
                for (int j = 0; j < NQ; ++j) {
                    const double b = ex[i] * ey[j];
#pragma unroll
                    for (int l = 0; l < NQ; ++l) acc[i][j][l] = fma(b, ez[l], acc[i][j][l]);
                }
        }
    }
    if (threadIdx.x == 0 && blockIdx.z == 0 && t1 > t0) {
        atomicAdd(cutstats, (unsigned long long)(t1 - t0));
        atomicAdd(cutstats + 1, (unsigned long long)nskip);
    }
    const size_t M = (size_t)NQ * NQ * NQ;
#pragma unroll
    for (int i = 0; i < NI; ++i)
#pragma unroll
        for (int j = 0; j < NQ; ++j)
#pragma unroll
            for (int l = 0; l < NQ; ++l) {
                const size_t node = ((size_t)(i0 + i) * NQ + j) * NQ + l;
                part[((size_t)blockIdx.y * M + node) * (size_t)npad_max + p] = acc[i][j][l];
            }
}

// Node sums -> G_p (unscaled: (1/w_p) dS_eps/dv_p) and s_p.  fact_mode: 0 = the node sums are the
// literal kernel's; 1 = they are the factorised kernel's if fact_usable() (automatic choice), else the
// literal kernel's; 2 = factorised forced (a cloud that is too wide raises LANDAU_ERANGE = -5).
// planar = 1: the factorised kernel summed only the n_q^2 nodes (k_i, k_j, 0) of the 2-V setting (v_z = 0, where
// the node sum does not depend on k_l beyond the factor exp(-k_l^2)); the z-quadrature is then done in closed form:
//   sum_l a_l k_l [1 + ln rho_ijl] = 0,   sum_l a_l [1 + ln rho_ijl] = (sum_l a_l)(1 + ln rho_ij0) - sum_l a_l k_l^2,
// the last term dropping out of G by the antisymmetry of the knots in i and j -- which gives the paper's 2-V Eq. (22)
// exactly and the same s_p as the n_q^3-node evaluation.
// One block = FIN_MARKERS consecutive slots; warp w takes the nodes w, w + FIN_SLICES, ... of all of them (coalesced reads
// of the node sums, n_q^3 / FIN_SLICES logarithms per thread), the slices meet in shared memory and are added in slice
// order (deterministic).  Round 1: one thread per marker walked all n_q^3 nodes x chunks serially -- 178 us for the
// 8192 markers of BASELINE config 1, as long as the contraction itself.
constexpr int FIN_MARKERS = 32, FIN_SLICES = 8, FIN_THREADS = FIN_MARKERS * FIN_SLICES;

__global__ void __launch_bounds__(FIN_THREADS)
entropy_finalize_kernel(const DevTable* __restrict__ T, DevLayout* __restrict__ L, int npad_max,
                        int nchunks, const int* __restrict__ perm, const double* __restrict__ part,
                        const double* __restrict__ px, const double* __restrict__ py,
                        const double* __restrict__ pz, int fact_mode, int planar,
                        double* __restrict__ Gx, double* __restrict__ Gy, double* __restrict__ Gz,
                        double* __restrict__ snode, const StepCtrl* __restrict__ stop) {
    if (stop && stop->done) return;
    const int lane = threadIdx.x & 31, slice = threadIdx.x >> 5;
    const int p = blockIdx.x * FIN_MARKERS + lane;
    if (blockIdx.x * FIN_MARKERS >= L->npad) return;                 // block-uniform
    const bool factorised = fact_mode != 0 && fact_usable(T, L);
    if (p == 0 && slice == 0) L->used_fact = factorised ? 1 : 0;
    if (fact_mode == 2 && !factorised) { if (p == 0 && slice == 0) atomicMin(&L->err, -5); return; }
    const bool real = p < L->npad && perm[p] >= 0;
    const int S = T->S, nq = T->n_q;
    const int s = species_of_slot(L, S, min(p, L->npad - 1));
    const double eps = T->eps[s];
    const double PI = 3.14159265358979323846;
    const double lognorm = -1.5 * log(2.0 * PI * eps);
    // factorised form: ln A_p(k) = -|k|^2 - 2 k.(p - c) + ln(sum); (p - c) in mollifier units
    double cx = 0.0, cy = 0.0, cz = 0.0;
    if (factorised && real) {
        const double inv = T->inv_sqrt_2eps[s];
        cx = (px[p] - L->center[s][0]) * inv;
        cy = (py[p] - L->center[s][1]) * inv;
        cz = (pz[p] - L->center[s][2]) * inv;
    }
    double gx = 0.0, gy = 0.0, gz = 0.0, sn = 0.0;
    if (real) {
        if (planar && factorised) {
            double az = 0.0, azk2 = 0.0, axy = 0.0;
            for (int l = 0; l < nq; ++l) { az += T->gw[l]; azk2 = fma(T->gw[l], T->knot[l] * T->knot[l], azk2); }
            const int M2 = nq * nq;
            for (int node = slice; node < M2; node += FIN_SLICES) {
                const int i = node / nq, j = node - i * nq;
                double a = 0.0;
                for (int c = 0; c < nchunks; ++c) a += part[((size_t)c * M2 + node) * (size_t)npad_max + p];
                const double ki = T->knot[i], kj = T->knot[j];
                const double lnrho = lognorm + log(a) - ((ki * ki + kj * kj) + 2.0 * (ki * cx + kj * cy));
                const double aa = T->gw[i] * T->gw[j];
                const double t = aa * az * (1.0 + lnrho);
                gx = fma(t, ki, gx); gy = fma(t, kj, gy);
                sn = fma(aa * az, lnrho, sn);
                axy += aa;
            }
            sn -= axy * azk2;
        } else {
            const int M = nq * nq * nq;
            for (int node = slice; node < M; node += FIN_SLICES) {
                const int i = node / (nq * nq), j = (node / nq) % nq, l = node % nq;
                double a = 0.0;
                for (int c = 0; c < nchunks; ++c) a += part[((size_t)c * M + node) * (size_t)npad_max + p];
                const double ki = T->knot[i], kj = T->knot[j], kl = T->knot[l];
                double lnrho = lognorm + log(a);
                if (factorised)
                    lnrho -= (ki * ki + kj * kj + kl * kl) + 2.0 * (ki * cx + kj * cy + kl * cz);
                const double aaa = T->gw[i] * T->gw[j] * T->gw[l];
                const double t = aaa * (1.0 + lnrho);
                gx = fma(t, ki, gx); gy = fma(t, kj, gy); gz = fma(t, kl, gz);
                sn = fma(aaa, lnrho, sn);
            }
        }
    }
    __shared__ double s_red[FIN_SLICES][4][FIN_MARKERS];
    s_red[slice][0][lane] = gx; s_red[slice][1][lane] = gy; s_red[slice][2][lane] = gz; s_red[slice][3][lane] = sn;
    __syncthreads();
    if (slice != 0 || p >= L->npad) return;
    gx = gy = gz = sn = 0.0;
#pragma unroll
    for (int k = 0; k < FIN_SLICES; ++k) { gx += s_red[k][0][lane]; gy += s_red[k][1][lane]; gz += s_red[k][2][lane]; sn += s_red[k][3][lane]; }
    if (!real) { Gx[p] = 0.0; Gy[p] = 0.0; Gz[p] = 0.0; snode[p] = 0.0; return; }
    const double pref = -sqrt(2.0 / eps) / (PI * sqrt(PI));
    gx *= pref; gy *= pref; gz *= pref;
    if (!(isfinite(gx) && isfinite(gy) && isfinite(gz) && isfinite(sn))) atomicMin(&L->err, -4);
    // 2-V mode (NEXT-2): with v_z = 0 the z-sum cancels analytically (knots are antisymmetric); storing an exact
    // zero keeps the v_z = 0 manifold invariant (g_z = 0 => every pair term has u_z = 0 exactly)
    Gx[p] = gx; Gy[p] = gy; Gz[p] = (T->dim == 2) ? 0.0 : gz; snode[p] = sn;
}

}  // namespace landau
