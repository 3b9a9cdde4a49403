// entropy_fact.cuh -- step a1 of the hot path, factorised form: ONE exponential per same-species pair.
//
// Eq. (22) (PAPER.md:130-134, 3-V restatement DESIGN.md section 3 D1) needs, for every marker p of
// species s and every tensor Gauss-Hermite node k = (k_i, k_j, k_l),
//     A_p(k) = sum_{q in s} w_q exp(-|k + d_pq|^2),     d_pq = (v_p - v_q)/sqrt(2 eps_s).
// With a per-species centre c_s and p' = (v_p - c_s)/sqrt(2 eps_s), q' likewise (d_pq = p' - q'):
//     exp(-|k + d|^2) = exp(-|k|^2) * prod_axis exp(-2 k_a p'_a)            (target only, applied in finalize)
//                     * exp(-|d|^2)                                          (the one per-pair exponential)
//                     * prod_axis exp(+2 k_a q'_a)                           (source only: per-marker table)
// so   F_p(i,j,l) = sum_q [w_q exp(-|d_pq|^2)] Tx_q(i) Ty_q(j) Tz_q(l),     T._q(i) = exp(2 k_i q'_.)
// and  ln A_p(k) = -|k|^2 - 2 k.p' + ln F_p(k)   (entropy_finalize_kernel, factorised = 1).
// Per pair: 1 exponential + NI + NI*NQ multiplies + NI*NQ^2 accumulate-FMAs (the algorithmic minimum of
// SURVEY.md section 8(d)), against 3 NQ exponentials in the literal kernel (entropy.cuh).
//
// Range (reading N3): the source tables grow like exp(2 k_max h_s) per axis, h_s the
// species' half-width in mollifier units.  entropy_bounds_kernel measures h_s; fact_usable() admits the
// factorised form only when 6 k_max h_s <= FACT_EXP_LIMIT for every species, which keeps every factor,
// every product and every node sum inside the FP64 range with ~200 in the exponent to spare.  Wider
// clouds take the literal kernel, whose factors are all <= 1.
#pragma once
#include "common.cuh"
#include "entropy.cuh"   // fact_usable()
#include "pair_sym.cuh"   // mbarrier / bulk-copy helpers

namespace landau {

constexpr int FACT_TILE = 64;        // sources per shared-memory stage
constexpr int FACT_THREADS = 128;    // one target per thread

template <int NQ>
struct FactCfg {
    static constexpr int REC = (4 + 3 * NQ + 1) & ~1;   // doubles per source record (even: 16-byte rows)
};

// One block per species: bounding box of its (real) markers -> centre and half-width.
__global__ void __launch_bounds__(1024)
entropy_bounds_kernel(const DevTable* __restrict__ T, DevLayout* __restrict__ L, const double* __restrict__ x,
                      const double* __restrict__ y, const double* __restrict__ z, const double* __restrict__ w,
                      int cutoff_on, const StepCtrl* __restrict__ stop, unsigned long long* __restrict__ cutstats) {
    if (stop && stop->done) return;
    const int s = blockIdx.x;
    if (s == 0 && threadIdx.x == 0) { cutstats[0] = 0ull; cutstats[1] = 0ull; }   // counters of this pass (Gaussian cutoff)
    const int p0 = L->off[s], p1 = L->off[s + 1];
    const double BIG = 1.7976931348623157e308;
    double lo[3] = {BIG, BIG, BIG}, hi[3] = {-BIG, -BIG, -BIG};
    double wlo = BIG, whi = 0.0;
    for (int p = p0 + threadIdx.x; p < p1; p += blockDim.x) {
        if (w[p] > 0.0) {
            const double a = x[p], b = y[p], c = z[p];
            lo[0] = fmin(lo[0], a); hi[0] = fmax(hi[0], a);
            lo[1] = fmin(lo[1], b); hi[1] = fmax(hi[1], b);
            lo[2] = fmin(lo[2], c); hi[2] = fmax(hi[2], c);
            wlo = fmin(wlo, w[p]); whi = fmax(whi, w[p]);
        }
    }
    __shared__ double slo[32][3], shi[32][3], swlo[32], swhi[32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        wlo = fmin(wlo, __shfl_xor_sync(0xffffffffu, wlo, o));
        whi = fmax(whi, __shfl_xor_sync(0xffffffffu, whi, o));
    }
    if ((threadIdx.x & 31) == 0) { swlo[threadIdx.x >> 5] = wlo; swhi[threadIdx.x >> 5] = whi; }
    const int lane = threadIdx.x & 31, wv = threadIdx.x >> 5;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            lo[d] = fmin(lo[d], __shfl_xor_sync(0xffffffffu, lo[d], o));
            hi[d] = fmax(hi[d], __shfl_xor_sync(0xffffffffu, hi[d], o));
        }
        if (lane == 0) { slo[wv][d] = lo[d]; shi[wv][d] = hi[d]; }
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double hw = 0.0;
        for (int d = 0; d < 3; ++d) {
            double a = BIG, b = -BIG;
            for (int k = 0; k < (int)(blockDim.x >> 5); ++k) { a = fmin(a, slo[k][d]); b = fmax(b, shi[k][d]); }
            if (a > b) { a = 0.0; b = 0.0; }                       // species without markers
            L->center[s][d] = 0.5 * a + 0.5 * b;
            hw = fmax(hw, 0.5 * b - 0.5 * a);
        }
        L->halfwidth[s] = hw * T->inv_sqrt_2eps[s];
        // Gaussian cutoff threshold of this species (entropy.cuh, tile_is_far)
        double a = BIG, b = 0.0;
        for (int k = 0; k < (int)(blockDim.x >> 5); ++k) { a = fmin(a, swlo[k]); b = fmax(b, swhi[k]); }
        const int cnt = L->count[s];
        L->cut_T[s] = (cutoff_on && cnt > 0 && a > 0.0 && b >= a)
                          ? 60.0 * 0.69314718055994531 + log(b / a) + log((double)cnt) : BIG;
    }
}

// Per-slot source record {x', y', z', w, Tx[NQ], Ty[NQ], Tz[NQ]}; dummies are all-zero records, so as
// sources they add exactly 0 whatever the centre is.
template <int NQ>
__global__ void entropy_fact_prep_kernel(const DevTable* __restrict__ T, const DevLayout* __restrict__ L,
                                         int npad_max, const double* __restrict__ x,
                                         const double* __restrict__ y, const double* __restrict__ z,
                                         const double* __restrict__ w, double* __restrict__ rec,
                                         const StepCtrl* __restrict__ stop) {
    if (stop && stop->done) return;
    constexpr int REC = FactCfg<NQ>::REC;
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= npad_max) return;
    if (!fact_usable(T, L)) return;
    double r[REC];
#pragma unroll
    for (int k = 0; k < REC; ++k) r[k] = 0.0;
    if (p < L->npad && w[p] > 0.0) {
        const int s = species_of_slot(L, T->S, p);
        const double inv = T->inv_sqrt_2eps[s];
        r[0] = (x[p] - L->center[s][0]) * inv;
        r[1] = (y[p] - L->center[s][1]) * inv;
        r[2] = (z[p] - L->center[s][2]) * inv;
        r[3] = w[p];
#pragma unroll
        for (int i = 0; i < NQ; ++i) {
            const double k2 = 2.0 * T->knot[i];
            r[4 + i] = exp(k2 * r[0]);
            r[4 + NQ + i] = exp(k2 * r[1]);
            r[4 + 2 * NQ + i] = exp(k2 * r[2]);
        }
    }
    double2* o = reinterpret_cast<double2*>(rec + (size_t)p * REC);
#pragma unroll
    for (int k = 0; k < REC / 2; ++k) o[k] = make_double2(r[2 * k], r[2 * k + 1]);
}

// exp(-r2) for r2 >= 0, FP64, ~1 ulp: n = round(-r2 log2 e), r = -r2 - n ln 2 (two-term Cody-Waite),
// degree-13 Taylor polynomial on |r| <= ln2/2 (truncation 4e-18 relative), scaling by 2^n through the
// exponent field.  Arguments beyond 708 return 0 (the literal term is < 1e-307 there; with the
// range guard above it cannot matter to any node sum).  17 FP64-pipe instructions.
__device__ __forceinline__ double exp_neg(double r2) {
    const double x = -r2;
    const double MAGIC = 6755399441055744.0;                      // 1.5 * 2^52: round-to-nearest by addition
    double t = fma(x, 1.4426950408889634074, MAGIC);
    const int n = __double2loint(t);
    t -= MAGIC;
    double r = fma(t, -6.93147180369123816490e-01, x);
    r = fma(t, -1.90821492927058770002e-10, r);
    double p = 1.6059043836821614599e-10;                          // 1/13!
    p = fma(p, r, 2.0876756987868098979e-09);                      // 1/12!
    p = fma(p, r, 2.5052108385441718775e-08);                      // 1/11!
    p = fma(p, r, 2.7557319223985890653e-07);                      // 1/10!
    p = fma(p, r, 2.7557319223985892511e-06);                      // 1/9!
    p = fma(p, r, 2.4801587301587301566e-05);                      // 1/8!
    p = fma(p, r, 1.9841269841269841253e-04);                      // 1/7!
    p = fma(p, r, 1.3888888888888889419e-03);                      // 1/6!
    p = fma(p, r, 8.3333333333333332177e-03);                      // 1/5!
    p = fma(p, r, 4.1666666666666664354e-02);                      // 1/4!
    p = fma(p, r, 1.6666666666666665741e-01);                      // 1/3!
    p = fma(p, r, 0.5);
    p = fma(p, r, 1.0);
    p = fma(p, r, 1.0);
    const double res = __hiloint2double(__double2hiint(p) + (n << 20), __double2loint(p));
    return r2 > 708.0 ? 0.0 : res;
}

// grid = (target tiles of 128 slots, source chunks, NQ/NI node groups).  Each thread owns one target
// and the NI*NQ*NQ node sums with i in [i0, i0+NI).  Source records arrive by TMA bulk copies
// (cp.async.bulk + mbarrier), double buffered.  Output layout as entropy_literal_kernel:
// part[((chunk * M + node) * npad_max) + slot].
template <int NQ, int NI>
__global__ void __launch_bounds__(FACT_THREADS)
entropy_fact_kernel(const DevTable* __restrict__ T, const DevLayout* __restrict__ L, int npad_max, int nchunks,
                    const double* __restrict__ rec, double* __restrict__ part, const StepCtrl* __restrict__ stop) {
    if (stop && stop->done) return;
    constexpr int REC = FactCfg<NQ>::REC;
    const int slot0 = blockIdx.x * FACT_THREADS;
    if (slot0 >= L->npad) return;
    if (!fact_usable(T, L)) return;
    const int S = T->S;
    const int s = species_of_slot(L, S, slot0);
    const int src0 = L->off[s], src1 = L->off[s + 1];
    const int ntiles = (src1 - src0) / FACT_TILE;
    const int tpc = ceil_div(ntiles, nchunks);
    const int t0 = blockIdx.y * tpc, t1 = min(ntiles, t0 + tpc);
    const int i0 = (NI == NQ) ? 0 : blockIdx.z * NI;

    __shared__ __align__(128) double s_rec[2][FACT_TILE * REC];
    __shared__ __align__(8) uint64_t s_bar[2];
    const int tid = threadIdx.x;
    if (tid == 0) {
        mbar_init(&s_bar[0], 1);
        mbar_init(&s_bar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    auto issue = [&](int t, int stage) {
        if (tid == 0) {
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            constexpr uint32_t BYTES = FACT_TILE * REC * (uint32_t)sizeof(double);
            mbar_expect_tx(&s_bar[stage], BYTES);
            bulk_g2s(&s_rec[stage][0], rec + ((size_t)src0 + (size_t)t * FACT_TILE) * REC, BYTES, &s_bar[stage]);
        }
    };

    const int p = slot0 + tid;
    const double px = rec[(size_t)p * REC], py = rec[(size_t)p * REC + 1], pz = rec[(size_t)p * REC + 2];
    double acc[NI][NQ][NQ];
#pragma unroll
    for (int i = 0; i < NI; ++i)
#pragma unroll
        for (int j = 0; j < NQ; ++j)
#pragma unroll
            for (int l = 0; l < NQ; ++l) acc[i][j][l] = 0.0;

    uint32_t phase_bits = 0;
    int stage = 0;
    if (t0 < t1) issue(t0, 0);
    for (int t = t0; t < t1; ++t) {
        if (t + 1 < t1) issue(t + 1, stage ^ 1);
        mbar_wait(&s_bar[stage], (phase_bits >> stage) & 1u);
        phase_bits ^= 1u << stage;
        const double* sr = &s_rec[stage][0];
#pragma unroll 2
        for (int q = 0; q < FACT_TILE; ++q) {
            const double* r = sr + q * REC;
            const double2 a = *reinterpret_cast<const double2*>(r);
            const double2 b = *reinterpret_cast<const double2*>(r + 2);
            const double dx = px - a.x, dy = py - a.y, dz = pz - b.x;
            const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
            const double c = b.y * exp_neg(r2);
            double ty[NQ], tz[NQ];
#pragma unroll
            for (int j = 0; j < NQ; ++j) { ty[j] = r[4 + NQ + j]; tz[j] = r[4 + 2 * NQ + j]; }
#pragma unroll
            for (int i = 0; i < NI; ++i) {
                const double cx = c * r[4 + i0 + i];
#pragma unroll
                for (int j = 0; j < NQ; ++j) {
                    const double cxy = cx * ty[j];
#pragma unroll
                    for (int l = 0; l < NQ; ++l) acc[i][j][l] = fma(cxy, tz[l], acc[i][j][l]);
                }
            }
        }
        __syncthreads();
        stage ^= 1;
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

}  // namespace landau
