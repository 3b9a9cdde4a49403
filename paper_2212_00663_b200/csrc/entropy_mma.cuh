// entropy_mma.cuh -- step a1 of the hot path as a dense FP64 contraction on the tensor pipe (DMMA).
//
// The factorised node sums of entropy_fact.cuh (Eq. (22); 3-V restatement DESIGN.md
// section 3 D1),
//     F_p(n) = sum_{q in s} C_pq * P_q(n),   C_pq = exp(-|p' - q'|^2),   P_q(n) = w_q Tx_q(i) Ty_q(j) Tz_q(l),
// with n = (i,j,l) a tensor Gauss-Hermite node, ARE a matrix product  F[targets x nodes] = C[targets x sources]
// * P[sources x nodes]  whose left factor is generated on the fly (one exponential per pair).  This kernel
// issues it as  mma.sync.m8n8k4.f64 (SASS DMMA.8x8x4):  a warp owns 8*MT targets x NL <= 64 nodes of
// accumulators in registers; per k-step of 4 sources each lane computes the MT entries C[lane/4 + 8 mt][lane%4]
// of the A fragments (its own exponentials), reads the NBG entries P[lane%4][8 nb + lane/4] of the B fragments
// from the product table in shared memory, and issues MT*NBG DMMAs.  Per pair the FP64 pipe sees
// 16 vector instructions (|d|^2, exponential) + n_q^3 tensor FMAs, against 108 vector instructions in
// entropy_fact_kernel; on B200 DMMA and DFMA share one pipe (profiles/r1_entropy_fact_v3_full.md), so the gain
// is the removed product/issue overhead and DMMA's 12/12 (vs DFMA's 11/12) pipe efficiency, not overlap.
//
// The product table is the SAME for every target tile, so it is built once per pass 1 in global memory
// (entropy_prod_kernel: row of slot q and node group g = { P_q(node0 + 0..NL), x', y', z', 0 }, ROW = NL + 4 doubles,
// the weight folded into the products) and a tile of 64 rows arrives as ONE TMA bulk copy (double buffered, one
// __syncthreads per tile).  Round 1-2 built the table inside every block from the per-marker factor records: a serial
// LDS -> DMUL -> STS chain that took 20 % of every warp's time (profiles/r2_entropy_mma_full.md).  A species' table
// (544 B per marker at n_q = 4) stays L2 resident while the co-resident blocks stream it.  ROW = NL + 4 is 4 or 12
// mod 16, so the B-fragment reads of a half-warp fall into 16 distinct bank pairs.
// Nodes beyond n_q^3 (padding of the last 8-node block) have P = 0.
// Output layout as the other pass-1 kernels: part[((chunk * M + node) * npad_max) + slot].
#pragma once
#include "common.cuh"
#include "entropy.cuh"
#include "entropy_fact.cuh"

namespace landau {

constexpr int MMA_THREADS = 128;   // 4 warps, 32 targets each
constexpr int MMA_TILE = 64;       // sources per stage
constexpr int MMA_MT = 4;          // 8-target blocks per warp
#ifndef LANDAU_MMA_STAGES            // tuning knob (build.py: LANDAU_NVCC_EXTRA); 3 measured: no gain
#define LANDAU_MMA_STAGES 2
#endif
constexpr int MMA_STAGES = LANDAU_MMA_STAGES;      // product-table tiles in shared memory
constexpr int MMA_LCAP = 1024;     // source tiles per segment of the active-tile list (Gaussian cutoff)

// NZ = NQ: the 3-V tensor grid of n_q^3 nodes.  NZ = 1: the paper's own 2-V setting (landau_set_dimension(2), v_z = 0):
// the z-factor of every node is exp(0) = 1 and the z-quadrature is done in closed form by entropy_finalize_kernel, so
// only the n_q^2 nodes (k_i, k_j, 0) are summed -- a quarter of the tensor work at n_q = 4.
template <int NQ, int NZ = NQ>
struct MmaCfg {
    static constexpr int M = NQ * NQ * NZ;
    static constexpr int NB = (M + 7) / 8;                          // 8-node blocks
    static constexpr int NBG = NB <= 8 ? NB : (NQ == 6 ? 7 : 8);    // blocks per node group (gridDim.z)
    static constexpr int GROUPS = (NB + NBG - 1) / NBG;
    static constexpr int NL = NBG * 8;                              // nodes per group (<= 64)
    static constexpr int ROW = NL + 4;                              // doubles per product-table row
    static constexpr int REC = FactCfg<NQ>::REC;
    static constexpr uint32_t TILE_BYTES = MMA_TILE * ROW * (uint32_t)sizeof(double);
    static constexpr size_t SMEM =
        sizeof(double) * (MMA_STAGES * MMA_TILE * ROW + 256) + MMA_STAGES * sizeof(uint64_t) +
        sizeof(int) * (MMA_LCAP + 8);
    static size_t table_bytes(size_t npad_max) { return sizeof(double) * ROW * npad_max * GROUPS; }
};

// Product table of pass 1 (one launch per pass): tab[(g * npad_max + q) * ROW + c] = w_q Tx_q(i) Ty_q(j) Tz_q(l) for
// node n = g * NL + c = (i, j, l), c < NL (0 beyond n_q^3), then {x', y', z', 0}; from the factor records of
// entropy_fact_prep_kernel.  Dummies have all-zero rows: as sources they add exactly 0.
template <int NQ, int NZ>
__global__ void entropy_prod_kernel(const DevTable* __restrict__ T, const DevLayout* __restrict__ L, int npad_max,
                                    const double* __restrict__ rec, double* __restrict__ tab,
                                    const StepCtrl* __restrict__ stop) {
    if (stop && stop->done) return;
    using C = MmaCfg<NQ, NZ>;
    const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (size_t)npad_max * C::ROW) return;
    if (!fact_usable(T, L)) return;
    const int q = (int)(idx / C::ROW), c = (int)(idx - (size_t)q * C::ROW);
    const double* r = rec + (size_t)q * C::REC;
    double v = 0.0;
    if (c < C::NL) {
        const int nd = blockIdx.y * C::NL + c;
        if (nd < C::M) {
            v = r[4 + nd / (NQ * NZ)] * r[4 + NQ + (nd / NZ) % NQ];
            if (NZ != 1) v *= r[4 + 2 * NQ + nd % NZ];
            v *= r[3];
        }
    } else if (c < C::NL + 3) {
        v = r[c - C::NL];
    }
    tab[((size_t)blockIdx.y * npad_max + q) * C::ROW + c] = v;
}

// exp(-r2) for r2 >= 0, FP64, ~1.5 ulp, 10 FP64-pipe instructions: N = round(-r2 * 64/ln 2),
// r = -r2 - N ln2/64 (two-term Cody-Waite, |r| <= ln2/128), exp(r) by its degree-5 Taylor polynomial
// (truncation r^6/720 < 3.5e-17), times 2^(j/64) from a 64-entry table (j = N mod 64) and 2^(N div 64)
// through the exponent field.  Arguments beyond 708 return 0.
__device__ __forceinline__ double exp_neg_tab(double r2, const double* __restrict__ s_e2) {
    const double x = -r2;
    const double MAGIC = 6755399441055744.0;                       // 1.5 * 2^52
    double t = fma(x, 92.332482616893656877, MAGIC);               // 64 / ln 2
    const int N = __double2loint(t);
    t -= MAGIC;
    double r = fma(t, -1.08304246932675596327e-02, x);             // ln2_hi / 64 (33 significant bits)
    r = fma(t, -2.98158582698529328128e-12, r);                    // ln2_lo / 64
    double p = 8.3333333333333332177e-03;                          // 1/5!
    p = fma(p, r, 4.1666666666666664354e-02);                      // 1/4!
    p = fma(p, r, 1.6666666666666665741e-01);                      // 1/3!
    p = fma(p, r, 0.5);
    p = fma(p, r, 1.0);
    p = fma(p, r, 1.0);
    p *= s_e2[N & 63];
    const int hi = __double2hiint(p) + ((N >> 6) << 20);
    const bool far = __double2hiint(r2) > 0x40862000;              // r2 > 708 (r2 >= 0: integer order)
    return __hiloint2double(far ? 0 : hi, far ? 0 : __double2loint(p));
}

// exp(-r2) for r2 >= 0 as used by the contraction kernel: <= 1.5 ulp with 9 FP64-pipe instructions (exp_neg_tab: 10).
// N = round(-r2 * 256/ln 2), r = -r2 - N ln2/256 (two-term Cody-Waite, |r| <= ln2/512 = 1.36e-3),
// exp(r) - 1 = r (1 + r (1/2 + r (1/6 + r/24)))  (dropped r^5/120 < 4e-17), times 2^(j/256) from a 256-entry table
// (j = N mod 256) and 2^(N div 256) through the exponent field.  Arguments beyond 708 return 0.
// (Measured and dropped: the cubic part in FP32 through the bit patterns -- 7 FP64 instructions, but the longer
// dependent chain FP64 -> integer -> FP32 -> FP64 costs more than the two FMAs: 68.0 against 62.8 ms per pass.)
__device__ __forceinline__ double exp_neg_t256(double r2, const double* __restrict__ s_e2) {
    const double x = -r2;
    const double MAGIC = 6755399441055744.0;                       // 1.5 * 2^52
    double t = fma(x, 369.32993046757462751, MAGIC);               // 256 / ln 2
    const int N = __double2loint(t);
    t -= MAGIC;
    double r = fma(t, -1.08304246932675596327e-02 / 4.0, x);       // ln2_hi / 256 (33 significant bits)
    r = fma(t, -2.98158582698529328128e-12 / 4.0, r);              // ln2_lo / 256
    double p = fma(r, 4.1666666666666664354e-02, 1.6666666666666665741e-01);
    p = fma(p, r, 0.5);
    p = fma(p, r, 1.0);
    p *= r;
    const double tab = s_e2[N & 255];
    p = fma(tab, p, tab);
    const int hi = __double2hiint(p) + ((N >> 8) << 20);
    const bool far = __double2hiint(r2) > 0x40862000;              // r2 > 708 (r2 >= 0: integer order)
    return __hiloint2double(far ? 0 : hi, far ? 0 : __double2loint(p));
}

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}

// grid = (target tiles of 128 slots, source chunks, MmaCfg<NQ, NZ>::GROUPS node groups).
template <int NQ, int NZ = NQ>
__global__ void __launch_bounds__(MMA_THREADS, 2)
entropy_mma_kernel(const DevTable* __restrict__ T, const DevLayout* __restrict__ L, int npad_max, int nchunks,
                   const double* __restrict__ tab, const TileBox* __restrict__ box,
                   unsigned long long* __restrict__ cutstats, double* __restrict__ part,
                   const StepCtrl* __restrict__ stop) {
    if (stop && stop->done) return;
    using C = MmaCfg<NQ, NZ>;
    constexpr int ROW = C::ROW, MT = MMA_MT, NBG = C::NBG, NL = C::NL, M = C::M;
    const int slot0 = blockIdx.x * MMA_THREADS;
    if (slot0 >= L->npad) return;
    if (!fact_usable(T, L)) return;
    const int S = T->S;
    const int s = species_of_slot(L, S, slot0);
    const int src0 = L->off[s], src1 = L->off[s + 1];
    const int ntiles = (src1 - src0) / MMA_TILE;
    const int tpc = ceil_div(ntiles, nchunks);
    const int t0 = blockIdx.y * tpc, t1 = min(ntiles, t0 + tpc);
    const int node0 = blockIdx.z * NL;
    const double* gtab = tab + (size_t)blockIdx.z * npad_max * ROW;   // this node group's table

    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* s_prod = reinterpret_cast<double*>(smem_raw);            // [MMA_STAGES][MMA_TILE][ROW]
    double* s_e2 = s_prod + MMA_STAGES * MMA_TILE * ROW;             // [256]  2^(j/256)
    uint64_t* s_bar = reinterpret_cast<uint64_t*>(s_e2 + 256);        // [MMA_STAGES]
    int* s_list = reinterpret_cast<int*>(s_bar + MMA_STAGES);        // [MMA_LCAP] active source tiles of a segment
    int* s_wcnt = s_list + MMA_LCAP;                                 // [4]
    const int tid = threadIdx.x, lane = tid & 31, wv = tid >> 5;
    const int lr = lane >> 2, lc = lane & 3;                         // fragment row / column of this lane
    for (int i = tid; i < 256; i += MMA_THREADS) s_e2[i] = T->exp2_tab256[i];
    if (tid == 0) {
#pragma unroll
        for (int b = 0; b < MMA_STAGES; ++b) mbar_init(&s_bar[b], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // gk counts the tiles loaded by this block so far (stage = gk % STAGES, mbarrier parity = (gk / STAGES) & 1);
    // li is the tile's position in the active list of the current segment
    auto issue = [&](int gk, int li) {
        if (tid == 0) {
            const int st = gk % MMA_STAGES;
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            mbar_expect_tx(&s_bar[st], C::TILE_BYTES);
            bulk_g2s(s_prod + (size_t)st * MMA_TILE * ROW,
                     gtab + ((size_t)src0 + (size_t)s_list[li] * MMA_TILE) * ROW, C::TILE_BYTES, &s_bar[st]);
        }
    };

    double px[MT], py[MT], pz[MT];
#pragma unroll
    for (int mt = 0; mt < MT; ++mt) {
        const double* r = gtab + (size_t)(slot0 + wv * 32 + mt * 8 + lr) * ROW + NL;
        px[mt] = r[0]; py[mt] = r[1]; pz[mt] = r[2];
    }
    double acc[MT][NBG][2];
#pragma unroll
    for (int mt = 0; mt < MT; ++mt)
#pragma unroll
        for (int nb = 0; nb < NBG; ++nb) acc[mt][nb][0] = acc[mt][nb][1] = 0.0;

    // Gaussian cutoff (entropy.cuh): source tiles whose box is far from this block's 128 targets are not visited
    static_assert(MMA_THREADS == 2 * MMA_TILE, "a target tile is two boxes");
    const TileBox tbox = box_union(box[slot0 / MMA_TILE], box[slot0 / MMA_TILE + 1]);
    const double cutT = L->cut_T[s], kmax3 = 1.7320508075688772 * fabs(T->knot[NQ - 1]);
    int gbase = 0, nskip = 0;
    for (int seg0 = t0; seg0 < t1; seg0 += MMA_LCAP) {
    const int seg1 = min(t1, seg0 + MMA_LCAP);
    int n = 0;
    for (int base = seg0; base < seg1; base += MMA_THREADS) {
        const int t = base + tid;
        const bool act = t < seg1 && !tile_is_far(tbox, box[src0 / MMA_TILE + t], cutT, kmax3);
        const unsigned m = __ballot_sync(0xffffffffu, act);
        if (lane == 0) s_wcnt[wv] = __popc(m);
        __syncthreads();
        int off = n;
        for (int q = 0; q < wv; ++q) off += s_wcnt[q];
        if (act) s_list[off + __popc(m & ((1u << lane) - 1u))] = t;
        n += s_wcnt[0] + s_wcnt[1] + s_wcnt[2] + s_wcnt[3];
        __syncthreads();
    }
    nskip += (seg1 - seg0) - n;
#pragma unroll
    for (int b = 0; b < MMA_STAGES; ++b)
        if (b < n) issue(gbase + b, b);
    for (int kk = 0; kk < n; ++kk) {
        const int k = gbase + kk;
        mbar_wait(&s_bar[k % MMA_STAGES], (uint32_t)(k / MMA_STAGES) & 1u);
        const double* pr = s_prod + (size_t)(k % MMA_STAGES) * MMA_TILE * ROW;
#ifndef LANDAU_MMA_UNROLL            // tuning knob (build.py: LANDAU_NVCC_EXTRA)
#define LANDAU_MMA_UNROLL 2
#endif
        constexpr int KS_UNROLL = LANDAU_MMA_UNROLL;
#pragma unroll KS_UNROLL
        for (int ks = 0; ks < MMA_TILE / 4; ++ks) {
            const double* row = pr + (ks * 4 + lc) * ROW;
            const double2 a = *reinterpret_cast<const double2*>(row + NL);
            const double qz = row[NL + 2];
            double A[MT], Bf[NBG];
#pragma unroll
            for (int nb = 0; nb < NBG; ++nb) Bf[nb] = row[nb * 8 + lr];
#pragma unroll
            for (int mt = 0; mt < MT; ++mt) {
                const double dx = px[mt] - a.x, dy = py[mt] - a.y, dz = pz[mt] - qz;
                const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
                A[mt] = exp_neg_t256(r2, s_e2);
            }
#pragma unroll
            for (int mt = 0; mt < MT; ++mt)
#pragma unroll
                for (int nb = 0; nb < NBG; ++nb) dmma884(acc[mt][nb][0], acc[mt][nb][1], A[mt], Bf[nb]);
        }
        __syncthreads();                                              // every warp is done with this stage
        if (kk + MMA_STAGES < n) issue(k + MMA_STAGES, kk + MMA_STAGES);
    }
    gbase += n;
    }
    if (tid == 0 && blockIdx.z == 0 && t1 > t0) {
        atomicAdd(cutstats, (unsigned long long)(t1 - t0));
        atomicAdd(cutstats + 1, (unsigned long long)nskip);
    }
#pragma unroll
    for (int mt = 0; mt < MT; ++mt) {
        const int p = slot0 + wv * 32 + mt * 8 + lr;
#pragma unroll
        for (int nb = 0; nb < NBG; ++nb)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int nd = node0 + nb * 8 + 2 * lc + e;
                if (nd < M) part[((size_t)blockIdx.y * M + nd) * (size_t)npad_max + p] = acc[mt][nb][e];
            }
    }
}

}  // namespace landau
