// entropy_mma.cuh -- step a1 of the hot path as a dense FP64 contraction on the tensor pipe (DMMA).
//
// The factorised node sums of entropy_fact.cuh (Eq. (22); 3-V restatement DESIGN.md
// section 3 D1),
//     F_p(n) = sum_{q in s} C_pq * P_q(n),   C_pq = w_q exp(-|p' - q'|^2),   P_q(n) = Tx_q(i) Ty_q(j) Tz_q(l),
// with n = (i,j,l) a tensor Gauss-Hermite node, ARE a matrix product  F[targets x nodes] = C[targets x sources]
// * P[sources x nodes]  whose left factor is generated on the fly (one exponential per pair).  This kernel
// issues it as  mma.sync.m8n8k4.f64 (SASS DMMA.8x8x4):  a warp owns 8*MT targets x NL <= 64 nodes of
// accumulators in registers; per k-step of 4 sources each lane computes the MT entries C[lane/4 + 8 mt][lane%4]
// of the A fragments (its own exponentials), reads the NBG entries P[lane%4][8 nb + lane/4] of the B fragments
// from a per-tile product table in shared memory, and issues MT*NBG DMMAs.  Per pair the FP64 pipe sees
// 17 vector instructions (|d|^2, exponential, weight) + n_q^3 tensor FMAs, against 108 vector instructions in
// entropy_fact_kernel; on B200 DMMA and DFMA share one pipe (profiles/r1_entropy_fact_v3_full.md), so the gain
// is the removed product/issue overhead and DMMA's 12/12 (vs DFMA's 11/12) pipe efficiency, not overlap.
//
// Source records {x',y',z',w,Tx[NQ],Ty[NQ],Tz[NQ]} are those of entropy_fact_prep_kernel, staged by TMA bulk
// copies (double buffered); the block turns each tile of 64 records into the product table
// s_prod[q][0..NL) = P_q(node0 + .), s_prod[q][64..68) = {x',y',z',w}  (row stride 68 doubles: the B-fragment
// reads of a half-warp fall into 16 distinct bank pairs), also double buffered, one __syncthreads per tile.
// Nodes beyond n_q^3 (padding of the last 8-node block) have P = 0 and are not written.
// Output layout as the other pass-1 kernels: part[((chunk * M + node) * npad_max) + slot].
#pragma once
#include "common.cuh"
#include "entropy.cuh"
#include "entropy_fact.cuh"

namespace landau {

constexpr int MMA_THREADS = 128;   // 4 warps, 32 targets each
constexpr int MMA_TILE = 64;       // sources per stage
constexpr int MMA_MT = 4;          // 8-target blocks per warp
constexpr int MMA_ROW = 68;        // doubles per product-table row
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
    static constexpr int REC = FactCfg<NQ>::REC;
    static constexpr size_t SMEM =
        sizeof(double) * (2 * MMA_TILE * MMA_ROW + 2 * MMA_TILE * REC + 64) + 2 * sizeof(uint64_t) +
        sizeof(int) * (MMA_LCAP + 8);
};

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

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}

// grid = (target tiles of 128 slots, source chunks, MmaCfg<NQ, NZ>::GROUPS node groups).
template <int NQ, int NZ = NQ>
__global__ void __launch_bounds__(MMA_THREADS, 2)
entropy_mma_kernel(const DevTable* __restrict__ T, const DevLayout* __restrict__ L, int npad_max, int nchunks,
                   const double* __restrict__ rec, const TileBox* __restrict__ box,
                   unsigned long long* __restrict__ cutstats, double* __restrict__ part,
                   const StepCtrl* __restrict__ stop) {
    if (stop && stop->done) return;
    using C = MmaCfg<NQ, NZ>;
    constexpr int REC = C::REC, MT = MMA_MT, NBG = C::NBG, NL = C::NL, M = C::M;
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

    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* s_prod = reinterpret_cast<double*>(smem_raw);            // [2][MMA_TILE][MMA_ROW]
    double* s_rec = s_prod + 2 * MMA_TILE * MMA_ROW;                 // [2][MMA_TILE * REC]
    double* s_e2 = s_rec + 2 * MMA_TILE * REC;                       // [64]  2^(j/64)
    uint64_t* s_bar = reinterpret_cast<uint64_t*>(s_e2 + 64);        // [2]
    int* s_list = reinterpret_cast<int*>(s_bar + 2);                 // [MMA_LCAP] active source tiles of a segment
    int* s_wcnt = s_list + MMA_LCAP;                                 // [4]
    const int tid = threadIdx.x, lane = tid & 31, wv = tid >> 5;
    const int lr = lane >> 2, lc = lane & 3;                         // fragment row / column of this lane
    if (tid < 64) s_e2[tid] = T->exp2_tab[tid];
    if (tid == 0) {
        mbar_init(&s_bar[0], 1);
        mbar_init(&s_bar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // gk counts the tiles loaded by this block so far (stage = gk & 1, mbarrier parity = (gk >> 1) & 1); li is the
    // tile's position in the active list of the current segment
    auto issue = [&](int gk, int li) {
        if (tid == 0) {
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            constexpr uint32_t BYTES = MMA_TILE * REC * (uint32_t)sizeof(double);
            mbar_expect_tx(&s_bar[gk & 1], BYTES);
            bulk_g2s(s_rec + (size_t)(gk & 1) * MMA_TILE * REC,
                     rec + ((size_t)src0 + (size_t)s_list[li] * MMA_TILE) * REC, BYTES, &s_bar[gk & 1]);
        }
    };
    // product-table builder: lane = node (conflict-free: a warp reads <= NQ distinct factors of ONE record per
    // load and writes 32 consecutive doubles of one row), the block's two warp pairs take alternate sources
    const int be = tid & 63, bq = tid >> 6;
    const int bnd = node0 + be;
    const bool bvalid = be < NL && bnd < M;
    const int oi = 4 + (bvalid ? bnd / (NQ * NZ) : 0), oj = 4 + NQ + (bvalid ? (bnd / NZ) % NQ : 0),
              ol = 4 + 2 * NQ + (bvalid ? bnd % NZ : 0);
    auto build = [&](int k) {                                        // records of tile k -> product table k & 1
        mbar_wait(&s_bar[k & 1], (uint32_t)(k >> 1) & 1u);
        const double* r = s_rec + (size_t)(k & 1) * MMA_TILE * REC + bq * REC;
        double* row = s_prod + ((size_t)(k & 1) * MMA_TILE + bq) * MMA_ROW;
#pragma unroll 8
        for (int qi = 0; qi < MMA_TILE / 2; ++qi) {
            const double v = NZ == 1 ? r[oi] * r[oj] : r[oi] * r[oj] * r[ol];
            if (be < NL) row[be] = bvalid ? v : 0.0;
            if (be < 4) row[64 + be] = r[be];
            r += 2 * REC;
            row += 2 * MMA_ROW;
        }
    };

    double px[MT], py[MT], pz[MT];
#pragma unroll
    for (int mt = 0; mt < MT; ++mt) {
        const size_t p = (size_t)(slot0 + wv * 32 + mt * 8 + lr) * REC;
        px[mt] = rec[p]; py[mt] = rec[p + 1]; pz[mt] = rec[p + 2];
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
    if (n > 0) {
        issue(gbase, 0);
        if (n > 1) issue(gbase + 1, 1);
        build(gbase);
        __syncthreads();
        if (n > 2) issue(gbase + 2, 2);
    }
    for (int kk = 0; kk < n; ++kk) {
        const int k = gbase + kk;
        if (kk + 1 < n) build(k + 1);
        const double* pr = s_prod + (size_t)(k & 1) * MMA_TILE * MMA_ROW;
#pragma unroll 2
        for (int ks = 0; ks < MMA_TILE / 4; ++ks) {
            const double* row = pr + (ks * 4 + lc) * MMA_ROW;
            const double2 a = *reinterpret_cast<const double2*>(row + 64);
            const double2 b = *reinterpret_cast<const double2*>(row + 66);
            double A[MT], Bf[NBG];
#pragma unroll
            for (int nb = 0; nb < NBG; ++nb) Bf[nb] = row[nb * 8 + lr];
#pragma unroll
            for (int mt = 0; mt < MT; ++mt) {
                const double dx = px[mt] - a.x, dy = py[mt] - a.y, dz = pz[mt] - b.x;
                const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
                A[mt] = b.y * exp_neg_tab(r2, s_e2);
            }
#pragma unroll
            for (int mt = 0; mt < MT; ++mt)
#pragma unroll
                for (int nb = 0; nb < NBG; ++nb) dmma884(acc[mt][nb][0], acc[mt][nb][1], A[mt], Bf[nb]);
        }
        __syncthreads();
        if (kk + 3 < n) issue(k + 3, kk + 3);
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
