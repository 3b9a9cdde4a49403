// pair_sym.cuh -- step a3, symmetric (action-reaction) form of the pairwise Landau sum.
//
// Eq. (23) is antisymmetric under p <-> q up to the weights (this is what the
// paper's conservation proofs use, Eqs. 27 and 29):
//     term(p <- q) = (nu_ss'/m_s ) w_q Q(z) (g_p - g_q)
//     term(q <- p) = -(nu_ss'/m_s') w_p Q(z) (g_p - g_q)          (Q(-z) = Q(z))
// so Q(z)(g_p - g_q)/|z| is computed ONCE per unordered pair and applied to both markers:
// 30 FP64-pipe instructions per unordered pair = 15 per ordered pair, against 26 in the one-sided
// kernel (pair.cuh).  That is what lets the kernel exceed "100 % pipe = 61-74 % of peak FLOP/s"
// of the one-sided form.
//
// Schedule.  Slots are cut into target tiles of BT = W*32*RT markers and source units of
// BS = W*32*RS markers (BT % BS == 0; the packed layout pads every species to a multiple of BT, so
// every tile and unit is species-uniform and nu_ss' is hoisted per task).  A task is (target tile
// I, source unit j) with j >= first unit of I:
//     j inside tile I  -> "diagonal" task, evaluated one-sidedly (every ordered pair by its target);
//     j beyond tile I  -> symmetric task, both sides accumulated.
// Tasks are numbered I-major and dealt to the G persistent CTAs in contiguous, equal runs (static
// schedule => deterministic summation order).  Inside a task warp w works through the W sub-tiles
// of 32*RS sources in the order (w + phase) % W (a Latin square: in any phase each sub-tile belongs
// to exactly one warp), and inside a sub-tile lane l visits source group (l + k) % 32 at step k;
// the source-side accumulators sit in shared memory next to their sources and are read, updated and
// written back by whichever lane holds the group (conflict free; no shuffles, no atomics).  Each
// lane keeps RT targets (and their accumulators) in registers.  Sources come from a structure-of-
// arrays copy {x,y,z,w,gx,gy,gz}[npad] staged into shared memory by TMA bulk copies
// (cp.async.bulk + mbarrier), double buffered across tasks.
//
// Output, O(N) memory and deterministic (no per-CTA slices, no floating-point atomics):
//   * target side: a CTA leaves tile I once per run; it stores the tile's accumulators (scaled by nu/m) as one
//     compact segment  tpart[I + cta][3][BT]  (plain stores; a tile's row of tasks is shared by <= a few
//     consecutive CTAs, and I + cta is unique per (cta, tile) because both grow along the task order);
//   * source side: the 3*BS sums of a task are added IN PLACE into  acc[3][npad_max]  (L2 resident).  The
//     additions to one source unit are ordered by a per-unit ticket: the visits of unit j by the tiles
//     I' < j/rho are ranked by (local time of the visit in its CTA's run, CTA index) -- a pure function of the
//     static schedule that every CTA evaluates for itself -- and a CTA adds only when ticket[j] equals its rank.
//     All CTAs of the persistent grid are co-resident (grid = SM count, 1 CTA/SM) and advance through their
//     equal runs at the same pace, so a visit's predecessors have (almost always) already passed; the order is
//     fixed, hence the sum is bit-reproducible.  The wait is bounded: on expiry the kernel raises the layout's
//     error flag instead of hanging.
//   sym_reset_kernel zeroes acc and the tickets before the launch; sym_combine_kernel adds, per slot, acc and the
//   tile's segments in CTA order into ONE field slice [3][npad_max] for the update / combine kernels.
#pragma once
#include "common.cuh"
#include "stiff_pairs.cuh"

namespace landau {

__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    uint32_t done = 0;
    while (!done) {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(done)
            : "r"(smem_u32(bar)), "r"(parity)
            : "memory");
    }
}

template <int W, int RT, int RS, typename F = double>
struct SymCfg {
    static constexpr int THREADS = W * 32;
    static constexpr int BT = W * 32 * RT;   // targets per tile (registers)
    static constexpr int BS = W * 32 * RS;   // sources per unit (shared memory)
    static constexpr int SUB = 32 * RS;      // sources per warp and phase
    static constexpr int NCOMP = 7;          // x y z w gx gy gz
    static constexpr size_t SMEM = sizeof(F) * (2 * NCOMP * BS + 3 * BS) + 64;
    static_assert(BT % BS == 0, "target tile must be a whole number of source units");
};

// Ticket waits of the output path: bound per wait (each spin sleeps >= 40 ns and reads one global word) and the value
// raised in DevLayout::err when it expires (= LANDAU_ECUDA; landau_api.cu finish() turns it into the call's status).
#ifndef LANDAU_SYM_TICKET_SPINS
#define LANDAU_SYM_TICKET_SPINS (1u << 26)
#endif
constexpr unsigned SYM_TICKET_SPINS = LANDAU_SYM_TICKET_SPINS;
constexpr int SYM_ABORT = -3;

// number of tasks before target tile I:  sum_{i<I} (TU - rho*i)
__device__ __host__ inline long long sym_tasks_before(int I, int TU, int rho) {
    return (long long)I * TU - (long long)rho * I * (I - 1) / 2;
}

// CTA that owns task k when task t belongs to CTA b iff ntasks*b/G <= t < ntasks*(b+1)/G
__device__ __host__ inline int sym_task_owner(long long k, int G, long long ntasks) {
    return (int)(((k + 1) * G - 1) / ntasks);
}

__device__ __forceinline__ int ld_acquire_gpu(const int* p) {
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_gpu(int* p, int v) {
    asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// FP32 flavour of rsqrt_or_zero (FP32 field variant of BASELINE config 4): MUFU.RSQ + one Newton step;
// a separation that underflows in FP32 contributes 0 (reading S5 in FP32).
__device__ __forceinline__ float rsqrt_or_zero(float x) {
    float y = rsqrtf(fmaxf(x, 1e-30f));
    y = y * fmaf(-0.5f * x * y, y, 1.5f);
    return x < 1e-30f ? 0.f : y;
}
__device__ __forceinline__ float sym_fma(float a, float b, float c) { return fmaf(a, b, c); }
__device__ __forceinline__ double sym_fma(double a, double b, double c) { return fma(a, b, c); }
template <typename F> struct SymVec2;
template <> struct SymVec2<double> { using type = double2; };
template <> struct SymVec2<float> { using type = float2; };

// DIM = 2: the paper's 2-V setting (v_z = 0, g_z = 0; landau_set_dimension(2)): the z components of z, g_p - g_q and
// of both accumulators are identically zero and are not computed -- 22 instead of 30 FP64 instructions per unordered
// pair, results bit-identical to the 3-V arithmetic on v_z = 0 data (fma(0, 0, x) = x).
// The 3-V step exactly as profiled in profiles/r2_pair_sym_full.md (the generic sym_step below compiles to a slower
// schedule for DIM = 3: 41.1 ms against 40.0 ms per launch at 3 x 2^16, so the headline instantiation keeps its own text).
template <bool SYM, int RT, int RS, typename F>
__device__ __forceinline__ void sym_step3(const F (&px)[RT], const F (&py)[RT], const F (&pz)[RT],
                                         const F (&gx)[RT], const F (&gy)[RT], const F (&gz)[RT],
                                         const F (&wp)[RT], F (&ax)[RT], F (&ay)[RT],
                                         F (&az)[RT], const F (&qx)[RS], const F (&qy)[RS],
                                         const F (&qz)[RS], const F (&hx)[RS], const F (&hy)[RS],
                                         const F (&hz)[RS], const F (&wq)[RS], F (&bx)[RS],
                                         F (&by)[RS], F (&bz)[RS]) {
#pragma unroll
    for (int s = 0; s < RS; ++s) {
#pragma unroll
        for (int r = 0; r < RT; ++r) {
            const F zx = px[r] - qx[s], zy = py[r] - qy[s], zz = pz[r] - qz[s];
            const F cx = gx[r] - hx[s], cy = gy[r] - hy[s], cz = gz[r] - hz[s];
            const F r2 = sym_fma(zz, zz, sym_fma(zy, zy, zx * zx));
            const F d = sym_fma(zz, cz, sym_fma(zy, cy, zx * cx));
            const F yv = rsqrt_or_zero(r2);
            const F h = d * (yv * yv);
            const F ux = sym_fma(-zx, h, cx), uy = sym_fma(-zy, h, cy), uz = sym_fma(-zz, h, cz);
            const F a = wq[s] * yv;
            ax[r] = sym_fma(a, ux, ax[r]); ay[r] = sym_fma(a, uy, ay[r]); az[r] = sym_fma(a, uz, az[r]);
            if (SYM) {
                const F b = wp[r] * yv;
                bx[s] = sym_fma(b, ux, bx[s]); by[s] = sym_fma(b, uy, by[s]); bz[s] = sym_fma(b, uz, bz[s]);
            }
        }
    }
}

// What the detection variant of the kernel (first pass-2 evaluation of a step, stiff_pairs.cuh) hands to sym_step.
struct StiffDetect {
    StiffCtrl* sc; int* mark;
    double thr2, im_p, im_q;
    int tslot, sslot;            // slot of target r = 0 (targets are 32 apart) and of source s = 0
};

template <bool SYM, int RT, int RS, typename F, int DIM, bool DETECT = false>
__device__ __forceinline__ void sym_step(const F (&px)[RT], const F (&py)[RT], const F (&pz)[RT],
                                         const F (&gx)[RT], const F (&gy)[RT], const F (&gz)[RT],
                                         const F (&wp)[RT], F (&ax)[RT], F (&ay)[RT],
                                         F (&az)[RT], const F (&qx)[RS], const F (&qy)[RS],
                                         const F (&qz)[RS], const F (&hx)[RS], const F (&hy)[RS],
                                         const F (&hz)[RS], const F (&wq)[RS], F (&bx)[RS],
                                         F (&by)[RS], F (&bz)[RS], const StiffDetect* det = nullptr) {
#pragma unroll
    for (int s = 0; s < RS; ++s) {
#pragma unroll
        for (int r = 0; r < RT; ++r) {
            const F zx = px[r] - qx[s], zy = py[r] - qy[s];
            const F cx = gx[r] - hx[s], cy = gy[r] - hy[s];
            F r2 = sym_fma(zy, zy, zx * zx), d = sym_fma(zy, cy, zx * cx);
            F zz = F(0), cz = F(0);
            if (DIM == 3) {
                zz = pz[r] - qz[s]; cz = gz[r] - hz[s];
                r2 = sym_fma(zz, zz, r2); d = sym_fma(zz, cz, d);
            }
            if (DETECT) {
                if ((double)r2 < det->thr2) {
                    const int pp = det->tslot + 32 * r, qq = det->sslot + s;
                    if (SYM || pp < qq)             // a diagonal task sees every pair from both sides
                        stiff_candidate(det->sc, det->mark, pp, qq, (double)r2, (double)cx, (double)cy, (double)cz,
                                        (double)wq[s], (double)wp[r], det->im_p, det->im_q);
                }
            }
            const F yv = rsqrt_or_zero(r2);
            const F h = d * (yv * yv);
            const F ux = sym_fma(-zx, h, cx), uy = sym_fma(-zy, h, cy);
            const F a = wq[s] * yv;
            ax[r] = sym_fma(a, ux, ax[r]); ay[r] = sym_fma(a, uy, ay[r]);
            F uz = F(0);
            if (DIM == 3) { uz = sym_fma(-zz, h, cz); az[r] = sym_fma(a, uz, az[r]); }
            if (SYM) {
                const F b = wp[r] * yv;
                bx[s] = sym_fma(b, ux, bx[s]); by[s] = sym_fma(b, uy, by[s]);
                if (DIM == 3) bz[s] = sym_fma(b, uz, bz[s]);
            }
        }
    }
}

template <int W, int RT, int RS, typename F = double, int DIM = 3, bool DETECT = false>
__global__ void __launch_bounds__(W * 32, 1)
pair_sym_kernel(const DevTable* __restrict__ T, const DevLayout* __restrict__ L,
                const StepCtrl* __restrict__ ctrl, int npad_max, const F* __restrict__ soa,
                double* acc, double* __restrict__ tpart, int* ticket, int* errflag, int gate = GATE_NONE,
                StiffCtrl* stiff = nullptr, int* stiff_mark = nullptr) {
    using C = SymCfg<W, RT, RS, F>;
    using F2 = typename SymVec2<F>::type;
    if (ctrl && ctrl->done) return;
    if (gate_closed(ctrl, gate)) return;      // mixed-precision / stiff-pair steps: the alternative kernel runs
    if (*(volatile int*)errflag == SYM_ABORT) return;   // an earlier launch gave up on a ticket: the queued ones exit at once
    extern __shared__ __align__(128) unsigned char smem_raw[];
    F* s_src = reinterpret_cast<F*>(smem_raw);                        // [2][NCOMP][BS]
    F* s_acc = s_src + 2 * C::NCOMP * C::BS;                          // [3][BS]
    uint64_t* s_bar = reinterpret_cast<uint64_t*>(s_acc + 3 * C::BS); // [2]
    __shared__ double s_nu[LD_MAX_SPECIES * LD_MAX_SPECIES];
    __shared__ double s_im[LD_MAX_SPECIES];
    __shared__ int s_rank[2];
    __shared__ int s_abort;                   // this CTA saw the abort flag: no more waits, no more in-place adds

    const int S = T->S;
    const int npad = L->npad;
    constexpr int rho = C::BT / C::BS;
    const int TI = npad / C::BT, TU = npad / C::BS;
    const long long ntasks = sym_tasks_before(TI, TU, rho);
    const long long t0 = ntasks * blockIdx.x / gridDim.x, t1 = ntasks * (blockIdx.x + 1) / gridDim.x;
    if (t0 >= t1) return;

    const int tid = threadIdx.x, lane = tid & 31, wv = tid >> 5;
    for (int i = tid; i < S * S; i += C::THREADS) s_nu[i] = T->nu[i];
    if (tid < S) s_im[tid] = T->inv_mass[tid];
    if (tid == 0) {
        s_rank[0] = 0; s_rank[1] = 0; s_abort = 0;
        mbar_init(&s_bar[0], 1);
        mbar_init(&s_bar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // decode the first task
    int I = 0;
    while (I + 1 < TI && sym_tasks_before(I + 1, TU, rho) <= t0) ++I;
    int j = rho * I + (int)(t0 - sym_tasks_before(I, TU, rho));

    auto issue_load = [&](int unit, int stage) {
        if (tid == 0) {
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            mbar_expect_tx(&s_bar[stage], (DIM == 3 ? C::NCOMP : C::NCOMP - 2) * C::BS * (uint32_t)sizeof(F));
#pragma unroll
            for (int c = 0; c < C::NCOMP; ++c)
                if (DIM == 3 || (c != 2 && c != 6))               // 2-V: the z rows are not needed
                bulk_g2s(s_src + ((size_t)stage * C::NCOMP + c) * C::BS,
                         soa + (size_t)c * npad_max + (size_t)unit * C::BS, C::BS * (uint32_t)sizeof(F),
                         &s_bar[stage]);
        }
    };

    const int G = (int)gridDim.x;
    auto store_targets = [&](int tile, int sp, const F (&ax)[RT], const F (&ay)[RT], const F (&az)[RT]) {
        const double im = s_im[sp];
        double* seg = tpart + (size_t)(tile + (int)blockIdx.x) * 3 * C::BT;
#pragma unroll
        for (int r = 0; r < RT; ++r) {
            const int q = wv * 32 * RT + r * 32 + lane;
            seg[q] = (double)ax[r] * im;
            seg[C::BT + q] = (double)ay[r] * im;
            seg[2 * C::BT + q] = DIM == 3 ? (double)az[r] * im : 0.0;
        }
    };
    F px[RT], py[RT], pz[RT], gx[RT], gy[RT], gz[RT], w0[RT], wp[RT], ax[RT], ay[RT], az[RT];
    int curI = -1, sI = 0;
    uint32_t phase_bits = 0;   // bit s = parity to wait for on stage s
    int stage = 0;
    issue_load(j, 0);

    for (long long t = t0; t < t1; ++t) {
        if (I != curI) {
            if (curI >= 0) store_targets(curI, sI, ax, ay, az);
            curI = I;
            sI = species_of_slot(L, S, I * C::BT);
#pragma unroll
            for (int r = 0; r < RT; ++r) {
                const int p = I * C::BT + wv * 32 * RT + r * 32 + lane;
                px[r] = soa[p]; py[r] = soa[(size_t)npad_max + p];
                pz[r] = DIM == 3 ? soa[2 * (size_t)npad_max + p] : F(0);
                w0[r] = soa[3 * (size_t)npad_max + p];
                gx[r] = soa[4 * (size_t)npad_max + p]; gy[r] = soa[5 * (size_t)npad_max + p];
                gz[r] = DIM == 3 ? soa[6 * (size_t)npad_max + p] : F(0);
                ax[r] = ay[r] = az[r] = F(0);
            }
        }
        // next task (prefetch its source unit into the other stage)
        int In = I, jn = j + 1;
        if (jn >= TU) { In = I + 1; jn = rho * In; }
        if (t + 1 < t1) issue_load(jn, stage ^ 1);

        const int sJ = species_of_slot(L, S, j * C::BS);
        const F nu = (F)s_nu[sI * S + sJ];
        const bool diag = j < rho * (I + 1);
#pragma unroll
        for (int r = 0; r < RT; ++r) wp[r] = w0[r] * nu;
        for (int i = tid; i < DIM * C::BS; i += C::THREADS) s_acc[i] = F(0);
        // rank of this visit of source unit j among the visits by all tiles I' < j/rho (header comment)
        const int par = (int)((t - t0) & 1);
        if (tid == 0) s_rank[par ^ 1] = 0;
        if (!diag) {
            const long long mytau = t - t0;
            int cnt = 0;
            for (int Ip = tid; Ip < j / rho; Ip += C::THREADS) {
                if (Ip == I) continue;
                const long long kp = sym_tasks_before(Ip, TU, rho) + (j - rho * Ip);
                const int bp = sym_task_owner(kp, G, ntasks);
                const long long taup = kp - ntasks * bp / G;
                cnt += (taup < mytau || (taup == mytau && bp < (int)blockIdx.x)) ? 1 : 0;
            }
            cnt = __reduce_add_sync(0xffffffffu, cnt);
            if (lane == 0 && cnt) atomicAdd(&s_rank[par], cnt);
        }
        mbar_wait(&s_bar[stage], (phase_bits >> stage) & 1u);
        phase_bits ^= 1u << stage;
        __syncthreads();

        const F* sx = s_src + (size_t)stage * C::NCOMP * C::BS;
        StiffDetect det;
        if (DETECT) {
            det.sc = stiff; det.mark = stiff_mark; det.thr2 = stiff->thr2[sI * S + sJ];
            det.im_p = s_im[sI]; det.im_q = s_im[sJ];
            det.tslot = I * C::BT + wv * 32 * RT + lane;
        }
        for (int ph = 0; ph < W; ++ph) {
            const int base = ((wv + ph) % W) * C::SUB;
            if (DIM == 3 && !DETECT) {
#pragma unroll 1
            for (int k = 0; k < 32; ++k) {
                const int g = base + ((lane + k) & 31) * RS;
                F qx[RS], qy[RS], qz[RS], qw[RS], hx[RS], hy[RS], hz[RS], bx[RS], by[RS], bz[RS];
                if (RS % 2 == 0) {
#pragma unroll
                    for (int s = 0; s < RS; s += 2) {
                        const F2 a0 = *reinterpret_cast<const F2*>(sx + 0 * C::BS + g + s);
                        const F2 a1 = *reinterpret_cast<const F2*>(sx + 1 * C::BS + g + s);
                        const F2 a2 = *reinterpret_cast<const F2*>(sx + 2 * C::BS + g + s);
                        const F2 a3 = *reinterpret_cast<const F2*>(sx + 3 * C::BS + g + s);
                        const F2 a4 = *reinterpret_cast<const F2*>(sx + 4 * C::BS + g + s);
                        const F2 a5 = *reinterpret_cast<const F2*>(sx + 5 * C::BS + g + s);
                        const F2 a6 = *reinterpret_cast<const F2*>(sx + 6 * C::BS + g + s);
                        qx[s] = a0.x; qx[s + 1] = a0.y; qy[s] = a1.x; qy[s + 1] = a1.y; qz[s] = a2.x; qz[s + 1] = a2.y;
                        qw[s] = a3.x * nu; qw[s + 1] = a3.y * nu;
                        hx[s] = a4.x; hx[s + 1] = a4.y; hy[s] = a5.x; hy[s + 1] = a5.y; hz[s] = a6.x; hz[s + 1] = a6.y;
                    }
                } else {
#pragma unroll
                    for (int s = 0; s < RS; ++s) {
                        qx[s] = sx[0 * C::BS + g + s]; qy[s] = sx[1 * C::BS + g + s]; qz[s] = sx[2 * C::BS + g + s];
                        qw[s] = sx[3 * C::BS + g + s] * nu;
                        hx[s] = sx[4 * C::BS + g + s]; hy[s] = sx[5 * C::BS + g + s]; hz[s] = sx[6 * C::BS + g + s];
                    }
                }
                if (diag) {
                    sym_step3<false, RT, RS, F>(px, py, pz, gx, gy, gz, wp, ax, ay, az, qx, qy, qz, hx, hy, hz, qw, bx, by, bz);
                } else {
                    // the source-side sums live in shared memory next to their sources: in this phase the sub-tile is
                    // this warp's alone and at step k every lane holds another group, so the read-modify-write is
                    // conflict free and ordered by the warp's program order (no shuffles, no atomics)
                    if (RS % 2 == 0) {
#pragma unroll
                        for (int s = 0; s < RS; s += 2) {
                            const F2 b0 = *reinterpret_cast<const F2*>(s_acc + g + s);
                            const F2 b1 = *reinterpret_cast<const F2*>(s_acc + C::BS + g + s);
                            const F2 b2 = *reinterpret_cast<const F2*>(s_acc + 2 * C::BS + g + s);
                            bx[s] = b0.x; bx[s + 1] = b0.y; by[s] = b1.x; by[s + 1] = b1.y; bz[s] = b2.x; bz[s + 1] = b2.y;
                        }
                    } else {
#pragma unroll
                        for (int s = 0; s < RS; ++s) { bx[s] = s_acc[g + s]; by[s] = s_acc[C::BS + g + s]; bz[s] = s_acc[2 * C::BS + g + s]; }
                    }
                    sym_step3<true, RT, RS, F>(px, py, pz, gx, gy, gz, wp, ax, ay, az, qx, qy, qz, hx, hy, hz, qw, bx, by, bz);
                    if (RS % 2 == 0) {
#pragma unroll
                        for (int s = 0; s < RS; s += 2) {
                            F2 b0, b1, b2;
                            b0.x = bx[s]; b0.y = bx[s + 1]; b1.x = by[s]; b1.y = by[s + 1]; b2.x = bz[s]; b2.y = bz[s + 1];
                            *reinterpret_cast<F2*>(s_acc + g + s) = b0;
                            *reinterpret_cast<F2*>(s_acc + C::BS + g + s) = b1;
                            *reinterpret_cast<F2*>(s_acc + 2 * C::BS + g + s) = b2;
                        }
                    } else {
#pragma unroll
                        for (int s = 0; s < RS; ++s) { s_acc[g + s] = bx[s]; s_acc[C::BS + g + s] = by[s]; s_acc[2 * C::BS + g + s] = bz[s]; }
                    }
                    __syncwarp();
                }
            }
            } else {
#pragma unroll 1
            for (int k = 0; k < 32; ++k) {
                const int g = base + ((lane + k) & 31) * RS;
                F qx[RS], qy[RS], qz[RS], qw[RS], hx[RS], hy[RS], hz[RS], bx[RS], by[RS], bz[RS];
                if (RS % 2 == 0) {
#pragma unroll
                    for (int s = 0; s < RS; s += 2) {
                        const F2 a0 = *reinterpret_cast<const F2*>(sx + 0 * C::BS + g + s);
                        const F2 a1 = *reinterpret_cast<const F2*>(sx + 1 * C::BS + g + s);
                        const F2 a3 = *reinterpret_cast<const F2*>(sx + 3 * C::BS + g + s);
                        const F2 a4 = *reinterpret_cast<const F2*>(sx + 4 * C::BS + g + s);
                        const F2 a5 = *reinterpret_cast<const F2*>(sx + 5 * C::BS + g + s);
                        qx[s] = a0.x; qx[s + 1] = a0.y; qy[s] = a1.x; qy[s + 1] = a1.y;
                        qw[s] = a3.x * nu; qw[s + 1] = a3.y * nu;
                        hx[s] = a4.x; hx[s + 1] = a4.y; hy[s] = a5.x; hy[s + 1] = a5.y;
                        qz[s] = qz[s + 1] = hz[s] = hz[s + 1] = F(0);
                        if (DIM == 3) {
                            const F2 a2 = *reinterpret_cast<const F2*>(sx + 2 * C::BS + g + s);
                            const F2 a6 = *reinterpret_cast<const F2*>(sx + 6 * C::BS + g + s);
                            qz[s] = a2.x; qz[s + 1] = a2.y; hz[s] = a6.x; hz[s + 1] = a6.y;
                        }
                    }
                } else {
#pragma unroll
                    for (int s = 0; s < RS; ++s) {
                        qx[s] = sx[0 * C::BS + g + s]; qy[s] = sx[1 * C::BS + g + s];
                        qz[s] = DIM == 3 ? sx[2 * C::BS + g + s] : F(0);
                        qw[s] = sx[3 * C::BS + g + s] * nu;
                        hx[s] = sx[4 * C::BS + g + s]; hy[s] = sx[5 * C::BS + g + s];
                        hz[s] = DIM == 3 ? sx[6 * C::BS + g + s] : F(0);
                    }
                }
                if (DETECT) det.sslot = j * C::BS + g;
                if (diag) {
                    sym_step<false, RT, RS, F, DIM, DETECT>(px, py, pz, gx, gy, gz, wp, ax, ay, az, qx, qy, qz, hx, hy, hz, qw,
                                                            bx, by, bz, &det);
                } else {
                    // the source-side sums live in shared memory next to their sources: in this phase the sub-tile is
                    // this warp's alone and at step k every lane holds another group, so the read-modify-write is
                    // conflict free and ordered by the warp's program order (no shuffles, no atomics)
                    if (RS % 2 == 0) {
#pragma unroll
                        for (int s = 0; s < RS; s += 2) {
                            const F2 b0 = *reinterpret_cast<const F2*>(s_acc + g + s);
                            const F2 b1 = *reinterpret_cast<const F2*>(s_acc + C::BS + g + s);
                            bx[s] = b0.x; bx[s + 1] = b0.y; by[s] = b1.x; by[s + 1] = b1.y; bz[s] = bz[s + 1] = F(0);
                            if (DIM == 3) {
                                const F2 b2 = *reinterpret_cast<const F2*>(s_acc + 2 * C::BS + g + s);
                                bz[s] = b2.x; bz[s + 1] = b2.y;
                            }
                        }
                    } else {
#pragma unroll
                        for (int s = 0; s < RS; ++s) {
                            bx[s] = s_acc[g + s]; by[s] = s_acc[C::BS + g + s];
                            bz[s] = DIM == 3 ? s_acc[2 * C::BS + g + s] : F(0);
                        }
                    }
                    sym_step<true, RT, RS, F, DIM, DETECT>(px, py, pz, gx, gy, gz, wp, ax, ay, az, qx, qy, qz, hx, hy, hz, qw,
                                                           bx, by, bz, &det);
                    if (RS % 2 == 0) {
#pragma unroll
                        for (int s = 0; s < RS; s += 2) {
                            F2 b0, b1, b2;
                            b0.x = bx[s]; b0.y = bx[s + 1]; b1.x = by[s]; b1.y = by[s + 1]; b2.x = bz[s]; b2.y = bz[s + 1];
                            *reinterpret_cast<F2*>(s_acc + g + s) = b0;
                            *reinterpret_cast<F2*>(s_acc + C::BS + g + s) = b1;
                            if (DIM == 3) *reinterpret_cast<F2*>(s_acc + 2 * C::BS + g + s) = b2;
                        }
                    } else {
#pragma unroll
                        for (int s = 0; s < RS; ++s) {
                            s_acc[g + s] = bx[s]; s_acc[C::BS + g + s] = by[s];
                            if (DIM == 3) s_acc[2 * C::BS + g + s] = bz[s];
                        }
                    }
                    __syncwarp();
                }
            }
            }
            __syncthreads();
        }
        if (!diag) {
            const double sc = -s_im[sJ];
            const int want = s_rank[par];
            // Wait for this unit's turn.  The wait is bounded, and the first CTA whose bound expires (its predecessor
            // is not running: the grid is not co-resident, or the schedule is wrong) raises SYM_ABORT for the whole
            // grid: every CTA polls the flag while it waits, and from then on adds nothing in place and passes no
            // ticket on -- the field is left incomplete and the call fails with LANDAU_ECUDA, it is never summed out
            // of order.  CTAs finish their remaining tasks without waiting, so the kernel ends within one evaluation.
            if (tid == 0) {
                unsigned spins = 0;
                int ab = s_abort;
                while (!ab && ld_acquire_gpu(ticket + j) != want) {
                    __nanosleep(40);
                    ++spins;
                    if ((spins & 63u) == 0 && *(volatile int*)errflag == SYM_ABORT) ab = 1;
                    if (spins > SYM_TICKET_SPINS) { atomicExch(errflag, SYM_ABORT); ab = 1; }
                }
                s_abort = ab;
            }
            __syncthreads();
            const bool aborted = s_abort != 0;
            if (!aborted)
                for (int i = tid; i < DIM * C::BS; i += C::THREADS) {
                    const int d = i / C::BS, e = i - d * C::BS;
                    double* o = acc + (size_t)d * npad_max + (size_t)j * C::BS + e;
                    __stcg(o, __ldcg(o) + sc * (double)s_acc[i]);
                }
            __threadfence();
            __syncthreads();
            if (tid == 0 && !aborted) st_release_gpu(ticket + j, want + 1);
        }
        I = In; j = jn; stage ^= 1;
    }
    store_targets(curI, sI, ax, ay, az);
}

// Before a launch of pair_sym_kernel: zero the in-place source-side accumulator and the per-unit tickets
// (skipped, like every kernel of an iteration, once the step is done).
__global__ void sym_reset_kernel(const StepCtrl* __restrict__ ctrl, double* __restrict__ acc, size_t n,
                                 int* __restrict__ ticket, int nticket, int gate = GATE_NONE) {
    if (ctrl && ctrl->done) return;
    if (gate_closed(ctrl, gate)) return;
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    const size_t i0 = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    for (size_t i = i0; i < n; i += stride) acc[i] = 0.0;
    for (size_t i = i0; i < (size_t)nticket; i += stride) ticket[i] = 0;
}

// After pair_sym_kernel: field slice out[3][npad_max] = in-place source-side sums + the target-side segments of
// the slot's tile, added in CTA order (the CTAs whose runs of tasks meet the tile's row).  G = grid of the pair kernel.
__global__ void sym_combine_kernel(const DevLayout* __restrict__ L, const StepCtrl* __restrict__ ctrl, int npad_max,
                                   int G, int BT, int BS, const double* __restrict__ acc,
                                   const double* __restrict__ tpart, double* __restrict__ out, int gate = GATE_NONE) {
    if (ctrl && ctrl->done) return;
    if (gate_closed(ctrl, gate)) return;
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= npad_max) return;
    const size_t np = (size_t)npad_max;
    const int npad = L->npad;
    double a = 0.0, b = 0.0, c = 0.0;
    if (p < npad) {
        const int rho = BT / BS, TI = npad / BT, TU = npad / BS;
        const long long ntasks = sym_tasks_before(TI, TU, rho);
        const int I = p / BT, q = p - I * BT;
        const long long k0 = sym_tasks_before(I, TU, rho), k1 = sym_tasks_before(I + 1, TU, rho);
        const int bf = sym_task_owner(k0, G, ntasks), bl = sym_task_owner(k1 - 1, G, ntasks);
        a = acc[p]; b = acc[np + p]; c = acc[2 * np + p];
        for (int cta = bf; cta <= bl; ++cta) {
            if (ntasks * cta / G >= ntasks * (cta + 1) / G) continue;      // a CTA without tasks wrote nothing
            const double* seg = tpart + (size_t)(I + cta) * 3 * BT + q;
            a += seg[0]; b += seg[BT]; c += seg[2 * BT];
        }
    }
    out[p] = a; out[np + p] = b; out[2 * np + p] = c;
}

// {x,y,z,w,G} (packed SoA) -> structure-of-arrays source copy {x,y,z,w,gx,gy,gz}[npad_max], g = G/m.
__global__ void build_soa_kernel(const DevTable* __restrict__ T, const DevLayout* __restrict__ L, int npad_max,
                                 const double* __restrict__ x, const double* __restrict__ y,
                                 const double* __restrict__ z, const double* __restrict__ w,
                                 const double* __restrict__ Gx, const double* __restrict__ Gy,
                                 const double* __restrict__ Gz, double* __restrict__ soa) {
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= npad_max) return;
    double v[7] = {0, 0, 0, 0, 0, 0, 0};
    if (p < L->npad) {
        const double im = T->inv_mass[species_of_slot(L, T->S, p)];
        v[0] = x[p]; v[1] = y[p]; v[2] = z[p]; v[3] = w[p];
        v[4] = Gx[p] * im; v[5] = Gy[p] * im; v[6] = Gz[p] * im;
    }
#pragma unroll
    for (int c = 0; c < 7; ++c) soa[(size_t)c * npad_max + p] = v[c];
}

// FP64 SoA source copy -> FP32 (FP32 field variant; mixed-precision step: only while ctrl->use_f32 is set).
__global__ void soa_to_f32_kernel(size_t n, const double* __restrict__ a, float* __restrict__ b,
                                  const StepCtrl* __restrict__ ctrl = nullptr) {
    if (ctrl && (ctrl->done || !ctrl->use_f32)) return;
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) b[i] = (float)a[i];
}

}  // namespace landau
