// cells.cuh -- SURVEY.md section 8(f) NEXT-3: many spatial collision cells in one launch.
//
// The paper's bracket couples only markers of the same collision cell (indicator 1(p, p-bar)) and
// "an efficient parallelization per each collision cell is elementary"; its tests use one cell
// (PAPER.md:110).  A PIC code calls the operator with thousands of small cells (10^2..10^3 markers each), a
// regime in which the large-N path of this library is bound by launch latency.  This kernel is the B200 answer
// for that regime: ONE persistent CTA per cell, the cell's whole state resident in shared memory, and the
// complete algorithm of Algorithm 1 for n_steps time steps inside a single launch:
//   load + stable bucketing by species  ->  per step { pass 1 (Eq. 22, factorised form of entropy_fact.cuh)
//   -> Jacobi fixed point of Eq. (24) with pass 2 (Eq. 23) per iteration, residual by a block reduction }
//   -> write back in caller order.
// No global-memory traffic, no kernel launch and no host synchronisation inside a step.  Cells are dealt to the
// CTAs through an atomic counter (cells are independent, so results do not depend on the assignment).
// Limits: markers per cell <= CellsCfg<NQ>::max_cap() (shared memory: 1024 for n_q <= 5, 970 / 878 / 802 for
// n_q = 6 / 7 / 8).  A cell that is too wide for the factorised pass 1 (reading N3) takes the literal-separable form
// of Eq. (22) (3 n_q exponentials per pair, every factor <= 1), as the single-cell path does.  n_q > 4: the n_q^3 node
// sums of a target are accumulated in slices of x-node indices (registers), the per-pair exponential recomputed per
// slice.  Arithmetic, stopping rule and readings are those of the single-cell path (S4, S5, S7, S8); tests compare
// every cell with the oracle.
#pragma once
#include "common.cuh"
#include "entropy.cuh"
#include "entropy_mma.cuh"   // exp_neg_tab
#include "pair.cuh"          // pair_accumulate
#include "pair_sym.cuh"      // sym_step3

namespace landau {

constexpr int CELLS_THREADS = 256;
constexpr int CELLS_CAP = 1024;                 // markers per cell (all species)
constexpr int CELLS_ROUNDS = CELLS_CAP / CELLS_THREADS;

struct CellRecord {          // mirrors landau_cell_info (host struct) field by field
    int status;              // 0 ok, 1 some step did not converge, < 0 error (cell left unchanged)
    int iterations;          // fixed-point iterations, summed over the steps
    int max_iterations;      // most iterations any step took
    int steps_not_converged;
    double residual;         // residual of the last step
};

template <int NQ>
struct CellsCfg {
    // doubles per marker: xn yn zn w | Gx Gy Gz | xk yk zk | 3 NQ table entries (pass 1) / one source record
    // {ux uy uz w gx gy gz 0} (pass 2, one-sided loop; 64 bytes: four LDS.128 per source instead of seven LDS.64) /
    // seven source arrays + three source-side accumulator arrays (pass 2, symmetric evaluation)
    static constexpr int TAB = 3 * NQ > 10 ? 3 * NQ : 10;
    static constexpr int DPM = 10 + TAB;
    // x-node indices per register slice of the node sums: NI * NQ^2 <= 64 accumulators
    static constexpr int NI = NQ <= 4 ? NQ : 1;
    static_assert(NQ % NI == 0, "slices must tile the x-node indices");
    static size_t smem(int cap) {
        return sizeof(double) * ((size_t)DPM * cap + 64 + 32 + 3 * CELLS_THREADS) + sizeof(int) * (size_t)cap;
    }
    static int max_cap() {                  // largest even cap whose state fits the 227 KB of a CTA
        int cap = CELLS_CAP;
        while (cap > 32 && smem(cap) > 227 * 1024 - 4096) cap -= 2;   // the kernel's static shared memory is ~2.2 KB
        return cap;
    }
};

// Fixed-order block sum of two values (warp shuffles, then warp 0 adds the warp totals in index order).
template <int NT = CELLS_THREADS>
__device__ __forceinline__ void cells_reduce2(double& a, double& b, double* s_red) {
    a = warp_sum(a); b = warp_sum(b);
    const int lane = threadIdx.x & 31, wv = threadIdx.x >> 5;
    __syncthreads();
    if (lane == 0) { s_red[2 * wv] = a; s_red[2 * wv + 1] = b; }
    __syncthreads();
    double x = 0.0, y = 0.0;
    for (int k = 0; k < NT / 32; ++k) { x += s_red[2 * k]; y += s_red[2 * k + 1]; }
    a = x; b = y;
}

// Pass 1 of one target against the sources [o0, o1) of its species, node slice i in [i0, i0 + NI): the partial
// sums  sum_{ijl} a_i a_j a_l k (1 + ln rho)  of Eq. (22) (without the prefactor).  NI = NQ is the whole gradient;
// NI < NQ lets several threads share one target (small cells), each recomputing the exponential.
template <int NQ, int NI, bool LITERAL>
__device__ __forceinline__ void cells_pass1_target(int i0, int o0, int o1, double px, double py, double pz,
                                                   const double* __restrict__ xk, const double* __restrict__ yk,
                                                   const double* __restrict__ zk, const double* __restrict__ ww,
                                                   const double* __restrict__ tab, const double* __restrict__ s_e2,
                                                   const double (&kn)[NQ], const double (&ga)[NQ], double lognorm,
                                                   double& gx, double& gy, double& gz) {
    double acc[NI][NQ][NQ];
#pragma unroll
    for (int i = 0; i < NI; ++i)
#pragma unroll
        for (int j = 0; j < NQ; ++j)
#pragma unroll
            for (int l = 0; l < NQ; ++l) acc[i][j][l] = 0.0;
#pragma unroll 2
    for (int q = o0; q < o1; ++q) {
        const double dx = px - xk[q], dy = py - yk[q], dz = pz - zk[q];
        double c, tx[NI], ty[NQ], tz[NQ];
        if (LITERAL) {
            // exp(-|k + d|^2) = prod_axis exp(-(k_a + d_a)^2): every factor <= 1 (wide cells, reading N3)
            c = ww[q];
#pragma unroll
            for (int i = 0; i < NI; ++i) {
                double ki = kn[0];
#pragma unroll
                for (int m = 1; m < NQ; ++m) if (m == i0 + i) ki = kn[m];
                const double a = ki + dx;
                tx[i] = exp_neg_tab(a * a, s_e2);
            }
#pragma unroll
            for (int j = 0; j < NQ; ++j) {
                const double a = kn[j] + dy, b = kn[j] + dz;
                ty[j] = exp_neg_tab(a * a, s_e2); tz[j] = exp_neg_tab(b * b, s_e2);
            }
        } else {
            const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
            c = ww[q] * exp_neg_tab(r2, s_e2);
            const double* t = tab + (size_t)q * 3 * NQ;
#pragma unroll
            for (int i = 0; i < NI; ++i) tx[i] = t[i0 + i];
#pragma unroll
            for (int j = 0; j < NQ; ++j) { ty[j] = t[NQ + j]; tz[j] = t[2 * NQ + j]; }
        }
#pragma unroll
        for (int i = 0; i < NI; ++i) {
            const double cx = c * tx[i];
#pragma unroll
            for (int j = 0; j < NQ; ++j) {
                const double cxy = cx * ty[j];
#pragma unroll
                for (int l = 0; l < NQ; ++l) acc[i][j][l] = fma(cxy, tz[l], acc[i][j][l]);
            }
        }
    }
    gx = gy = gz = 0.0;
#pragma unroll
    for (int i = 0; i < NI; ++i) {
        double ki = kn[0], gi = ga[0];                                // kn[i0 + i] without dynamic register indexing
#pragma unroll
        for (int m = 1; m < NQ; ++m) if (m == i0 + i) { ki = kn[m]; gi = ga[m]; }
#pragma unroll
        for (int j = 0; j < NQ; ++j)
#pragma unroll
            for (int l = 0; l < NQ; ++l) {
                double lnrho = lognorm + log(acc[i][j][l]);
                if (!LITERAL) lnrho -= (ki * ki + kn[j] * kn[j] + kn[l] * kn[l]) + 2.0 * (ki * px + kn[j] * py + kn[l] * pz);
                const double t = gi * ga[j] * ga[l] * (1.0 + lnrho);
                gx = fma(t, ki, gx); gy = fma(t, kn[j], gy); gz = fma(t, kn[l], gz);
            }
    }
}

// Pass 1 of one species of a cell as an FP64 tensor contraction (n_q = 4, factorised form; the in-cell version of
// entropy_mma.cuh): F[targets x 64 nodes] = C[targets x sources] * P[sources x nodes], C_pq = exp(-|p' - q'|^2),
// P_q(n) = w_q Tx_q(i) Ty_q(j) Tz_q(l).  A warp owns 32 targets x 64 nodes of accumulators (mma.sync.m8n8k4.f64, SASS
// DMMA.8x8x4); per k-step of 4 sources a lane computes its 4 exponentials (A fragments) and builds its 8 B-fragment
// entries P[source lane%4][node 8 nb + lane/4] from the source's factor table in shared memory (10 multiplies: the
// node index splits as i = nb/2, j = 2 (nb%2) + (lane/4)/4, l = (lane/4)%4) -- there is no room for a product table next
// to the cell's state.  64 + 10 vector instructions and 32 DMMAs per 128 pairs, against 101 vector instructions per
// pair in cells_pass1_target.  The logarithms and the node sum of Eq. (22) are taken in the accumulator layout (a lane
// holds 16 nodes of each of its 4 targets) and the 4 lanes of a target are added by two shuffles (fixed order).
__device__ __forceinline__ void cells_pass1_dmma4(int o0, int o1, const double* __restrict__ xk,
                                                  const double* __restrict__ yk, const double* __restrict__ zk,
                                                  const double* __restrict__ ww, const double* __restrict__ tab,
                                                  const double* __restrict__ s_e2, const double (&kn)[4],
                                                  const double (&ga)[4], double lognorm, double pref, bool planar,
                                                  double* __restrict__ Gx, double* __restrict__ Gy,
                                                  double* __restrict__ Gz, int* s_status) {
    constexpr int MT = 4, NBG = 8;
    const int lane = threadIdx.x & 31, wv = threadIdx.x >> 5;
    const int lr = lane >> 2, lc = lane & 3;
    const int nks = (o1 - o0 + 3) >> 2;
    const int j0 = lr >> 2, l0 = lr & 3;                     // B fragment: j = 2 (nb & 1) + j0, l = l0
    for (int base = o0; base < o1; base += CELLS_THREADS) {
        const int t0 = base + wv * 32;
        if (t0 >= o1) continue;                              // warp-uniform; no block barrier inside this function
        double px[MT], py[MT], pz[MT];
#pragma unroll
        for (int mt = 0; mt < MT; ++mt) {
            const int p = min(t0 + mt * 8 + lr, o1 - 1);     // clamped duplicate; not written
            px[mt] = xk[p]; py[mt] = yk[p]; pz[mt] = zk[p];
        }
        double acc[MT][NBG][2];
#pragma unroll
        for (int mt = 0; mt < MT; ++mt)
#pragma unroll
            for (int nb = 0; nb < NBG; ++nb) acc[mt][nb][0] = acc[mt][nb][1] = 0.0;
#pragma unroll 1
        for (int ks = 0; ks < nks; ++ks) {
            const int q = o0 + ks * 4 + lc;
            const bool ok = q < o1;
            const int qq = ok ? q : o1 - 1;
            const double qx = xk[qq], qy = yk[qq], qz = zk[qq];
            const double* t = tab + (size_t)qq * 12;
            const double2 ta = *reinterpret_cast<const double2*>(t), tb = *reinterpret_cast<const double2*>(t + 2);
            const double tzw = ok ? t[8 + l0] * ww[qq] : 0.0;  // a source beyond the species adds exactly 0
            const double u0 = t[4 + j0] * tzw, u1 = t[6 + j0] * tzw;
            double A[MT], Bf[NBG];
            Bf[0] = ta.x * u0; Bf[1] = ta.x * u1; Bf[2] = ta.y * u0; Bf[3] = ta.y * u1;
            Bf[4] = tb.x * u0; Bf[5] = tb.x * u1; Bf[6] = tb.y * u0; Bf[7] = tb.y * u1;
#pragma unroll
            for (int mt = 0; mt < MT; ++mt) {
                const double dx = px[mt] - qx, dy = py[mt] - qy, dz = pz[mt] - qz;
                A[mt] = exp_neg_tab(fma(dz, dz, fma(dy, dy, dx * dx)), s_e2);
            }
#pragma unroll
            for (int mt = 0; mt < MT; ++mt)
#pragma unroll
                for (int nb = 0; nb < NBG; ++nb) dmma884(acc[mt][nb][0], acc[mt][nb][1], A[mt], Bf[nb]);
        }
        // accumulator layout: acc[mt][nb][e] = F[target 8 mt + lr][node 8 nb + 2 lc + e], node = 16 i + 4 j + l
#pragma unroll
        for (int mt = 0; mt < MT; ++mt) {
            double gx = 0.0, gy = 0.0, gz = 0.0;
#pragma unroll
            for (int nb = 0; nb < NBG; ++nb) {
                const double ki = kn[nb >> 1], gi = ga[nb >> 1];
                const double kj = (lc & 2) ? kn[2 * (nb & 1) + 1] : kn[2 * (nb & 1)];
                const double gj = (lc & 2) ? ga[2 * (nb & 1) + 1] : ga[2 * (nb & 1)];
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const double kl = (lc & 1) ? kn[2 + e] : kn[e], gl = (lc & 1) ? ga[2 + e] : ga[e];
                    const double lnrho = lognorm + log(acc[mt][nb][e]) -
                                         ((ki * ki + kj * kj + kl * kl) + 2.0 * (ki * px[mt] + kj * py[mt] + kl * pz[mt]));
                    const double tt = gi * gj * gl * (1.0 + lnrho);
                    gx = fma(tt, ki, gx); gy = fma(tt, kj, gy); gz = fma(tt, kl, gz);
                }
            }
            gx += __shfl_xor_sync(0xffffffffu, gx, 1); gy += __shfl_xor_sync(0xffffffffu, gy, 1); gz += __shfl_xor_sync(0xffffffffu, gz, 1);
            gx += __shfl_xor_sync(0xffffffffu, gx, 2); gy += __shfl_xor_sync(0xffffffffu, gy, 2); gz += __shfl_xor_sync(0xffffffffu, gz, 2);
            const int p = t0 + mt * 8 + lr;
            if (lc == 0 && p < o1) {
                gx *= pref; gy *= pref; gz *= pref;
                if (!(isfinite(gx) && isfinite(gy) && isfinite(gz))) *s_status = -4;
                Gx[p] = gx; Gy[p] = gy; Gz[p] = planar ? 0.0 : gz;
            }
        }
    }
}

// Pass 2 of NT targets of one thread against every source of the cell (a source record is read once per NT targets:
// NT = 4 quarters the shared-memory traffic per pair).  t? = sum_s' nu_ss' sum_q w_q Q(u_p - u_q)(g_p - g_q).
// rec: [n][8] = {ux uy uz w gx gy gz 0}.
template <int NT>
__device__ __forceinline__ void cells_field(const double* __restrict__ rec, const int* __restrict__ s_off,
                                            const double* __restrict__ s_nu, int S, const int (&pc)[NT],
                                            const int (&sp)[NT], double (&tx)[NT], double (&ty)[NT], double (&tz)[NT]) {
    double px[NT], py[NT], pz[NT], hx[NT], hy[NT], hz[NT];
#pragma unroll
    for (int t = 0; t < NT; ++t) {
        const double* r = rec + (size_t)pc[t] * 8;
        px[t] = r[0]; py[t] = r[1]; pz[t] = r[2];
        hx[t] = r[4]; hy[t] = r[5]; hz[t] = r[6];
        tx[t] = ty[t] = tz[t] = 0.0;
    }
    for (int sb = 0; sb < S; ++sb) {
        const int q0 = s_off[sb], q1 = s_off[sb + 1];
        double ax[NT], ay[NT], az[NT];
#pragma unroll
        for (int t = 0; t < NT; ++t) ax[t] = ay[t] = az[t] = 0.0;
#pragma unroll 4
        for (int q = q0; q < q1; ++q) {
            const double2* r2 = reinterpret_cast<const double2*>(rec + (size_t)q * 8);
            const double2 a = r2[0], b = r2[1], c = r2[2], d = r2[3];
            const double qx = a.x, qy = a.y, qz = b.x, wq = b.y, gx = c.x, gy = c.y, gz = d.x;
#pragma unroll
            for (int t = 0; t < NT; ++t)
                pair_accumulate(px[t] - qx, py[t] - qy, pz[t] - qz, hx[t] - gx, hy[t] - gy, hz[t] - gz, wq, ax[t], ay[t],
                                az[t]);
        }
#pragma unroll
        for (int t = 0; t < NT; ++t) {
            const double nu = s_nu[sp[t] * S + sb];
            tx[t] = fma(nu, ax[t], tx[t]); ty[t] = fma(nu, ay[t], ty[t]); tz[t] = fma(nu, az[t], tz[t]);
        }
    }
}

// Slot of a thread's r-th target in the symmetric evaluation: warp w owns the G R slots of sub-tile w (G <= 32 groups,
// lanes >= G idle), stored as R / RS blocks of G groups of RS consecutive slots, so that the lanes of a warp read
// consecutive 8 RS-byte vectors whatever R is (R = 4 as two blocks of pairs: four consecutive slots per lane would be a
// 2-way bank conflict).  G = the even number of groups per warp that just covers the cell: a cell of 320 markers walks
// 20 lane steps per phase, not 32.
__device__ __forceinline__ int cells_sym_slot(int R, int RS, int G, int wv, int lane, int r) {
    return wv * G * R + (r / RS) * G * RS + lane * RS + (r % RS);
}

// Pass 2 of a whole cell in the symmetric (action-reaction) form of pair_sym.cuh: Q(z)(g_p - g_q)/|z| once per
// unordered pair, applied to both markers -- 15 instead of 26 FP64 instructions per ordered pair.  Needs
// nu_ss' = c_s c_s' (DevTable::nu_rank1; c_s is folded into the weights, W = w c_s, and applied to the target at the
// end).  Thread tid owns R = ceil(n / 256) slots of its warp's sub-tile (cells_sym_slot; registers: position, g, W,
// target-side sums); warp w's 32 R slots are also "sub-tile" w of the sources.  Phase 0: every warp its own sub-tile (the
// lane's own group one-sided, every unordered pair of different groups once, both sides).
// Phases 1..3: warp w against sub-tile (w + ph) % 8, both sides.  Phase 4: the pairs {w, w + 4} are split between the
// two warps (steps 0..G/2-1 / 1..G/2 of the lane rotation).  Inside a phase lane l visits source group (l + k) % G at
// step k -- R consecutive slots, read as 16-byte vectors -- and adds the source-side sums into the shared-memory
// accumulators next to the sources: in a phase a sub-tile belongs to one warp and at a step every lane holds another
// group, so there are no conflicts, no atomics, and the order is the program's (deterministic).
// sx: seven arrays [cap] {ux uy uz W gx gy gz}; sa: [3][cap]; slots n .. n2 (n2 even, <= cap) hold zero dummies.
template <int R, int RS>
__device__ __forceinline__ void cells_field_sym(const double* __restrict__ sx, double* __restrict__ sa, int cap, int n,
                                                int n2, int G, double (&tx)[R], double (&ty)[R], double (&tz)[R]) {
    static_assert(R % RS == 0, "sources of a group are taken RS at a time");
    const int tid = threadIdx.x, lane = tid & 31, wv = tid >> 5;
    const double* X = sx; const double* Y = sx + cap; const double* Z = sx + 2 * (size_t)cap;
    const double* Wt = sx + 3 * (size_t)cap;
    const double* HX = sx + 4 * (size_t)cap; const double* HY = sx + 5 * (size_t)cap; const double* HZ = sx + 6 * (size_t)cap;
    double* AX = sa; double* AY = sa + cap; double* AZ = sa + 2 * (size_t)cap;
    double px[R], py[R], pz[R], gx[R], gy[R], gz[R], wp[R], ax[R], ay[R], az[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int p = cells_sym_slot(R, RS, G, wv, lane, r);
        const bool ok = lane < G && p < n2;
        px[r] = ok ? X[p] : 0.0; py[r] = ok ? Y[p] : 0.0; pz[r] = ok ? Z[p] : 0.0;
        gx[r] = ok ? HX[p] : 0.0; gy[r] = ok ? HY[p] : 0.0; gz[r] = ok ? HZ[p] : 0.0;
        wp[r] = ok ? Wt[p] : 0.0;
        ax[r] = ay[r] = az[r] = 0.0;
        if (ok) { AX[p] = 0.0; AY[p] = 0.0; AZ[p] = 0.0; }
    }
    __syncthreads();
    constexpr int NW = CELLS_THREADS / 32;
#pragma unroll 1
    for (int ph = 0; ph <= NW / 2; ++ph) {
        const int u = (wv + ph) & (NW - 1);
        // phase 0 (own sub-tile): step 0 = the lane's own group, one-sided; steps 1..G/2-1 both sides; step G/2 both
        // sides by the lower half of the lanes only (the pair of groups {l, l + G/2} is seen from both ends)
        const int GH = G >> 1;
        int k0 = 0, k1 = G;
        if (ph == 0) k1 = GH + 1;
        if (ph == NW / 2) { if (wv < NW / 2) k1 = GH; else { k0 = 1; k1 = GH + 1; } }
#pragma unroll 1
        for (int k = k0; k < k1; ++k) {
            const int gk = lane + k;
            const int gl = gk >= G ? gk - G : gk;                      // the group this lane visits: (lane + k) mod G
            const bool one = ph == 0 && k == 0;
            const bool act = lane < G && !(ph == 0 && k == GH && lane >= GH);
#pragma unroll
            for (int h = 0; h < R; h += RS) {
                double qx[RS], qy[RS], qz[RS], qw[RS], hx[RS], hy[RS], hz[RS], bx[RS], by[RS], bz[RS];
                const int q = cells_sym_slot(R, RS, G, u, gl, h);
                if (RS == 2) {
                    // q and n2 are even: both slots exist or neither
                    const bool ok = q < n2 && act;
                    const double2 zero = make_double2(0.0, 0.0);
                    const double2 a0 = ok ? *reinterpret_cast<const double2*>(X + q) : zero;
                    const double2 a1 = ok ? *reinterpret_cast<const double2*>(Y + q) : zero;
                    const double2 a2 = ok ? *reinterpret_cast<const double2*>(Z + q) : zero;
                    const double2 a3 = ok ? *reinterpret_cast<const double2*>(Wt + q) : zero;
                    const double2 a4 = ok ? *reinterpret_cast<const double2*>(HX + q) : zero;
                    const double2 a5 = ok ? *reinterpret_cast<const double2*>(HY + q) : zero;
                    const double2 a6 = ok ? *reinterpret_cast<const double2*>(HZ + q) : zero;
                    qx[0] = a0.x; qx[RS - 1] = a0.y; qy[0] = a1.x; qy[RS - 1] = a1.y; qz[0] = a2.x; qz[RS - 1] = a2.y;
                    qw[0] = a3.x; qw[RS - 1] = a3.y;
                    hx[0] = a4.x; hx[RS - 1] = a4.y; hy[0] = a5.x; hy[RS - 1] = a5.y; hz[0] = a6.x; hz[RS - 1] = a6.y;
                    if (one) {
                        sym_step3<false, R, RS, double>(px, py, pz, gx, gy, gz, wp, ax, ay, az, qx, qy, qz, hx, hy, hz, qw, bx, by, bz);
                    } else {
                        const double2 b0 = ok ? *reinterpret_cast<const double2*>(AX + q) : zero;
                        const double2 b1 = ok ? *reinterpret_cast<const double2*>(AY + q) : zero;
                        const double2 b2 = ok ? *reinterpret_cast<const double2*>(AZ + q) : zero;
                        bx[0] = b0.x; bx[RS - 1] = b0.y; by[0] = b1.x; by[RS - 1] = b1.y; bz[0] = b2.x; bz[RS - 1] = b2.y;
                        sym_step3<true, R, RS, double>(px, py, pz, gx, gy, gz, wp, ax, ay, az, qx, qy, qz, hx, hy, hz, qw, bx, by, bz);
                        if (ok) {
                            *reinterpret_cast<double2*>(AX + q) = make_double2(bx[0], bx[RS - 1]);
                            *reinterpret_cast<double2*>(AY + q) = make_double2(by[0], by[RS - 1]);
                            *reinterpret_cast<double2*>(AZ + q) = make_double2(bz[0], bz[RS - 1]);
                        }
                    }
                } else {
#pragma unroll
                    for (int s2 = 0; s2 < RS; ++s2) {
                        const bool ok = q + s2 < n2 && act;
                        qx[s2] = ok ? X[q + s2] : 0.0; qy[s2] = ok ? Y[q + s2] : 0.0; qz[s2] = ok ? Z[q + s2] : 0.0;
                        qw[s2] = ok ? Wt[q + s2] : 0.0;
                        hx[s2] = ok ? HX[q + s2] : 0.0; hy[s2] = ok ? HY[q + s2] : 0.0; hz[s2] = ok ? HZ[q + s2] : 0.0;
                    }
                    if (one) {
                        sym_step3<false, R, RS, double>(px, py, pz, gx, gy, gz, wp, ax, ay, az, qx, qy, qz, hx, hy, hz, qw, bx, by, bz);
                    } else {
#pragma unroll
                        for (int s2 = 0; s2 < RS; ++s2) {
                            const bool ok = q + s2 < n2 && act;
                            bx[s2] = ok ? AX[q + s2] : 0.0; by[s2] = ok ? AY[q + s2] : 0.0; bz[s2] = ok ? AZ[q + s2] : 0.0;
                        }
                        sym_step3<true, R, RS, double>(px, py, pz, gx, gy, gz, wp, ax, ay, az, qx, qy, qz, hx, hy, hz, qw, bx, by, bz);
#pragma unroll
                        for (int s2 = 0; s2 < RS; ++s2)
                            if (q + s2 < n2 && act) { AX[q + s2] = bx[s2]; AY[q + s2] = by[s2]; AZ[q + s2] = bz[s2]; }
                    }
                }
            }
            if (!one) __syncwarp();
        }
        __syncthreads();
    }
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int p = cells_sym_slot(R, RS, G, wv, lane, r);
        const bool ok = lane < G && p < n2;
        tx[r] = ax[r] - (ok ? AX[p] : 0.0); ty[r] = ay[r] - (ok ? AY[p] : 0.0); tz[r] = az[r] - (ok ? AZ[p] : 0.0);
    }
}

// MINB = 1: any cell up to the shared-memory capacity, one CTA of 256 threads per SM (255 registers: register-tiled pair
// loops, DMMA accumulators).  MINB > 1 (n_q = 4, every cell of the batch <= NT / 2 markers): only the small-cell paths (2
// or 4 threads per target) are compiled, 128 registers; <4, 2, 256>: cells of <= 128 markers, two CTAs per SM;
// <4, 4, 128>: cells of <= 64 markers, four CTAs of 128 threads per SM -- such cells are bound by the latencies of their
// barriers and reductions, not by the FP64 pipe, and more resident cells fill the gaps.
constexpr int CELLS_SMALL = CELLS_THREADS / 2;

template <int NQ, int MINB = 1, int NT = CELLS_THREADS>
__global__ void __launch_bounds__(NT, MINB)
cells_run_kernel(const DevTable* __restrict__ T, int n_cells, int cap, const long long* __restrict__ cell_off,
                 const double* __restrict__ v, const double* __restrict__ w, const int32_t* __restrict__ sid,
                 double* __restrict__ v_out, int n_steps, double dt, double tol, int max_iter,
                 int* __restrict__ next_cell, CellRecord* __restrict__ records) {
    static_assert(MINB > 1 || NT == CELLS_THREADS, "the register-tiled paths are written for 256 threads");
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* xn = reinterpret_cast<double*>(smem_raw);
    double* yn = xn + cap; double* zn = yn + cap; double* ww = zn + cap;
    double* Gx = ww + cap; double* Gy = Gx + cap; double* Gz = Gy + cap;
    double* xk = Gz + cap; double* yk = xk + cap; double* zk = yk + cap;
    double* tab = zk + cap;                               // [cap][3 NQ] in pass 1; source records [cap][8] in pass 2
    double* srec = tab;
    double* s_e2 = tab + (size_t)CellsCfg<NQ>::TAB * cap; // [64]
    double* s_red = s_e2 + 64;                            // [32]
    double* s_part = s_red + 32;                          // [GF][3][TPG] partial sums of split targets (small cells)
    int* idx = reinterpret_cast<int*>(s_part + 3 * NT);   // [cap] caller index (within the cell) of slot p
    __shared__ int s_off[LD_MAX_SPECIES + 1];
    __shared__ int s_wcnt[NT / 32];
    __shared__ int s_cell, s_status;
    __shared__ double s_nu[LD_MAX_SPECIES * LD_MAX_SPECIES];

    const int tid = threadIdx.x, lane = tid & 31, wv = tid >> 5;
    const int S = T->S;
    if (tid < 64) s_e2[tid] = T->exp2_tab[tid];
    for (int i = tid; i < S * S; i += NT) s_nu[i] = T->nu[i];
    double kn[NQ], ga[NQ];
#pragma unroll
    for (int i = 0; i < NQ; ++i) { kn[i] = T->knot[i]; ga[i] = T->gw[i]; }
    const double kmax = fabs(kn[NQ - 1]);
    const double PI = 3.14159265358979323846;

    for (;;) {
        __syncthreads();
        if (tid == 0) { s_cell = atomicAdd(next_cell, 1); s_status = 0; }
        __syncthreads();
        const int cell = s_cell;
        if (cell >= n_cells) return;
        const long long g0 = cell_off[cell];
        const int n = (int)(cell_off[cell + 1] - g0);
        CellRecord rec;
        rec.status = 0; rec.iterations = 0; rec.max_iterations = 0; rec.steps_not_converged = 0; rec.residual = 0.0;
        auto pass_through = [&]() {                                    // failed cell: output = input
            if (v_out != v && n > 0)
                for (long long i = tid; i < 3LL * n; i += NT) v_out[3 * g0 + i] = v[3 * g0 + i];
        };
        if (n < 1 || n > cap || (MINB > 1 && n > NT / 2)) {
            pass_through();
            if (tid == 0) { rec.status = n == 0 ? 0 : -1; records[cell] = rec; }
            continue;
        }
        // ---- load + stable bucketing by species (caller order preserved inside a species)
        int base = 0;
        for (int s = 0; s < S; ++s) {
            if (tid == 0) s_off[s] = base;
            for (int c0 = 0; c0 < n; c0 += NT) {
                const int i = c0 + tid;
                int si = -2;
                if (i < n) { si = sid[g0 + i]; if (si < 0 || si >= S) { si = -2; s_status = -1; } }
                const bool mine = si == s;
                const unsigned m = __ballot_sync(0xffffffffu, mine);
                if (lane == 0) s_wcnt[wv] = __popc(m);
                __syncthreads();
                int before = 0, total = 0;
                for (int k = 0; k < NT / 32; ++k) { if (k < wv) before += s_wcnt[k]; total += s_wcnt[k]; }
                if (mine) {
                    const int p = base + before + __popc(m & ((1u << lane) - 1u));
                    const double a = v[3 * (g0 + i)], b = v[3 * (g0 + i) + 1], c = v[3 * (g0 + i) + 2], wi = w[g0 + i];
                    if (!(isfinite(a) && isfinite(b) && isfinite(c) && isfinite(wi))) s_status = -4;
                    else if (!(wi > 0.0)) s_status = -1;
                    xn[p] = a; yn[p] = b; zn[p] = c; ww[p] = wi; idx[p] = i;
                }
                base += total;
                __syncthreads();
            }
        }
        if (tid == 0) for (int s = S; s <= LD_MAX_SPECIES; ++s) s_off[s] = base;
        __syncthreads();
        if (s_status != 0 || base != n) {
            pass_through();
            if (tid == 0) { rec.status = s_status != 0 ? s_status : -1; records[cell] = rec; }
            continue;
        }
        // threads per target: small cells (NQ = 4 only) put 2 or 4 threads on every target
        const int GF = (NQ == 4) ? (n <= NT / 4 ? 4 : (n <= NT / 2 ? 2 : 1)) : 1;
        const int TPG = NT / GF, part = tid / TPG, tg = tid % TPG;
        for (int step = 0; step < n_steps && s_status == 0; ++step) {
            // ---- pass 1 (Eq. 22, factorised): G_p for every species, sources = same species of this cell
            for (int s = 0; s < S; ++s) {
                const int o0 = s_off[s], o1 = s_off[s + 1];
                if (o0 == o1) continue;
                const double eps = T->eps[s], inv = T->inv_sqrt_2eps[s];
                // bounding box -> centre and half-width in mollifier units
                double lo[3] = {1.7976931348623157e308, 1.7976931348623157e308, 1.7976931348623157e308};
                double hi[3] = {-1.7976931348623157e308, -1.7976931348623157e308, -1.7976931348623157e308};
                for (int p = o0 + tid; p < o1; p += NT) {
                    lo[0] = fmin(lo[0], xn[p]); hi[0] = fmax(hi[0], xn[p]);
                    lo[1] = fmin(lo[1], yn[p]); hi[1] = fmax(hi[1], yn[p]);
                    lo[2] = fmin(lo[2], zn[p]); hi[2] = fmax(hi[2], zn[p]);
                }
                double cen[3], hw = 0.0;
#pragma unroll
                for (int d = 0; d < 3; ++d) {
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1) {
                        lo[d] = fmin(lo[d], __shfl_xor_sync(0xffffffffu, lo[d], o));
                        hi[d] = fmax(hi[d], __shfl_xor_sync(0xffffffffu, hi[d], o));
                    }
                    __syncthreads();
                    if (lane == 0) { s_red[2 * wv] = lo[d]; s_red[2 * wv + 1] = hi[d]; }
                    __syncthreads();
                    double a = s_red[0], b = s_red[1];
                    for (int k = 1; k < NT / 32; ++k) { a = fmin(a, s_red[2 * k]); b = fmax(b, s_red[2 * k + 1]); }
                    cen[d] = 0.5 * a + 0.5 * b;
                    hw = fmax(hw, 0.5 * b - 0.5 * a);
                }
                // a cell too wide for the factorised form (reading N3) takes the literal-separable one
                const bool literal = !(6.0 * kmax * hw * inv <= FACT_EXP_LIMIT);
                // scaled coordinates (alias of xk..zk) and the per-marker exponential tables
                for (int p = o0 + tid; p < o1; p += NT) {
                    const double a = (xn[p] - cen[0]) * inv, b = (yn[p] - cen[1]) * inv, c = (zn[p] - cen[2]) * inv;
                    xk[p] = a; yk[p] = b; zk[p] = c;
                    if (!literal) {
                        double* t = tab + (size_t)p * 3 * NQ;
#pragma unroll
                        for (int i = 0; i < NQ; ++i) {
                            const double k2 = 2.0 * kn[i];
                            t[i] = exp(k2 * a); t[NQ + i] = exp(k2 * b); t[2 * NQ + i] = exp(k2 * c);
                        }
                    }
                }
                __syncthreads();
                const double lognorm = -1.5 * log(2.0 * PI * eps);
                const double pref = -sqrt(2.0 / eps) / (PI * sqrt(PI));
                if (GF > 1) {
                    // small cell: GF threads per target, each a slice of NQ/GF x-node indices; partial sums meet in
                    // shared memory and are added in part order (deterministic)
                    const int pt = o0 + tg;
                    const int p = min(pt, o1 - 1);
                    const double px = xk[p], py = yk[p], pz = zk[p];
                    double gx, gy, gz;
                    if (GF == 2) {
                        if (literal)
                            cells_pass1_target<NQ, (NQ >= 2 ? NQ / 2 : 1), true>(part * (NQ / 2), o0, o1, px, py, pz, xk, yk, zk,
                                                                                 ww, tab, s_e2, kn, ga, lognorm, gx, gy, gz);
                        else
                            cells_pass1_target<NQ, (NQ >= 2 ? NQ / 2 : 1), false>(part * (NQ / 2), o0, o1, px, py, pz, xk, yk, zk,
                                                                                  ww, tab, s_e2, kn, ga, lognorm, gx, gy, gz);
                    } else {
                        if (literal)
                            cells_pass1_target<NQ, (NQ >= 4 ? NQ / 4 : 1), true>(part * (NQ / 4), o0, o1, px, py, pz, xk, yk, zk,
                                                                                 ww, tab, s_e2, kn, ga, lognorm, gx, gy, gz);
                        else
                            cells_pass1_target<NQ, (NQ >= 4 ? NQ / 4 : 1), false>(part * (NQ / 4), o0, o1, px, py, pz, xk, yk, zk,
                                                                                  ww, tab, s_e2, kn, ga, lognorm, gx, gy, gz);
                    }
                    s_part[(part * 3 + 0) * TPG + tg] = gx;
                    s_part[(part * 3 + 1) * TPG + tg] = gy;
                    s_part[(part * 3 + 2) * TPG + tg] = gz;
                    __syncthreads();
                    if (part == 0 && pt < o1) {
                        double a = 0.0, b = 0.0, c = 0.0;
                        for (int g2 = 0; g2 < GF; ++g2) {
                            a += s_part[(g2 * 3 + 0) * TPG + tg]; b += s_part[(g2 * 3 + 1) * TPG + tg];
                            c += s_part[(g2 * 3 + 2) * TPG + tg];
                        }
                        a *= pref; b *= pref; c *= pref;
                        if (!(isfinite(a) && isfinite(b) && isfinite(c))) s_status = -4;
                        Gx[p] = a; Gy[p] = b; Gz[p] = (T->dim == 2) ? 0.0 : c;
                    }
                } else if (MINB == 1 && NQ == 4 && !literal) {
                    if constexpr (NQ == 4 && MINB == 1)
                        cells_pass1_dmma4(o0, o1, xk, yk, zk, ww, tab, s_e2, kn, ga, lognorm, pref, T->dim == 2, Gx, Gy, Gz,
                                          &s_status);
                } else if constexpr (MINB == 1) {
                    for (int r0 = o0; r0 < o1; r0 += NT) {
                        const int pt = r0 + tid;
                        const int p = min(pt, o1 - 1);                 // clamped duplicate; not written
                        const double px = xk[p], py = yk[p], pz = zk[p];
                        double gx = 0.0, gy = 0.0, gz = 0.0;
                        constexpr int NI = CellsCfg<NQ>::NI;
#pragma unroll 1
                        for (int i0 = 0; i0 < NQ; i0 += NI) {          // n_q > 4: slices of x-node indices
                            double sx, sy, sz;
                            if (literal)
                                cells_pass1_target<NQ, NI, true>(i0, o0, o1, px, py, pz, xk, yk, zk, ww, tab, s_e2, kn, ga,
                                                                 lognorm, sx, sy, sz);
                            else
                                cells_pass1_target<NQ, NI, false>(i0, o0, o1, px, py, pz, xk, yk, zk, ww, tab, s_e2, kn, ga,
                                                                  lognorm, sx, sy, sz);
                            gx += sx; gy += sy; gz += sz;
                        }
                        gx *= pref; gy *= pref; gz *= pref;
                        if (pt < o1) {
                            if (!(isfinite(gx) && isfinite(gy) && isfinite(gz))) s_status = -4;
                            Gx[p] = gx; Gy[p] = gy; Gz[p] = (T->dim == 2) ? 0.0 : gz;
                        }
                    }
                }
                __syncthreads();
            }
            __syncthreads();
            if (s_status != 0) break;
            // ---- Eq. (24): Jacobi fixed point, G^n frozen (g = G/m in place), v^(0) = v^n
            // symmetric in-cell evaluation (cells_field_sym) when nu_ss' = c_s c_s' and the cell has more than one slot per
            // thread (> 256 markers; with one slot per thread the one-sided loop and its broadcast reads are faster)
            const int rounds = ceil_div(n, NT);
#ifndef LANDAU_CELLS_SYM_MIN     // tuning knob (build.py: LANDAU_NVCC_EXTRA): smallest cell taking the symmetric evaluation
#define LANDAU_CELLS_SYM_MIN 257
#endif
            const bool use_sym = GF == 1 && T->nu_rank1 != 0 && n >= LANDAU_CELLS_SYM_MIN;
            // groups of `rounds` slots per warp: the even count that just covers the cell (<= 32)
            const int symG = min(32, (ceil_div(ceil_div(n, rounds), NT / 32) + 1) & ~1);
            const int n2 = min((NT / 32) * symG * rounds, cap);        // cap is even: pairs of slots exist or not together
            double* const sxa = tab;                                   // [7][cap] sources, then [3][cap] source-side sums
            double* const saa = tab + 7 * (size_t)cap;
            // slot of this thread's r-th target: consecutive slots in the symmetric evaluation, strided otherwise
            auto slot_of = [&](int r) {
                return use_sym ? ((r < rounds && lane < symG) ? cells_sym_slot(rounds, rounds == 3 ? 3 : 2, symG, wv, lane, r) : n)
                               : r * NT + tid;
            };
            int sp[CELLS_ROUNDS];
            double im[CELLS_ROUNDS], wm[CELLS_ROUNDS];
#pragma unroll
            for (int r = 0; r < CELLS_ROUNDS; ++r) {
                const int p = slot_of(r);
                sp[r] = 0; im[r] = 0.0; wm[r] = 0.0;
                if (p < n) {
                    int s = 0;
                    for (int t = 1; t < S; ++t) s += (p >= s_off[t]) ? 1 : 0;
                    sp[r] = s; im[r] = T->inv_mass[s]; wm[r] = ww[p] * T->mass[s];
                    xk[p] = xn[p]; yk[p] = yn[p]; zk[p] = zn[p];
                }
            }
            __syncthreads();                                           // pass 1 has read its tables: the region is free
#pragma unroll
            for (int r = 0; r < CELLS_ROUNDS; ++r) {
                const int p = slot_of(r);
                if (p < n) {
                    if (use_sym) {
                        sxa[p] = xn[p]; sxa[cap + p] = yn[p]; sxa[2 * (size_t)cap + p] = zn[p];
                        sxa[3 * (size_t)cap + p] = ww[p] * T->nu_fac[sp[r]];
                        sxa[4 * (size_t)cap + p] = Gx[p] * im[r]; sxa[5 * (size_t)cap + p] = Gy[p] * im[r];
                        sxa[6 * (size_t)cap + p] = Gz[p] * im[r];
                    } else {
                        double2* o = reinterpret_cast<double2*>(srec + (size_t)p * 8);
                        o[0] = make_double2(xn[p], yn[p]);
                        o[1] = make_double2(zn[p], ww[p]);
                        o[2] = make_double2(Gx[p] * im[r], Gy[p] * im[r]);
                        o[3] = make_double2(Gz[p] * im[r], 0.0);
                    }
                }
            }
            if (use_sym)                                               // zero dummies behind the cell's last marker
                for (int p = n + tid; p < n2; p += NT)
                    for (int c = 0; c < 7; ++c) sxa[(size_t)c * cap + p] = 0.0;
            __syncthreads();
            int it = 0, conv = 0;
            double res = 0.0;
            while (it < max_iter) {
                double nx[CELLS_ROUNDS], ny[CELLS_ROUNDS], nz[CELLS_ROUNDS];
                double num = 0.0, den = 0.0;
#pragma unroll
                for (int r = 0; r < CELLS_ROUNDS; ++r) nx[r] = ny[r] = nz[r] = 0.0;
                auto finish_target = [&](int r, double tx, double ty, double tz) {
                    const int p = slot_of(r);
                    if (p < n) {
                        const double a = fma(dt, tx * im[r], xn[p]), b = fma(dt, ty * im[r], yn[p]),
                                     c = fma(dt, tz * im[r], zn[p]);
                        const double dx = a - xk[p], dy = b - yk[p], dz = c - zk[p];
                        num += wm[r] * (dx * dx + dy * dy + dz * dz);
                        den += wm[r] * (a * a + b * b + c * c);
                        nx[r] = a; ny[r] = b; nz[r] = c;
                    }
                };
                if (GF > 1) {
                    // small cell: the GF threads of a target take consecutive slices of every source species
                    const int pc = min(tg, n - 1);
                    int spt = 0;
                    for (int t = 1; t < S; ++t) spt += (pc >= s_off[t]) ? 1 : 0;
                    const double* rp = srec + (size_t)pc * 8;
                    const double px = rp[0], py = rp[1], pz = rp[2], hx = rp[4], hy = rp[5], hz = rp[6];
                    double tx = 0.0, ty = 0.0, tz = 0.0;
                    for (int sb = 0; sb < S; ++sb) {
                        const int q0 = s_off[sb], len = s_off[sb + 1] - q0;
                        const int qa = q0 + (len * part) / GF, qb = q0 + (len * (part + 1)) / GF;
                        double ax = 0.0, ay = 0.0, az = 0.0;
#pragma unroll 4
                        for (int q = qa; q < qb; ++q) {
                            const double2* r2 = reinterpret_cast<const double2*>(srec + (size_t)q * 8);
                            const double2 a = r2[0], b = r2[1], c = r2[2], d = r2[3];
                            pair_accumulate(px - a.x, py - a.y, pz - b.x, hx - c.x, hy - c.y, hz - d.x, b.y, ax, ay, az);
                        }
                        const double nu = s_nu[spt * S + sb];
                        tx = fma(nu, ax, tx); ty = fma(nu, ay, ty); tz = fma(nu, az, tz);
                    }
                    s_part[(part * 3 + 0) * TPG + tg] = tx;
                    s_part[(part * 3 + 1) * TPG + tg] = ty;
                    s_part[(part * 3 + 2) * TPG + tg] = tz;
                    __syncthreads();
                    if (part == 0) {
                        double a = 0.0, b = 0.0, c = 0.0;
                        for (int g2 = 0; g2 < GF; ++g2) {
                            a += s_part[(g2 * 3 + 0) * TPG + tg]; b += s_part[(g2 * 3 + 1) * TPG + tg];
                            c += s_part[(g2 * 3 + 2) * TPG + tg];
                        }
                        finish_target(0, a, b, c);
                    }
                } else if constexpr (MINB == 1) {
                if (use_sym) {
                    // block-uniform branch on the cell size: R slots per thread
                    if (rounds == 4) {
                        double tx[4], ty[4], tz[4];
                        cells_field_sym<4, 2>(sxa, saa, cap, n, n2, symG, tx, ty, tz);
#pragma unroll
                        for (int r = 0; r < 4; ++r) { const double cf = T->nu_fac[sp[r]]; finish_target(r, tx[r] * cf, ty[r] * cf, tz[r] * cf); }
                    } else if (rounds == 3) {
                        double tx[3], ty[3], tz[3];
                        cells_field_sym<3, 3>(sxa, saa, cap, n, n2, symG, tx, ty, tz);
#pragma unroll
                        for (int r = 0; r < 3; ++r) { const double cf = T->nu_fac[sp[r]]; finish_target(r, tx[r] * cf, ty[r] * cf, tz[r] * cf); }
                    } else {
                        double tx[2], ty[2], tz[2];
                        cells_field_sym<2, 2>(sxa, saa, cap, n, n2, symG, tx, ty, tz);
#pragma unroll
                        for (int r = 0; r < 2; ++r) { const double cf = T->nu_fac[sp[r]]; finish_target(r, tx[r] * cf, ty[r] * cf, tz[r] * cf); }
                    }
                } else
                {
                    // all rounds of targets of a thread share every source read (block-uniform branch on the cell size)
                    static_assert(CELLS_ROUNDS == 4, "one branch per number of rounds");
                    int pc4[4], sp4[4];
#pragma unroll
                    for (int r = 0; r < 4; ++r) { pc4[r] = min(r * NT + tid, n - 1); sp4[r] = sp[r]; }
                    if (rounds == 4) {
                        double tx[4], ty[4], tz[4];
                        cells_field<4>(srec, s_off, s_nu, S, pc4, sp4, tx, ty, tz);
#pragma unroll
                        for (int r = 0; r < 4; ++r) finish_target(r, tx[r], ty[r], tz[r]);
                    } else if (rounds == 3) {
                        const int pc[3] = {pc4[0], pc4[1], pc4[2]}, spc[3] = {sp4[0], sp4[1], sp4[2]};
                        double tx[3], ty[3], tz[3];
                        cells_field<3>(srec, s_off, s_nu, S, pc, spc, tx, ty, tz);
#pragma unroll
                        for (int r = 0; r < 3; ++r) finish_target(r, tx[r], ty[r], tz[r]);
                    } else if (rounds == 2) {
                        const int pc[2] = {pc4[0], pc4[1]}, spc[2] = {sp4[0], sp4[1]};
                        double tx[2], ty[2], tz[2];
                        cells_field<2>(srec, s_off, s_nu, S, pc, spc, tx, ty, tz);
                        finish_target(0, tx[0], ty[0], tz[0]);
                        finish_target(1, tx[1], ty[1], tz[1]);
                    } else {
                        const int pc[1] = {pc4[0]}, spc[1] = {sp4[0]};
                        double tx[1], ty[1], tz[1];
                        cells_field<1>(srec, s_off, s_nu, S, pc, spc, tx, ty, tz);
                        finish_target(0, tx[0], ty[0], tz[0]);
                    }
                }
                }   // MINB == 1
                cells_reduce2<NT>(num, den, s_red);                        // also the barrier after all reads of u
#pragma unroll
                for (int r = 0; r < CELLS_ROUNDS; ++r) {
                    const int p = slot_of(r);
                    if (p < n) {
                        xk[p] = nx[r]; yk[p] = ny[r]; zk[p] = nz[r];
                        const double ux = 0.5 * (xn[p] + nx[r]), uy = 0.5 * (yn[p] + ny[r]), uz = 0.5 * (zn[p] + nz[r]);
                        if (use_sym) { sxa[p] = ux; sxa[cap + p] = uy; sxa[2 * (size_t)cap + p] = uz; }
                        else { double* o = srec + (size_t)p * 8; o[0] = ux; o[1] = uy; o[2] = uz; }
                    }
                }
                __syncthreads();
                res = sqrt(num / den);
                ++it;
                if (!isfinite(res)) { if (tid == 0) s_status = -4; break; }
                if (res <= tol) { conv = 1; break; }
            }
            __syncthreads();
            if (s_status != 0) break;
            // commit (also when not converged, reading S8)
            for (int p = tid; p < n; p += NT) { xn[p] = xk[p]; yn[p] = yk[p]; zn[p] = zk[p]; }
            rec.iterations += it;
            rec.max_iterations = max(rec.max_iterations, it);
            rec.steps_not_converged += conv ? 0 : 1;
            rec.residual = res;
            __syncthreads();
        }
        __syncthreads();
        if (s_status != 0) {                                           // error: the cell is left unchanged
            pass_through();
            if (tid == 0) { rec.status = s_status; records[cell] = rec; }
            continue;
        }
        for (int p = tid; p < n; p += NT) {
            double* o = v_out + 3 * (g0 + idx[p]);
            o[0] = xn[p]; o[1] = yn[p]; o[2] = zn[p];
        }
        if (tid == 0) { rec.status = rec.steps_not_converged ? 1 : 0; records[cell] = rec; }
    }
}

}  // namespace landau
