// common.cuh -- shared device-side definitions of the CUDA path (NOT shared with oracle/).
//
// Packed marker layout.  Markers are bucketed by species
// (stable), each species padded with zero-weight dummies to a multiple of `pad`; slot index
// p in [0, npad).  Structure of arrays, FP64:
//     x[p], y[p], z[p]   velocity                      w[p]  weight (0 for dummies)
//     perm[p]            caller index of the marker in slot p, -1 for dummies
// A dummy has v = 0, w = 0, G = 0: as a source it contributes exactly 0 to both passes, as a
// target its result is discarded.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define LD_MAX_SPECIES 16
#define LD_MAX_NQ 8

namespace landau {

// Per-context species / quadrature table, lives in device global memory (one copy per context).
struct DevTable {
    int S;
    int n_q;
    int pad;                          // padding granularity of the packed layout (slots)
    int dim;                          // 3 (default) or 2: 2-V mode, v_z = 0 is kept exactly (landau_set_dimension)
    double mass[LD_MAX_SPECIES];
    double inv_mass[LD_MAX_SPECIES];
    double eps[LD_MAX_SPECIES];
    double inv_sqrt_2eps[LD_MAX_SPECIES];   // 1/sqrt(2 eps_s): velocity -> mollifier units
    double nu[LD_MAX_SPECIES * LD_MAX_SPECIES];
    double knot[LD_MAX_NQ];           // Gauss-Hermite knots k_i (weight exp(-k^2))
    double gw[LD_MAX_NQ];             // Gauss-Hermite weights a_i
    double exp2_tab[64];              // 2^(j/64), j = 0..63 (table of exp_neg_tab, entropy_mma.cuh)
    double exp2_tab256[256];          // 2^(j/256) (table of exp_neg_t256, entropy_mma.cuh)
    double nu_fac[LD_MAX_SPECIES];    // nu_ss' = nu_fac[s] nu_fac[s'] when nu_rank1 (the default nu0 q_s^2 q_s'^2 is)
    int nu_rank1;
    int _r0;
};

// Per-pack layout, written on the device by the pack kernels (no host round trip needed).
struct DevLayout {
    int count[LD_MAX_SPECIES];        // markers of species s
    int off[LD_MAX_SPECIES + 1];      // first slot of species s; off[S] = npad (all multiples of pad)
    int npad;
    int err;                          // 0, or LANDAU_E* found by a kernel (validation, non-finite)
    int used_fact;                    // 1 if the last pass 1 took the factorised kernel
    int _r1;
    double center[LD_MAX_SPECIES][3]; // bounding-box centre of species s (factorised pass 1)
    double halfwidth[LD_MAX_SPECIES]; // max_p |v_p - center|_inf / sqrt(2 eps_s), written once per pass 1
    double cut_T[LD_MAX_SPECIES];     // Gaussian cutoff of pass 1 (entropy.cuh, tile_is_far): a source tile at box
                                      // distance d (mollifier units) is skipped when d^2 - 2 d |k|_max >= cut_T[s]
};

// Device-side control block of the fixed-point loop.
struct StepCtrl {
    int done;            // 1 once r_k <= tol (or a non-finite residual was seen): later launches exit
    int iterations;
    int converged;
    int err;
    double residual;
    unsigned int ticket; // last-block-done counter of the residual reduction
    int hold;            // 1: step_commit keeps v^n when the step did not converge (adaptive sub-stepping)
    int use_f32;         // mixed-precision step (landau_set_mixed_precision): 1 = the next pass 2 runs in FP32
    int _r;
};

struct StepRecord {      // mirrors landau_step_info (host struct) field by field
    int iterations;
    double residual;
    int converged;
};

__host__ __device__ inline int ceil_div(int a, int b) { return (a + b - 1) / b; }

// Which of several alternative kernels enqueued for one iteration of a device-driven step actually runs.
// 0: always; 1 / 2: only if the mixed-precision flag is set / clear; 3 / 4: only for the first / a later iteration.
constexpr int GATE_NONE = 0, GATE_F32 = 1, GATE_F64 = 2, GATE_FIRST = 3, GATE_LATER = 4;
__device__ __forceinline__ bool gate_closed(const StepCtrl* __restrict__ ctrl, int gate) {
    if (!ctrl || gate == GATE_NONE) return false;
    if (gate == GATE_F32) return ctrl->use_f32 != 1;
    if (gate == GATE_F64) return ctrl->use_f32 != 0;
    if (gate == GATE_FIRST) return ctrl->iterations != 0;
    return ctrl->iterations == 0;
}

__device__ __forceinline__ int species_of_slot(const DevLayout* __restrict__ L, int S, int slot) {
    int s = 0;
#pragma unroll 1
    for (int t = 1; t < S; ++t) s += (slot >= L->off[t]) ? 1 : 0;
    return s;
}

// FP64 reciprocal square root to < 1 ulp-ish: hardware seed (MUFU.RSQ64H, ~2^-20 relative after
// the operand's low word is ignored) + one third-order (Halley) correction, 5 FP64-pipe
// instructions.  With e = 1 - x y^2:  x^(-1/2) = y (1 + e/2 + 3 e^2/8 + O(e^3)); the dropped term
// is (5/16) e^3 < 2^-58.  x = 0 and subnormal x return 0 (reading S5: a coincident pair contributes
// nothing); callers rely on that to skip the self pair without a branch.
__device__ __forceinline__ double rsqrt_or_zero(double x) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    if (__double2hiint(x) < 0x00100000) y = 0.0;   // +0 / subnormal (x >= 0 always here)
    const double t = x * y;
    const double e = fma(-t, y, 1.0);
    const double p = fma(0.375, e, 0.5);
    const double ye = y * e;
    return fma(ye, p, y);
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

}  // namespace landau
