/*
 * landau_ref.h -- C ABI of the CPU ORACLE (test infrastructure, not the product).
 *
 * Plain, slow, literal restatement of the multispecies particle Landau scheme of
 * Zonta, Pusztay, Hirvijoki, arXiv:2212.00663, in the 3-V form of SURVEY.md
 * section 8(c) (readings D1, D2, S1-S10, U1-U3 are listed in DESIGN.md).
 *
 * ONLY tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may call this library.  It shares no code with the CUDA path (paper_2212_00663_b200/csrc,
 * include/landau.h): no common header, table generator, helper or constant.
 *
 * All pointers are HOST pointers.  v is [N x 3] row-major, w is [N], species_id is [N] in
 * 0..S-1 in any order.  Every function returns 0 on success, 1 = step not converged (the
 * step is still committed), -1 invalid argument, -2 out of memory,
 * -4 non-finite input or result.
 */
#ifndef LANDAU_REF_H
#define LANDAU_REF_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct landau_ref_ctx landau_ref_ctx;

typedef struct {
    int iterations;
    double residual;
    int converged;
} landau_ref_step_info;

/* O1: n-point Gauss-Hermite rule for weight exp(-k^2). */
int landau_ref_gauss_hermite(int n, double* knots, double* weights);

/* nu (S x S, symmetric) may be NULL: nu_ss' = nu0 * q_s^2 * q_s'^2 (reading U1). */
int landau_ref_create(landau_ref_ctx** out, int n_species, const double* mass, const double* charge,
                      const double* eps, int n_q, double nu0, const double* nu);
void landau_ref_destroy(landau_ref_ctx* ctx);
int landau_ref_num_threads(void);
void landau_ref_set_num_threads(int n);

/* O2: G_p = (1/w_p) dS_eps/dv_p, 3-V Eq. (22); S_eps_out (S entries, Eq. 20) may be NULL. */
int landau_ref_entropy_grad(landau_ref_ctx* ctx, int64_t N, const double* v, const double* w,
                            const int32_t* species_id, double* G_out, double* S_eps_out);
/* same, but only for the n_rows target markers listed in rows[]; G_out is [n_rows x 3]. */
int landau_ref_entropy_grad_rows(landau_ref_ctx* ctx, int64_t N, const double* v, const double* w,
                                 const int32_t* species_id, int64_t n_rows, const int64_t* rows,
                                 double* G_out);

/* O3: V_p of Eq. (23) with the entropy gradient G_in supplied. */
int landau_ref_pair_field(landau_ref_ctx* ctx, int64_t N, const double* v, const double* w,
                          const int32_t* species_id, const double* G_in, double* out);
int landau_ref_pair_field_rows(landau_ref_ctx* ctx, int64_t N, const double* v, const double* w,
                               const int32_t* species_id, const double* G_in, int64_t n_rows,
                               const int64_t* rows, double* out);

/* O2 then O3. */
int landau_ref_eval_field(landau_ref_ctx* ctx, int64_t N, const double* v, const double* w,
                          const int32_t* species_id, double* out);

/* context-held state for time stepping */
int landau_ref_set_markers(landau_ref_ctx* ctx, int64_t N, const double* v, const double* w,
                           const int32_t* species_id);
int landau_ref_get_markers(landau_ref_ctx* ctx, double* v_out);
/* O4: one step of Eq. (24)-(25) by Jacobi fixed-point iteration. */
int landau_ref_step(landau_ref_ctx* ctx, double dt, double tol, int max_iter,
                    landau_ref_step_info* info);
/* O4b: one step of the discrete-gradient scheme, Eqs. (46)-(49), with Gonzalez' midpoint discrete
 * gradient of S_eps (reading DG1); same fixed point, residual and status conventions as O4. */
int landau_ref_step_dg(landau_ref_ctx* ctx, double dt, double tol, int max_iter,
                       landau_ref_step_info* info);
/* O5: n_s, P_s (S x 3), K_s, S_eps,s of the held markers; any output may be NULL. */
int landau_ref_moments(landau_ref_ctx* ctx, double* n, double* P, double* K, double* S_eps);
/* stress: S x 6 = m_s sum w v_i v_j in order xx,yy,zz,xy,xz,yz; m4: S x 3 = sum w (v_i-u_i)^4 */
int landau_ref_moments_ext(landau_ref_ctx* ctx, double* stress, double* m4);

#ifdef __cplusplus
}
#endif
#endif
