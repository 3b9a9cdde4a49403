// landau_api.cu -- the C ABI of include/landau.h: context, scratch management, launch logic.
// Every arithmetic step of the path runs in the kernels of this directory; there is no CPU
// fallback and nothing here touches oracle/.
#include "../../include/landau.h"

#include <cuda_runtime.h>
#include <nvtx3/nvToolsExt.h>
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <cmath>
#include <new>
#include <vector>

#include "common.cuh"
#include "entropy.cuh"
#include "entropy_fact.cuh"
#include "entropy_mma.cuh"
#include "moments.cuh"
#include "pack.cuh"
#include "pair.cuh"
#include "pair_sym.cuh"
#include "step.cuh"
#include "step_small.cuh"
#include "step_dg.cuh"
#include "step_anderson.cuh"
#include "step_newton.cuh"
#include "stiff_pairs.cuh"
#include "cells.cuh"

using namespace landau;

namespace {

struct Buf {
    void* p = nullptr;
    size_t cap = 0;
};

// Packed marker cloud (device).  Two live in a context: `tmp` for the stateless calls and `state`
// for the markers held by landau_set_markers.
struct Cloud {
    int64_t N = 0;
    int npad_max = 0;
    int pad = 0;
    Buf lay, xyzw, perm, G, rec, soa;
    bool G_valid = false;   // G / snode hold pass 1 of the CURRENT x, y, z (lets a step reuse the pass 1 of landau_moments)
    int sym = 0;   // 1: the symmetric pair kernel's layout (pad = its target tile) and SoA source copy
    DevLayout* L() const { return (DevLayout*)lay.p; }
    double* x() const { return (double*)xyzw.p; }
    double* y() const { return x() + npad_max; }
    double* z() const { return x() + 2 * (size_t)npad_max; }
    double* w() const { return x() + 3 * (size_t)npad_max; }
    int* prm() const { return (int*)perm.p; }
    double* Gx() const { return (double*)G.p; }
    double* Gy() const { return Gx() + npad_max; }
    double* Gz() const { return Gx() + 2 * (size_t)npad_max; }
    double* snode() const { return Gx() + 3 * (size_t)npad_max; }
    double* recs() const { return (double*)rec.p; }
    double* soas() const { return (double*)soa.p; }
};

}  // namespace

struct landau_ctx {
    int S = 0;
    int n_q = 4;
    int precision = 0;
    int pair_kernel = 0;
    int entropy_kernel = 0;
    int device = 0;
    int sm_count = 148;
    cudaStream_t stream = nullptr;
    double mass[LD_MAX_SPECIES], charge[LD_MAX_SPECIES], eps[LD_MAX_SPECIES];
    double nu[LD_MAX_SPECIES * LD_MAX_SPECIES];
    double knot[LD_MAX_NQ], gw[LD_MAX_NQ];
    DevTable* d_tab = nullptr;
    StepCtrl* d_ctrl = nullptr;
    int* d_cursor = nullptr;
    double* d_momout = nullptr;           // S x MOM_OUT
    void* h_pin = nullptr;                // pinned read-back area
    Cloud tmp, state;
    Buf blockcnt, blockoff, part, vpart, blockpart, vk, V, records, stage_v, stage_w, stage_s, stage_o;
    Buf facttab, prodtab, tilebox;
    Buf cellkey, cellrank, chunkcnt, binoff, spbox;   // Morton bucketing of pack (pack.cuh)
    int morton_on = 1;                                // landau_set_cutoff(.., morton)
    size_t attr_cellcount = 0;
    unsigned long long* d_cutstats = nullptr;   // pass 1 Gaussian cutoff: {source tiles considered, skipped}
    int cutoff_on = 1;                          // landau_set_cutoff
    double mixed_until = 0.0;                   // landau_set_mixed_precision: FP32 pass 2 while the residual exceeds it
    double stiff_dt = 0.0;                      // dt of the step being enqueued (stiff_begin_kernel)
    double stiff_theta = 0.0;                   // landau_set_stiff_pairs: pairs with stiffness above it are solved implicitly
    StiffCtrl* d_stiff = nullptr;
    Buf stiff_mark, stiff_scratch;
    bool attr_sym64_det = false, attr_sym64_2v_det = false;
    Buf sym_acc, sym_tpart, sym_ticket;   // symmetric pair kernel: in-place source sums, target segments, unit tickets
    // cudaFuncAttributeMaxDynamicSharedMemorySize is a per-device attribute: remembered per context (= per device)
    bool attr_sym64 = false, attr_sym32 = false, attr_mma[LD_MAX_NQ + 1] = {}, attr_mma2v[LD_MAX_NQ + 1] = {};
    bool attr_sym64_2v = false;
    size_t attr_cells[LD_MAX_NQ + 1] = {}, attr_cells_small[2] = {};
    int small_occ[2][2] = {};                    // resident CTAs per SM of step_small_kernel<R, DIM> (0 = not asked yet)
    bool coop_ok = false;                        // the device supports cooperative launches
    bool sym_refused = false;                    // the symmetric pair kernel's grid does not fit this device at once
    size_t prodtab_budget = (size_t)16 << 30;    // pass 1: largest product table the automatic choice allocates
    bool mma_declined = false;                   // the last pass 1 took the vector-pipe form because of that budget
    int dim = 3;                          // landau_set_dimension
    int substep = 0;                      // landau_set_substep: levels of step halving for unconverged steps
    int solver = 0, aa_depth = 3;         // landau_set_solver: 0 Jacobi (the paper's), 1 Anderson, 2 Newton-Krylov (NEXT-4)
    int nk_m = 20;                        // GMRES restart length of the Newton-Krylov solver
    AndersonCtrl* d_aa = nullptr;
    NewtonCtrl* d_nk = nullptr;
    DgCtrl* d_dg = nullptr;
    Buf aa_hist;
    Buf cells_off, cells_rec, soa32;
    // CUDA-graph form of a whole step for launch-bound (small) clouds, landau_set_step_graph
    int graph_mode = 1;                   // 0 off, 1 automatic (npad <= 65536 slots), 2 always
    unsigned long long alloc_gen = 0;
    cudaStream_t body_stream = nullptr, cap_stream = nullptr;
    struct StepGraph {
        cudaGraph_t graph = nullptr; cudaGraphExec_t exec = nullptr;
        unsigned long long gen = 0; int64_t N = 0; int npm = 0, max_iter = 0, fixed_nodes = 0, body_nodes = 0;
        double dt = 0.0, tol = 0.0, mixed = 0.0, stiff = 0.0; int ek = 0, pk = 0, solver = 0, depth = 0; bool failed = false;
    } sg;
    Buf dg_u, dg_Gu, dg_Gk, dg_part;      // discrete-gradient step (step_dg.cuh)
    int64_t launches = 0;
    // optional per-kernel timing (landau_profile_*): CUDA events around the two all-pairs kernels
    bool entropy_ran = false;             // a pass 1 ran since the last finish() (for landau_last_kernels)
    bool prof_on = false;
    bool in_run = false;
    struct ProfEv { cudaEvent_t e0, e1; int kind; int step; int iter; };
    std::vector<ProfEv> prof_events;
    std::vector<cudaEvent_t> prof_pool;
    int prof_step = 0, prof_iter = 0;
    double prof_ms[2] = {0.0, 0.0};
    int64_t prof_n[2] = {0, 0};
    char err[512];
    char kernels[128];
    const char* k_pair = "-";
    const char* k_entropy = "-";
    const char* k_step = "-";
};

namespace {

constexpr size_t PIN_BYTES = 1 << 16;
// pinned read-back area: [0, 8) finish()'s {err, used_fact}; [PIN_CTRL, +sizeof(StepCtrl)) the step control block;
// [PIN_MOM, ...) per-species moment sums
constexpr size_t PIN_CTRL = 128, PIN_MOM = 512;
static_assert(PIN_CTRL >= 2 * sizeof(int) && PIN_CTRL + 96 + 16 <= PIN_MOM && sizeof(StepCtrl) <= 64,
              "pinned read-back areas overlap");
static_assert(PIN_MOM + sizeof(double) * LD_MAX_SPECIES * 16 <= PIN_BYTES, "pinned read-back area too small");

int fail(landau_ctx* c, int code, const char* fmt, ...) {
    if (c) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(c->err, sizeof(c->err), fmt, ap);
        va_end(ap);
    }
    return code;
}

// NVTX range around a phase of the path (visible in Nsight timelines; a no-op without a profiler attached)
struct NvtxRange {
    explicit NvtxRange(const char* name) { nvtxRangePushA(name); }
    ~NvtxRange() { nvtxRangePop(); }
};

// Every entry point runs on the context's device and leaves the caller's current device as it found it.
struct DevGuard {
    int prev = -1;
    bool switched = false;
    explicit DevGuard(const landau_ctx* c) {
        if (!c) return;
        if (cudaGetDevice(&prev) == cudaSuccess && prev != c->device) switched = cudaSetDevice(c->device) == cudaSuccess;
    }
    ~DevGuard() { if (switched) cudaSetDevice(prev); }
    DevGuard(const DevGuard&) = delete;
    DevGuard& operator=(const DevGuard&) = delete;
};

#define CU(call)                                                                              \
    do {                                                                                      \
        cudaError_t e_ = (call);                                                              \
        if (e_ != cudaSuccess)                                                                \
            return fail(c, e_ == cudaErrorMemoryAllocation ? LANDAU_ENOMEM : LANDAU_ECUDA,    \
                        "%s: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__); \
    } while (0)

#define RC(call)             \
    do {                     \
        int rc_ = (call);    \
        if (rc_ < 0) return rc_; \
    } while (0)

int ensure(landau_ctx* c, Buf& b, size_t bytes) {
    if (bytes <= b.cap) return 0;
    if (b.p) CU(cudaFree(b.p));
    b.p = nullptr; b.cap = 0;
    ++c->alloc_gen;                       // invalidates a cached step graph (kernel arguments are baked in)
    size_t want = bytes + bytes / 8 + 256;
    CU(cudaMalloc(&b.p, want));
    b.cap = want;
    return 0;
}

void release(Buf& b) {
    if (b.p) cudaFree(b.p);
    b.p = nullptr; b.cap = 0;
}

cudaEvent_t prof_get_event(landau_ctx* c) {
    cudaEvent_t e = nullptr;
    if (!c->prof_pool.empty()) { e = c->prof_pool.back(); c->prof_pool.pop_back(); }
    else cudaEventCreate(&e);
    return e;
}

// kind 0 = pairwise kernel (pass 2), 1 = entropy node-sum kernel (pass 1)
struct ProfScope {
    landau_ctx* c; int kind; cudaEvent_t e0 = nullptr;
    ProfScope(landau_ctx* c_, int kind_) : c(c_), kind(kind_) {
        if (c->prof_on) { e0 = prof_get_event(c); cudaEventRecord(e0, c->stream); }
    }
    ~ProfScope() {
        if (!e0) return;
        cudaEvent_t e1 = prof_get_event(c);
        cudaEventRecord(e1, c->stream);
        c->prof_events.push_back({e0, e1, kind, c->prof_step, c->prof_iter});
    }
};

// Resolve recorded events after a synchronisation.  iters_per_step (may be NULL) gives, for step
// records of the call just finished, how many fixed-point iterations really ran: pair launches
// beyond that exited at once and are not counted.
void prof_resolve(landau_ctx* c, const int* iters_per_step, int n_steps) {
    for (auto& ev : c->prof_events) {
        float ms = 0.f;
        bool count = true;
        if (ev.kind == 0 && iters_per_step && ev.step < n_steps && ev.iter >= iters_per_step[ev.step]) count = false;
        if (count && cudaEventElapsedTime(&ms, ev.e0, ev.e1) == cudaSuccess) {
            c->prof_ms[ev.kind] += ms;
            c->prof_n[ev.kind] += 1;
        }
        c->prof_pool.push_back(ev.e0);
        c->prof_pool.push_back(ev.e1);
    }
    c->prof_events.clear();
}

// Gauss-Hermite rule for the weight exp(-k^2) by Golub-Welsch: knots are the eigenvalues of the
// symmetric tridiagonal Jacobi matrix J (zero diagonal, off-diagonal sqrt(i/2)), weights are
// sqrt(pi) times the squared first components of the normalised eigenvectors.  Eigen-decomposition
// by cyclic Jacobi rotations in long double (n <= 8).
void gauss_hermite_gw(int n, double* knots, double* weights) {
    long double A[LD_MAX_NQ][LD_MAX_NQ] = {}, V[LD_MAX_NQ][LD_MAX_NQ] = {};
    for (int i = 0; i < n; ++i) V[i][i] = 1.0L;
    for (int i = 1; i < n; ++i) A[i][i - 1] = A[i - 1][i] = sqrtl(0.5L * i);
    for (int sweep = 0; sweep < 100; ++sweep) {
        long double off = 0.0L;
        for (int i = 0; i < n; ++i)
            for (int j = i + 1; j < n; ++j) off += A[i][j] * A[i][j];
        if (off < 1e-40L) break;
        for (int p = 0; p < n; ++p)
            for (int q = p + 1; q < n; ++q) {
                if (fabsl(A[p][q]) < 1e-300L) continue;
                const long double theta = (A[q][q] - A[p][p]) / (2.0L * A[p][q]);
                const long double t = (theta >= 0 ? 1.0L : -1.0L) / (fabsl(theta) + sqrtl(theta * theta + 1.0L));
                const long double cs = 1.0L / sqrtl(t * t + 1.0L), sn = t * cs;
                for (int k = 0; k < n; ++k) {
                    const long double akp = A[k][p], akq = A[k][q];
                    A[k][p] = cs * akp - sn * akq;
                    A[k][q] = sn * akp + cs * akq;
                }
                for (int k = 0; k < n; ++k) {
                    const long double apk = A[p][k], aqk = A[q][k];
                    A[p][k] = cs * apk - sn * aqk;
                    A[q][k] = sn * apk + cs * aqk;
                }
                for (int k = 0; k < n; ++k) {
                    const long double vkp = V[k][p], vkq = V[k][q];
                    V[k][p] = cs * vkp - sn * vkq;
                    V[k][q] = sn * vkp + cs * vkq;
                }
            }
    }
    int idx[LD_MAX_NQ];
    for (int i = 0; i < n; ++i) idx[i] = i;
    std::sort(idx, idx + n, [&](int a, int b) { return A[a][a] < A[b][b]; });
    const long double sqrt_pi = 1.77245385090551602729816748334114518L;
    for (int i = 0; i < n; ++i) {
        knots[i] = (double)A[idx[i]][idx[i]];
        weights[i] = (double)(sqrt_pi * V[0][idx[i]] * V[0][idx[i]]);
    }
    // enforce the exact antisymmetry of the knot set (k_i = -k_{n-1-i}; middle knot 0 for odd n)
    for (int i = 0; i < n / 2; ++i) {
        const double k = 0.5 * (knots[n - 1 - i] - knots[i]);
        const double a = 0.5 * (weights[n - 1 - i] + weights[i]);
        knots[i] = -k; knots[n - 1 - i] = k;
        weights[i] = a; weights[n - 1 - i] = a;
    }
    if (n & 1) knots[n / 2] = 0.0;
}

// The symmetric pair kernel (pair_sym.cuh) in its large configuration: 8 warps, 4 targets per
// lane, 2 sources per lane and step: target tiles of 1024 slots, source units of 512.
#ifndef LANDAU_SYM_W      // tuning knobs: -DLANDAU_SYM_W=.. -DLANDAU_SYM_RT=.. -DLANDAU_SYM_RS=.. (build.py: LANDAU_NVCC_EXTRA)
#define LANDAU_SYM_W 8
#endif
#ifndef LANDAU_SYM_RT
#define LANDAU_SYM_RT 4
#endif
#ifndef LANDAU_SYM_RS
#define LANDAU_SYM_RS 2
#endif
constexpr int SYM_W = LANDAU_SYM_W, SYM_RT = LANDAU_SYM_RT, SYM_RS = LANDAU_SYM_RS;
using SymL = SymCfg<SYM_W, SYM_RT, SYM_RS>;
constexpr int64_t SYM_MIN_MARKERS = 16384;

int want_sym(const landau_ctx* c, int64_t N) {
    if (c->pair_kernel == 1) return 0;
    if (c->pair_kernel == 2) return 1;
    if (c->sym_refused) return 0;              // a cooperative launch of the symmetric kernel was refused (launch_pair_sym)
    return N >= SYM_MIN_MARKERS;
}

int choose_pad(const landau_ctx* c, int64_t N) { return want_sym(c, N) ? SymL::BT : 128; }

int npad_upper(int64_t N, int S, int pad) {
    const int64_t up = N + (int64_t)S * (pad - 1);
    return (int)(((up + pad - 1) / pad) * pad);
}


// ---- optimised kernels -----------------------------------------------------------------------
int pair_sym_available(landau_ctx* c, Cloud& cl) { (void)c; return cl.sym; }
// mixed-precision implicit step: Jacobi solver, 3-V, symmetric kernel (>= 16384 markers)
bool stiff_active(const landau_ctx* c) { return c->stiff_theta > 0.0 && c->solver != 2; }
bool mixed_step_active(const landau_ctx* c, const Cloud& cl) {
    return c->mixed_until > 0.0 && c->solver == 0 && c->dim == 3 && cl.sym && c->precision == 0 && !stiff_active(c);
}
// Buffers of the symmetric kernel's output path (pair_sym.cuh): O(N), whatever the grid.
int ensure_sym_buffers(landau_ctx* c, const Cloud& cl, int G) {
    const size_t npm = (size_t)cl.npad_max;
    RC(ensure(c, c->vpart, sizeof(double) * 3 * npm));
    RC(ensure(c, c->sym_acc, sizeof(double) * 3 * npm));
    RC(ensure(c, c->sym_tpart, sizeof(double) * 3 * SymL::BT * (npm / SymL::BT + (size_t)G)));
    RC(ensure(c, c->sym_ticket, sizeof(int) * (npm / SymL::BS + 1)));
    return 0;
}

template <typename F, int DIM = 3, bool DETECT = false>
int launch_pair_sym(landau_ctx* c, Cloud& cl, const StepCtrl* ctrl, const F* soa, bool& attr_done, int* nparts,
                    int gate = GATE_NONE) {
    using Cfg = SymCfg<SYM_W, SYM_RT, SYM_RS, F>;
    const int G = c->sm_count;                 // persistent grid, 1 CTA per SM: all CTAs co-resident (ticket waits)
    RC(ensure_sym_buffers(c, cl, G));
    auto kern = pair_sym_kernel<SYM_W, SYM_RT, SYM_RS, F, DIM, DETECT>;
    if (!attr_done) {
        CU(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::SMEM));
        attr_done = true;
    }
    const int npm = cl.npad_max;
    sym_reset_kernel<<<c->sm_count, 256, 0, c->stream>>>(ctrl, (double*)c->sym_acc.p, 3 * (size_t)npm,
                                                          (int*)c->sym_ticket.p, npm / SymL::BS + 1, gate);
    // The ticket waits of the output path need every CTA resident at once.  Outside stream capture the launch is
    // cooperative, so that a device which cannot hold the grid (an MPS SM limit, a green context) refuses it here
    // instead of spinning there; a captured step graph replays what a cooperative launch of this context already ran.
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    CU(cudaStreamIsCapturing(c->stream, &cap));
    if (c->coop_ok && cap == cudaStreamCaptureStatusNone) {
        const DevTable* a_T = c->d_tab; const DevLayout* a_L = cl.L(); const StepCtrl* a_ctrl = ctrl; int a_npm = npm;
        const F* a_soa = soa; double* a_acc = (double*)c->sym_acc.p; double* a_tpart = (double*)c->sym_tpart.p;
        int* a_ticket = (int*)c->sym_ticket.p; int* a_err = &cl.L()->err; int a_gate = gate;
        StiffCtrl* a_stiff = c->d_stiff; int* a_mark = (int*)c->stiff_mark.p;
        void* args[] = {&a_T, &a_L, &a_ctrl, &a_npm, &a_soa, &a_acc, &a_tpart, &a_ticket, &a_err, &a_gate, &a_stiff,
                        &a_mark};
        const cudaError_t ce = cudaLaunchCooperativeKernel((const void*)kern, dim3(G), dim3(Cfg::THREADS), args,
                                                           Cfg::SMEM, c->stream);
        if (ce == cudaErrorCooperativeLaunchTooLarge || ce == cudaErrorNotSupported) {
            cudaGetLastError();
            c->sym_refused = true;             // want_sym(): automatic selection takes the one-sided kernel from now on
            return fail(c, LANDAU_ECUDA,
                        "the symmetric pair kernel needs its %d thread blocks resident at once and this device cannot "
                        "hold them (%s); later calls of this context use the one-sided kernel (or set pair_kernel = 1)",
                        G, cudaGetErrorString(ce));
        }
        CU(ce);
    } else {
        kern<<<G, Cfg::THREADS, Cfg::SMEM, c->stream>>>(c->d_tab, cl.L(), ctrl, npm, soa, (double*)c->sym_acc.p,
                                                        (double*)c->sym_tpart.p, (int*)c->sym_ticket.p, &cl.L()->err,
                                                        gate, c->d_stiff, (int*)c->stiff_mark.p);
    }
    sym_combine_kernel<<<ceil_div(npm, 256), 256, 0, c->stream>>>(cl.L(), ctrl, npm, G, SymL::BT, SymL::BS,
                                                                   (const double*)c->sym_acc.p,
                                                                   (const double*)c->sym_tpart.p, (double*)c->vpart.p,
                                                                   gate);
    c->launches += 3;
    *nparts = 1;
    return 0;
}

// ---- a0: pack -----------------------------------------------------------------------------
int pack(landau_ctx* c, Cloud& cl, int64_t N, const double* v, const double* w, const int32_t* sid) {
    if (!c) return LANDAU_EINVAL;
    NvtxRange nvtx("landau:a0 pack");
    if (N < 1 || !v || !w || !sid) return fail(c, LANDAU_EINVAL, "pack: NULL array or N < 1");
    if (N > (int64_t)1 << 24) return fail(c, LANDAU_EINVAL, "pack: N = %lld exceeds 2^24 markers", (long long)N);
    const int S = c->S;
    const int pad = choose_pad(c, N);
    const int npm = npad_upper(N, S, pad);
    cl.N = N; cl.npad_max = npm; cl.pad = pad; cl.sym = want_sym(c, N); cl.G_valid = false;
    if (cl.sym) RC(ensure(c, cl.soa, sizeof(double) * 7 * (size_t)npm));
    RC(ensure(c, cl.lay, sizeof(DevLayout)));
    RC(ensure(c, cl.xyzw, sizeof(double) * 4 * (size_t)npm));
    RC(ensure(c, cl.perm, sizeof(int) * (size_t)npm));
    RC(ensure(c, cl.G, sizeof(double) * 4 * (size_t)npm));
    RC(ensure(c, cl.rec, sizeof(double) * 8 * (size_t)npm));
    const int nb = ceil_div((int)N, PACK_THREADS);
    RC(ensure(c, c->blockcnt, sizeof(int) * (size_t)nb * S));
    RC(ensure(c, c->blockoff, sizeof(int) * (size_t)nb * S));
    cudaStream_t st = c->stream;
    CU(cudaMemsetAsync(cl.lay.p, 0, sizeof(DevLayout), st));
    CU(cudaMemsetAsync(cl.xyzw.p, 0, sizeof(double) * 4 * (size_t)npm, st));
    CU(cudaMemsetAsync(cl.perm.p, 0xFF, sizeof(int) * (size_t)npm, st));
    pack_count_kernel<<<nb, PACK_THREADS, 0, st>>>((int)N, v, w, sid, S, (int*)c->blockcnt.p, cl.L());
    pack_scan_kernel<<<1, 32, 0, st>>>(nb, S, pad, (const int*)c->blockcnt.p, (int*)c->blockoff.p, cl.L());
    c->launches += 2;
    // clouds with many tiles: order every species along a Morton curve (compact tiles for pass 1's Gaussian cutoff)
    if (c->morton_on && N >= 4096 && N <= ((int64_t)1 << 21)) {
        // cell level: >= 32 markers per cell on average, the histogram fits the count kernel's shared memory, and the
        // per-chunk histograms (nchunks x nbins ints, the sort's only super-linear scratch) stay under 32 MiB -- at
        // N = 2^21, S = 1 that is 4096 cells and 16 MiB instead of 32768 cells and 128 MiB
        const int nchunks = ceil_div((int)N, CELL_CHUNK);
        int LC = 0;
        while (LC < 7 && (N / S) >> (3 * LC) > 32 && ((int64_t)S << (3 * (LC + 1))) <= CELL_MAX_BINS &&
               (size_t)nchunks * ((size_t)S << (3 * (LC + 1))) * sizeof(int) <= CELL_SCRATCH_MAX_BYTES)
            ++LC;
        const int nbins = S << (3 * LC);
        RC(ensure(c, c->cellkey, sizeof(int) * (size_t)N));
        RC(ensure(c, c->cellrank, sizeof(int) * (size_t)N));
        RC(ensure(c, c->chunkcnt, sizeof(int) * (size_t)nchunks * nbins));
        RC(ensure(c, c->binoff, sizeof(int) * (2 * (size_t)nbins + 2)));
        RC(ensure(c, c->spbox, sizeof(SpeciesBox)));
        const size_t smem = sizeof(int) * (size_t)nbins;
        if (smem > 48 * 1024 && smem > c->attr_cellcount) {
            CU(cudaFuncSetAttribute(pack_cell_count_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            c->attr_cellcount = smem;
        }
        int* binoff = (int*)c->binoff.p;
        int* bintot = binoff + nbins + 1;
        pack_box_init_kernel<<<1, 64, 0, st>>>((SpeciesBox*)c->spbox.p);
        pack_box_kernel<<<nb, PACK_THREADS, 0, st>>>((int)N, v, sid, S, (SpeciesBox*)c->spbox.p);
        pack_cell_count_kernel<<<nchunks, PACK_THREADS, smem, st>>>((int)N, v, sid, S, LC, nbins,
                                                                    (const SpeciesBox*)c->spbox.p, (int*)c->cellkey.p,
                                                                    (int*)c->cellrank.p, (int*)c->chunkcnt.p);
        pack_cell_scan_chunks_kernel<<<ceil_div(nbins, 256), 256, 0, st>>>(nchunks, nbins, (int*)c->chunkcnt.p, bintot);
        pack_cell_scan_bins_kernel<<<1, 1024, 0, st>>>(nbins, bintot, binoff);
        pack_cell_scatter_kernel<<<nb, PACK_THREADS, 0, st>>>((int)N, v, w, S, LC, nbins, (const int*)c->cellkey.p,
                                                              (const int*)c->cellrank.p, (const int*)c->chunkcnt.p,
                                                              binoff, cl.L(), cl.x(), cl.y(), cl.z(), cl.w(), cl.prm());
        c->launches += 6;
    } else {
        pack_scatter_kernel<<<nb, PACK_THREADS, 0, st>>>((int)N, v, w, sid, S, (const int*)c->blockoff.p, cl.L(),
                                                          cl.x(), cl.y(), cl.z(), cl.w(), cl.prm());
        c->launches += 1;
    }
    CU(cudaGetLastError());
    return 0;
}

// ---- a1/a2: entropy gradient of a packed cloud ---------------------------------------------
template <int NQ, int NI>
void launch_entropy_literal(landau_ctx* c, Cloud& cl, int nchunks, int skip_if_fact, const StepCtrl* stop) {
    dim3 grid(cl.npad_max / ENT_THREADS, nchunks, NQ / NI);
    entropy_literal_kernel<NQ, NI><<<grid, ENT_THREADS, 0, c->stream>>>(
        c->d_tab, cl.L(), cl.npad_max, nchunks, skip_if_fact, cl.x(), cl.y(), cl.z(), cl.w(),
        (const TileBox*)c->tilebox.p, c->d_cutstats, (double*)c->part.p, stop);
}

template <int NQ, int NI>
int launch_entropy_fact(landau_ctx* c, Cloud& cl, int nchunks, const StepCtrl* stop) {
    RC(ensure(c, c->facttab, sizeof(double) * FactCfg<NQ>::REC * (size_t)cl.npad_max));
    entropy_fact_prep_kernel<NQ><<<ceil_div(cl.npad_max, 128), 128, 0, c->stream>>>(
        c->d_tab, cl.L(), cl.npad_max, cl.x(), cl.y(), cl.z(), cl.w(), (double*)c->facttab.p, stop);
    dim3 grid(cl.npad_max / FACT_THREADS, nchunks, NQ / NI);
    entropy_fact_kernel<NQ, NI><<<grid, FACT_THREADS, 0, c->stream>>>(c->d_tab, cl.L(), cl.npad_max, nchunks,
                                                                      (const double*)c->facttab.p, (double*)c->part.p, stop);
    return 0;
}

template <int NQ, int NZ>
int launch_entropy_mma_nz(landau_ctx* c, Cloud& cl, int nchunks, const StepCtrl* stop) {
    using M = MmaCfg<NQ, NZ>;
    RC(ensure(c, c->facttab, sizeof(double) * M::REC * (size_t)cl.npad_max));
    RC(ensure(c, c->prodtab, M::table_bytes((size_t)cl.npad_max)));
    entropy_fact_prep_kernel<NQ><<<ceil_div(cl.npad_max, 128), 128, 0, c->stream>>>(
        c->d_tab, cl.L(), cl.npad_max, cl.x(), cl.y(), cl.z(), cl.w(), (double*)c->facttab.p, stop);
    // the product table every block of the contraction streams (built once per pass, entropy_mma.cuh)
    dim3 pgrid((unsigned)(((size_t)cl.npad_max * M::ROW + 255) / 256), M::GROUPS);
    entropy_prod_kernel<NQ, NZ><<<pgrid, 256, 0, c->stream>>>(c->d_tab, cl.L(), cl.npad_max, (const double*)c->facttab.p,
                                                             (double*)c->prodtab.p, stop);
    c->launches += 1;
    auto kern = entropy_mma_kernel<NQ, NZ>;
    bool& attr = NZ == 1 ? c->attr_mma2v[NQ] : c->attr_mma[NQ];
    if (!attr) {
        CU(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)M::SMEM));
        attr = true;
    }
    dim3 grid(cl.npad_max / MMA_THREADS, nchunks, M::GROUPS);
    kern<<<grid, MMA_THREADS, M::SMEM, c->stream>>>(c->d_tab, cl.L(), cl.npad_max, nchunks,
                                                    (const double*)c->prodtab.p, (const TileBox*)c->tilebox.p,
                                                    c->d_cutstats, (double*)c->part.p, stop);
    return 0;
}

// 2-V mode (landau_set_dimension(2)): the native planar node grid, n_q^2 nodes instead of n_q^3
template <int NQ>
int launch_entropy_mma(landau_ctx* c, Cloud& cl, int nchunks, const StepCtrl* stop) {
    return c->dim == 2 ? launch_entropy_mma_nz<NQ, 1>(c, cl, nchunks, stop) : launch_entropy_mma_nz<NQ, NQ>(c, cl, nchunks, stop);
}

// node groups (gridDim.z) each kernel splits the n_q^3 node sums into
int literal_groups(int nq) { return nq <= 4 ? 1 : nq; }
int fact_groups(int nq) { return nq <= 4 ? 1 : (nq == 6 ? 3 : nq); }
int mma_groups(int nq) {
    switch (nq) { case 5: return MmaCfg<5>::GROUPS; case 6: return MmaCfg<6>::GROUPS; case 7: return MmaCfg<7>::GROUPS;
                  case 8: return MmaCfg<8>::GROUPS; default: return 1; }
}

size_t mma_table_bytes(int nq, int dim, size_t npad_max) {
#define LD_TB(Q) (dim == 2 ? MmaCfg<Q, 1>::table_bytes(npad_max) : MmaCfg<Q, Q>::table_bytes(npad_max))
    switch (nq) {
        case 2: return LD_TB(2); case 3: return LD_TB(3); case 4: return LD_TB(4); case 5: return LD_TB(5);
        case 6: return LD_TB(6); case 7: return LD_TB(7); case 8: return LD_TB(8); default: return 0;
    }
#undef LD_TB
}

// stop != nullptr: every kernel of the pass exits at once when stop->done is set (device-driven loops)
int entropy(landau_ctx* c, Cloud& cl, const StepCtrl* stop = nullptr) {
    NvtxRange nvtx("landau:a1-a2 pass 1 (entropy gradient)");
    const int nq = c->n_q;
    const size_t M = (size_t)nq * nq * nq;
    const int ttiles = cl.npad_max / ENT_THREADS;
    // 0 automatic (DMMA contraction when the cloud is narrow enough, decided on the device, else literal),
    // 1 literal, 2 factorised on the vector pipe, 3 factorised as a DMMA contraction
    const int mode = c->entropy_kernel;
    bool use_mma = mode == 0 || mode == 3;
    // The DMMA form streams a per-pass product table of ROW x GROUPS doubles per marker (544 B at n_q = 4, 4352 B at
    // n_q = 8: 9 GB / 73 GB at 2^24 markers).  Beyond the context's budget the automatic choice takes the factorised
    // vector-pipe kernel (same arithmetic, 216 B per marker at most) instead of failing with LANDAU_ENOMEM.
    c->mma_declined = false;
    if (use_mma) {
        const size_t tb = mma_table_bytes(nq, c->dim, (size_t)cl.npad_max);
        if (tb > c->prodtab_budget) {
            if (mode == 3)
                return fail(c, LANDAU_ENOMEM, "entropy_kernel = 3: the product table of the DMMA form needs %.1f MB for %d "
                            "slots at n_q = %d, over the budget of %.1f MB (LANDAU_PRODTAB_BUDGET_MB / a quarter of "
                            "the device memory); use entropy_kernel = 0 or 2", tb / 1048576.0, cl.npad_max, nq,
                            c->prodtab_budget / 1048576.0);
            use_mma = false;
            c->mma_declined = true;
        }
    }
    const int ig = mode == 1 ? literal_groups(nq)
                             : std::min(literal_groups(nq), use_mma ? mma_groups(nq) : fact_groups(nq));
    // enough blocks for >= ~20 waves of 2 resident blocks per SM, so that the last wave costs < 5 %
    int nchunks = ceil_div(40 * c->sm_count, ttiles * ig);
#ifndef LANDAU_PASS1_MIN_TILES   // tuning knob (build.py: LANDAU_NVCC_EXTRA): source tiles of 64 per chunk, at least
#define LANDAU_PASS1_MIN_TILES 4
#endif
    // (launch-bound clouds of <= 4096 slots: half of that -- more, smaller blocks; measured on the paper's 2048-marker tests)
    const int min_tiles = cl.npad_max <= 4096 ? std::max(1, LANDAU_PASS1_MIN_TILES / 2) : LANDAU_PASS1_MIN_TILES;
    const int chunk_cap = std::max(1, cl.npad_max / (c->S * 64 * min_tiles));
    nchunks = std::max(1, std::min(nchunks, chunk_cap));
    nchunks = std::min(nchunks, 64);
    while (nchunks > 1 && (size_t)nchunks * M * cl.npad_max * sizeof(double) > ((size_t)2 << 30)) --nchunks;
    if (use_mma && nchunks >= 3) {
        // wave quantisation: 2 blocks are resident per SM, and a last wave that fills a few SMs costs a whole block
        // time (3 x 2^16 markers: 4 chunks = 21.08 waves, the 22nd wave 4 % of the kernel).  Take the chunk count
        // near the first guess whose block count is closest below a whole number of waves.
        const int hi = std::min({64, 2 * nchunks, chunk_cap});
        double best = 1e30;
        int pick = nchunks;
        for (int k = std::max(2, nchunks - 1); k <= hi; ++k) {
            if ((size_t)k * M * cl.npad_max * sizeof(double) > ((size_t)2 << 30)) break;
            const double waves = (double)ttiles * mma_groups(nq) * k / (2.0 * c->sm_count);
            const double cost = std::ceil(waves) / waves + 0.002 * k;      // larger k: more partial sums to store
            if (cost < best) { best = cost; pick = k; }
        }
        nchunks = pick;
    }
    RC(ensure(c, c->part, (size_t)nchunks * M * cl.npad_max * sizeof(double)));
    RC(ensure(c, c->tilebox, sizeof(TileBox) * ((size_t)cl.npad_max / ENT_SRC_TILE + 2)));
    {
    ProfScope prof(c, 1);
    // species extents (range guard of the factorised forms) and weights (Gaussian cutoff threshold); tile boxes
    entropy_bounds_kernel<<<c->S, 1024, 0, c->stream>>>(c->d_tab, cl.L(), cl.x(), cl.y(), cl.z(), cl.w(), c->cutoff_on, stop,
                                                         c->d_cutstats);
    entropy_tilebox_kernel<<<cl.npad_max / ENT_SRC_TILE, 64, 0, c->stream>>>(c->d_tab, cl.L(), cl.npad_max, cl.x(), cl.y(),
                                                                             cl.z(), cl.w(), (TileBox*)c->tilebox.p, stop);
    c->launches += 2;
    if (mode != 1) {
        if (use_mma) switch (nq) {
            case 2: RC((launch_entropy_mma<2>(c, cl, nchunks, stop))); break;
            case 3: RC((launch_entropy_mma<3>(c, cl, nchunks, stop))); break;
            case 4: RC((launch_entropy_mma<4>(c, cl, nchunks, stop))); break;
            case 5: RC((launch_entropy_mma<5>(c, cl, nchunks, stop))); break;
            case 6: RC((launch_entropy_mma<6>(c, cl, nchunks, stop))); break;
            case 7: RC((launch_entropy_mma<7>(c, cl, nchunks, stop))); break;
            case 8: RC((launch_entropy_mma<8>(c, cl, nchunks, stop))); break;
            default: return fail(c, LANDAU_EINVAL, "n_q = %d unsupported", nq);
        }
        else switch (nq) {
            case 2: RC((launch_entropy_fact<2, 2>(c, cl, nchunks, stop))); break;
            case 3: RC((launch_entropy_fact<3, 3>(c, cl, nchunks, stop))); break;
            case 4: RC((launch_entropy_fact<4, 4>(c, cl, nchunks, stop))); break;
            case 5: RC((launch_entropy_fact<5, 1>(c, cl, nchunks, stop))); break;
            case 6: RC((launch_entropy_fact<6, 2>(c, cl, nchunks, stop))); break;
            case 7: RC((launch_entropy_fact<7, 1>(c, cl, nchunks, stop))); break;
            case 8: RC((launch_entropy_fact<8, 1>(c, cl, nchunks, stop))); break;
            default: return fail(c, LANDAU_EINVAL, "n_q = %d unsupported", nq);
        }
        c->launches += 2;
    }
    if (mode != 2 && mode != 3) {
        const int skip = mode == 0 ? 1 : 0;
        switch (nq) {
            case 2: launch_entropy_literal<2, 2>(c, cl, nchunks, skip, stop); break;
            case 3: launch_entropy_literal<3, 3>(c, cl, nchunks, skip, stop); break;
            case 4: launch_entropy_literal<4, 4>(c, cl, nchunks, skip, stop); break;
            case 5: launch_entropy_literal<5, 1>(c, cl, nchunks, skip, stop); break;
            case 6: launch_entropy_literal<6, 1>(c, cl, nchunks, skip, stop); break;
            case 7: launch_entropy_literal<7, 1>(c, cl, nchunks, skip, stop); break;
            case 8: launch_entropy_literal<8, 1>(c, cl, nchunks, skip, stop); break;
            default: return fail(c, LANDAU_EINVAL, "n_q = %d unsupported", nq);
        }
        c->launches += 1;
    }
    }
    entropy_finalize_kernel<<<ceil_div(cl.npad_max, FIN_MARKERS), FIN_THREADS, 0, c->stream>>>(
        c->d_tab, cl.L(), cl.npad_max, nchunks, cl.prm(), (const double*)c->part.p, cl.x(), cl.y(), cl.z(),
        mode == 1 ? 0 : (mode >= 2 ? 2 : 1), (c->dim == 2 && use_mma) ? 1 : 0, cl.Gx(), cl.Gy(), cl.Gz(), cl.snode(), stop);
    c->launches += 1;
    CU(cudaGetLastError());
    cl.G_valid = true;
    c->entropy_ran = true;
    return 0;
}

#ifndef LANDAU_ONESIDED_WAVES  // tuning knob (build.py: LANDAU_NVCC_EXTRA): blocks per SM the source chunking aims at
#define LANDAU_ONESIDED_WAVES 8
#endif
// Grid of the one-sided pair kernel for a cloud: targets per thread, target tiles, source chunks.
void onesided_grid(const landau_ctx* c, const Cloud& cl, int* R, int* ttiles, int* nchunks) {
    // targets per thread: 2, or 1 for the smallest clouds (more blocks matter more than source reuse there)
#ifndef LANDAU_ONESIDED_R1_MAX   // tuning knob (build.py: LANDAU_NVCC_EXTRA)
#define LANDAU_ONESIDED_R1_MAX 4096
#endif
    *R = cl.npad_max <= LANDAU_ONESIDED_R1_MAX ? 1 : 2;
    *ttiles = ceil_div(cl.npad_max, PAIR_THREADS * *R);
    const int stiles = cl.npad_max / PAIR_SRC_TILE;
    *nchunks = std::min(32, std::max(1, std::min(stiles, ceil_div(LANDAU_ONESIDED_WAVES * c->sm_count, *ttiles))));
}

// ---- a3: pairwise field of source records -> partial fields ---------------------------------
// Returns the number of partial slices written to c->vpart (to be summed in index order).
// detect: 0 = plain evaluation; 1 = this is the first evaluation of a step with the stiff-pair treatment on (find
// the pairs); 2 = enqueue both flavours, gated on the device by the iteration count (CUDA-graph body)
int pair(landau_ctx* c, Cloud& cl, const StepCtrl* ctrl, int* nparts_out, int detect = 0) {
    NvtxRange nvtx("landau:a3 pass 2 (pairwise Landau sum)");
    int use_sym = 0;
    if (c->pair_kernel == 2 || c->pair_kernel == 0) use_sym = pair_sym_available(c, cl);
    ProfScope prof(c, 0);
    c->k_pair = use_sym ? "sym" : "onesided";
    snprintf(c->kernels, sizeof(c->kernels), "pair=%s entropy=%s", c->k_pair, c->k_entropy);
    const bool fp32_field = c->precision == 1 && !ctrl;     // FP32 variant: field evaluation only
    if (use_sym && !fp32_field && ctrl && mixed_step_active(c, cl)) {
        // mixed-precision step (landau_set_mixed_precision): both flavours are enqueued, the device flag
        // StepCtrl::use_f32 (set by step_update_kernel from the last residual) decides which one runs
        const size_t n7 = 7 * (size_t)cl.npad_max;
        RC(ensure(c, c->soa32, sizeof(float) * n7));
        soa_to_f32_kernel<<<c->sm_count * 4, 256, 0, c->stream>>>(n7, cl.soas(), (float*)c->soa32.p, ctrl);
        c->launches += 1;
        c->k_pair = "sym_mixed";
        snprintf(c->kernels, sizeof(c->kernels), "pair=%s entropy=%s", c->k_pair, c->k_entropy);
        RC(launch_pair_sym<float>(c, cl, ctrl, (const float*)c->soa32.p, c->attr_sym32, nparts_out, GATE_F32));
        RC(launch_pair_sym<double>(c, cl, ctrl, cl.soas(), c->attr_sym64, nparts_out, GATE_F64));
        return 0;
    }
    if (use_sym && !fp32_field) {
        const int g_det = detect == 2 ? GATE_FIRST : GATE_NONE, g_plain = detect == 2 ? GATE_LATER : GATE_NONE;
        if (c->dim == 2) {                     // native 2-V arithmetic (landau_set_dimension(2))
            c->k_pair = "sym2v";
            snprintf(c->kernels, sizeof(c->kernels), "pair=%s entropy=%s", c->k_pair, c->k_entropy);
            if (detect) RC((launch_pair_sym<double, 2, true>(c, cl, ctrl, cl.soas(), c->attr_sym64_2v_det, nparts_out, g_det)));
            if (detect != 1) RC((launch_pair_sym<double, 2>(c, cl, ctrl, cl.soas(), c->attr_sym64_2v, nparts_out, g_plain)));
        } else {
            if (detect) RC((launch_pair_sym<double, 3, true>(c, cl, ctrl, cl.soas(), c->attr_sym64_det, nparts_out, g_det)));
            if (detect != 1) RC(launch_pair_sym<double>(c, cl, ctrl, cl.soas(), c->attr_sym64, nparts_out, g_plain));
        }
        return 0;
    }
    if (c->precision == 1 && !ctrl && cl.sym) {             // FP32 field variant, symmetric kernel in FP32
        const size_t n7 = 7 * (size_t)cl.npad_max;
        RC(ensure(c, c->soa32, sizeof(float) * n7));
        soa_to_f32_kernel<<<c->sm_count * 4, 256, 0, c->stream>>>(n7, cl.soas(), (float*)c->soa32.p);
        c->launches += 1;
        RC(launch_pair_sym<float>(c, cl, nullptr, (const float*)c->soa32.p, c->attr_sym32, nparts_out));
        c->k_pair = "sym_f32";
        snprintf(c->kernels, sizeof(c->kernels), "pair=%s entropy=%s", c->k_pair, c->k_entropy);
        return 0;
    }
    if (c->precision == 1 && !ctrl) {                       // FP32 field variant below the symmetric kernel's size
        constexpr int RF = 4;
        const int ttiles = ceil_div(cl.npad_max, PAIR_THREADS * RF);
        const int stiles = cl.npad_max / PAIR_SRC_TILE;
        int nchunks = std::max(1, std::min(stiles, ceil_div(8 * c->sm_count, ttiles)));
        nchunks = std::min(nchunks, 32);
        RC(ensure(c, c->vpart, sizeof(double) * 3 * (size_t)nchunks * cl.npad_max));
        dim3 grid(ttiles, nchunks);
        pair_onesided_f32_kernel<RF><<<grid, PAIR_THREADS, 0, c->stream>>>(c->d_tab, cl.L(), cl.npad_max, nchunks,
                                                                        cl.recs(), (double*)c->vpart.p);
        c->k_pair = "onesided_f32";
        snprintf(c->kernels, sizeof(c->kernels), "pair=%s entropy=%s", c->k_pair, c->k_entropy);
        c->launches += 1;
        *nparts_out = nchunks;
        return 0;
    }
    int R, ttiles, nchunks;
    onesided_grid(c, cl, &R, &ttiles, &nchunks);
    RC(ensure(c, c->vpart, sizeof(double) * 3 * (size_t)nchunks * cl.npad_max));
    dim3 grid(ttiles, nchunks);
    if (detect) {
        // stiff-pair steps (landau_set_stiff_pairs): the first evaluation of a step also finds the stiff pairs
        const int g_det = detect == 2 ? GATE_FIRST : GATE_NONE;
        StiffCtrl* sc = c->d_stiff;
        int* mk = (int*)c->stiff_mark.p;
        double* vp = (double*)c->vpart.p;
#define LD_ONESIDED(RR, DD, DET, GATE) pair_onesided_kernel<RR, DD, DET><<<grid, PAIR_THREADS, 0, c->stream>>>( \
            c->d_tab, cl.L(), ctrl, cl.npad_max, nchunks, cl.recs(), vp, GATE, sc, mk)
        if (c->dim == 2) { if (R == 1) LD_ONESIDED(1, 2, true, g_det); else LD_ONESIDED(2, 2, true, g_det); }
        else             { if (R == 1) LD_ONESIDED(1, 3, true, g_det); else LD_ONESIDED(2, 3, true, g_det); }
        c->launches += 1;
        if (detect == 2) {
            if (c->dim == 2) { if (R == 1) LD_ONESIDED(1, 2, false, GATE_LATER); else LD_ONESIDED(2, 2, false, GATE_LATER); }
            else             { if (R == 1) LD_ONESIDED(1, 3, false, GATE_LATER); else LD_ONESIDED(2, 3, false, GATE_LATER); }
            c->launches += 1;
        }
#undef LD_ONESIDED
        c->k_pair = c->dim == 2 ? "onesided2v" : "onesided";
        snprintf(c->kernels, sizeof(c->kernels), "pair=%s entropy=%s", c->k_pair, c->k_entropy);
        *nparts_out = nchunks;
        return 0;
    }
    if (c->dim == 2) {                         // native 2-V arithmetic (landau_set_dimension(2))
        c->k_pair = "onesided2v";
        snprintf(c->kernels, sizeof(c->kernels), "pair=%s entropy=%s", c->k_pair, c->k_entropy);
        if (R == 1)
            pair_onesided_kernel<1, 2><<<grid, PAIR_THREADS, 0, c->stream>>>(c->d_tab, cl.L(), ctrl, cl.npad_max, nchunks,
                                                                            cl.recs(), (double*)c->vpart.p);
        else
            pair_onesided_kernel<2, 2><<<grid, PAIR_THREADS, 0, c->stream>>>(c->d_tab, cl.L(), ctrl, cl.npad_max, nchunks,
                                                                            cl.recs(), (double*)c->vpart.p);
    } else if (R == 1)
        pair_onesided_kernel<1><<<grid, PAIR_THREADS, 0, c->stream>>>(c->d_tab, cl.L(), ctrl, cl.npad_max, nchunks,
                                                                     cl.recs(), (double*)c->vpart.p);
    else
        pair_onesided_kernel<2><<<grid, PAIR_THREADS, 0, c->stream>>>(c->d_tab, cl.L(), ctrl, cl.npad_max, nchunks,
                                                                     cl.recs(), (double*)c->vpart.p);
    c->launches += 1;
    *nparts_out = nchunks;
    return 0;
}

// Read the layout's error flag and which pass-1 kernel ran (one synchronisation).
int finish(landau_ctx* c, Cloud& cl, const char* where) {
    int* h = (int*)c->h_pin;
    CU(cudaMemcpyAsync(h, &cl.L()->err, 2 * sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    CU(cudaGetLastError());
    if (c->prof_on && !c->in_run) prof_resolve(c, nullptr, 0);
    if (c->entropy_ran)
        c->k_entropy = h[1] ? (((c->entropy_kernel == 0 && !c->mma_declined) || c->entropy_kernel == 3) ? "mma" : "fact")
                            : "literal";
    c->entropy_ran = false;
    snprintf(c->kernels, sizeof(c->kernels), "pair=%s entropy=%s", c->k_pair, c->k_entropy);
    if (*h) cl.G_valid = false;
    if (*h == LANDAU_EINVAL) return fail(c, LANDAU_EINVAL, "%s: species_id out of range or weight <= 0", where);
    if (*h == LANDAU_ENONFINITE) return fail(c, LANDAU_ENONFINITE, "%s: non-finite input or result", where);
    if (*h == LANDAU_ERANGE)
        return fail(c, LANDAU_ERANGE, "%s: marker cloud too wide for the factorised entropy kernel (entropy_kernel = 2 or 3)", where);
    if (*h == LANDAU_ECUDA)
        return fail(c, LANDAU_ECUDA, "%s: a device-side wait timed out (thread blocks of a kernel that orders its "
                    "output by tickets or grid barriers were not all resident); the output was not completed", where);
    if (*h) return fail(c, *h, "%s: device-side error %d", where, *h);
    return 0;
}

int field_of_cloud(landau_ctx* c, Cloud& cl, double* out) {
    int nparts = 0;
    c->prof_step = 0; c->prof_iter = 0;
    if (cl.sym)
        build_soa_kernel<<<ceil_div(cl.npad_max, 256), 256, 0, c->stream>>>(c->d_tab, cl.L(), cl.npad_max, cl.x(), cl.y(),
                                                                            cl.z(), cl.w(), cl.Gx(), cl.Gy(), cl.Gz(),
                                                                            cl.soas());
    else
        build_rec_kernel<<<ceil_div(cl.npad_max, 256), 256, 0, c->stream>>>(c->d_tab, cl.L(), cl.npad_max, cl.x(), cl.y(),
                                                                            cl.z(), cl.w(), cl.Gx(), cl.Gy(), cl.Gz(),
                                                                            cl.recs());
    RC(pair(c, cl, nullptr, &nparts));
    RC(ensure(c, c->V, sizeof(double) * 3 * (size_t)cl.npad_max));
    double* Vx = (double*)c->V.p;
    double* Vy = Vx + cl.npad_max;
    double* Vz = Vy + cl.npad_max;
    combine_field_kernel<<<ceil_div(cl.npad_max, 256), 256, 0, c->stream>>>(cl.L(), cl.npad_max, nparts,
                                                                            (const double*)c->vpart.p, Vx, Vy, Vz);
    scatter3_kernel<<<ceil_div(cl.npad_max, 256), 256, 0, c->stream>>>(cl.npad_max, cl.L(), cl.prm(), Vx, Vy, Vz, out);
    c->launches += 3;
    CU(cudaGetLastError());
    return 0;
}

int species_sums(landau_ctx* c, Cloud& cl, bool with_entropy, bool with_m4, double* h_out /* S x MOM_OUT */) {
    NvtxRange nvtx("landau:a6 moments");
    const int nb = cl.npad_max / MOM_THREADS;
    RC(ensure(c, c->blockpart, sizeof(double) * (size_t)std::max(nb * MOM_NQ, 4096)));
    CU(cudaMemsetAsync(c->d_momout, 0, sizeof(double) * LD_MAX_SPECIES * MOM_OUT, c->stream));
    moments_block_kernel<<<nb, MOM_THREADS, 0, c->stream>>>(cl.L(), cl.npad_max, cl.x(), cl.y(), cl.z(), cl.w(),
                                                            with_entropy ? cl.snode() : nullptr,
                                                            (double*)c->blockpart.p);
    moments_species_kernel<<<c->S, MOM_THREADS, 0, c->stream>>>(cl.L(), (const double*)c->blockpart.p, MOM_NQ, 0,
                                                               c->d_momout);
    c->launches += 2;
    if (with_m4) {
        moments_m4_block_kernel<<<nb, MOM_THREADS, 0, c->stream>>>(c->d_tab, cl.L(), cl.npad_max, cl.x(), cl.y(),
                                                                   cl.z(), cl.w(), c->d_momout,
                                                                   (double*)c->blockpart.p);
        moments_species_kernel<<<c->S, MOM_THREADS, 0, c->stream>>>(cl.L(), (const double*)c->blockpart.p, 3, 12,
                                                                   c->d_momout);
        c->launches += 2;
    }
    CU(cudaMemcpyAsync(h_out, c->d_momout, sizeof(double) * c->S * MOM_OUT, cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    CU(cudaGetLastError());
    return 0;
}

int stage_in(landau_ctx* c, int64_t N, const double* v, const double* w, const int32_t* sid, const double** dv,
             const double** dw, const int32_t** ds) {
    if (N < 1 || !v || !w || !sid) return fail(c, LANDAU_EINVAL, "NULL array or N < 1");
    RC(ensure(c, c->stage_v, sizeof(double) * 3 * (size_t)N));
    RC(ensure(c, c->stage_w, sizeof(double) * (size_t)N));
    RC(ensure(c, c->stage_s, sizeof(int32_t) * (size_t)N));
    CU(cudaMemcpyAsync(c->stage_v.p, v, sizeof(double) * 3 * (size_t)N, cudaMemcpyHostToDevice, c->stream));
    CU(cudaMemcpyAsync(c->stage_w.p, w, sizeof(double) * (size_t)N, cudaMemcpyHostToDevice, c->stream));
    CU(cudaMemcpyAsync(c->stage_s.p, sid, sizeof(int32_t) * (size_t)N, cudaMemcpyHostToDevice, c->stream));
    *dv = (const double*)c->stage_v.p; *dw = (const double*)c->stage_w.p; *ds = (const int32_t*)c->stage_s.p;
    return 0;
}

__global__ void fp64_peak_kernel(double* out, int iters, double a, double b) {
    double x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
#pragma unroll 1
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int k = 0; k < 16; ++k) {
            x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
            x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
        }
    }
    const double s = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
    if (s == 123.456) out[0] = s;
}

// FP64 tensor-pipe peak: dependent-free DMMA.8x8x4 streams (8 accumulator pairs per thread), 2*8*8*4 flop per warp MMA.
__global__ void fp64_dmma_peak_kernel(double* out, int iters, double a, double b) {
    double c0[8], c1[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) { c0[k] = threadIdx.x + k; c1[k] = threadIdx.x - k; }
#pragma unroll 1
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
            for (int k = 0; k < 8; ++k) dmma884(c0[k], c1[k], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < 8; ++k) s += c0[k] + c1[k];
    if (s == 123.456) out[0] = s;
}
}  // namespace


namespace {
// ---- a4: the kernels of one implicit step, shared by the plain launch sequence and the CUDA-graph capture ------
struct StepBufs {
    int npm, nub;
    double *xk, *yk, *zk;          // current iterate x (Jacobi: v^(k))
    double* hist;                  // solver history (Anderson: dF, dG, fprev, gcur; Newton-Krylov: Q, gcur)
    double* commit;                // [3][npm] state committed at the end of the step
};

StepBufs step_bufs(landau_ctx* c, const Cloud& cl) {
    StepBufs b;
    b.npm = cl.npad_max; b.nub = ceil_div(b.npm, UPD_THREADS);
    b.xk = (double*)c->vk.p; b.yk = b.xk + b.npm; b.zk = b.yk + b.npm;
    b.hist = (double*)c->aa_hist.p;
    b.commit = b.xk;
    if (c->solver == 1) b.commit = b.hist + (2 * (size_t)c->aa_depth + 1) * 3 * (size_t)b.npm;
    if (c->solver == 2) b.commit = b.hist + ((size_t)c->nk_m + 1) * 3 * (size_t)b.npm;
    return b;
}

size_t step_hist_doubles(const landau_ctx* c, int npm) {
    if (c->solver == 1) return (2 * (size_t)c->aa_depth + 2) * 3 * (size_t)npm;
    if (c->solver == 2) return ((size_t)c->nk_m + 4) * 3 * (size_t)npm;
    return 0;
}

int step_blockpart_doubles(const landau_ctx* c, int nub) {
    return std::max(std::max(AA_NRED, NK_NRED) * nub, 4096);
}

int enqueue_step_begin(landau_ctx* c, Cloud& cl, const StepBufs& b, int max_iter) {
    cudaStream_t st = c->stream;
    step_begin_kernel<<<ceil_div(b.npm, 256), 256, 0, st>>>(c->d_tab, cl.L(), c->d_ctrl, b.npm, cl.x(), cl.y(), cl.z(),
                                                             cl.w(), cl.Gx(), cl.Gy(), cl.Gz(), b.xk, b.yk, b.zk,
                                                             cl.sym ? nullptr : cl.recs(), cl.sym ? cl.soas() : nullptr,
                                                             mixed_step_active(c, cl) && max_iter > 1 ? 1 : 0);
    c->launches += 1;
    if (c->solver == 1) {
        anderson_begin_kernel<<<1, 32, 0, st>>>(c->d_aa, c->aa_depth);
        c->launches += 1;
    }
    if (c->solver == 2) {
        nk_begin_kernel<<<1, 32, 0, st>>>(c->d_nk, c->nk_m);
        c->launches += 1;
    }
    if (stiff_active(c)) {
        double* scr = (double*)c->stiff_scratch.p;
        stiff_begin_kernel<<<c->S, 256, 0, st>>>(c->d_tab, cl.L(), c->d_stiff, (int*)c->stiff_mark.p, b.npm, c->stiff_dt,
                                                 c->stiff_theta, cl.w(), cl.Gx(), cl.Gy(), cl.Gz(), scr,
                                                 (unsigned int*)(scr + 2 * LD_MAX_SPECIES));
        c->launches += 1;
    }
    return 0;
}

// One iteration = one pass 2 at the current sources + the solver's update kernels.  `first` skips work that
// step_begin has already done.  cond != 0: the kernel that decides convergence also drives the WHILE node.
int enqueue_step_iteration(landau_ctx* c, Cloud& cl, const StepBufs& b, double dt, double tol, int max_iter, bool first,
                           cudaGraphConditionalHandle cond) {
    NvtxRange nvtx("landau:a4-a5 fixed-point iteration");
    cudaStream_t st = c->stream;
    const int npm = b.npm;
    double* rec = cl.sym ? nullptr : cl.recs();
    double* soa = cl.sym ? cl.soas() : nullptr;
    int nparts = 0;
    if (c->solver == 2 && !first) {
        nk_sources_kernel<<<ceil_div(npm, 256), 256, 0, st>>>(cl.L(), c->d_ctrl, c->d_nk, npm, cl.x(), cl.y(), cl.z(),
                                                               b.xk, b.yk, b.zk, b.hist, rec, soa);
        c->launches += 1;
    }
    const bool stiff = stiff_active(c);
    RC(pair(c, cl, c->d_ctrl, &nparts, !stiff ? 0 : (cond ? 2 : (first ? 1 : 0))));
    st = c->stream;
    if (stiff) {
        stiff_fix_kernel<<<STIFF_CAP / 128, 128, 0, st>>>(c->d_tab, cl.L(), c->d_ctrl, c->d_stiff, (const int*)c->stiff_mark.p,
                                                         npm, nparts, dt, cl.x(), cl.y(), cl.z(), rec, soa,
                                                         (double*)c->vpart.p);
        c->launches += 1;
    }
    if (c->solver == 0) {
        step_update_kernel<<<b.nub, UPD_THREADS, 0, st>>>(c->d_tab, cl.L(), c->d_ctrl, npm, nparts, dt, tol, max_iter,
                                                           (const double*)c->vpart.p, cl.x(), cl.y(), cl.z(), cl.w(),
                                                           b.xk, b.yk, b.zk, rec, soa, (double*)c->blockpart.p, cond,
                                                           mixed_step_active(c, cl) ? c->mixed_until : 0.0);
        c->launches += 1;
    } else if (c->solver == 1) {
        // NEXT-4: Anderson-accelerated fixed point (step_anderson.cuh); commits g(x_k) of the last evaluation
        double* dF = b.hist;
        double* dG = dF + (size_t)c->aa_depth * 3 * npm;
        double* fprev = dG + (size_t)c->aa_depth * 3 * npm;
        double* gcur = fprev + 3 * (size_t)npm;
        anderson_update_kernel<<<b.nub, UPD_THREADS, 0, st>>>(
            c->d_tab, cl.L(), c->d_ctrl, c->d_aa, npm, nparts, dt, tol, max_iter, (const double*)c->vpart.p, cl.x(),
            cl.y(), cl.z(), cl.w(), b.xk, b.yk, b.zk, dF, dG, fprev, gcur, (double*)c->blockpart.p, cond);
        anderson_mix_kernel<<<ceil_div(npm, 256), 256, 0, st>>>(cl.L(), c->d_ctrl, c->d_aa, npm, cl.x(), cl.y(), cl.z(),
                                                                 gcur, dG, b.xk, b.yk, b.zk, rec, soa);
        c->launches += 2;
    } else {
        // NEXT-4: Jacobian-free Newton-Krylov (step_newton.cuh); commits g(x) of the last phase-0 evaluation
        double* Q = b.hist;
        double* gcur = Q + ((size_t)c->nk_m + 1) * 3 * (size_t)npm;
        double* Vcur = gcur + 3 * (size_t)npm;
        double* fvec = Vcur + 3 * (size_t)npm;
        nk_post_kernel<<<b.nub, UPD_THREADS, 0, st>>>(c->d_tab, cl.L(), c->d_ctrl, c->d_nk, npm, nparts, dt, tol,
                                                       max_iter, (const double*)c->vpart.p, cl.x(), cl.y(), cl.z(),
                                                       cl.w(), b.xk, b.yk, b.zk, Q, gcur, Vcur, fvec,
                                                       (double*)c->blockpart.p, cond);
        nk_update_kernel<<<ceil_div(npm, 256), 256, 0, st>>>(cl.L(), c->d_ctrl, c->d_nk, npm, Q, fvec, b.xk, b.yk, b.zk);
        c->launches += 2;
    }
    return 0;
}

void enqueue_step_commit(landau_ctx* c, Cloud& cl, const StepBufs& b) {
    const size_t np = (size_t)b.npm;
    step_commit_kernel<<<ceil_div(b.npm, 256), 256, 0, c->stream>>>(cl.L(), c->d_ctrl, b.npm, cl.x(), cl.y(), cl.z(),
                                                                     b.commit, b.commit + np, b.commit + 2 * np,
                                                                     (StepRecord*)c->records.p, c->d_cursor);
    c->launches += 1;
}
}  // namespace

// =============================================================================================
namespace {
// ---- a4 for launch-bound clouds: one step as a CUDA graph with a conditional WHILE node ----------------------
// Nodes: step_begin, WHILE { (zero_slices,) pair, step_update -> cudaGraphSetConditional }, commit.  Pass 1 stays
// outside (ordinary launches just before the graph) so that a pass 1 already done by landau_moments is reused.
// Built by stream capture of the very launch sequence landau_run issues otherwise, after one ordinary step has
// sized every buffer (nothing may be allocated during capture).  Returns 0 and leaves sg.exec == nullptr with
// sg.failed set if the capture is refused; the ordinary launch sequence is then used (same kernels, same results).
void destroy_step_graph(landau_ctx* c) {
    if (c->sg.exec) cudaGraphExecDestroy(c->sg.exec);
    if (c->sg.graph) cudaGraphDestroy(c->sg.graph);
    c->sg.exec = nullptr; c->sg.graph = nullptr;
}

bool step_graph_matches(const landau_ctx* c, const Cloud& cl, double dt, double tol, int max_iter) {
    const auto& g = c->sg;
    return g.exec && g.gen == c->alloc_gen && g.N == cl.N && g.npm == cl.npad_max && g.dt == dt && g.tol == tol &&
           g.max_iter == max_iter && g.ek == c->entropy_kernel && g.pk == c->pair_kernel && g.solver == c->solver &&
           g.mixed == c->mixed_until && g.stiff == c->stiff_theta &&
           g.depth == (c->solver == 1 ? c->aa_depth : c->solver == 2 ? c->nk_m : 0);
}

int build_step_graph(landau_ctx* c, Cloud& cl, double dt, double tol, int max_iter) {
    destroy_step_graph(c);
    if ((!c->body_stream && cudaStreamCreateWithFlags(&c->body_stream, cudaStreamNonBlocking) != cudaSuccess) ||
        (!c->cap_stream && cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking) != cudaSuccess)) {
        c->sg.failed = true; cudaGetLastError(); return 0;
    }
    const int npm = cl.npad_max;
    const StepBufs sb = step_bufs(c, cl);
    // capture on a private stream (the context's stream may be the legacy default stream, which cannot be captured)
    cudaStream_t user_stream = c->stream;
    cudaStream_t st = c->cap_stream;
    c->stream = st;
    const unsigned long long gen0 = c->alloc_gen;
    const int64_t launches0 = c->launches;
    const bool g_valid0 = cl.G_valid, ran0 = c->entropy_ran;
    const char* stage = "begin capture";
    cudaError_t ce = cudaStreamBeginCapture(st, cudaStreamCaptureModeRelaxed);
    bool ok = ce == cudaSuccess;
    cudaGraph_t graph = nullptr;
    int fixed = 0, body_nodes = 0;
    if (ok) {
        if (ok) ok = enqueue_step_begin(c, cl, sb, max_iter) == 0;
        cudaStreamCaptureStatus status;
        cudaGraph_t g = nullptr;
        const cudaGraphNode_t* deps = nullptr;
        size_t ndeps = 0;
        cudaGraphConditionalHandle handle = 0;
        cudaGraphNode_t cond_node = nullptr;
        cudaGraphNodeParams params = {cudaGraphNodeTypeConditional};
#define SG_TRY(what, call) if (ok) { ce = (call); if (ce != cudaSuccess) { ok = false; stage = what; } }
        SG_TRY("capture info", cudaStreamGetCaptureInfo(st, &status, nullptr, &g, &deps, &ndeps));
        if (ok && status != cudaStreamCaptureStatusActive) { ok = false; stage = "capture not active"; }
        SG_TRY("conditional handle", cudaGraphConditionalHandleCreate(&handle, g, 1, cudaGraphCondAssignDefault));
        if (ok) {
            params.type = cudaGraphNodeTypeConditional;
            params.conditional.handle = handle;
            params.conditional.type = cudaGraphCondTypeWhile;
            params.conditional.size = 1;
            SG_TRY("conditional node", cudaGraphAddNode(&cond_node, g, deps, ndeps, &params));
        }
        fixed = (int)(c->launches - launches0);
        if (ok) {
            cudaGraph_t body = params.conditional.phGraph_out[0];
            SG_TRY("body capture", cudaStreamBeginCaptureToGraph(c->body_stream, body, nullptr, nullptr, 0,
                                                                 cudaStreamCaptureModeRelaxed));
            if (ok) {
                const int64_t l1 = c->launches;
                c->stream = c->body_stream;
                // the body always rebuilds its sources (first = false): it is replayed for every iteration
                ok = enqueue_step_iteration(c, cl, sb, dt, tol, max_iter, false, handle) == 0;
                c->stream = st;
                body_nodes = (int)(c->launches - l1);
                cudaGraph_t tmp = nullptr;
                ce = cudaStreamEndCapture(c->body_stream, &tmp);
                if (ce != cudaSuccess && ok) { ok = false; stage = "end body capture"; }
            }
        }
        SG_TRY("update dependencies", cudaStreamUpdateCaptureDependencies(st, &cond_node, 1, cudaStreamSetCaptureDependencies));
        if (ok) {
            const int64_t l2 = c->launches;
            enqueue_step_commit(c, cl, sb);
            fixed += (int)(c->launches - l2);
        }
        ce = cudaStreamEndCapture(st, &graph);
        if ((ce != cudaSuccess || !graph) && ok) { ok = false; stage = "end capture"; }
    }
    c->stream = user_stream;
    c->launches = launches0;                    // nothing was launched: capture only records
    cl.G_valid = g_valid0; c->entropy_ran = ran0;
    cudaGraphExec_t exec = nullptr;
    if (ok && c->alloc_gen != gen0) { ok = false; stage = "a buffer was reallocated during capture"; }
    SG_TRY("instantiate", cudaGraphInstantiate(&exec, graph, 0));
#undef SG_TRY
    if (!ok) {
        cudaGetLastError();
        if (exec) cudaGraphExecDestroy(exec);
        if (graph) cudaGraphDestroy(graph);
        c->sg.failed = true;
        snprintf(c->err, sizeof(c->err), "step graph not built (%s: %s); using the plain launch sequence", stage,
                 cudaGetErrorString(ce));
        return 0;
    }
    auto& g = c->sg;
    g.graph = graph; g.exec = exec; g.gen = c->alloc_gen; g.N = cl.N; g.npm = npm; g.dt = dt; g.tol = tol;
    g.max_iter = max_iter; g.ek = c->entropy_kernel; g.pk = c->pair_kernel; g.fixed_nodes = fixed; g.body_nodes = body_nodes;
    g.solver = c->solver; g.depth = c->solver == 1 ? c->aa_depth : c->solver == 2 ? c->nk_m : 0;
    g.mixed = c->mixed_until; g.stiff = c->stiff_theta;
    return 0;
}
}  // namespace

namespace {
// Launch-bound clouds (step_small.cuh): all Jacobi iterations of a step in one persistent kernel.  Returns 1 if the
// kernel was launched, 0 if this cloud / configuration does not qualify (the caller takes the graph or the launch
// sequence), < 0 on error.
template <int R, int DIM>
int launch_step_small_rd(landau_ctx* c, Cloud& cl, const StepBufs& b, int ttiles, int nchunks, double dt, double tol,
                                int max_iter) {
    auto kern = step_small_kernel<R, DIM>;
    int& occ = c->small_occ[R - 1][DIM - 2];
    if (!occ) {
        CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, PAIR_THREADS, 0));
        if (occ < 1) occ = -1;
    }
    const int G = ttiles * nchunks;
    if (occ < 0 || G > occ * c->sm_count) return 0;               // every CTA must be resident (grid-wide barriers)
    const DevTable* T = c->d_tab; DevLayout* L = cl.L(); StepCtrl* ctrl = c->d_ctrl;
    int npm = b.npm;
    double* rec = cl.recs(); double* vpart = (double*)c->vpart.p;
    const double *xn = cl.x(), *yn = cl.y(), *zn = cl.z(), *w = cl.w();
    double *xk = b.xk, *yk = b.yk, *zk = b.zk, *bp = (double*)c->blockpart.p;
    unsigned int* bar = &c->d_ctrl->ticket;                        // zeroed by step_begin_kernel
    void* args[] = {&T, &L, &ctrl, &npm, &ttiles, &nchunks, &dt, &tol, &max_iter, &rec, &vpart, &xn, &yn, &zn, &w,
                    &xk, &yk, &zk, &bp, &bar};
    const cudaError_t ce = cudaLaunchCooperativeKernel((const void*)kern, dim3(G), dim3(PAIR_THREADS), args, 0, c->stream);
    if (ce == cudaErrorCooperativeLaunchTooLarge || ce == cudaErrorNotSupported) {
        // fewer SMs than the occupancy query assumed (e.g. an MPS partition): the graph / launch sequence instead
        cudaGetLastError();
        occ = -1;
        return 0;
    }
    CU(ce);
    c->launches += 1;
    return 1;
}

bool step_small_eligible(const landau_ctx* c, const Cloud& cl) {
    return c->graph_mode == 1 && !c->prof_on && c->solver == 0 && !stiff_active(c) && !cl.sym && c->precision == 0 &&
           c->coop_ok && cl.npad_max <= PAIR_THREADS * UPD_THREADS;
}

int launch_step_small(landau_ctx* c, Cloud& cl, const StepBufs& b, double dt, double tol, int max_iter) {
    int R, ttiles, nchunks;
    onesided_grid(c, cl, &R, &ttiles, &nchunks);
    RC(ensure(c, c->vpart, sizeof(double) * 3 * (size_t)nchunks * cl.npad_max));
    int rc;
    if (c->dim == 2) rc = R == 1 ? launch_step_small_rd<1, 2>(c, cl, b, ttiles, nchunks, dt, tol, max_iter)
                                 : launch_step_small_rd<2, 2>(c, cl, b, ttiles, nchunks, dt, tol, max_iter);
    else             rc = R == 1 ? launch_step_small_rd<1, 3>(c, cl, b, ttiles, nchunks, dt, tol, max_iter)
                                 : launch_step_small_rd<2, 3>(c, cl, b, ttiles, nchunks, dt, tol, max_iter);
    if (rc == 1) {
        c->k_pair = c->dim == 2 ? "onesided2v" : "onesided";
        snprintf(c->kernels, sizeof(c->kernels), "pair=%s entropy=%s", c->k_pair, c->k_entropy);
    }
    return rc;
}

}  // namespace

namespace {
// NEXT-3: many collision cells, one persistent CTA per cell, whole run in one launch (cells.cuh).
template <int NQ, int MINB, int NT>
int launch_cells_v(landau_ctx* c, int n_cells, int cap, const double* v, const double* w, const int32_t* sid,
                   double* v_out, int n_steps, double dt, double tol, int max_iter) {
    auto kern = cells_run_kernel<NQ, MINB, NT>;
    const size_t smem = CellsCfg<NQ>::smem(cap);
    size_t& attr = MINB == 1 ? c->attr_cells[NQ] : c->attr_cells_small[MINB == 2 ? 0 : 1];
    if (smem > attr) {
        CU(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        attr = smem;
    }
    int* counter = (int*)((char*)c->cells_off.p + sizeof(long long) * ((size_t)n_cells + 1));
    const int grid = std::min(n_cells, MINB * c->sm_count);
    kern<<<grid, NT, smem, c->stream>>>(c->d_tab, n_cells, cap, (const long long*)c->cells_off.p, v, w, sid,
                                        v_out, n_steps, dt, tol, max_iter, counter, (CellRecord*)c->cells_rec.p);
    c->launches += 1;
    return 0;
}

template <int NQ>
int launch_cells(landau_ctx* c, int n_cells, int cap, const double* v, const double* w, const int32_t* sid,
                 double* v_out, int n_steps, double dt, double tol, int max_iter) {
    // batches of small cells (n_q = 4): builds of the kernel with only the small-cell paths and several CTAs per SM
    if (NQ == 4 && cap <= CELLS_THREADS / 4 && n_cells > 2 * c->sm_count)
        return launch_cells_v<4, 4, CELLS_THREADS / 2>(c, n_cells, cap, v, w, sid, v_out, n_steps, dt, tol, max_iter);
    if (NQ == 4 && cap <= CELLS_SMALL && n_cells > c->sm_count)
        return launch_cells_v<4, 2, CELLS_THREADS>(c, n_cells, cap, v, w, sid, v_out, n_steps, dt, tol, max_iter);
    return launch_cells_v<NQ, 1, CELLS_THREADS>(c, n_cells, cap, v, w, sid, v_out, n_steps, dt, tol, max_iter);
}

}  // namespace

extern "C" {

void landau_default_opts(landau_opts* o) {
    if (!o) return;
    memset(o, 0, sizeof(*o));
    o->n_q = 4; o->nu0 = 1.0; o->nu = nullptr; o->precision = 0; o->stream = nullptr;
    o->pair_kernel = 0; o->entropy_kernel = 0; o->device = -1;
}

const char* landau_version(void) { return "landau-b200 0.1 (sm_100a)"; }

const char* landau_last_error(const landau_ctx* c) { return c ? c->err : "NULL context"; }
const char* landau_last_kernels(const landau_ctx* c) { return c ? c->kernels : ""; }
int64_t landau_launch_count(const landau_ctx* c) { return c ? c->launches : 0; }

int landau_create(landau_ctx** out, int S, const double* mass, const double* charge, const double* eps,
                  const landau_opts* opts) {
    if (!out) return LANDAU_EINVAL;
    *out = nullptr;
    if (S < 1 || S > LD_MAX_SPECIES || !mass || !charge || !eps) return LANDAU_EINVAL;
    landau_opts o;
    landau_default_opts(&o);
    if (opts) o = *opts;
    if (o.n_q == 0) o.n_q = 4;
    if (o.nu0 == 0.0) o.nu0 = 1.0;
    if (o.n_q < 2 || o.n_q > LD_MAX_NQ) return LANDAU_EINVAL;
    if (o.precision < 0 || o.precision > 1 || o.pair_kernel < 0 || o.pair_kernel > 2 || o.entropy_kernel < 0 ||
        o.entropy_kernel > 3)
        return LANDAU_EINVAL;
    for (int s = 0; s < S; ++s)
        if (!(mass[s] > 0.0) || !(eps[s] > 0.0) || !isfinite(charge[s]) || !isfinite(mass[s]) || !isfinite(eps[s]))
            return LANDAU_EINVAL;
    landau_ctx* c = new (std::nothrow) landau_ctx();
    if (!c) return LANDAU_ENOMEM;
    c->err[0] = 0; c->kernels[0] = 0;
    c->S = S; c->n_q = o.n_q; c->precision = o.precision; c->pair_kernel = o.pair_kernel;
    c->entropy_kernel = o.entropy_kernel; c->stream = (cudaStream_t)o.stream;
    for (int s = 0; s < S; ++s) { c->mass[s] = mass[s]; c->charge[s] = charge[s]; c->eps[s] = eps[s]; }
    for (int s = 0; s < S; ++s)
        for (int t = 0; t < S; ++t)
            c->nu[s * S + t] = o.nu ? o.nu[s * S + t] : o.nu0 * charge[s] * charge[s] * charge[t] * charge[t];
    for (int s = 0; s < S; ++s)
        for (int t = 0; t < S; ++t)
            if (c->nu[s * S + t] != c->nu[t * S + s] || !isfinite(c->nu[s * S + t])) { delete c; return LANDAU_EINVAL; }
    gauss_hermite_gw(c->n_q, c->knot, c->gw);

    auto bail = [&](int code) { landau_destroy(c); return code; };
    int ndev = 0, caller_dev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { delete c; return LANDAU_ECUDA; }
    if (cudaGetDevice(&caller_dev) != cudaSuccess) { delete c; return LANDAU_ECUDA; }
    c->device = o.device >= 0 ? o.device : caller_dev;
    if (c->device >= ndev) { delete c; return LANDAU_ECUDA; }
    DevGuard dev_guard(c);                 // the caller's current device is left untouched
    { int cur = -1; if (cudaGetDevice(&cur) != cudaSuccess || cur != c->device) { delete c; return LANDAU_ECUDA; } }
    cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, c->device);
    { int coop = 0; cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, c->device); c->coop_ok = coop != 0; }
    DevTable t;
    memset(&t, 0, sizeof(t));
    t.S = S; t.n_q = c->n_q; t.pad = 128; t.dim = 3;
    for (int s = 0; s < S; ++s) {
        t.mass[s] = mass[s]; t.inv_mass[s] = 1.0 / mass[s]; t.eps[s] = eps[s];
        t.inv_sqrt_2eps[s] = 1.0 / sqrt(2.0 * eps[s]);
    }
    for (int i = 0; i < S * S; ++i) t.nu[i] = c->nu[i];
    // nu_ss' = c_s c_s' (true of the default nu0 q_s^2 q_s'^2): the symmetric in-cell pair evaluation of
    // cells.cuh folds c_s into the weights; any other table keeps the one-sided loop
    t.nu_rank1 = 1;
    for (int a = 0; a < S; ++a) { t.nu_fac[a] = sqrt(c->nu[a * S + a]); if (!(c->nu[a * S + a] > 0.0)) t.nu_rank1 = 0; }
    for (int a = 0; a < S && t.nu_rank1; ++a)
        for (int b = 0; b < S; ++b)
            if (fabs(t.nu_fac[a] * t.nu_fac[b] - c->nu[a * S + b]) > 4e-16 * fabs(c->nu[a * S + b])) t.nu_rank1 = 0;
    for (int i = 0; i < c->n_q; ++i) { t.knot[i] = c->knot[i]; t.gw[i] = c->gw[i]; }
    for (int j = 0; j < 64; ++j) t.exp2_tab[j] = exp2((double)j / 64.0);
    for (int j = 0; j < 256; ++j) t.exp2_tab256[j] = exp2((double)j / 256.0);
    {   // product-table budget of pass 1's DMMA form: a quarter of the device memory, or LANDAU_PRODTAB_BUDGET_MB
        cudaDeviceProp prop;
        if (cudaGetDeviceProperties(&prop, c->device) == cudaSuccess) c->prodtab_budget = prop.totalGlobalMem / 4;
        if (const char* e = getenv("LANDAU_PRODTAB_BUDGET_MB")) {
            const double mb = atof(e);
            if (mb > 0.0) c->prodtab_budget = (size_t)(mb * 1048576.0);
        }
    }
    if (cudaMalloc(&c->d_tab, sizeof(DevTable)) != cudaSuccess) return bail(LANDAU_ECUDA);
    if (cudaMalloc(&c->d_ctrl, sizeof(StepCtrl)) != cudaSuccess) return bail(LANDAU_ECUDA);
    if (cudaMalloc(&c->d_cursor, sizeof(int)) != cudaSuccess) return bail(LANDAU_ECUDA);
    if (cudaMalloc(&c->d_aa, sizeof(AndersonCtrl)) != cudaSuccess) return bail(LANDAU_ECUDA);
    if (cudaMalloc(&c->d_nk, sizeof(NewtonCtrl)) != cudaSuccess) return bail(LANDAU_ECUDA);
    if (cudaMalloc(&c->d_dg, sizeof(DgCtrl)) != cudaSuccess) return bail(LANDAU_ECUDA);
    if (cudaMalloc(&c->d_stiff, sizeof(StiffCtrl)) != cudaSuccess) return bail(LANDAU_ECUDA);
    if (cudaMemset(c->d_stiff, 0, sizeof(StiffCtrl)) != cudaSuccess) return bail(LANDAU_ECUDA);
    if (cudaMalloc(&c->d_cutstats, 2 * sizeof(unsigned long long)) != cudaSuccess) return bail(LANDAU_ECUDA);
    if (cudaMemset(c->d_cutstats, 0, 2 * sizeof(unsigned long long)) != cudaSuccess) return bail(LANDAU_ECUDA);
    if (cudaMalloc(&c->d_momout, sizeof(double) * LD_MAX_SPECIES * MOM_OUT) != cudaSuccess) return bail(LANDAU_ECUDA);
    if (cudaMallocHost(&c->h_pin, PIN_BYTES) != cudaSuccess) return bail(LANDAU_ECUDA);
    if (cudaMemcpy(c->d_tab, &t, sizeof(t), cudaMemcpyHostToDevice) != cudaSuccess) return bail(LANDAU_ECUDA);
    if (cudaMemset(c->d_ctrl, 0, sizeof(StepCtrl)) != cudaSuccess) return bail(LANDAU_ECUDA);
    *out = c;
    return LANDAU_OK;
}

void landau_destroy(landau_ctx* c) {
    if (!c) return;
    DevGuard dev_guard(c);
    for (auto& ev : c->prof_events) { cudaEventDestroy(ev.e0); cudaEventDestroy(ev.e1); }
    for (auto e : c->prof_pool) cudaEventDestroy(e);
    if (c->d_tab) cudaFree(c->d_tab);
    if (c->d_ctrl) cudaFree(c->d_ctrl);
    if (c->d_cursor) cudaFree(c->d_cursor);
    if (c->d_aa) cudaFree(c->d_aa);
    if (c->d_nk) cudaFree(c->d_nk);
    if (c->d_dg) cudaFree(c->d_dg);
    if (c->d_stiff) cudaFree(c->d_stiff);
    if (c->d_cutstats) cudaFree(c->d_cutstats);
    destroy_step_graph(c);
    if (c->body_stream) cudaStreamDestroy(c->body_stream);
    if (c->cap_stream) cudaStreamDestroy(c->cap_stream);
    if (c->d_momout) cudaFree(c->d_momout);
    if (c->h_pin) cudaFreeHost(c->h_pin);
    for (Cloud* cl : {&c->tmp, &c->state}) {
        release(cl->lay); release(cl->xyzw); release(cl->perm); release(cl->G); release(cl->rec); release(cl->soa);
    }
    for (Buf* b : {&c->blockcnt, &c->blockoff, &c->part, &c->vpart, &c->blockpart, &c->vk, &c->V, &c->records,
                   &c->stage_v, &c->stage_w, &c->stage_s, &c->stage_o, &c->facttab, &c->prodtab, &c->dg_u, &c->dg_Gu,
                   &c->dg_Gk, &c->dg_part, &c->aa_hist, &c->cells_off, &c->cells_rec, &c->soa32, &c->sym_acc,
                   &c->sym_tpart, &c->sym_ticket, &c->tilebox, &c->cellkey,
                   &c->cellrank, &c->chunkcnt, &c->binoff, &c->spbox, &c->stiff_mark, &c->stiff_scratch})
        release(*b);
    delete c;
}

int landau_get_quadrature(const landau_ctx* c, double* knots, double* weights) {
    if (!c || !knots || !weights) return LANDAU_EINVAL;
    for (int i = 0; i < c->n_q; ++i) { knots[i] = c->knot[i]; weights[i] = c->gw[i]; }
    return 0;
}

int landau_entropy_grad(landau_ctx* c, int64_t N, const double* v, const double* w, const int32_t* sid, double* G_out,
                        double* S_eps_out) {
    if (!c) return LANDAU_EINVAL;
    DevGuard dev_guard(c);
    if (!G_out) return fail(c, LANDAU_EINVAL, "entropy_grad: NULL output");
    Cloud& cl = c->tmp;
    RC(pack(c, cl, N, v, w, sid));
    RC(entropy(c, cl));
    scatter3_kernel<<<ceil_div(cl.npad_max, 256), 256, 0, c->stream>>>(cl.npad_max, cl.L(), cl.prm(), cl.Gx(), cl.Gy(),
                                                                       cl.Gz(), G_out);
    c->launches += 1;
    if (S_eps_out) {
        double* h = (double*)((char*)c->h_pin + PIN_MOM);
        RC(species_sums(c, cl, true, false, h));
        const double PI = 3.14159265358979323846;
        for (int s = 0; s < c->S; ++s) S_eps_out[s] = -h[s * MOM_OUT + 11] / (PI * sqrt(PI));
    }
    return finish(c, cl, "entropy_grad");
}

int landau_pair_field(landau_ctx* c, int64_t N, const double* v, const double* w, const int32_t* sid,
                      const double* G_in, double* out) {
    if (!c) return LANDAU_EINVAL;
    DevGuard dev_guard(c);
    if (!G_in || !out) return fail(c, LANDAU_EINVAL, "pair_field: NULL array");
    Cloud& cl = c->tmp;
    c->k_entropy = "-";                       // the entropy gradient is supplied: no pass 1 in this call
    RC(pack(c, cl, N, v, w, sid));
    gather3_kernel<<<ceil_div(cl.npad_max, 256), 256, 0, c->stream>>>(cl.npad_max, cl.L(), cl.prm(), G_in, cl.Gx(),
                                                                      cl.Gy(), cl.Gz());
    c->launches += 1;
    RC(field_of_cloud(c, cl, out));
    return finish(c, cl, "pair_field");
}

int landau_eval_field(landau_ctx* c, int64_t N, const double* v, const double* w, const int32_t* sid, double* out) {
    if (!c) return LANDAU_EINVAL;
    DevGuard dev_guard(c);
    if (!out) return fail(c, LANDAU_EINVAL, "eval_field: NULL output");
    Cloud& cl = c->tmp;
    RC(pack(c, cl, N, v, w, sid));
    RC(entropy(c, cl));
    RC(field_of_cloud(c, cl, out));
    return finish(c, cl, "eval_field");
}

int landau_eval_field_host(landau_ctx* c, int64_t N, const double* v, const double* w, const int32_t* sid,
                           double* out) {
    if (!c) return LANDAU_EINVAL;
    DevGuard dev_guard(c);
    if (!out) return fail(c, LANDAU_EINVAL, "eval_field_host: NULL output");
    const double *dv, *dw;
    const int32_t* ds;
    RC(stage_in(c, N, v, w, sid, &dv, &dw, &ds));
    RC(ensure(c, c->stage_o, sizeof(double) * 3 * (size_t)N));
    Cloud& cl = c->tmp;
    RC(pack(c, cl, N, dv, dw, ds));
    RC(entropy(c, cl));
    RC(field_of_cloud(c, cl, (double*)c->stage_o.p));
    CU(cudaMemcpyAsync(out, c->stage_o.p, sizeof(double) * 3 * (size_t)N, cudaMemcpyDeviceToHost, c->stream));
    return finish(c, cl, "eval_field_host");
}

int landau_set_markers(landau_ctx* c, int64_t N, const double* v, const double* w, const int32_t* sid) {
    if (!c) return LANDAU_EINVAL;
    DevGuard dev_guard(c);
    Cloud& cl = c->state;
    cl.N = 0;
    RC(pack(c, cl, N, v, w, sid));
    int rc = finish(c, cl, "set_markers");
    if (rc < 0) cl.N = 0;
    return rc;
}

int landau_set_markers_host(landau_ctx* c, int64_t N, const double* v, const double* w, const int32_t* sid) {
    if (!c) return LANDAU_EINVAL;
    DevGuard dev_guard(c);
    const double *dv, *dw;
    const int32_t* ds;
    RC(stage_in(c, N, v, w, sid, &dv, &dw, &ds));
    return landau_set_markers(c, N, dv, dw, ds);
}

int landau_get_markers(landau_ctx* c, double* v_out) {
    if (!c) return LANDAU_EINVAL;
    DevGuard dev_guard(c);
    Cloud& cl = c->state;
    if (cl.N < 1) return fail(c, LANDAU_EINVAL, "get_markers: no markers held");
    if (!v_out) return fail(c, LANDAU_EINVAL, "get_markers: NULL output");
    scatter3_kernel<<<ceil_div(cl.npad_max, 256), 256, 0, c->stream>>>(cl.npad_max, cl.L(), cl.prm(), cl.x(), cl.y(),
                                                                       cl.z(), v_out);
    c->launches += 1;
    return finish(c, cl, "get_markers");
}

int landau_get_markers_host(landau_ctx* c, double* v_out) {
    if (!c) return LANDAU_EINVAL;
    DevGuard dev_guard(c);
    Cloud& cl = c->state;
    if (cl.N < 1) return fail(c, LANDAU_EINVAL, "get_markers: no markers held");
    if (!v_out) return fail(c, LANDAU_EINVAL, "get_markers: NULL output");
    RC(ensure(c, c->stage_o, sizeof(double) * 3 * (size_t)cl.N));
    scatter3_kernel<<<ceil_div(cl.npad_max, 256), 256, 0, c->stream>>>(cl.npad_max, cl.L(), cl.prm(), cl.x(), cl.y(),
                                                                       cl.z(), (double*)c->stage_o.p);
    c->launches += 1;
    CU(cudaMemcpyAsync(v_out, c->stage_o.p, sizeof(double) * 3 * (size_t)cl.N, cudaMemcpyDeviceToHost, c->stream));
    return finish(c, cl, "get_markers_host");
}

static int run_steps(landau_ctx* c, int n_steps, double dt, double tol, int max_iter, landau_step_info* info, int hold) {
    if (!c) return LANDAU_EINVAL;
    DevGuard dev_guard(c);
    Cloud& cl = c->state;
    if (cl.N < 1) return fail(c, LANDAU_EINVAL, "step: no markers held (landau_set_markers first)");
    if (n_steps < 1 || max_iter < 1 || !(dt > 0.0) || !(tol >= 0.0) || !isfinite(dt))
        return fail(c, LANDAU_EINVAL, "step: need n_steps >= 1, max_iter >= 1, dt > 0, tol >= 0");
    const int npm = cl.npad_max;
    RC(ensure(c, c->vk, sizeof(double) * 3 * (size_t)npm));
    RC(ensure(c, c->records, sizeof(StepRecord) * (size_t)n_steps));
    const int nub = ceil_div(npm, UPD_THREADS);
    RC(ensure(c, c->blockpart, sizeof(double) * (size_t)step_blockpart_doubles(c, nub)));
    if (c->solver != 0) RC(ensure(c, c->aa_hist, sizeof(double) * step_hist_doubles(c, npm)));
    if (stiff_active(c)) {
        RC(ensure(c, c->stiff_mark, sizeof(int) * (size_t)npm));
        if (!c->stiff_scratch.p) {
            RC(ensure(c, c->stiff_scratch, sizeof(double) * (2 * LD_MAX_SPECIES + 2)));
            CU(cudaMemsetAsync(c->stiff_scratch.p, 0, sizeof(double) * (2 * LD_MAX_SPECIES + 2), c->stream));
        }
        c->stiff_dt = dt;
    }
    const StepBufs sb = step_bufs(c, cl);
    cudaStream_t st = c->stream;
    CU(cudaMemsetAsync(c->d_cursor, 0, sizeof(int), st));
    CU(cudaMemsetAsync(c->d_ctrl, 0, sizeof(StepCtrl), st));
    if (hold) {
        const int one = 1;
        CU(cudaMemcpyAsync(&c->d_ctrl->hold, &one, sizeof(int), cudaMemcpyHostToDevice, st));
    }
    const bool graph_ok = !hold && c->graph_mode != 0 && !c->sg.failed && !c->prof_on &&
                          (c->graph_mode == 2 || npm <= 65536);
    std::vector<char> via_graph(n_steps, 0), via_small(n_steps, 0);
    bool small_ok = step_small_eligible(c, cl);
    for (int n = 0; n < n_steps; ++n) {
        c->prof_step = n; c->prof_iter = 0;
        if (!cl.G_valid) RC(entropy(c, cl));     // a preceding landau_moments(S_eps) already evaluated pass 1 here
        cl.G_valid = false;                      // the step moves the markers
        if (small_ok) {
            // vpart must have its final size before step_begin (nothing else allocates in a fused step)
            RC(enqueue_step_begin(c, cl, sb, max_iter));
            const int rs = launch_step_small(c, cl, sb, dt, tol, max_iter);
            if (rs < 0) return rs;
            if (rs == 1) { enqueue_step_commit(c, cl, sb); via_small[n] = 1; continue; }
            small_ok = false;                    // not resident: the graph / launch sequence from here on (begin is idempotent)
        }
        if (graph_ok && step_graph_matches(c, cl, dt, tol, max_iter)) {
            CU(cudaGraphLaunch(c->sg.exec, st));
            c->launches += c->sg.fixed_nodes;
            via_graph[n] = 1;
            continue;
        }
        RC(enqueue_step_begin(c, cl, sb, max_iter));
        for (int k = 0; k < max_iter; ++k) {
            c->prof_iter = k;
            RC(enqueue_step_iteration(c, cl, sb, dt, tol, max_iter, k == 0, 0));
        }
        enqueue_step_commit(c, cl, sb);
        // every buffer now has its size: capture the same sequence as a graph for the steps that follow
        if (graph_ok && !step_graph_matches(c, cl, dt, tol, max_iter)) RC(build_step_graph(c, cl, dt, tol, max_iter));
    }
    CU(cudaGetLastError());
    // one synchronisation: records + error flags
    std::vector<StepRecord> h(n_steps);
    StepCtrl* hc = (StepCtrl*)((char*)c->h_pin + PIN_CTRL);
    CU(cudaMemcpyAsync(hc, c->d_ctrl, sizeof(StepCtrl), cudaMemcpyDeviceToHost, st));
    CU(cudaMemcpyAsync(h.data(), c->records.p, sizeof(StepRecord) * (size_t)n_steps, cudaMemcpyDeviceToHost, st));
    c->in_run = true;
    int rc = finish(c, cl, "step");
    c->in_run = false;
    if (rc < 0) { if (c->prof_on) prof_resolve(c, nullptr, 0); return rc; }
    if (hc->err) return fail(c, hc->err, "step: non-finite residual");
    if (c->prof_on) {
        std::vector<int> its(n_steps);
        for (int n = 0; n < n_steps; ++n) its[n] = h[n].iterations;
        prof_resolve(c, its.data(), n_steps);
    }
    c->k_step = via_small[n_steps - 1] ? "fused" : (via_graph[n_steps - 1] ? "graph" : "launch");
    snprintf(c->kernels, sizeof(c->kernels), "pair=%s entropy=%s step=%s", c->k_pair, c->k_entropy, c->k_step);
    int any_unconverged = 0;
    for (int n = 0; n < n_steps; ++n) {
        if (via_graph[n]) c->launches += (int64_t)h[n].iterations * c->sg.body_nodes;   // WHILE body launches
        if (info) { info[n].iterations = h[n].iterations; info[n].residual = h[n].residual; info[n].converged = h[n].converged; }
        if (!h[n].converged) any_unconverged = 1;
    }
    return any_unconverged ? LANDAU_NOT_CONVERGED : LANDAU_OK;
}

int landau_set_dimension(landau_ctx* c, int dim) {
    if (!c) return LANDAU_EINVAL;
    DevGuard dev_guard(c);
    if (dim != 2 && dim != 3) return fail(c, LANDAU_EINVAL, "set_dimension: dim must be 2 or 3");
    c->dim = dim;
    c->state.G_valid = false; c->tmp.G_valid = false;
    ++c->alloc_gen;                              // a captured step graph holds the other dimension's kernels
    CU(cudaMemcpyAsync(&c->d_tab->dim, &c->dim, sizeof(int), cudaMemcpyHostToDevice, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    return 0;
}

// One step of length dt with up to `depth` levels of halving: a step whose fixed point does not converge is not
// committed (StepCtrl::hold) and is redone as two steps of dt/2.  Every sub-step is a step of Eq. (24), so momentum
// and energy are conserved by each of them.  At depth 0 the step is committed whatever happens (reading S8).
static int advance_adaptive(landau_ctx* c, double dt, double tol, int max_iter, int depth, landau_step_info* acc) {
    landau_step_info one = {0, 0.0, 0};
    const int rc = run_steps(c, 1, dt, tol, max_iter, &one, depth > 0 ? 1 : 0);
    if (rc < 0) return rc;
    acc->iterations += one.iterations;
    if (one.converged || depth == 0) {
        acc->residual = one.residual > acc->residual ? one.residual : acc->residual;
        if (!one.converged) acc->converged = 0;
        return 0;
    }
    c->state.G_valid = true;            // nothing moved: G^n of the refused step is still the entropy gradient of v^n
    for (int half = 0; half < 2; ++half) {
        const int r2 = advance_adaptive(c, 0.5 * dt, tol, max_iter, depth - 1, acc);
        if (r2 < 0) return r2;
    }
    return 0;
}

int landau_run(landau_ctx* c, int n_steps, double dt, double tol, int max_iter, landau_step_info* info) {
    if (!c) return LANDAU_EINVAL;
    if (c->substep == 0) return run_steps(c, n_steps, dt, tol, max_iter, info, 0);
    if (n_steps < 1) return fail(c, LANDAU_EINVAL, "step: need n_steps >= 1");
    int any_unconverged = 0;
    for (int n = 0; n < n_steps; ++n) {
        landau_step_info acc = {0, 0.0, 1};
        const int rc = advance_adaptive(c, dt, tol, max_iter, c->substep, &acc);
        if (rc < 0) return rc;
        if (info) info[n] = acc;
        if (!acc.converged) any_unconverged = 1;
    }
    return any_unconverged ? LANDAU_NOT_CONVERGED : LANDAU_OK;
}

int landau_set_substep(landau_ctx* c, int max_halvings) {
    if (!c) return LANDAU_EINVAL;
    if (max_halvings < 0 || max_halvings > 10) return fail(c, LANDAU_EINVAL, "set_substep: max_halvings must be 0..10");
    c->substep = max_halvings;
    return 0;
}

int landau_set_stiff_pairs(landau_ctx* c, double theta) {
    if (!c) return LANDAU_EINVAL;
    if (!(theta >= 0.0) || !isfinite(theta))
        return fail(c, LANDAU_EINVAL, "set_stiff_pairs: the stiffness threshold must be >= 0 (0 = off)");
    c->stiff_theta = theta;
    return 0;
}

int landau_stiff_pairs_last(landau_ctx* c, int* n_pairs, int* n_skipped) {
    if (!c) return LANDAU_EINVAL;
    DevGuard dev_guard(c);
    int* h = (int*)((char*)c->h_pin + PIN_CTRL + 96);
    CU(cudaMemcpyAsync(h, c->d_stiff, 4 * sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    if (n_pairs) *n_pairs = h[0] < STIFF_CAP ? h[0] : STIFF_CAP;
    if (n_skipped) *n_skipped = h[2] + h[3] + (h[1] ? 1 : 0);
    return 0;
}

int landau_set_mixed_precision(landau_ctx* c, double f32_until) {
    if (!c) return LANDAU_EINVAL;
    if (!(f32_until >= 0.0) || !isfinite(f32_until))
        return fail(c, LANDAU_EINVAL, "set_mixed_precision: the switch-over residual must be >= 0 (0 = off)");
    // Below FP32's own resolution of the iterate (2^-23 ~ 1.2e-7 relative in V, times dt / |v| << 1 in v) the residual
    // of an FP32 evaluation cannot fall any further, so the switch to FP64 would never happen and every step would
    // burn max_iter iterations: refuse such a threshold instead of looping.
    if (f32_until > 0.0 && f32_until < 1e-10)
        return fail(c, LANDAU_EINVAL, "set_mixed_precision: a switch-over residual below 1e-10 is under the FP32 noise "
                    "floor of the iterate; use >= 1e-10 (1e-7 is typical) or 0 = off");
    c->mixed_until = f32_until;
    return 0;
}

int landau_set_cutoff(landau_ctx* c, int on, int morton) {
    if (!c) return LANDAU_EINVAL;
    c->cutoff_on = on != 0;
    c->morton_on = morton != 0;
    c->state.G_valid = false; c->tmp.G_valid = false;
    ++c->alloc_gen;                                  // a captured step graph has the old setting baked in
    return 0;
}

int landau_cutoff_stats(landau_ctx* c, int64_t* tiles_considered, int64_t* tiles_skipped) {
    if (!c) return LANDAU_EINVAL;
    DevGuard dev_guard(c);
    unsigned long long* h = (unsigned long long*)((char*)c->h_pin + PIN_CTRL + 64);
    CU(cudaMemcpyAsync(h, c->d_cutstats, 2 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    if (tiles_considered) *tiles_considered = (int64_t)h[0];
    if (tiles_skipped) *tiles_skipped = (int64_t)h[1];
    return 0;
}

int landau_set_step_graph(landau_ctx* c, int mode) {
    if (!c) return LANDAU_EINVAL;
    if (mode < 0 || mode > 2) return fail(c, LANDAU_EINVAL, "set_step_graph: mode must be 0 (off), 1 (automatic) or 2 (always)");
    c->graph_mode = mode;
    c->sg.failed = false;
    return 0;
}

int landau_set_solver(landau_ctx* c, int solver, int depth) {
    if (!c) return LANDAU_EINVAL;
    if (solver < 0 || solver > 2)
        return fail(c, LANDAU_EINVAL, "set_solver: solver must be 0 (Jacobi), 1 (Anderson) or 2 (Newton-Krylov)");
    if (solver == 1 && (depth < 1 || depth > AA_MAXM))
        return fail(c, LANDAU_EINVAL, "set_solver: Anderson depth must be 1..%d", AA_MAXM);
    if (solver == 2 && (depth < 1 || depth > NK_MAXM))
        return fail(c, LANDAU_EINVAL, "set_solver: Newton-Krylov restart length must be 1..%d", NK_MAXM);
    c->solver = solver;
    if (solver == 1) c->aa_depth = depth;
    if (solver == 2) c->nk_m = depth;
    return 0;
}

int landau_step(landau_ctx* c, double dt, double tol, int max_iter, landau_step_info* info) {
    return landau_run(c, 1, dt, tol, max_iter, info);
}

// NEXT-1: one discrete-gradient step (Eqs. 46-49; step_dg.cuh).  Device driven: the entropies, Gonzalez' lambda and the
// residual are reduced on the device and every kernel of an iteration exits at once when StepCtrl::done is set; the
// host enqueues the iterations in chunks of DG_CHUNK and reads the done flag once per chunk (no read-back inside an
// iteration).
int landau_step_dg(landau_ctx* c, double dt, double tol, int max_iter, landau_step_info* info) {
    if (!c) return LANDAU_EINVAL;
    DevGuard dev_guard(c);
    Cloud& cl = c->state;
    if (cl.N < 1) return fail(c, LANDAU_EINVAL, "step_dg: no markers held (landau_set_markers first)");
    if (max_iter < 1 || !(dt > 0.0) || !(tol >= 0.0) || !isfinite(dt))
        return fail(c, LANDAU_EINVAL, "step_dg: need max_iter >= 1, dt > 0, tol >= 0");
    constexpr int DG_CHUNK = 8;
    const int npm = cl.npad_max;
    const size_t B4 = sizeof(double) * 4 * (size_t)npm;
    RC(ensure(c, c->vk, B4));
    RC(ensure(c, c->dg_u, B4));
    RC(ensure(c, c->dg_Gu, B4));
    RC(ensure(c, c->dg_Gk, B4));
    RC(ensure(c, c->records, sizeof(StepRecord)));
    const int nub = ceil_div(npm, UPD_THREADS), ndb = ceil_div(npm, DG_THREADS);
    RC(ensure(c, c->blockpart, sizeof(double) * (size_t)step_blockpart_doubles(c, nub)));
    RC(ensure(c, c->dg_part, sizeof(double) * 2 * (size_t)ndb));
    const bool anderson = c->solver == 1;          // landau_set_solver(1, depth) also accelerates this fixed point
    if (anderson) RC(ensure(c, c->aa_hist, sizeof(double) * (2 * (size_t)c->aa_depth + 2) * 3 * (size_t)npm));
    double* aa_dF = (double*)c->aa_hist.p;
    double* aa_dG = anderson ? aa_dF + (size_t)c->aa_depth * 3 * npm : nullptr;
    double* aa_fprev = anderson ? aa_dG + (size_t)c->aa_depth * 3 * npm : nullptr;
    double* aa_gcur = anderson ? aa_fprev + 3 * (size_t)npm : nullptr;
    double* xk = (double*)c->vk.p;
    double* yk = xk + npm;
    double* zk = yk + npm;
    cudaStream_t st = c->stream;
    // cloud-shaped views that share the state's layout and permutation
    Cloud U = cl;  U.xyzw = c->dg_u;  U.G = c->dg_Gu;        // midpoint u, G(u)
    Cloud VK = cl; VK.xyzw = c->vk;   VK.G = c->dg_Gk;       // iterate v^(k), its entropy integrand
    double* rec = cl.sym ? nullptr : cl.recs();
    double* soa = cl.sym ? cl.soas() : nullptr;
    CU(cudaMemsetAsync(c->d_cursor, 0, sizeof(int), st));
    CU(cudaMemsetAsync(c->d_ctrl, 0, sizeof(StepCtrl), st));
    c->prof_step = 0; c->prof_iter = 0;
    if (!cl.G_valid) RC(entropy(c, cl));                      // G(v^n), entropy integrand at v^n
    cl.G_valid = false;
    dg_begin_kernel<<<1, 32, 0, st>>>(c->d_dg);
    step_begin_kernel<<<ceil_div(npm, 256), 256, 0, st>>>(c->d_tab, cl.L(), c->d_ctrl, npm, cl.x(), cl.y(), cl.z(),
                                                           cl.w(), cl.Gx(), cl.Gy(), cl.Gz(), xk, yk, zk, rec, soa);
    dg_entropy_total_kernel<<<ndb, DG_THREADS, 0, st>>>(cl.L(), c->d_ctrl, npm, cl.w(), cl.snode(), (double*)c->dg_part.p,
                                                         c->d_dg, 0);
    CU(cudaMemcpyAsync(xk + 3 * (size_t)npm, cl.w(), sizeof(double) * (size_t)npm, cudaMemcpyDeviceToDevice, st));
    c->launches += 3;
    if (anderson) {
        anderson_begin_kernel<<<1, 32, 0, st>>>(c->d_aa, c->aa_depth);
        c->launches += 1;
    }
    StepCtrl* hc = (StepCtrl*)((char*)c->h_pin + PIN_CTRL);
    for (int k = 0; k < max_iter; ++k) {
        int nparts = 0;
        c->prof_iter = k;
        if (k > 0) {
            dg_midpoint_kernel<<<ceil_div(npm, 256), 256, 0, st>>>(cl.L(), c->d_ctrl, npm, cl.x(), cl.y(), cl.z(), cl.w(),
                                                                    xk, yk, zk, U.x());
            RC(entropy(c, U, c->d_ctrl));
            RC(entropy(c, VK, c->d_ctrl));
            dg_entropy_total_kernel<<<ndb, DG_THREADS, 0, st>>>(cl.L(), c->d_ctrl, npm, VK.w(), VK.snode(),
                                                                 (double*)c->dg_part.p, c->d_dg, 1);
            dg_lambda_kernel<<<ndb, DG_THREADS, 0, st>>>(cl.L(), c->d_ctrl, c->d_dg, npm, cl.x(), cl.y(), cl.z(), cl.w(),
                                                          xk, yk, zk, U.Gx(), U.Gy(), U.Gz(), (double*)c->dg_part.p);
            dg_build_kernel<<<ceil_div(npm, 256), 256, 0, st>>>(c->d_tab, cl.L(), c->d_ctrl, c->d_dg, npm, U.x(), cl.x(),
                                                                 cl.y(), cl.z(), xk, yk, zk, U.Gx(), U.Gy(), U.Gz(), rec, soa);
            c->launches += 4;
        }
        RC(pair(c, cl, c->d_ctrl, &nparts));
        if (anderson) {
            anderson_update_kernel<<<nub, UPD_THREADS, 0, st>>>(
                c->d_tab, cl.L(), c->d_ctrl, c->d_aa, npm, nparts, dt, tol, max_iter, (const double*)c->vpart.p, cl.x(),
                cl.y(), cl.z(), cl.w(), xk, yk, zk, aa_dF, aa_dG, aa_fprev, aa_gcur, (double*)c->blockpart.p, 0);
            anderson_mix_kernel<<<ceil_div(npm, 256), 256, 0, st>>>(cl.L(), c->d_ctrl, c->d_aa, npm, cl.x(), cl.y(), cl.z(),
                                                                     aa_gcur, aa_dG, xk, yk, zk, rec, soa);
            c->launches += 2;
        } else {
            step_update_kernel<<<nub, UPD_THREADS, 0, st>>>(c->d_tab, cl.L(), c->d_ctrl, npm, nparts, dt, tol, max_iter,
                                                             (const double*)c->vpart.p, cl.x(), cl.y(), cl.z(), cl.w(),
                                                             xk, yk, zk, rec, soa, (double*)c->blockpart.p, 0);
            c->launches += 1;
        }
        if ((k + 1) % DG_CHUNK == 0 && k + 1 < max_iter) {    // one look at the flag per chunk of iterations
            CU(cudaMemcpyAsync(hc, c->d_ctrl, sizeof(StepCtrl), cudaMemcpyDeviceToHost, st));
            CU(cudaStreamSynchronize(st));
            if (hc->done) break;
        }
    }
    {
        const double* cm = anderson ? aa_gcur : xk;
        step_commit_kernel<<<ceil_div(npm, 256), 256, 0, st>>>(cl.L(), c->d_ctrl, npm, cl.x(), cl.y(), cl.z(), cm,
                                                                cm + npm, cm + 2 * (size_t)npm,
                                                                (StepRecord*)c->records.p, c->d_cursor);
    }
    c->launches += 1;
    CU(cudaGetLastError());
    CU(cudaMemcpyAsync(hc, c->d_ctrl, sizeof(StepCtrl), cudaMemcpyDeviceToHost, st));
    c->in_run = true;
    int rc = finish(c, cl, "step_dg");
    c->in_run = false;
    if (c->prof_on) {
        const int its = hc->iterations;
        prof_resolve(c, &its, 1);
    }
    if (rc < 0) return rc;
    if (hc->err) return fail(c, hc->err, "step_dg: non-finite residual");
    if (info) { info->iterations = hc->iterations; info->residual = hc->residual; info->converged = hc->converged; }
    return hc->converged ? LANDAU_OK : LANDAU_NOT_CONVERGED;
}

int landau_cells_max_markers(int n_q) {
    switch (n_q) {
        case 2: case 3: case 4: return CELLS_CAP;
        case 5: return CellsCfg<5>::max_cap();
        case 6: return CellsCfg<6>::max_cap();
        case 7: return CellsCfg<7>::max_cap();
        case 8: return CellsCfg<8>::max_cap();
        default: return 0;
    }
}

int landau_cells_run(landau_ctx* c, int n_cells, const int64_t* cell_offset, const double* v, const double* w,
                     const int32_t* sid, double* v_out, int n_steps, double dt, double tol, int max_iter,
                     landau_cell_info* info) {
    if (!c) return LANDAU_EINVAL;
    DevGuard dev_guard(c);
    if (n_cells < 1 || !cell_offset || !v || !w || !sid || !v_out)
        return fail(c, LANDAU_EINVAL, "cells_run: NULL array or n_cells < 1");
    if (n_steps < 1 || max_iter < 1 || !(dt > 0.0) || !(tol >= 0.0) || !isfinite(dt))
        return fail(c, LANDAU_EINVAL, "cells_run: need n_steps >= 1, max_iter >= 1, dt > 0, tol >= 0");
    const int cap_max = landau_cells_max_markers(c->n_q);
    int cap = 0;
    for (int k = 0; k < n_cells; ++k) {
        const int64_t nk = cell_offset[k + 1] - cell_offset[k];
        if (nk < 0) return fail(c, LANDAU_EINVAL, "cells_run: cell_offset must be non-decreasing");
        if (nk > cap_max)
            return fail(c, LANDAU_EINVAL, "cells_run: cell %d has %lld markers, limit %d per cell at n_q = %d", k,
                        (long long)nk, cap_max, c->n_q);
        cap = std::max(cap, (int)nk);
    }
    cap = std::max(32, (cap + 1) & ~1);
    cudaStream_t st = c->stream;
    RC(ensure(c, c->cells_off, sizeof(long long) * ((size_t)n_cells + 1) + 64));
    RC(ensure(c, c->cells_rec, sizeof(CellRecord) * (size_t)n_cells));
    static_assert(sizeof(long long) == sizeof(int64_t), "offset type");
    CU(cudaMemcpyAsync(c->cells_off.p, cell_offset, sizeof(int64_t) * ((size_t)n_cells + 1), cudaMemcpyHostToDevice, st));
    CU(cudaMemsetAsync((char*)c->cells_off.p + sizeof(long long) * ((size_t)n_cells + 1), 0, sizeof(int), st));
    switch (c->n_q) {
        case 2: RC((launch_cells<2>(c, n_cells, cap, v, w, sid, v_out, n_steps, dt, tol, max_iter))); break;
        case 3: RC((launch_cells<3>(c, n_cells, cap, v, w, sid, v_out, n_steps, dt, tol, max_iter))); break;
        case 4: RC((launch_cells<4>(c, n_cells, cap, v, w, sid, v_out, n_steps, dt, tol, max_iter))); break;
        case 5: RC((launch_cells<5>(c, n_cells, cap, v, w, sid, v_out, n_steps, dt, tol, max_iter))); break;
        case 6: RC((launch_cells<6>(c, n_cells, cap, v, w, sid, v_out, n_steps, dt, tol, max_iter))); break;
        case 7: RC((launch_cells<7>(c, n_cells, cap, v, w, sid, v_out, n_steps, dt, tol, max_iter))); break;
        default: RC((launch_cells<8>(c, n_cells, cap, v, w, sid, v_out, n_steps, dt, tol, max_iter))); break;
    }
    CU(cudaGetLastError());
    std::vector<CellRecord> h(n_cells);
    CU(cudaMemcpyAsync(h.data(), c->cells_rec.p, sizeof(CellRecord) * (size_t)n_cells, cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    CU(cudaGetLastError());
    snprintf(c->kernels, sizeof(c->kernels), "cells=fused");
    int worst = 0, any_unconv = 0;
    for (int k = 0; k < n_cells; ++k) {
        if (info) {
            info[k].status = h[k].status; info[k].iterations = h[k].iterations;
            info[k].max_iterations = h[k].max_iterations; info[k].steps_not_converged = h[k].steps_not_converged;
            info[k].residual = h[k].residual;
        }
        worst = std::min(worst, h[k].status);
        if (h[k].status == 1) any_unconv = 1;
    }
    if (worst < 0) return fail(c, worst, "cells_run: at least one cell failed (status %d); see landau_cell_info.status", worst);
    return any_unconv ? LANDAU_NOT_CONVERGED : LANDAU_OK;
}

int landau_moments(landau_ctx* c, double* n, double* P, double* K, double* S_eps) {
    if (!c) return LANDAU_EINVAL;
    DevGuard dev_guard(c);
    Cloud& cl = c->state;
    if (cl.N < 1) return fail(c, LANDAU_EINVAL, "moments: no markers held");
    if (S_eps && !cl.G_valid) RC(entropy(c, cl));
    double* h = (double*)((char*)c->h_pin + PIN_MOM);
    RC(species_sums(c, cl, S_eps != nullptr, false, h));
    const double PI = 3.14159265358979323846;
    for (int s = 0; s < c->S; ++s) {
        const double* r = h + s * MOM_OUT;
        if (n) n[s] = r[0];
        if (P) { P[3 * s] = c->mass[s] * r[1]; P[3 * s + 1] = c->mass[s] * r[2]; P[3 * s + 2] = c->mass[s] * r[3]; }
        if (K) K[s] = 0.5 * c->mass[s] * r[4];
        if (S_eps) S_eps[s] = -r[11] / (PI * sqrt(PI));
    }
    return finish(c, cl, "moments");
}

int landau_moments_ext(landau_ctx* c, double* stress, double* m4) {
    if (!c) return LANDAU_EINVAL;
    DevGuard dev_guard(c);
    Cloud& cl = c->state;
    if (cl.N < 1) return fail(c, LANDAU_EINVAL, "moments_ext: no markers held");
    double* h = (double*)((char*)c->h_pin + PIN_MOM);
    RC(species_sums(c, cl, false, m4 != nullptr, h));
    for (int s = 0; s < c->S; ++s) {
        const double* r = h + s * MOM_OUT;
        if (stress) for (int i = 0; i < 6; ++i) stress[6 * s + i] = c->mass[s] * r[5 + i];
        if (m4) for (int i = 0; i < 3; ++i) m4[3 * s + i] = r[12 + i];
    }
    return finish(c, cl, "moments_ext");
}

int landau_profile_enable(landau_ctx* c, int on) {
    if (!c) return LANDAU_EINVAL;
    c->prof_on = on != 0;
    c->prof_ms[0] = c->prof_ms[1] = 0.0;
    c->prof_n[0] = c->prof_n[1] = 0;
    return 0;
}

int landau_profile_read(landau_ctx* c, double* pair_ms, int64_t* pair_launches, double* entropy_ms,
                        int64_t* entropy_launches) {
    if (!c) return LANDAU_EINVAL;
    if (pair_ms) *pair_ms = c->prof_ms[0];
    if (pair_launches) *pair_launches = c->prof_n[0];
    if (entropy_ms) *entropy_ms = c->prof_ms[1];
    if (entropy_launches) *entropy_launches = c->prof_n[1];
    return 0;
}

int landau_fp64_peak_dmma(landau_ctx* c, int reps, double* flops_out) {
    if (!c || !flops_out || reps < 1) return LANDAU_EINVAL;
    DevGuard dev_guard(c);
    RC(ensure(c, c->V, 1024));
    const int blocks = c->sm_count * 4, threads = 256, iters = 4096;
    cudaEvent_t e0, e1;
    CU(cudaEventCreate(&e0));
    CU(cudaEventCreate(&e1));
    double best = 0.0;
    for (int r = 0; r < reps + 1; ++r) {
        CU(cudaEventRecord(e0, c->stream));
        fp64_dmma_peak_kernel<<<blocks, threads, 0, c->stream>>>((double*)c->V.p, iters, 1e-3, 1e-3);
        CU(cudaEventRecord(e1, c->stream));
        CU(cudaEventSynchronize(e1));
        float ms = 0.f;
        CU(cudaEventElapsedTime(&ms, e0, e1));
        // per warp and MMA: m8 n8 k4 -> 2*8*8*4 = 512 flop; 32 MMAs per loop iteration
        const double fl = 512.0 * 32.0 * (double)iters * blocks * (threads / 32) / (ms * 1e-3);
        if (r > 0 && fl > best) best = fl;
    }
    c->launches += reps + 1;
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    *flops_out = best;
    return 0;
}

int landau_fp64_peak(landau_ctx* c, int reps, double* flops_out) {
    if (!c || !flops_out || reps < 1) return LANDAU_EINVAL;
    DevGuard dev_guard(c);
    RC(ensure(c, c->V, 1024));
    const int blocks = c->sm_count * 4, threads = 256, iters = 4096;
    cudaEvent_t e0, e1;
    CU(cudaEventCreate(&e0));
    CU(cudaEventCreate(&e1));
    double best = 0.0;
    for (int r = 0; r < reps + 1; ++r) {
        CU(cudaEventRecord(e0, c->stream));
        fp64_peak_kernel<<<blocks, threads, 0, c->stream>>>((double*)c->V.p, iters, 0.999999, 1e-9);
        CU(cudaEventRecord(e1, c->stream));
        CU(cudaEventSynchronize(e1));
        float ms = 0.f;
        CU(cudaEventElapsedTime(&ms, e0, e1));
        const double fl = 2.0 * 8.0 * 16.0 * (double)iters * blocks * threads / (ms * 1e-3);
        if (r > 0 && fl > best) best = fl;
    }
    c->launches += reps + 1;
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    *flops_out = best;
    return 0;
}

}  // extern "C"
