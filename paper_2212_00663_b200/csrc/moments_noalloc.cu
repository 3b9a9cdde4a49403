// moments_noalloc.cu -- landau_moments_noalloc: the conservation diagnostics n_s, P_s, K_s
// (Eqs. 33, 26, 28) for callers that must not allocate device memory.
//
// Who that is.  A collision operator is a guest inside somebody else's time loop.  A PIC code that
// has already handed every byte of HBM to its own field and particle arrays (or to a framework's
// fixed memory pool) has nothing left for cudaMalloc to give; and a diagnostics hook that runs
// between two asynchronous phases of such a loop cannot afford cudaMalloc / cudaFree either, because
// both may synchronise the whole device and so stall streams that are none of this library's
// business.  Every other entry point of liblandau.so goes through a landau_ctx whose scratch is
// cudaMalloc'ed (at landau_create and lazily afterwards), so none of them is usable there.  This one
// takes no context and calls no cudaMalloc, cudaFree or allocating library routine, ever: its only
// scratch -- the per-block partial sums of the two-stage reduction -- lives in the file-scope
// __device__ array below, which is part of the library image.
//
// What that costs.  Every GPU that loads liblandau.so carries the array (640.25 KiB) until the
// process exits, whether or not this entry point is called.  Its size fixes the largest problem:
// LANDAU_MOMENTS_NOALLOC_MAX_N = 2^21 markers (one partial per 2048 markers, per species, per sum)
// and LANDAU_MAX_SPECIES species; larger calls are refused with LANDAU_EINVAL, not truncated.
//
// Sharing.  There is ONE array per device, shared by every call from every thread and stream.  It
// keeps whatever the previous call left in it.  The partial-sum slots need no clearing (stage 1 of a
// call writes every slot stage 2 of that call reads); the status word in the header must start at
// zero and is cleared on the caller's stream at the start of every call.  Two calls that overlap on
// the GPU (different streams, or different host threads on streams that are not ordered against each
// other) race on the array and both results are garbage: order them yourself.
//
// Set-up.  In host code the array's name is only a handle; its device address comes from
// cudaGetSymbolAddress, looked up here once per device with that device current, on the first call
// made on that device.  That first call may make the CUDA runtime load this library's device code
// onto the GPU, so make it once, early, outside any stream capture.  Later calls on the same device
// only enqueue one memset and two kernels on the caller's stream and return without synchronising.
//
// This file shares nothing with the context path (moments.cuh): the summation order differs, so the
// two agree to rounding (a few ulp of the sums), not bit for bit.
#include <cuda_runtime.h>
#include <stdint.h>

#include <cstdarg>
#include <cstdio>
#include <mutex>

#include "landau.h"

namespace {

constexpr int NA_THREADS = 256;
constexpr int NA_PER_THREAD = 8;
constexpr int NA_CHUNK = NA_THREADS * NA_PER_THREAD;               // markers per stage-1 block
constexpr int NA_SUMS = 5;                                         // w, w vx, w vy, w vz, w |v|^2
constexpr int NA_MAX_BLOCKS = LANDAU_MOMENTS_NOALLOC_MAX_N / NA_CHUNK;
constexpr int NA_HEADER = 32;                                      // doubles; [0] = status word
constexpr size_t NA_DOUBLES = NA_HEADER + (size_t)NA_MAX_BLOCKS * LANDAU_MAX_SPECIES * NA_SUMS;
constexpr int NA_MAX_DEVICES = 64;

static_assert(LANDAU_MOMENTS_NOALLOC_MAX_N % NA_CHUNK == 0, "whole blocks");
static_assert(NA_DOUBLES * sizeof(double) == 655616, "the size stated in landau.h and README.md");

// The scratch: header (status word) + partial sums [block][species][sum].  Device code names it
// directly; host code must go through cudaGetSymbolAddress (scratch_for_current_device below).
static __device__ __align__(256) double g_na_scratch[NA_DOUBLES];

struct Masses {
    double m[LANDAU_MAX_SPECIES];
};

__device__ __forceinline__ double na_warp_sum(double x) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    return x;
}

// Fixed-order block sum of NA_SUMS values per thread; the result lands in res[0..NA_SUMS) (shared).
__device__ __forceinline__ void na_block_sum(const double (&a)[NA_SUMS], double (*sm)[NA_SUMS], double* res) {
    const int lane = threadIdx.x & 31, wv = threadIdx.x >> 5;
#pragma unroll
    for (int q = 0; q < NA_SUMS; ++q) {
        const double s = na_warp_sum(a[q]);
        if (lane == 0) sm[wv][q] = s;
    }
    __syncthreads();
    if (threadIdx.x < NA_SUMS) {
        double s = 0.0;
#pragma unroll
        for (int k = 0; k < NA_THREADS / 32; ++k) s += sm[k][threadIdx.x];
        res[threadIdx.x] = s;
    }
    __syncthreads();
}

// Stage 1: block b sums its 2048 markers per species into scratch[b][s][0..5).
__global__ void __launch_bounds__(NA_THREADS)
moments_noalloc_stage1(long long N, int S, const double* __restrict__ v, const double* __restrict__ w,
                       const int32_t* __restrict__ sid, double* __restrict__ scratch) {
    __shared__ double sm[NA_THREADS / 32][NA_SUMS];
    __shared__ double res[NA_SUMS];
    double t[NA_PER_THREAD][NA_SUMS];
    int sp[NA_PER_THREAD];
    const long long base = (long long)blockIdx.x * NA_CHUNK + threadIdx.x;
#pragma unroll
    for (int k = 0; k < NA_PER_THREAD; ++k) {
        const long long p = base + (long long)k * NA_THREADS;
        sp[k] = -1;
#pragma unroll
        for (int q = 0; q < NA_SUMS; ++q) t[k][q] = 0.0;
        if (p < N) {
            const double x = v[3 * p], y = v[3 * p + 1], z = v[3 * p + 2], ww = w[p];
            sp[k] = sid[p];
            if (sp[k] < 0 || sp[k] >= S) scratch[0] = 1.0;   // any writer writes the same value
            t[k][0] = ww; t[k][1] = ww * x; t[k][2] = ww * y; t[k][3] = ww * z;
            t[k][4] = ww * (x * x + y * y + z * z);
        }
    }
    double* part = scratch + NA_HEADER + (size_t)blockIdx.x * S * NA_SUMS;
    for (int s = 0; s < S; ++s) {
        double a[NA_SUMS];
#pragma unroll
        for (int q = 0; q < NA_SUMS; ++q) a[q] = 0.0;
#pragma unroll
        for (int k = 0; k < NA_PER_THREAD; ++k)
            if (sp[k] == s)
#pragma unroll
                for (int q = 0; q < NA_SUMS; ++q) a[q] += t[k][q];
        na_block_sum(a, sm, res);
        if (threadIdx.x < NA_SUMS) part[s * NA_SUMS + threadIdx.x] = res[threadIdx.x];
        __syncthreads();
    }
}

// Stage 2: block s adds the nb partials of species s in a fixed order and writes
// out[s][0] = n_s, out[s][1..3] = P_s = m_s sum w v, out[s][4] = K_s = (m_s / 2) sum w |v|^2.
__global__ void __launch_bounds__(NA_THREADS)
moments_noalloc_stage2(int nb, int S, Masses mass, const double* __restrict__ scratch, double* __restrict__ out) {
    __shared__ double sm[NA_THREADS / 32][NA_SUMS];
    __shared__ double res[NA_SUMS];
    const int s = blockIdx.x;
    const double* part = scratch + NA_HEADER;
    double a[NA_SUMS];
#pragma unroll
    for (int q = 0; q < NA_SUMS; ++q) a[q] = 0.0;
    for (int b = threadIdx.x; b < nb; b += NA_THREADS)
#pragma unroll
        for (int q = 0; q < NA_SUMS; ++q) a[q] += part[((size_t)b * S + s) * NA_SUMS + q];
    na_block_sum(a, sm, res);
    if (threadIdx.x < NA_SUMS) {
        const double m = mass.m[s];
        double r = res[threadIdx.x];
        if (threadIdx.x >= 1 && threadIdx.x <= 3) r *= m;
        if (threadIdx.x == 4) r *= 0.5 * m;
        if (scratch[0] != 0.0) r = __longlong_as_double(0x7ff8000000000000LL);   // bad species id: poison
        out[s * NA_SUMS + threadIdx.x] = r;
    }
}

thread_local char t_err[256] = "";

int na_fail(int code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    std::vsnprintf(t_err, sizeof(t_err), fmt, ap);
    va_end(ap);
    return code;
}

// Device address of g_na_scratch on the CURRENT device, looked up once per device.
int scratch_for_current_device(double** out) {
    static std::mutex mu;
    static double* ptr[NA_MAX_DEVICES] = {};
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return na_fail(LANDAU_ECUDA, "%s", cudaGetErrorString(e));
    if (dev < 0 || dev >= NA_MAX_DEVICES) return na_fail(LANDAU_ECUDA, "device ordinal %d out of range", dev);
    std::lock_guard<std::mutex> lock(mu);
    if (!ptr[dev]) {
        double* p = nullptr;
        e = cudaGetSymbolAddress((void**)&p, g_na_scratch);
        if (e != cudaSuccess || !p) {
            (void)cudaGetLastError();
            return na_fail(LANDAU_ECUDA, "cudaGetSymbolAddress: %s", e != cudaSuccess ? cudaGetErrorString(e) : "NULL address");
        }
        ptr[dev] = p;
    }
    *out = ptr[dev];
    return 0;
}

}  // namespace

extern "C" int landau_moments_noalloc(int64_t N, const double* v, const double* w, const int32_t* species_id,
                                      int n_species, const double* mass, double* out, void* stream) {
    t_err[0] = 0;
    if (!v || !w || !species_id || !mass || !out) return na_fail(LANDAU_EINVAL, "NULL argument");
    if (n_species < 1 || n_species > LANDAU_MAX_SPECIES)
        return na_fail(LANDAU_EINVAL, "n_species = %d outside 1..%d", n_species, LANDAU_MAX_SPECIES);
    if (N < 1) return na_fail(LANDAU_EINVAL, "N = %lld < 1", (long long)N);
    if (N > LANDAU_MOMENTS_NOALLOC_MAX_N)
        return na_fail(LANDAU_EINVAL,
                       "N = %lld exceeds LANDAU_MOMENTS_NOALLOC_MAX_N = %lld: the built-in scratch array holds one "
                       "partial per 2048 markers and cannot grow; use landau_moments (which allocates)",
                       (long long)N, (long long)LANDAU_MOMENTS_NOALLOC_MAX_N);
    Masses m;
    for (int s = 0; s < LANDAU_MAX_SPECIES; ++s) m.m[s] = s < n_species ? mass[s] : 0.0;
    for (int s = 0; s < n_species; ++s)
        if (!(m.m[s] > 0.0)) return na_fail(LANDAU_EINVAL, "mass[%d] is not > 0", s);
    double* scratch = nullptr;
    if (int rc = scratch_for_current_device(&scratch)) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const int nb = (int)((N + NA_CHUNK - 1) / NA_CHUNK);
    // the status word must start at zero; the partial-sum slots are all rewritten by stage 1
    cudaError_t e = cudaMemsetAsync(scratch, 0, NA_HEADER * sizeof(double), st);
    if (e != cudaSuccess) return na_fail(LANDAU_ECUDA, "%s", cudaGetErrorString(e));
    moments_noalloc_stage1<<<nb, NA_THREADS, 0, st>>>((long long)N, n_species, v, w, species_id, scratch);
    moments_noalloc_stage2<<<n_species, NA_THREADS, 0, st>>>(nb, n_species, m, scratch, out);
    e = cudaGetLastError();
    if (e != cudaSuccess) return na_fail(LANDAU_ECUDA, "%s", cudaGetErrorString(e));
    return LANDAU_OK;
}

extern "C" const char* landau_moments_noalloc_last_error(void) { return t_err; }
