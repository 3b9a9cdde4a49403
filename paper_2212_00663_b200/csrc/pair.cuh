// pair.cuh -- step a3 of the hot path: the pairwise Landau sum, Eq. (23) with the
// projection tensor Q of Eq. (4) and Gamma^h of Eq. (16):
//
//   V_p = (1/m_s) sum_s' nu_ss' sum_{q in s', q != p} w_q Q(v_p - v_q) (g_p - g_q),   g = G/m,
//   Q(z) c = (c - z (z.c)/|z|^2) / |z|.
//
// Source markers are records of 8 doubles {x, y, z, w, gx, gy, gz, 0} (one 64-byte line each) so a
// tile is one contiguous block of global memory.  One-sided kernel: every ordered pair is
// evaluated by its target's thread (26 FP64-pipe instructions per pair); the symmetric
// (action-reaction) kernel is in pair_sym.cuh.
#pragma once
#include "common.cuh"
#include "stiff_pairs.cuh"

namespace landau {

constexpr int PAIR_THREADS = 128;
constexpr int PAIR_SRC_TILE = 128;   // sources per shared-memory tile (species-uniform: pad % 128 == 0)

// One ordered pair.  z = v_p - v_q, c = g_p - g_q; adds w_q Q(z) c to acc.
__device__ __forceinline__ void pair_accumulate(double zx, double zy, double zz, double cx, double cy,
                                                double cz, double wq, double& ax, double& ay,
                                                double& az) {
    const double r2 = fma(zz, zz, fma(zy, zy, zx * zx));
    const double d = fma(zz, cz, fma(zy, cy, zx * cx));
    const double yv = rsqrt_or_zero(r2);          // 1/|z|, or 0 for a coincident pair (reading S5)
    const double h = d * (yv * yv);               // (z.c)/|z|^2
    const double a = wq * yv;
    ax = fma(a, fma(-zx, h, cx), ax);
    ay = fma(a, fma(-zy, h, cy), ay);
    az = fma(a, fma(-zz, h, cz), az);
}

// 2-V form of pair_accumulate (landau_set_dimension(2): v_z = 0, g_z = 0): the z terms vanish identically; the x, y
// results are bit-identical to the 3-V arithmetic on such data.
__device__ __forceinline__ void pair_accumulate2(double zx, double zy, double cx, double cy, double wq, double& ax,
                                                 double& ay) {
    const double r2 = fma(zy, zy, zx * zx);
    const double d = fma(zy, cy, zx * cx);
    const double yv = rsqrt_or_zero(r2);
    const double h = d * (yv * yv);
    const double a = wq * yv;
    ax = fma(a, fma(-zx, h, cx), ax);
    ay = fma(a, fma(-zy, h, cy), ay);
}

// Loads of data another CTA of the SAME launch may have written (the fused small-cloud step, step_small.cuh) bypass L1.
template <bool COH>
__device__ __forceinline__ double2 ld_d2(const double2* p) { return COH ? __ldcg(p) : *p; }

// Body of the one-sided kernel for target tile bx and source chunk by.  Each thread owns R targets (slots
// bx*128R + r*128 + tid).  Partial fields are written chunk-major: vpart[((chunk*3 + d) * npad_max) + slot], already
// scaled by nu_ss'/m_s, so that the combine step is a fixed-order sum over chunks.  sm: [PAIR_SRC_TILE * 8] doubles.
template <int R, int DIM, bool DETECT, bool COH>
__device__ __forceinline__ void pair_onesided_body(const DevTable* __restrict__ T, const DevLayout* __restrict__ L,
                                                   int npad_max, int nchunks, const double* rec, double* vpart,
                                                   StiffCtrl* stiff, int* stiff_mark, int bx, int by, double* sm,
                                                   const double* s_nu) {
    const int npad = L->npad;
    const int slot0 = bx * (PAIR_THREADS * R);
    if (slot0 >= npad) return;
    const int S = T->S;
    double px[R], py[R], pz[R], gx[R], gy[R], gz[R];
    double tx[R], ty[R], tz[R], pw[R];
    int sp[R], ps[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        int p = slot0 + r * PAIR_THREADS + threadIdx.x;
        ps[r] = p < npad ? p : -1;
        if (p >= npad) p = npad - 1;              // clamped duplicate; its result is not written
        const double2* rp = reinterpret_cast<const double2*>(rec + (size_t)p * 8);
        const double2 a = ld_d2<COH>(rp), b = ld_d2<COH>(rp + 1), c = ld_d2<COH>(rp + 2), d = ld_d2<COH>(rp + 3);
        px[r] = a.x; py[r] = a.y; pz[r] = b.x; pw[r] = b.y;   // (the weight is only used by the stiff-pair detection)
        gx[r] = c.x; gy[r] = c.y; gz[r] = d.x;
        tx[r] = ty[r] = tz[r] = 0.0;
        sp[r] = species_of_slot(L, S, p);
    }

    const int ntiles = npad / PAIR_SRC_TILE;
    const int tpc = ceil_div(ntiles, nchunks);
    const int t0 = by * tpc, t1 = min(ntiles, t0 + tpc);
    for (int t = t0; t < t1; ++t) {
        __syncthreads();
        {
            const double2* src = reinterpret_cast<const double2*>(rec + (size_t)t * PAIR_SRC_TILE * 8);
            double2* dst = reinterpret_cast<double2*>(sm);
#pragma unroll
            for (int k = 0; k < 4; ++k) dst[threadIdx.x + k * PAIR_THREADS] = ld_d2<COH>(src + threadIdx.x + k * PAIR_THREADS);
        }
        __syncthreads();
        const int sb = species_of_slot(L, S, t * PAIR_SRC_TILE);
        double ax[R], ay[R], az[R];
#pragma unroll
        for (int r = 0; r < R; ++r) ax[r] = ay[r] = az[r] = 0.0;
#pragma unroll 4
        for (int j = 0; j < PAIR_SRC_TILE; ++j) {
            const double2* q = reinterpret_cast<const double2*>(sm + j * 8);
            const double2 a = q[0], b = q[1], c = q[2], d = q[3];
#pragma unroll
            for (int r = 0; r < R; ++r) {
                if (DETECT) {
                    // first evaluation of a step: stiff pairs (stiff_pairs.cuh); every pair is seen from both sides
                    const double zx = px[r] - a.x, zy = py[r] - a.y, zz = pz[r] - b.x;
                    const double r2 = fma(zz, zz, fma(zy, zy, zx * zx));
                    const int q = t * PAIR_SRC_TILE + j;
                    if (r2 < stiff->thr2[sp[r] * S + sb] && ps[r] >= 0 && ps[r] < q) {
                        const double nu = s_nu[sp[r] * S + sb];
                        stiff_candidate(stiff, stiff_mark, ps[r], q, r2, gx[r] - c.x, gy[r] - c.y, gz[r] - d.x, nu * b.y,
                                        nu * pw[r], T->inv_mass[sp[r]], T->inv_mass[sb]);
                    }
                }
                if (DIM == 3)
                    pair_accumulate(px[r] - a.x, py[r] - a.y, pz[r] - b.x, gx[r] - c.x, gy[r] - c.y,
                                    gz[r] - d.x, b.y, ax[r], ay[r], az[r]);
                else
                    pair_accumulate2(px[r] - a.x, py[r] - a.y, gx[r] - c.x, gy[r] - c.y, b.y, ax[r], ay[r]);
            }
        }
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const double nu = s_nu[sp[r] * S + sb];
            tx[r] = fma(nu, ax[r], tx[r]); ty[r] = fma(nu, ay[r], ty[r]); tz[r] = fma(nu, az[r], tz[r]);
        }
    }
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int p = slot0 + r * PAIR_THREADS + threadIdx.x;
        if (p < npad) {
            const double im = T->inv_mass[sp[r]];
            double* o = vpart + (size_t)by * 3 * (size_t)npad_max + p;
            o[0] = tx[r] * im;
            o[(size_t)npad_max] = ty[r] * im;
            o[2 * (size_t)npad_max] = tz[r] * im;
        }
    }
}

// grid = (target tiles, source chunks).
template <int R, int DIM = 3, bool DETECT = false>
__global__ void __launch_bounds__(PAIR_THREADS)
pair_onesided_kernel(const DevTable* __restrict__ T, const DevLayout* __restrict__ L,
                     const StepCtrl* __restrict__ ctrl, int npad_max, int nchunks,
                     const double* __restrict__ rec, double* __restrict__ vpart, int gate = GATE_NONE,
                     StiffCtrl* stiff = nullptr, int* stiff_mark = nullptr) {
    if (ctrl && ctrl->done) return;
    if (gate_closed(ctrl, gate)) return;
    __shared__ __align__(16) double sm[PAIR_SRC_TILE * 8];
    __shared__ double s_nu[LD_MAX_SPECIES * LD_MAX_SPECIES];
    for (int i = threadIdx.x; i < T->S * T->S; i += PAIR_THREADS) s_nu[i] = T->nu[i];
    pair_onesided_body<R, DIM, DETECT, false>(T, L, npad_max, nchunks, rec, vpart, stiff, stiff_mark, blockIdx.x, blockIdx.y,
                                              sm, s_nu);
}

// FP32 variant of the one-sided kernel (BASELINE config 4, "plus an FP32 field variant"; landau_opts.precision = 1,
// field evaluation only, never the implicit step).  Same tiling; records are converted to FP32 while they are
// staged into shared memory, every per-pair operation (differences included) is FP32 on the FMA pipe with
// MUFU.RSQ + one Newton step, the per-tile sums (128 sources) are FP32, and tiles are accumulated in FP64.
// A pair whose FP32 separation underflows (|z|^2 < 1e-30) contributes 0 (reading S5 in FP32).
// Expected error vs the FP64 oracle: ~1e-6 relative L2 (tests/test_gpu_parity.py, bench.py report it).
template <int R>
__global__ void __launch_bounds__(PAIR_THREADS)
pair_onesided_f32_kernel(const DevTable* __restrict__ T, const DevLayout* __restrict__ L, int npad_max, int nchunks,
                         const double* __restrict__ rec, double* __restrict__ vpart) {
    const int npad = L->npad;
    const int slot0 = blockIdx.x * (PAIR_THREADS * R);
    if (slot0 >= npad) return;
    const int S = T->S;
    __shared__ float4 sa[PAIR_SRC_TILE], sb[PAIR_SRC_TILE];
    __shared__ double s_nu[LD_MAX_SPECIES * LD_MAX_SPECIES];
    for (int i = threadIdx.x; i < S * S; i += PAIR_THREADS) s_nu[i] = T->nu[i];

    float px[R], py[R], pz[R], gx[R], gy[R], gz[R];
    double tx[R], ty[R], tz[R];
    int sp[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        int p = slot0 + r * PAIR_THREADS + threadIdx.x;
        if (p >= npad) p = npad - 1;
        const double2* rp = reinterpret_cast<const double2*>(rec + (size_t)p * 8);
        const double2 a = rp[0], b = rp[1], c = rp[2], d = rp[3];
        px[r] = (float)a.x; py[r] = (float)a.y; pz[r] = (float)b.x;
        gx[r] = (float)c.x; gy[r] = (float)c.y; gz[r] = (float)d.x;
        tx[r] = ty[r] = tz[r] = 0.0;
        sp[r] = species_of_slot(L, S, p);
    }
    const int ntiles = npad / PAIR_SRC_TILE;
    const int tpc = ceil_div(ntiles, nchunks);
    const int t0 = blockIdx.y * tpc, t1 = min(ntiles, t0 + tpc);
    for (int t = t0; t < t1; ++t) {
        __syncthreads();
        {
            const double2* src = reinterpret_cast<const double2*>(rec + ((size_t)t * PAIR_SRC_TILE + threadIdx.x) * 8);
            const double2 a = src[0], b = src[1], c = src[2], d = src[3];
            sa[threadIdx.x] = make_float4((float)a.x, (float)a.y, (float)b.x, (float)b.y);
            sb[threadIdx.x] = make_float4((float)c.x, (float)c.y, (float)d.x, 0.f);
        }
        __syncthreads();
        const int sbs = species_of_slot(L, S, t * PAIR_SRC_TILE);
        float ax[R], ay[R], az[R];
#pragma unroll
        for (int r = 0; r < R; ++r) ax[r] = ay[r] = az[r] = 0.f;
#pragma unroll 4
        for (int j = 0; j < PAIR_SRC_TILE; ++j) {
            const float4 a = sa[j], b = sb[j];
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const float zx = px[r] - a.x, zy = py[r] - a.y, zz = pz[r] - a.z;
                const float cx = gx[r] - b.x, cy = gy[r] - b.y, cz = gz[r] - b.z;
                const float r2 = fmaf(zz, zz, fmaf(zy, zy, zx * zx));
                const float d = fmaf(zz, cz, fmaf(zy, cy, zx * cx));
                float y = rsqrtf(fmaxf(r2, 1e-30f));
                y = y * fmaf(-0.5f * r2 * y, y, 1.5f);            // one Newton step
                y = r2 < 1e-30f ? 0.f : y;
                const float h = d * (y * y);
                const float wy = a.w * y;
                ax[r] = fmaf(wy, fmaf(-zx, h, cx), ax[r]);
                ay[r] = fmaf(wy, fmaf(-zy, h, cy), ay[r]);
                az[r] = fmaf(wy, fmaf(-zz, h, cz), az[r]);
            }
        }
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const double nu = s_nu[sp[r] * S + sbs];
            tx[r] = fma(nu, (double)ax[r], tx[r]); ty[r] = fma(nu, (double)ay[r], ty[r]);
            tz[r] = fma(nu, (double)az[r], tz[r]);
        }
    }
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int p = slot0 + r * PAIR_THREADS + threadIdx.x;
        if (p < npad) {
            const double im = T->inv_mass[sp[r]];
            double* o = vpart + (size_t)blockIdx.y * 3 * (size_t)npad_max + p;
            o[0] = tx[r] * im;
            o[(size_t)npad_max] = ty[r] * im;
            o[2 * (size_t)npad_max] = tz[r] * im;
        }
    }
}

// {x,y,z,w,G} (packed SoA) -> source records with g = G/m_s.
__global__ void build_rec_kernel(const DevTable* __restrict__ T, const DevLayout* __restrict__ L,
                                 int npad_max, const double* __restrict__ x, const double* __restrict__ y,
                                 const double* __restrict__ z, const double* __restrict__ w,
                                 const double* __restrict__ Gx, const double* __restrict__ Gy,
                                 const double* __restrict__ Gz, double* __restrict__ rec) {
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= npad_max || p >= L->npad) return;
    const double im = T->inv_mass[species_of_slot(L, T->S, p)];
    double2* o = reinterpret_cast<double2*>(rec + (size_t)p * 8);
    o[0] = make_double2(x[p], y[p]);
    o[1] = make_double2(z[p], w[p]);
    o[2] = make_double2(Gx[p] * im, Gy[p] * im);
    o[3] = make_double2(Gz[p] * im, 0.0);
}

// Fixed-order sum of the chunk partials -> packed SoA field.
__global__ void combine_field_kernel(const DevLayout* __restrict__ L, int npad_max, int nchunks,
                                     const double* __restrict__ vpart, double* __restrict__ Vx,
                                     double* __restrict__ Vy, double* __restrict__ Vz) {
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= npad_max || p >= L->npad) return;
    double a = 0.0, b = 0.0, c = 0.0;
    for (int k = 0; k < nchunks; ++k) {
        const double* o = vpart + (size_t)k * 3 * (size_t)npad_max + p;
        a += o[0]; b += o[(size_t)npad_max]; c += o[2 * (size_t)npad_max];
    }
    Vx[p] = a; Vy[p] = b; Vz[p] = c;
}

}  // namespace landau
