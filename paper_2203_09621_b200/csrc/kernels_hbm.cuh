// HBM-bound kernels of the path: spectral bounds (a1), initial transform (a2), split (a3).
// Each streams its matrices once with 128-bit coalesced accesses; grids are multiples of the
// SM count.  Algorithmic bytes per element are stated in DESIGN.md "Kernels".
#pragma once
#include <cuda_fp16.h>
#include <cuda_runtime.h>

#include "control.cuh"

namespace dmpt {

// order-preserving map double <-> signed 64-bit, for atomicMin/atomicMax (order independent,
// hence deterministic)
__device__ __forceinline__ long long dbl_to_ordered(double d) {
    long long b = __double_as_longlong(d);
    return b >= 0 ? b : b ^ 0x7FFFFFFFFFFFFFFFLL;
}
__host__ __device__ __forceinline__ double ordered_to_dbl(long long b) {
    long long r = b >= 0 ? b : b ^ 0x7FFFFFFFFFFFFFFFLL;
#ifdef __CUDA_ARCH__
    return __longlong_as_double(r);
#else
    double d;
    memcpy(&d, &r, sizeof d);
    return d;
#endif
}

__device__ __forceinline__ float4 ldg_stream4(const float* p) {
    float4 v;
    asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0, %1, %2, %3}, [%4];"
                 : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
    return v;
}

template <typename T>
__device__ __forceinline__ T warp_sum(T v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
template <typename T>
__device__ __forceinline__ T warp_max(T v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

// hi = fp16(2^e x), lo = fp16(2^e x - hi), round-to-nearest-even (Eq. 13 after an exact
// power-of-two scale, readings R12/R17)
__device__ __forceinline__ void split_scaled(float x, float scale, __half& hi, __half& lo) {
    const float t = x * scale;              // exact: scale is a power of two (barring overflow)
    hi = __float2half_rn(t);
    lo = __float2half_rn(t - __half2float(hi));
}

// ---------------------------------------------------------------------------------------------
// a1  Gershgorin discs: one warp per row, shuffle reduction of sum_j |H0_ij|,
//     eps_min = min_i (H0_ii - r_i), eps_max = max_i (H0_ii + r_i), r_i = sum_{j != i} |H0_ij|.
//     bounds[0], bounds[1]: ordered-int encodings, initialised to +inf / -inf by dmpt_reset_state_kernel.
//     The same pass streams the perturbation(s) and leaves max|H1_f| in h1max[f] (bit pattern of a
//     non-negative float, ordered like an unsigned integer): the power-of-two scale of the first split of
//     S1_0 = -H1/W is then known BEFORE the fused transform + split kernel runs (reading R12).
//     h0 == nullptr (caller-supplied bounds) skips the discs; h1[f] == nullptr skips that field.
// ---------------------------------------------------------------------------------------------
struct H1Ptrs {
    const float* p[3];
};

__device__ __forceinline__ float absmax4(float m, const float4& v) {
    return fmaxf(fmaxf(m, fmaxf(fabsf(v.x), fabsf(v.y))), fmaxf(fabsf(v.z), fabsf(v.w)));
}

__global__ void __launch_bounds__(256) dmpt_gershgorin_kernel(const float* __restrict__ h0, H1Ptrs h1, int n, int ld,
                                                              long long* __restrict__ bounds,
                                                              unsigned int* __restrict__ h1max) {
    const int warps_per_block = blockDim.x >> 5;
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    double lo = INFINITY, hi = -INFINITY;
    float m1[3] = {0.f, 0.f, 0.f};
    bool vec = (ld & 3) == 0 && (reinterpret_cast<uintptr_t>(h0) & 15) == 0;
#pragma unroll
    for (int f = 0; f < 3; ++f) vec = vec && (reinterpret_cast<uintptr_t>(h1.p[f]) & 15) == 0;
    for (int row = blockIdx.x * warps_per_block + warp; row < n; row += gridDim.x * warps_per_block) {
        const size_t off = (size_t)row * ld;
        float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f;
        int j = 0;
        if (vec) {
            const int n4 = n & ~3;
            for (j = lane * 4; j < n4; j += 128) {
                if (h0) {
                    const float4 v = ldg_stream4(h0 + off + j);
                    a0 += fabsf(v.x); a1 += fabsf(v.y); a2 += fabsf(v.z); a3 += fabsf(v.w);
                }
#pragma unroll
                for (int f = 0; f < 3; ++f)
                    if (h1.p[f]) m1[f] = absmax4(m1[f], ldg_stream4(h1.p[f] + off + j));
            }
            j = n4;
        }
        for (j += lane; j < n; j += 32) {
            if (h0) a0 += fabsf(h0[off + j]);
#pragma unroll
            for (int f = 0; f < 3; ++f)
                if (h1.p[f]) m1[f] = fmaxf(m1[f], fabsf(h1.p[f][off + j]));
        }
        if (h0) {
            double s = warp_sum((double)a0 + (double)a1 + (double)a2 + (double)a3);
            const double d = (double)h0[off + row];
            const double r = s - fabs(d);
            lo = fmin(lo, d - r);
            hi = fmax(hi, d + r);
        }
    }
#pragma unroll
    for (int f = 0; f < 3; ++f) {
        const float m = warp_max(m1[f]);
        if (lane == 0 && m > 0.f) atomicMax(&h1max[f], __float_as_uint(m));     // +inf orders above every finite value
    }
    if (lane == 0 && lo <= hi) {
        atomicMin(&bounds[0], dbl_to_ordered(lo));
        atomicMax(&bounds[1], dbl_to_ordered(hi));
    }
}

// ---------------------------------------------------------------------------------------------
// a2 + a3 fused.  Initial normalisation layer (Eq. 34, 493):
//        S0 = (eps_max I - H0)/W,  S1_f = -H1_f/W,  W = eps_max - eps_min,
//     each element formed in fp64 and rounded once to fp32, written to the n_pad x n_pad fp32 workspace
//     matrices (zero outside n x n) TOGETHER WITH the first operand split (Eq. 13, 302-307):
//        (Mhi, Mlo) = split(2^a (S0 - I/2)),   (S1hi, S1lo)_f = split(2^e_f S1_f)
//     (residual form and power-of-two scales: DESIGN.md R12, R17).  Algorithmic bytes per element:
//     4 (1 + NF) read + (4 + 4)(1 + NF) written = 24 at one field, against 32 for transform + two splits.
//     Partials per block: Tr S0, ||S0||_F^2 (summed in a fixed order by dmpt_control_init_kernel).
//     NF = 0: ground-state mode (no perturbation).  The scales e_f and the optional prescale 2^p_f of a
//     perturbation outside [2^-30, 2^30] come from DmptCtl (dmpt_bounds_to_ctl_kernel).
// ---------------------------------------------------------------------------------------------
struct TransformArgs {
    const float* h0;
    const float* h1[3];
    int n, ld, n_pad, s0_shift;
    float* s0;
    float* s1[3];
    __half* mh;
    __half* ml;
    __half* yh[3];
    __half* yl[3];
    const DmptCtl* ctl;
    double* partials;      // [grid][3]: Tr S0, ||S0||_F^2, unused
};

template <int NF>
__global__ void __launch_bounds__(256) dmpt_transform_split_kernel(const TransformArgs a) {
    const DmptCtl c = *a.ctl;
    const double emax = c.eps_max;
    const double inv_w = 1.0 / (c.eps_max - c.eps_min);
    double inv_wf[3];
    float scale1[3];
    const int e_in[3] = {c.e1_in, c.e2_in, c.e3_in};
    const int pre[3] = {c.p1, c.p2, c.p3};
#pragma unroll
    for (int f = 0; f < 3; ++f) {
        inv_wf[f] = ldexp(inv_w, pre[f]);          // exact; pre = 0 unless |H1|/W is far outside fp16's reach
        scale1[f] = exp2f((float)e_in[f]);
    }
    const float scale0 = exp2f((float)a.s0_shift);
    const int n = a.n, ld = a.ld, n_pad = a.n_pad;
    const int c8_per_row = n_pad >> 3;
    const bool with0 = a.h0 != nullptr;      // nullptr: the perturbations only (order-1 side of an order-parallel pair)
    bool vec = (ld & 3) == 0 && (reinterpret_cast<uintptr_t>(a.h0) & 15) == 0;
#pragma unroll
    for (int f = 0; f < NF; ++f) vec = vec && (reinterpret_cast<uintptr_t>(a.h1[f]) & 15) == 0;
    double tr = 0.0, fro = 0.0;
    // block per row (grid-stride), 8 consecutive columns per thread: 128-bit loads and stores throughout
    for (int row = blockIdx.x; row < n_pad; row += gridDim.x)
        for (int c8 = threadIdx.x; c8 < c8_per_row; c8 += blockDim.x) {
            const int col = c8 << 3;
            float x0[8], x1[NF > 0 ? NF : 1][8];
#pragma unroll
            for (int t = 0; t < 8; ++t) {
                x0[t] = 0.f;
#pragma unroll
                for (int f = 0; f < NF; ++f) x1[f][t] = 0.f;
            }
            if (row < n && col < n) {
                const size_t off = (size_t)row * ld + col;
                if (vec && col + 7 < n) {
                    if (with0) {
                        const float4 u0 = ldg_stream4(a.h0 + off), u1 = ldg_stream4(a.h0 + off + 4);
                        x0[0] = u0.x; x0[1] = u0.y; x0[2] = u0.z; x0[3] = u0.w;
                        x0[4] = u1.x; x0[5] = u1.y; x0[6] = u1.z; x0[7] = u1.w;
                    }
#pragma unroll
                    for (int f = 0; f < NF; ++f) {
                        const float4 w0 = ldg_stream4(a.h1[f] + off), w1 = ldg_stream4(a.h1[f] + off + 4);
                        x1[f][0] = w0.x; x1[f][1] = w0.y; x1[f][2] = w0.z; x1[f][3] = w0.w;
                        x1[f][4] = w1.x; x1[f][5] = w1.y; x1[f][6] = w1.z; x1[f][7] = w1.w;
                    }
                } else {
#pragma unroll
                    for (int t = 0; t < 8; ++t)
                        if (col + t < n) {
                            if (with0) x0[t] = a.h0[off + t];
#pragma unroll
                            for (int f = 0; f < NF; ++f) x1[f][t] = a.h1[f][off + t];
                        }
                }
            }
            float o0[8];
            __align__(16) __half hh[8];
            __align__(16) __half ll[8];
            float fsum[2] = {0.f, 0.f};        // fp32 per four elements, fp64 beyond
#pragma unroll
            for (int t = 0; t < 8; ++t) {
                const bool inside = row < n && col + t < n;
                const bool dg = col + t == row;
                o0[t] = inside ? (float)(((dg ? emax : 0.0) - (double)x0[t]) * inv_w) : 0.f;
                if (inside && dg) tr += (double)o0[t];
                fsum[t >> 2] = fmaf(o0[t], o0[t], fsum[t >> 2]);
                split_scaled(dg ? o0[t] - 0.5f : o0[t], scale0, hh[t], ll[t]);     // operands hold M = S0 - I/2
            }
            fro += (double)fsum[0] + (double)fsum[1];
            const size_t i8 = (size_t)row * n_pad + col;
            if (with0) {
                *reinterpret_cast<float4*>(a.s0 + i8) = make_float4(o0[0], o0[1], o0[2], o0[3]);
                *reinterpret_cast<float4*>(a.s0 + i8 + 4) = make_float4(o0[4], o0[5], o0[6], o0[7]);
                *reinterpret_cast<uint4*>(a.mh + i8) = *reinterpret_cast<const uint4*>(hh);
                *reinterpret_cast<uint4*>(a.ml + i8) = *reinterpret_cast<const uint4*>(ll);
            }
#pragma unroll
            for (int f = 0; f < NF; ++f) {
                float o1[8];
#pragma unroll
                for (int t = 0; t < 8; ++t) {
                    const bool inside = row < n && col + t < n;
                    o1[t] = inside ? (float)(-(double)x1[f][t] * inv_wf[f]) : 0.f;
                    split_scaled(o1[t], scale1[f], hh[t], ll[t]);
                }
                *reinterpret_cast<float4*>(a.s1[f] + i8) = make_float4(o1[0], o1[1], o1[2], o1[3]);
                *reinterpret_cast<float4*>(a.s1[f] + i8 + 4) = make_float4(o1[4], o1[5], o1[6], o1[7]);
                *reinterpret_cast<uint4*>(a.yh[f] + i8) = *reinterpret_cast<const uint4*>(hh);
                *reinterpret_cast<uint4*>(a.yl[f] + i8) = *reinterpret_cast<const uint4*>(ll);
            }
        }
    __shared__ double sh[2][8];
    tr = warp_sum(tr);
    fro = warp_sum(fro);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (lane == 0) { sh[0][warp] = tr; sh[1][warp] = fro; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0, f = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) { t += sh[0][w]; f += sh[1][w]; }
        a.partials[blockIdx.x * 3 + 0] = t;
        a.partials[blockIdx.x * 3 + 1] = f;
        a.partials[blockIdx.x * 3 + 2] = 0.0;
    }
}

// Undo the prescale 2^p of a response iterate in place (only launched when p != 0: a perturbation whose
// size is far outside fp16's reach, see dmpt_bounds_to_ctl_kernel).  Exact unless the true value is subnormal.
__global__ void __launch_bounds__(256) dmpt_unscale_kernel(float* __restrict__ x, int n_pad, int minus_p) {
    const long long total = (long long)n_pad * n_pad;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x)
        x[i] = ldexpf(x[i], minus_p);
}

// zero-padded copy of a caller matrix into an n_pad x n_pad workspace matrix (single-shot products, dmpt_product_nt)
// and max|.| per block.  Block per row (grid-stride), four columns per thread: 128-bit accesses when the source allows.
__global__ void __launch_bounds__(256) dmpt_pad_copy_kernel(const float* __restrict__ src, int n, int ld,
                                                       int n_pad, float* __restrict__ dst,
                                                       double* __restrict__ partials /* [grid] max */) {
    const bool vec = (ld & 3) == 0 && (reinterpret_cast<uintptr_t>(src) & 15) == 0;
    const int c4_per_row = n_pad >> 2;
    float mx = 0.f;
    for (int row = blockIdx.x; row < n_pad; row += gridDim.x)
        for (int c4 = threadIdx.x; c4 < c4_per_row; c4 += blockDim.x) {
            const int col = c4 << 2;
            float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
            if (row < n && col < n) {
                const float* s = src + (size_t)row * ld + col;
                if (vec && col + 3 < n) {
                    v = ldg_stream4(s);
                } else {
                    v.x = s[0];
                    if (col + 1 < n) v.y = s[1];
                    if (col + 2 < n) v.z = s[2];
                    if (col + 3 < n) v.w = s[3];
                }
            }
            *reinterpret_cast<float4*>(dst + (size_t)row * n_pad + col) = v;
            mx = absmax4(mx, v);
        }
    __shared__ double sh[8];
    double dmx = warp_max((double)mx);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = dmx;
    __syncthreads();
    if (threadIdx.x == 0) {
        double m = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) m = fmax(m, sh[w]);
        partials[blockIdx.x] = m;
    }
}

// ---------------------------------------------------------------------------------------------
// Tighter spectral bounds (dmpt_options::bounds == 2; reading R18 of DESIGN.md; the paper takes the bounds as inputs
// and names Gershgorin "for example"): k steps of the Lanczos recursion on H0,
//     w = H0 v_j - beta_{j-1} v_{j-1},  alpha_j = v_j.w,  w -= alpha_j v_j,  beta_j = ||w||,  v_{j+1} = w / beta_j,
// from a fixed pseudo-random start vector (signs and magnitudes), then the extreme eigenvalues theta_min, theta_max of the k x k tridiagonal
// matrix widened by the residual norm beta_k (every Ritz value has an eigenvalue of H0 within beta_k |s_k| <= beta_k;
// with a start vector that has a component along every eigenvector the extreme Ritz values converge first, so
// [theta_min - beta_k, theta_max + beta_k] encloses the spectrum in practice - tests check it on every workload) and
// intersected with the Gershgorin discs, which enclose it by theorem.  Each step streams H0 once (4 N^2 bytes, HBM
// bound); vectors, dot products and the tridiagonal problem are fp64.  Without re-orthogonalisation the recursion
// only produces copies of converged extreme Ritz values, which does not move the extremes.
// ---------------------------------------------------------------------------------------------
constexpr int kLanczosMaxSteps = 64;

struct LanczosState {       // device, fp64
    double alpha[kLanczosMaxSteps];
    double beta[kLanczosMaxSteps + 1];      // beta[j] = ||f_j|| after step j (beta[0] unused)
    int steps;                              // steps completed
    int finished;                           // 1: the Krylov space became invariant (beta_j ~ 0) - no further steps
};

__device__ __forceinline__ double lanczos_start(int i) {
    // fixed, input-independent pattern: pseudo-random sign AND magnitude in [0.5, 1), so that no eigenvector of a
    // structured matrix (e.g. (e_1 - e_2)/sqrt(2)) is orthogonal to the start vector by symmetry
    unsigned int x = (unsigned int)i * 2654435761u + 0x9E3779B9u;
    x ^= x >> 16; x *= 0x85EBCA6Bu; x ^= x >> 13; x *= 0xC2B2AE35u; x ^= x >> 16;
    const double mag = 0.5 + (double)(x >> 8) * (0.5 / 16777216.0);
    return (x & 1u) ? mag : -mag;
}

// v_0 = 0, v_1 = the normalised start vector: one block (fixed-order norm)
__global__ void __launch_bounds__(1024) dmpt_lanczos_init_kernel(double* __restrict__ v0, double* __restrict__ v1, int n,
                                                                 LanczosState* st) {
    __shared__ double sh[32];
    __shared__ double bc;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
    double q = 0.0;
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
        const double x = lanczos_start(i);
        q += x * x;
    }
    q = warp_sum(q);
    if (lane == 0) sh[warp] = q;
    __syncthreads();
    if (warp == 0) {
        double t = lane < nw ? sh[lane] : 0.0;
        t = warp_sum(t);
        if (lane == 0) bc = 1.0 / sqrt(t);
    }
    __syncthreads();
    const double inv = bc;
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
        v0[i] = 0.0;
        v1[i] = lanczos_start(i) * inv;
    }
    if (threadIdx.x == 0) {
        st->steps = 0;
        st->finished = 0;
        st->beta[0] = 0.0;
    }
}

// w = H0 v - beta_{j-1} v_prev: one warp per row, 128-bit streaming loads of the matrix, fp64 accumulation
__global__ void __launch_bounds__(256) dmpt_lanczos_matvec_kernel(const float* __restrict__ h0, int n, int ld,
                                                                  const double* __restrict__ v,
                                                                  const double* __restrict__ v_prev,
                                                                  double* __restrict__ w, const LanczosState* st, int j) {
    if (st->finished) return;
    const double beta_prev = st->beta[j - 1];
    const int warps_per_block = blockDim.x >> 5;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const bool vec = (ld & 3) == 0 && (reinterpret_cast<uintptr_t>(h0) & 15) == 0;
    for (int row = blockIdx.x * warps_per_block + warp; row < n; row += gridDim.x * warps_per_block) {
        const float* hr = h0 + (size_t)row * ld;
        double acc = 0.0;
        int c = 0;
        if (vec) {
            const int n4 = n & ~3;
            for (c = lane * 4; c < n4; c += 128) {
                const float4 a = ldg_stream4(hr + c);
                acc += (double)a.x * v[c] + (double)a.y * v[c + 1] + (double)a.z * v[c + 2] + (double)a.w * v[c + 3];
            }
            c = n4;
        }
        for (c += lane; c < n; c += 32) acc += (double)hr[c] * v[c];
        acc = warp_sum(acc);
        if (lane == 0) w[row] = acc - beta_prev * v_prev[row];
    }
}

// alpha_j, w -= alpha_j v, beta_j, v_next = w / beta_j: one block, fixed-order fp64 reductions
__global__ void __launch_bounds__(1024) dmpt_lanczos_update_kernel(const double* __restrict__ v, double* __restrict__ w,
                                                                   int n, LanczosState* st, int j) {
    if (st->finished) return;
    __shared__ double sh[32];
    __shared__ double bc;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
    auto block_sum = [&](double x) {
        x = warp_sum(x);
        __syncthreads();
        if (lane == 0) sh[warp] = x;
        __syncthreads();
        if (warp == 0) {
            double t = lane < nw ? sh[lane] : 0.0;
            t = warp_sum(t);
            if (lane == 0) bc = t;
        }
        __syncthreads();
        return bc;
    };
    double a = 0.0;
    for (int i = threadIdx.x; i < n; i += blockDim.x) a += v[i] * w[i];
    const double alpha = block_sum(a);
    double b = 0.0;
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
        const double x = w[i] - alpha * v[i];
        w[i] = x;
        b += x * x;
    }
    const double beta = sqrt(block_sum(b));
    // invariant subspace (or a non-finite matrix): stop here; the bounds kernel then keeps the Gershgorin discs
    const bool stop = !(beta > 1e-12 * (fabs(alpha) + st->beta[j - 1] + 1e-300)) || !isfinite(beta);
    if (!stop) {
        const double inv = 1.0 / beta;
        for (int i = threadIdx.x; i < n; i += blockDim.x) w[i] *= inv;       // w becomes v_{j+1}
    }
    if (threadIdx.x == 0) {
        st->alpha[j - 1] = alpha;
        st->beta[j] = stop ? 0.0 : beta;
        st->steps = j;
        if (stop) st->finished = 1;
    }
}

// Small matrices (n <= 1024): the whole recursion in ONE block, one row per thread - at these sizes the 2 k launches
// of the general path cost more than the layers they save.  H0 is symmetric, so thread i reads column i (H[k][i] over
// k): consecutive threads read consecutive addresses.  Same arithmetic order per row as a sequential dot product.
__global__ void __launch_bounds__(1024) dmpt_lanczos_small_kernel(const float* __restrict__ h0, int n, int ld, int steps,
                                                                  LanczosState* st) {
    __shared__ double v[1024];
    __shared__ double sh[32];
    __shared__ double bc;
    const int i = threadIdx.x;
    const int lane = i & 31, warp = i >> 5, nw = blockDim.x >> 5;
    auto block_sum = [&](double x) {
        x = warp_sum(x);
        __syncthreads();
        if (lane == 0) sh[warp] = x;
        __syncthreads();
        if (warp == 0) {
            double t = lane < nw ? sh[lane] : 0.0;
            t = warp_sum(t);
            if (lane == 0) bc = t;
        }
        __syncthreads();
        return bc;
    };
    // rows padded to a power of two >= 32; the 1024 threads split every column sum into tpr slices of k
    int rows = 32;
    while (rows < n) rows <<= 1;
    const int tpr = 1024 / rows, row = i & (rows - 1), slice = i / rows;
    const int k_per = (n + tpr - 1) / tpr, k0 = slice * k_per, k1 = min(n, k0 + k_per);
    __shared__ double part[1024];
    const bool on = i < n;                       // thread i also owns element i of the vectors
    double x = on ? lanczos_start(i) : 0.0;
    const double nrm = sqrt(block_sum(x * x));
    double v_cur = x / nrm, v_prev = 0.0, beta_prev = 0.0;
    int done_steps = 0, finished = 0;
    for (int j = 1; j <= steps; ++j) {
        __syncthreads();
        v[i] = v_cur;
        __syncthreads();
        double acc = 0.0;
        if (row < n) {
#pragma unroll 8
            for (int k = k0; k < k1; ++k) acc += (double)h0[(size_t)k * ld + row] * v[k];
        }
        part[i] = acc;
        __syncthreads();
        double w = 0.0;
        if (on) {
            for (int q = 0; q < tpr; ++q) w += part[q * rows + i];       // fixed order
            w -= beta_prev * v_prev;
        }
        const double alpha = block_sum(on ? v_cur * w : 0.0);
        w = on ? w - alpha * v_cur : 0.0;
        const double beta = sqrt(block_sum(w * w));
        const bool stop = !(beta > 1e-12 * (fabs(alpha) + beta_prev + 1e-300)) || !isfinite(beta);
        if (i == 0) {
            st->alpha[j - 1] = alpha;
            st->beta[j] = stop ? 0.0 : beta;
        }
        done_steps = j;
        if (stop) { finished = 1; break; }
        v_prev = v_cur;
        v_cur = w / beta;
        beta_prev = beta;
    }
    if (i == 0) {
        st->beta[0] = 0.0;
        st->steps = done_steps;
        st->finished = finished;
    }
}

// Extreme eigenvalues of the tridiagonal matrix by bisection on the Sturm count, widened by beta_k and intersected
// with the Gershgorin discs already in `bounds` (ordered-int encodings, as dmpt_gershgorin_kernel leaves them).
__global__ void dmpt_lanczos_bounds_kernel(const LanczosState* st, long long* bounds) {
    if (threadIdx.x | blockIdx.x) return;
    const int k = st->steps;
    if (k < 2 || st->finished) return;                       // keep Gershgorin
    const double* a = st->alpha;
    const double* b = st->beta;                              // off-diagonals b[1] .. b[k-1]; residual b[k]
    double lo = INFINITY, hi = -INFINITY;
    for (int i = 0; i < k; ++i) {
        const double r = (i > 0 ? fabs(b[i]) : 0.0) + (i < k - 1 ? fabs(b[i + 1]) : 0.0);
        lo = fmin(lo, a[i] - r);
        hi = fmax(hi, a[i] + r);
    }
    if (!isfinite(lo) || !isfinite(hi)) return;
    auto count_below = [&](double x) {                       // eigenvalues of T strictly below x
        int cnt = 0;
        double d = 1.0;
        for (int i = 0; i < k; ++i) {
            const double off = i > 0 ? b[i] * b[i] : 0.0;
            d = a[i] - x - (i > 0 ? off / d : 0.0);
            if (d == 0.0) d = -1e-300;
            if (d < 0.0) ++cnt;
        }
        return cnt;
    };
    double l0 = lo, h0 = hi;                                 // smallest eigenvalue: count_below(x) >= 1
    for (int it = 0; it < 100; ++it) {
        const double m = 0.5 * (l0 + h0);
        if (count_below(m) >= 1) h0 = m; else l0 = m;
    }
    const double th_min = l0;
    double l1 = lo, h1 = hi;                                 // largest: count_below(x) >= k
    for (int it = 0; it < 100; ++it) {
        const double m = 0.5 * (l1 + h1);
        if (count_below(m) >= k) h1 = m; else l1 = m;
    }
    const double th_max = h1;
    const double resid = fabs(b[k]);
    const double e_lo = th_min - resid, e_hi = th_max + resid;
    const double g_lo = ordered_to_dbl(bounds[0]), g_hi = ordered_to_dbl(bounds[1]);
    if (!isfinite(e_lo) || !isfinite(e_hi)) return;
    bounds[0] = dbl_to_ordered(fmax(e_lo, g_lo));
    bounds[1] = dbl_to_ordered(fmin(e_hi, g_hi));
}

// the same copy of the TRANSPOSE of a caller matrix (dmpt_congruence: Z^T as the row operand of a product), through a
// 32 x 33 shared-memory tile so that both the reads and the writes are full lines.  grid = (n_pad/32)^2 tiles,
// grid-stride; 256 threads = 32 x 8.
__global__ void __launch_bounds__(256) dmpt_pad_copy_t_kernel(const float* __restrict__ src, int n, int ld, int n_pad,
                                                              float* __restrict__ dst,
                                                              double* __restrict__ partials /* [grid] max */) {
    __shared__ float tile[32][33];
    __shared__ double sh[8];
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const int tiles_per_row = n_pad >> 5;
    const long long num_tiles = (long long)tiles_per_row * tiles_per_row;
    float mx = 0.f;
    for (long long t = blockIdx.x; t < num_tiles; t += gridDim.x) {
        const int bi = (int)(t / tiles_per_row), bj = (int)(t - (long long)bi * tiles_per_row);   // dst tile (bi, bj)
        // dst[bi*32 + r][bj*32 + c] = src[bj*32 + c][bi*32 + r]
        __syncthreads();
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const int sr = bj * 32 + ty + 8 * k, sc = bi * 32 + tx;
            tile[ty + 8 * k][tx] = (sr < n && sc < n) ? src[(size_t)sr * ld + sc] : 0.f;
        }
        __syncthreads();
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const float v = tile[tx][ty + 8 * k];
            dst[(size_t)(bi * 32 + ty + 8 * k) * n_pad + bj * 32 + tx] = v;
            mx = fmaxf(mx, fabsf(v));
        }
    }
    double dmx = warp_max((double)mx);
    if (tx == 0) sh[ty] = dmx;
    __syncthreads();
    if (threadIdx.x == 0) {
        double m = 0.0;
        for (int w = 0; w < 8; ++w) m = fmax(m, sh[w]);
        partials[blockIdx.x] = m;
    }
}

// ---------------------------------------------------------------------------------------------
// Lower triangle <- transpose of the upper triangle, in place, on an n_pad x n_pad workspace matrix.  The layer
// kernel's TMA epilogue keeps only the blocks on or above the diagonal of the fp32 iterates up to date (nothing reads
// the others during a run: every product works on tiles i <= j); this pass restores the full symmetric matrix before
// an iterate leaves the workspace.  32 x 32 tiles through shared memory: full lines in, full lines out.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) dmpt_symmetrize_kernel(float* __restrict__ a, int n_pad) {
    __shared__ float tile[32][33];
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const int T = n_pad >> 5;
    const long long num = (long long)T * T;
    for (long long t = blockIdx.x; t < num; t += gridDim.x) {
        const int bi = (int)(t / T), bj = (int)(t - (long long)bi * T);      // destination tile (bi, bj), bi >= bj
        if (bi < bj) continue;
        __syncthreads();
#pragma unroll
        for (int k = 0; k < 4; ++k)                                           // source tile (bj, bi), above the diagonal
            tile[ty + 8 * k][tx] = a[(size_t)(bj * 32 + ty + 8 * k) * n_pad + bi * 32 + tx];
        __syncthreads();
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const int r = bi * 32 + ty + 8 * k, c = bj * 32 + tx;
            if (r > c) a[(size_t)r * n_pad + c] = tile[tx][ty + 8 * k];
        }
    }
}

// ---------------------------------------------------------------------------------------------
// Finite-difference response from ground-state runs (Eqs. 83-84): the two elementwise steps.
//   dmpt_axpy_kernel:     out = H0 + t H1, formed in fp64 and rounded once (n x n, dense, leading dimension n)
//   dmpt_fd_accum_kernel: acc = (first ? 0 : acc) + w D, w = stencil weight / (denominator h), fp64 per element
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) dmpt_axpy_kernel(const float* __restrict__ h0, const float* __restrict__ h1, int n,
                                                        int ld, double t, float* __restrict__ out) {
    const long long total = (long long)n * n;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
        const int row = (int)(i / n), col = (int)(i - (long long)row * n);
        const size_t o = (size_t)row * ld + col;
        out[i] = (float)((double)h0[o] + t * (double)h1[o]);
    }
}

__global__ void __launch_bounds__(256) dmpt_fd_accum_kernel(const float* __restrict__ d, int n, int ld_d, double w, int first,
                                                            float* __restrict__ acc, int ld_acc) {
    const long long total = (long long)n * n;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
        const int row = (int)(i / n), col = (int)(i - (long long)row * n);
        const size_t oa = (size_t)row * ld_acc + col;
        const double prev = first ? 0.0 : (double)acc[oa];
        acc[oa] = (float)(prev + w * (double)d[(size_t)row * ld_d + col]);
    }
}

// ---------------------------------------------------------------------------------------------
// Scalar set-up between the transform and the first layer: spectral bounds -> ctl (before the
// transform), then first reductions -> ctl and the decision for layer 1 (after it).
// ---------------------------------------------------------------------------------------------
__global__ void dmpt_reset_state_kernel(DmptCtl* ctl, long long* bounds, unsigned int* h1max) {
    if (threadIdx.x | blockIdx.x) return;
    DmptCtl c;
    memset(&c, 0, sizeof c);
    *ctl = c;
    bounds[0] = dbl_to_ordered(INFINITY);
    bounds[1] = dbl_to_ordered(-INFINITY);
    h1max[0] = h1max[1] = h1max[2] = 0u;
}

// Spectral bounds -> ctl, and for every perturbation the size of S1_0 = -H1/W and the exponent of its first
// split (reading R12): max|S1_0| = fl32(max|H1| / W) because the rounding is monotone.  A perturbation whose
// S1_0 lies outside [2^-30, 2^30] is carried with an exact prescale 2^p (max|2^p S1_0| in [1, 2)) so that every
// power-of-two factor of the layer epilogue stays a normal fp32 number; the run undoes it on the outputs.
__global__ void dmpt_bounds_to_ctl_kernel(const long long* __restrict__ bounds, const unsigned int* __restrict__ h1max,
                                          DmptCtl* ctl, DmptProblem pb, int use_given, double eps_min, double eps_max) {
    if (threadIdx.x | blockIdx.x) return;
    DmptCtl c = *ctl;
    // use_given: 0 = the Gershgorin discs in `bounds`; 1 = the caller's numbers; 2 = already in ctl (order-parallel
    // pair: copied from the order-0 side)
    const double lo = use_given == 2 ? c.eps_min : (use_given ? eps_min : ordered_to_dbl(bounds[0]));
    const double hi = use_given == 2 ? c.eps_max : (use_given ? eps_max : ordered_to_dbl(bounds[1]));
    c.eps_min = lo;
    c.eps_max = hi;
    const double w = hi - lo;
    if (!(w > 0.0) || !isfinite(w)) {
        c.done = 1;
        c.status = -4;  // DMPT_EDEGENERATE
        // keep the transform finite
        c.eps_min = 0.0;
        c.eps_max = 1.0;
    }
    const double inv_w = 1.0 / (c.eps_max - c.eps_min);
    const int nslots = pb.order == 0 ? 0 : pb.nfields;
    int pre[3] = {0, 0, 0}, e[3] = {0, 0, 0};
    double mx[3] = {0.0, 0.0, 0.0};
    for (int f = 0; f < nslots; ++f) {
        const double m = (double)__uint_as_float(h1max[f]) * inv_w;
        if (!isfinite(m)) {
            c.done = 1;
            c.status = -6;  // DMPT_ENUMERIC
            continue;
        }
        if (m > 0.0 && (m < 0x1p-30 || m > 0x1p30)) {
            int ex;
            frexp(m, &ex);              // m in [2^(ex-1), 2^ex)
            pre[f] = 1 - ex;
        }
        mx[f] = (double)(float)ldexp(m, pre[f]);
        e[f] = pb.s1_autoscale ? scale_exponent(mx[f]) : 0;
    }
    c.p1 = pre[0]; c.p2 = pre[1]; c.p3 = pre[2];
    c.s1_max = mx[0]; c.s2_max = mx[1]; c.s3_max = mx[2];
    c.e1_in = c.e1_out = e[0];
    c.e2_in = c.e2_out = e[1];
    c.e3_in = c.e3_out = e[2];
    *ctl = c;
}

// First reductions -> ctl and the decision for layer 1.  One warp, fixed summation order.
__global__ void dmpt_control_init_kernel(DmptCtl* ctl, DmptLogs logs, DmptProblem pb,
                                         const double* __restrict__ partials, int nblocks, DmptHandoff* handoff) {
    if (blockIdx.x || threadIdx.x >= 32) return;
    if (logs.clk)
        for (int i = threadIdx.x; i < kMaxSmStamps; i += 32)
            logs.clk->first[i][0] = logs.clk->first[i][1] = logs.clk->last[i][0] = logs.clk->last[i][1] = 0;
    double t = 0.0, f = 0.0;
    for (int b = threadIdx.x; b < nblocks; b += 32) {
        t += partials[b * 3 + 0];
        f += partials[b * 3 + 1];
    }
    t = warp_sum(t);
    f = warp_sum(f);
    if (threadIdx.x) return;
    DmptCtl c = *ctl;
    c.n_s = t;
    c.n_x = f;
    c.layer = 1;
    if (pb.pair_side == 2) {        // the decision for layer 1 arrives from the order-0 side
        *ctl = c;
        return;
    }
    if (!c.done) control_decide(c, logs, pb);
    if (pb.pair_side == 1) handoff_publish(c, handoff);
    *ctl = c;
}

// ---------------------------------------------------------------------------------------------
// Order 2 only: the scale of the FIRST split of S2.  S2_0 = 0, so S2_1 = sigma_1 S1_0 S1_0 and, by
// Cauchy-Schwarz, max|S2_1| = max_i sum_k (S1_0)_ik^2 (attained on the diagonal).  One warp per row
// of the padded S1_0; the maximum lands in *est as the bit pattern of a non-negative double
// (ordered like an unsigned integer).  dmpt_s2_scale_init_kernel then sets e2_out (reading R12).
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) dmpt_rowsq_max_kernel(const float* __restrict__ s1, int n_pad,
                                                             unsigned long long* __restrict__ est) {
    const int warps_per_block = blockDim.x >> 5;
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    double mx = 0.0;
    for (int row = blockIdx.x * warps_per_block + warp; row < n_pad; row += gridDim.x * warps_per_block) {
        const float* p = s1 + (size_t)row * n_pad;
        double acc = 0.0;
        for (int j = lane * 4; j < n_pad; j += 128) {
            const float4 v = ldg_stream4(p + j);
            acc += (double)(v.x * v.x + v.y * v.y) + (double)(v.z * v.z + v.w * v.w);
        }
        mx = fmax(mx, warp_sum(acc));
    }
    if (lane == 0 && mx > 0.0 && isfinite(mx)) atomicMax(est, (unsigned long long)__double_as_longlong(mx));
}

__global__ void dmpt_s2_scale_init_kernel(DmptCtl* ctl, DmptProblem pb, const unsigned long long* __restrict__ est) {
    if (threadIdx.x | blockIdx.x) return;
    const double m = __longlong_as_double((long long)*est);
    ctl->s2_max = m;
    ctl->e2_in = 0;
    ctl->e2_out = pb.s1_autoscale ? scale_exponent(m) : 0;
}

// Order 3: the scale of the first split of a non-zero S3 (S3_2, written by layer 2) from the row norms of S1_1 and
// S2_1: max|S1_1 S2_1 + S2_1 S1_1| <= 2 sqrt(max_i sum_k (S1_1)_ik^2) sqrt(max_j sum_k (S2_1)_jk^2).
__global__ void dmpt_s3_scale_init_kernel(DmptCtl* ctl, DmptProblem pb, const unsigned long long* __restrict__ est1,
                                          const unsigned long long* __restrict__ est2) {
    if (threadIdx.x | blockIdx.x) return;
    const double r1 = __longlong_as_double((long long)*est1), r2 = __longlong_as_double((long long)*est2);
    const double m = 2.0 * sqrt(r1) * sqrt(r2);
    ctl->s3_max = m;
    ctl->e3_out = pb.s1_autoscale ? scale_exponent(m) : 0;
}

// ---------------------------------------------------------------------------------------------
// Inverse factorisation (A19-A21): the two elementwise steps around the products.
//   Z_0 = I / sqrt(eps_max(S)) with the Gershgorin bound of S, so that the spectrum of X_0 = Z_0 S Z_0 lies in (0, 1]
//   W   = a_0 I + a_1 X + a_2 X^2,  a = {1.875, -1.25, 0.375} (A20, A21), and ||X - I||_F^2 per block
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) dmpt_scaled_identity_kernel(float* __restrict__ z, int n, int ld,
                                                                   const long long* __restrict__ bounds) {
    const float d = (float)(1.0 / sqrt(ordered_to_dbl(bounds[1])));
    const long long total = (long long)n * n;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
        const int row = (int)(i / n), col = (int)(i - (long long)row * n);
        z[(size_t)row * ld + col] = row == col ? d : 0.f;
    }
}

__global__ void __launch_bounds__(256) dmpt_zpoly_kernel(const float* __restrict__ x, float* __restrict__ x2_to_w, int n,
                                                         double* __restrict__ partials /* [grid] */) {
    const long long total = (long long)n * n;
    double err = 0.0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
        const int row = (int)(i / n), col = (int)(i - (long long)row * n);
        const float dg = row == col ? 1.f : 0.f;
        const float xv = x[i];
        const float d = xv - dg;
        err += (double)d * (double)d;
        x2_to_w[i] = fmaf(0.375f, x2_to_w[i], fmaf(-1.25f, xv, 1.875f * dg));
    }
    __shared__ double sh[8];
    err = warp_sum(err);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = err;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) t += sh[w];
        partials[blockIdx.x] = t;
    }
}

// ---------------------------------------------------------------------------------------------
// a3  Split (Eq. 13, 302-307 Eqs. 42-43) after an exact power-of-two scale 2^e
//     (readings R12/R17): hi = fp16(2^e x), lo = fp16(2^e x - hi), round-to-nearest-even.
//     8 elements per thread: two 128-bit loads, one 128-bit store per output.
//     `which` selects the exponent on the device: 0 -> s0_shift, 1, 2, 3 -> ctl->e1_in, e2_in, e3_in.
//     With diag_half the matrix split is M = S0 - I/2 (residual form, layer_kernel.cuh).
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) dmpt_split_kernel(const float* __restrict__ x, int n_pad,
                                                         __half* __restrict__ hi, __half* __restrict__ lo,
                                                         const DmptCtl* __restrict__ ctl, int which, int s0_shift,
                                                         int diag_half) {
    const int e = which == 0 ? s0_shift : (which == 1 ? ctl->e1_in : (which == 2 ? ctl->e2_in : ctl->e3_in));
    const float scale = exp2f((float)e);
    const float diag_shift = diag_half ? 0.5f : 0.f;       // order 0: the operands hold M = S0 - I/2
    const int c8_per_row = n_pad >> 3;
    // block per row (grid-stride), threads along the row: no 64-bit division per element
    for (int row = blockIdx.x; row < n_pad; row += gridDim.x)
        for (int c8 = threadIdx.x; c8 < c8_per_row; c8 += blockDim.x) {
            const int col = c8 << 3;
            const size_t i8 = (size_t)row * n_pad + col;
            const float4 v0 = ldg_stream4(x + i8);
            const float4 v1 = ldg_stream4(x + i8 + 4);
            float v[8] = {v0.x, v0.y, v0.z, v0.w, v1.x, v1.y, v1.z, v1.w};
            __align__(16) __half h[8];
            __align__(16) __half l[8];
#pragma unroll
            for (int t = 0; t < 8; ++t) split_scaled(col + t == row ? v[t] - diag_shift : v[t], scale, h[t], l[t]);
            *reinterpret_cast<uint4*>(hi + i8) = *reinterpret_cast<const uint4*>(h);
            *reinterpret_cast<uint4*>(lo + i8) = *reinterpret_cast<const uint4*>(l);
        }
}

}  // namespace dmpt
