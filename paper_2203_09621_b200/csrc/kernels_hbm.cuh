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

// ---------------------------------------------------------------------------------------------
// a1  Gershgorin discs: one warp per row, shuffle reduction of sum_j |H0_ij|,
//     eps_min = min_i (H0_ii - r_i), eps_max = max_i (H0_ii + r_i), r_i = sum_{j != i} |H0_ij|.
//     bounds[0], bounds[1]: ordered-int encodings, initialised to +inf / -inf by the host.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) dmpt_gershgorin_kernel(const float* __restrict__ h0, int n, int ld,
                                                         long long* __restrict__ bounds) {
    const int warps_per_block = blockDim.x >> 5;
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    double lo = INFINITY, hi = -INFINITY;
    const bool vec = ((ld & 3) == 0) && ((reinterpret_cast<uintptr_t>(h0) & 15) == 0);
    for (int row = blockIdx.x * warps_per_block + warp; row < n; row += gridDim.x * warps_per_block) {
        const float* p = h0 + (size_t)row * ld;
        float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f;
        int j = 0;
        if (vec) {
            const int n4 = n & ~3;
            for (j = lane * 4; j < n4; j += 128) {
                float4 v = ldg_stream4(p + j);
                a0 += fabsf(v.x); a1 += fabsf(v.y); a2 += fabsf(v.z); a3 += fabsf(v.w);
            }
            j = n4;
        }
        for (j += lane; j < n; j += 32) a0 += fabsf(p[j]);
        double s = warp_sum((double)a0 + (double)a1 + (double)a2 + (double)a3);
        const double d = (double)p[row];
        const double r = s - fabs(d);
        lo = fmin(lo, d - r);
        hi = fmax(hi, d + r);
    }
    if (lane == 0 && lo <= hi) {
        atomicMin(&bounds[0], dbl_to_ordered(lo));
        atomicMax(&bounds[1], dbl_to_ordered(hi));
    }
}

// ---------------------------------------------------------------------------------------------
// a2  Initial normalisation layer (Eq. 34, 493):
//        S0 = (eps_max I - H0)/W,  S1 = -H1/W,  W = eps_max - eps_min,
//     written to n_pad x n_pad fp32 workspace matrices (zero outside n x n), together with the
//     first reductions: Tr S0, ||S0||_F^2, max|S1| as per-block partials (summed in a fixed order
//     by dmpt_control_init_kernel).  Each element is formed in fp64 and rounded once to fp32.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) dmpt_transform_kernel(const float* __restrict__ h0,
                                                        const float* __restrict__ h1, int n, int ld,
                                                        int n_pad, float* __restrict__ s0,
                                                        float* __restrict__ s1,
                                                        const DmptCtl* __restrict__ ctl,
                                                        double* __restrict__ partials /* [grid][3] */) {
    const double emax = ctl->eps_max;
    const double inv_w = 1.0 / (ctl->eps_max - ctl->eps_min);
    const int q_per_row = n_pad >> 2;
    const bool with_h1 = h1 != nullptr;        // order 0 (ground state only): S1 = 0
    const bool vec = ((ld & 3) == 0) && ((reinterpret_cast<uintptr_t>(h0) & 15) == 0) &&
                     ((reinterpret_cast<uintptr_t>(h1) & 15) == 0);
    double tr = 0.0, fro = 0.0;
    float mx = 0.f;
    // block per row (grid-stride), threads along the row: no 64-bit division per element
    for (int row = blockIdx.x; row < n_pad; row += gridDim.x)
    for (int qc = threadIdx.x; qc < q_per_row; qc += blockDim.x) {
        const int col = qc << 2;
        float a[4] = {0.f, 0.f, 0.f, 0.f}, b[4] = {0.f, 0.f, 0.f, 0.f};
        if (row < n) {
            if (vec && col + 3 < n) {
                float4 va = ldg_stream4(h0 + (size_t)row * ld + col);
                float4 vb = with_h1 ? ldg_stream4(h1 + (size_t)row * ld + col) : make_float4(0.f, 0.f, 0.f, 0.f);
                a[0] = va.x; a[1] = va.y; a[2] = va.z; a[3] = va.w;
                b[0] = vb.x; b[1] = vb.y; b[2] = vb.z; b[3] = vb.w;
            } else {
#pragma unroll
                for (int t = 0; t < 4; ++t)
                    if (col + t < n) {
                        a[t] = h0[(size_t)row * ld + col + t];
                        b[t] = with_h1 ? h1[(size_t)row * ld + col + t] : 0.f;
                    }
            }
        }
        float o0[4], o1[4];
        float fsum = 0.f;
#pragma unroll
        for (int t = 0; t < 4; ++t) {
            const bool inside = row < n && col + t < n;
            const double diag = (inside && col + t == row) ? emax : 0.0;
            o0[t] = inside ? (float)((diag - (double)a[t]) * inv_w) : 0.f;
            o1[t] = inside ? (float)(-(double)b[t] * inv_w) : 0.f;
            if (inside && col + t == row) tr += (double)o0[t];
            fsum = fmaf(o0[t], o0[t], fsum);
            mx = fmaxf(mx, fabsf(o1[t]));
        }
        fro += (double)fsum;
        *reinterpret_cast<float4*>(s0 + (size_t)row * n_pad + col) = make_float4(o0[0], o0[1], o0[2], o0[3]);
        *reinterpret_cast<float4*>(s1 + (size_t)row * n_pad + col) = make_float4(o1[0], o1[1], o1[2], o1[3]);
    }
    __shared__ double sh[3][8];
    tr = warp_sum(tr);
    fro = warp_sum(fro);
    double dmx = warp_max((double)mx);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (lane == 0) { sh[0][warp] = tr; sh[1][warp] = fro; sh[2][warp] = dmx; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0, f = 0.0, m = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) { t += sh[0][w]; f += sh[1][w]; m = fmax(m, sh[2][w]); }
        partials[blockIdx.x * 3 + 0] = t;
        partials[blockIdx.x * 3 + 1] = f;
        partials[blockIdx.x * 3 + 2] = m;
    }
}

// zero-padded copy of a caller matrix into an n_pad x n_pad workspace matrix (dmpt_layer_products)
__global__ void __launch_bounds__(256) dmpt_pad_copy_kernel(const float* __restrict__ src, int n, int ld,
                                                       int n_pad, float* __restrict__ dst,
                                                       double* __restrict__ partials /* [grid] max */) {
    const long long total = (long long)n_pad * n_pad;
    float mx = 0.f;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total;
         i += (long long)gridDim.x * blockDim.x) {
        const int row = (int)(i / n_pad), col = (int)(i - (long long)row * n_pad);
        const float v = (row < n && col < n) ? src[(size_t)row * ld + col] : 0.f;
        dst[i] = v;
        mx = fmaxf(mx, fabsf(v));
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
// Scalar set-up between the transform and the first layer: spectral bounds -> ctl (before the
// transform), then first reductions -> ctl and the decision for layer 1 (after it).
// ---------------------------------------------------------------------------------------------
__global__ void dmpt_reset_state_kernel(DmptCtl* ctl, long long* bounds) {
    if (threadIdx.x | blockIdx.x) return;
    DmptCtl c;
    memset(&c, 0, sizeof c);
    *ctl = c;
    bounds[0] = dbl_to_ordered(INFINITY);
    bounds[1] = dbl_to_ordered(-INFINITY);
}

__global__ void dmpt_bounds_to_ctl_kernel(const long long* __restrict__ bounds, DmptCtl* ctl, int use_given,
                                     double eps_min, double eps_max) {
    if (threadIdx.x | blockIdx.x) return;
    const double lo = use_given ? eps_min : ordered_to_dbl(bounds[0]);
    const double hi = use_given ? eps_max : ordered_to_dbl(bounds[1]);
    ctl->eps_min = lo;
    ctl->eps_max = hi;
    const double w = hi - lo;
    if (!(w > 0.0) || !isfinite(w)) {
        ctl->done = 1;
        ctl->status = -4;  // DMPT_EDEGENERATE
        // keep the transform finite
        ctl->eps_min = 0.0;
        ctl->eps_max = 1.0;
    }
}

__global__ void dmpt_control_init_kernel(DmptCtl* ctl, DmptLogs logs, DmptProblem pb,
                                    const double* __restrict__ partials, int nblocks) {
    if (threadIdx.x | blockIdx.x) return;
    DmptCtl c = *ctl;
    double t = 0.0, f = 0.0, m = 0.0;
    for (int b = 0; b < nblocks; ++b) {
        t += partials[b * 3 + 0];
        f += partials[b * 3 + 1];
        m = fmax(m, partials[b * 3 + 2]);
    }
    c.n_s = t;
    c.n_x = f;
    c.s1_max = m;
    c.e1_in = c.e1_out = pb.s1_autoscale ? scale_exponent(m) : 0;
    c.e2_in = c.e2_out = 0;
    c.layer = 1;
    if (!c.done) control_decide(c, logs, pb);
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

// Multi-field runs: first scale of response slot 2 or 3 from max|S1_0| of that field (the third of the
// per-block partials the transform kernel wrote for it).
__global__ void dmpt_field_init_kernel(DmptCtl* ctl, DmptProblem pb, const double* __restrict__ partials, int nblocks,
                                       int slot) {
    if (threadIdx.x | blockIdx.x) return;
    double m = 0.0;
    for (int b = 0; b < nblocks; ++b) m = fmax(m, partials[b * 3 + 2]);
    const int e = pb.s1_autoscale ? scale_exponent(m) : 0;
    if (slot == 2) { ctl->s2_max = m; ctl->e2_in = ctl->e2_out = e; }
    else { ctl->s3_max = m; ctl->e3_in = ctl->e3_out = e; }
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
__device__ __forceinline__ void split_scaled(float x, float scale, __half& hi, __half& lo) {
    const float t = x * scale;              // exact: scale is a power of two (barring overflow)
    hi = __float2half_rn(t);
    lo = __float2half_rn(t - __half2float(hi));
}

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
