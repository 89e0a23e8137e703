// One deep layer of DNN-SP2-PT in ONE launch (steps a4-a8 of DESIGN.md):
//
//   X0 = S0^2               = hi0.hi0 + hi0.lo0 + lo0.hi0                  PAPER.md:124-136 (Eqs. 14-16)
//   X1 = S0 S1 + S1 S0      = sum of the 3 dual-half terms of each product PAPER.md:309-329 (Eqs. 44-46)
//   S0 <- sigma X0 + (1 - sigma) S0,  S1 <- sigma X1 + (1 - sigma) S1      PAPER.md:182, 193 (Eqs. 23, 25)
//   re-split of the new iterates to (hi, lo) fp16                          PAPER.md:120 (Eq. 13)
//   Tr S0, ||S0||_F^2, ||S0 - X0||_F^2, ||S1 - X1||_F^2, max|S1|
//   Algorithms 2 and 3 + the decision for the next layer (last CTA)
//
// Design (sm_100a).  All iterates are exactly symmetric, so C[i,j] = sum_k A[i,k] B[j,k]: both
// operands of every product are K-major row panels of the same fp16 matrices ("TN" GEMM, the
// natural TMA/UMMA layout), and only output tiles on or above the diagonal are computed; each
// is stored twice (direct and mirrored), which keeps the iterates bit-symmetric.  A tile of X0
// and the matching tile of X1 are accumulated side by side in TMEM from the SAME eight operand
// tiles per k-block (S0hi, S0lo, S1hi, S1lo for row panel I and for row panel J): 9 MMAs per 8
// tiles loaded, against 1 per 2 for a plain GEMM.  Executed tensor work per layer is
// 4.5 N^3 FMA (3 N^3 once S0 froze) against the paper's 5 N^3 (3 N^3).
//
// Warp roles: warp 0 TMA producer, warp 1 MMA issuer (one elected lane) and TMEM owner,
// warps 2-5 epilogue (one TMEM lane quadrant each).  TMEM holds two accumulator stages
// (2 x [X0 | X1] x 128 columns) so the epilogue of tile t overlaps the MMAs of tile t+1.
#pragma once
#include <cuda_fp16.h>

#include "control.cuh"
#include "kernels_hbm.cuh"
#include "ptx.cuh"

namespace dmpt {

constexpr int kTile = 128;                 // output tile edge (rows of panel I x rows of panel J)
constexpr int kBK = 32;                    // fp16 per k-block: 64-byte rows, SWIZZLE_64B
constexpr int kRowBytes = kBK * 2;
constexpr int kStages = 3;
constexpr int kOpBytes = kTile * kRowBytes;          // 8 KiB per operand tile
constexpr int kOpsPerStage = 8;
constexpr int kStageBytes = kOpBytes * kOpsPerStage; // 64 KiB
constexpr int kAccStages = 2;
constexpr int kTmemCols = 512;
constexpr int kNumThreads = 192;
constexpr int kEpiWarp0 = 2;
constexpr int kNumEpiWarps = 4;
constexpr int kSmemBytes = kStages * kStageBytes + 1024 /* alignment slack */ + 256 /* barriers */;

// operand slots inside a stage
enum Op : int { A0H = 0, A0L = 1, A1H = 2, A1L = 3, B0H = 4, B0L = 5, B1H = 6, B1L = 7 };

struct LayerParams {
    CUtensorMap maps[2][4];     // [buffer][S0hi, S0lo, S1hi, S1lo], box = kBK x kTile, SWIZZLE_64B
    float* s0;                  // fp32 S0, updated in place, ld = n_pad
    float* s1[2];               // fp32 S1, ping-pong
    __half* h[2][4];            // fp16 operand matrices the epilogue writes, same order as maps
    const uint32_t* tiles;      // (I | J << 16), I <= J, in launch order
    int num_tiles;
    int n_pad;
    DmptCtl* ctl;
    DmptLogs logs;
    DmptProblem pb;
    double* partials;           // [gridDim.x][kNumEpiWarps][RED_COUNT]
};

__device__ __forceinline__ void st_f4(float* p, float a, float b, float c, float d) {
    *reinterpret_cast<float4*>(p) = make_float4(a, b, c, d);
}
__device__ __forceinline__ uint32_t pack2(__half a, __half b) {
    return (uint32_t)__half_as_ushort(a) | ((uint32_t)__half_as_ushort(b) << 16);
}
// 32 fp16 of one row (packed two per register) -> four 128-bit stores
__device__ __forceinline__ void st_h32(__half* p, const uint32_t (&w)[16]) {
#pragma unroll
    for (int j = 0; j < 16; j += 4)
        *reinterpret_cast<uint4*>(p + 2 * j) = make_uint4(w[j], w[j + 1], w[j + 2], w[j + 3]);
}

__global__ void __launch_bounds__(kNumThreads, 1)
dmpt_layer_kernel(const __grid_constant__ LayerParams p) {
    // ---- the decision for this layer, taken by the previous launch
    const DmptCtl c = *p.ctl;
    if (c.done) return;

    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t bar_base = smem_base + kStages * kStageBytes;
    auto full_bar = [&](int s) { return bar_base + 8u * s; };
    auto empty_bar = [&](int s) { return bar_base + 8u * (kStages + s); };
    auto tfull_bar = [&](int s) { return bar_base + 8u * (2 * kStages + s); };
    auto tempty_bar = [&](int s) { return bar_base + 8u * (2 * kStages + kAccStages + s); };
    const uint32_t tmem_slot = bar_base + 8u * (2 * kStages + 2 * kAccStages);
    uint8_t* smem_gen = smem_raw + (smem_base - smem_u32(smem_raw));
    volatile uint32_t* tmem_slot_ptr =
        reinterpret_cast<volatile uint32_t*>(smem_gen + kStages * kStageBytes + 8 * (2 * kStages + 2 * kAccStages));

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;
    const int num_kb = p.n_pad / kBK;
    const bool with_x0 = c.mode0 != MODE_FROZEN;

    if (warp == 0 && lane == 0) {
        for (int m = 0; m < 4; ++m) {
            prefetch_tensormap(&p.maps[c.s0_buf][m]);
            prefetch_tensormap(&p.maps[c.s1_buf][m]);
        }
        for (int s = 0; s < kStages; ++s) {
            mbar_init(full_bar(s), 1);
            mbar_init(empty_bar(s), 1);
        }
        for (int s = 0; s < kAccStages; ++s) {
            mbar_init(tfull_bar(s), 1);
            mbar_init(tempty_bar(s), kNumEpiWarps);
        }
        fence_mbar_init();
    }
    if (warp == 1) {
        tmem_alloc<1>(tmem_slot, kTmemCols);
        tmem_relinquish<1>();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_ptr;

    if (warp == 0) {
        // =========================== TMA producer ===========================
        if (lane == 0) {
            const CUtensorMap* m0h = &p.maps[c.s0_buf][0];
            const CUtensorMap* m0l = &p.maps[c.s0_buf][1];
            const CUtensorMap* m1h = &p.maps[c.s1_buf][2];
            const CUtensorMap* m1l = &p.maps[c.s1_buf][3];
            int stage = 0;
            uint32_t phase = 0;
            for (int t = blockIdx.x; t < p.num_tiles; t += gridDim.x) {
                const uint32_t tl = p.tiles[t];
                const int row_i = (int)(tl & 0xFFFF) * kTile, row_j = (int)(tl >> 16) * kTile;
                for (int kb = 0; kb < num_kb; ++kb) {
                    mbar_wait(empty_bar(stage), phase ^ 1);
                    const uint32_t fb = full_bar(stage);
                    const uint32_t base = smem_base + stage * kStageBytes;
                    mbar_arrive_expect_tx(fb, kStageBytes);
                    const int k0 = kb * kBK;
                    tma_load_2d(base + A0H * kOpBytes, m0h, fb, k0, row_i);
                    tma_load_2d(base + B0H * kOpBytes, m0h, fb, k0, row_j);
                    tma_load_2d(base + A0L * kOpBytes, m0l, fb, k0, row_i);
                    tma_load_2d(base + B0L * kOpBytes, m0l, fb, k0, row_j);
                    tma_load_2d(base + A1H * kOpBytes, m1h, fb, k0, row_i);
                    tma_load_2d(base + B1H * kOpBytes, m1h, fb, k0, row_j);
                    tma_load_2d(base + A1L * kOpBytes, m1l, fb, k0, row_i);
                    tma_load_2d(base + B1L * kOpBytes, m1l, fb, k0, row_j);
                    if (++stage == kStages) { stage = 0; phase ^= 1; }
                }
            }
        }
    } else if (warp == 1) {
        // =========================== MMA issuer ===========================
        if (lane == 0) {
            constexpr uint32_t idesc = make_idesc_f16(kTile, kTile);
            int stage = 0;
            uint32_t phase = 0;
            int acc = 0;
            uint32_t acc_phase = 0;
            for (int t = blockIdx.x; t < p.num_tiles; t += gridDim.x) {
                mbar_wait(tempty_bar(acc), acc_phase ^ 1);
                tc_fence_after();
                const uint32_t d0 = tmem_base + acc * 256;        // X0 accumulator columns
                const uint32_t d1 = d0 + 128;                     // X1 accumulator columns
                for (int kb = 0; kb < num_kb; ++kb) {
                    mbar_wait(full_bar(stage), phase);
                    tc_fence_after();
                    const uint32_t base = smem_base + stage * kStageBytes;
                    uint64_t d[kOpsPerStage];
#pragma unroll
                    for (int o = 0; o < kOpsPerStage; ++o) d[o] = make_smem_desc<kRowBytes>(base + o * kOpBytes);
#pragma unroll
                    for (int ks = 0; ks < kBK / 16; ++ks) {
                        const uint64_t adv = (uint64_t)(ks * 32 >> 4);     // 16 fp16 = 32 bytes along K
                        const uint32_t first = (kb | ks) != 0;
                        if (with_x0) {
                            umma_f16<1>(d0, d[A0H] + adv, d[B0H] + adv, idesc, first);   // hi.hi
                            umma_f16<1>(d0, d[A0H] + adv, d[B0L] + adv, idesc, 1);       // hi.lo
                            umma_f16<1>(d0, d[A0L] + adv, d[B0H] + adv, idesc, 1);       // lo.hi
                        }
                        umma_f16<1>(d1, d[A0H] + adv, d[B1H] + adv, idesc, first);       // S0.S1
                        umma_f16<1>(d1, d[A1H] + adv, d[B0H] + adv, idesc, 1);           // S1.S0
                        umma_f16<1>(d1, d[A0H] + adv, d[B1L] + adv, idesc, 1);
                        umma_f16<1>(d1, d[A0L] + adv, d[B1H] + adv, idesc, 1);
                        umma_f16<1>(d1, d[A1H] + adv, d[B0L] + adv, idesc, 1);
                        umma_f16<1>(d1, d[A1L] + adv, d[B0H] + adv, idesc, 1);
                    }
                    umma_commit(empty_bar(stage));                 // frees the smem stage
                    if (++stage == kStages) { stage = 0; phase ^= 1; }
                }
                umma_commit(tfull_bar(acc));                       // accumulators complete
                if (++acc == kAccStages) { acc = 0; acc_phase ^= 1; }
            }
        }
    } else {
        // =========================== epilogue ===========================
        const int q = warp & 3;                         // TMEM lane quadrant this warp may read
        const int ld = p.n_pad;
        const float sig = (float)c.sigma;
        const float keep = 1.f - sig;                   // (1 - sigma): 0 or 2
        const float unscale0 = exp2f(-2.f * (float)p.pb.s0_shift);
        const float unscale1 = exp2f(-(float)(p.pb.s0_shift + c.e1_in));
        const float scale0 = exp2f((float)p.pb.s0_shift);
        const float scale1 = exp2f((float)c.e1_out);
        const bool upd0 = c.mode0 == MODE_ACTIVE;
        const bool need_old0 = (upd0 && c.sigma < 0) || c.mode0 == MODE_STOP;
        const bool conv0 = c.conv0 != 0;                // FroErr1 wanted (stop layer or frozen)
        float* s0 = p.s0;
        const float* s1_old = p.s1[c.s1_buf];
        float* s1_new = p.s1[c.s1_buf ^ 1];
        __half* o0h = p.h[c.s0_buf ^ 1][0];
        __half* o0l = p.h[c.s0_buf ^ 1][1];
        __half* o1h = p.h[c.s1_buf ^ 1][2];
        __half* o1l = p.h[c.s1_buf ^ 1][3];

        double r_tr = 0.0, r_fs0 = 0.0, r_f0 = 0.0, r_f1 = 0.0;
        float r_mx1 = 0.f;
        int acc = 0;
        uint32_t acc_phase = 0;
        for (int t = blockIdx.x; t < p.num_tiles; t += gridDim.x) {
            const uint32_t tl = p.tiles[t];
            const int ti = (int)(tl & 0xFFFF), tj = (int)(tl >> 16);
            const bool diag = ti == tj;
            const int gr = ti * kTile + q * 32 + lane;  // global row of this thread's TMEM lane
            mbar_wait(tfull_bar(acc), acc_phase);
            tc_fence_after();
            const uint32_t trow = tmem_base + ((uint32_t)(q * 32) << 16) + acc * 256;
            for (int ch = 0; ch < kTile / 32; ++ch) {
                if (diag && ch < q) continue;           // chunk strictly below the diagonal
                const int gc0 = tj * kTile + ch * 32;
                uint32_t v[32];
                float f_tr = 0.f, f_fs0 = 0.f, f_f0 = 0.f, f_f1 = 0.f;
                // ------------------------------------------------ order 0
                if (with_x0) {
                    tmem_ld_32x32(trow + ch * 32, v);
                    float old[32];
                    if (need_old0) {
#pragma unroll
                        for (int j = 0; j < 32; j += 4) {
                            const float4 o = *reinterpret_cast<const float4*>(s0 + (size_t)gr * ld + gc0 + j);
                            old[j] = o.x; old[j + 1] = o.y; old[j + 2] = o.z; old[j + 3] = o.w;
                        }
                    }
                    tmem_ld_wait();
                    if (upd0) {
                        __half hh[32], ll[32];
                        uint32_t ph[16], pl[16];
                        float nw[32];
#pragma unroll
                        for (int j = 0; j < 32; ++j) {
                            const float x = __uint_as_float(v[j]) * unscale0;
                            const float s = need_old0 ? fmaf(keep, old[j], sig * x) : x;
                            nw[j] = s;
                            split_scaled(s, scale0, hh[j], ll[j]);
                            if (j & 1) { ph[j >> 1] = pack2(hh[j - 1], hh[j]); pl[j >> 1] = pack2(ll[j - 1], ll[j]); }
                            const int gc = gc0 + j;
                            const float w = gr < gc ? 2.f : (gr == gc ? 1.f : 0.f);
                            f_fs0 = fmaf(w * s, s, f_fs0);
                            if (gr == gc) f_tr += s;
                        }
                        if (!diag) {
#pragma unroll
                            for (int j = 0; j < 32; j += 4)
                                st_f4(s0 + (size_t)gr * ld + gc0 + j, nw[j], nw[j + 1], nw[j + 2], nw[j + 3]);
                            st_h32(o0h + (size_t)gr * ld + gc0, ph);
                            st_h32(o0l + (size_t)gr * ld + gc0, pl);
#pragma unroll
                            for (int j = 0; j < 32; ++j) {
                                const size_t m = (size_t)(gc0 + j) * ld + gr;
                                s0[m] = nw[j];
                                o0h[m] = hh[j];
                                o0l[m] = ll[j];
                            }
                        } else {
#pragma unroll
                            for (int j = 0; j < 32; ++j) {
                                const int gc = gc0 + j;
                                if (gr <= gc) {
                                    const size_t dct = (size_t)gr * ld + gc;
                                    s0[dct] = nw[j]; o0h[dct] = hh[j]; o0l[dct] = ll[j];
                                }
                                if (gr < gc) {
                                    const size_t m = (size_t)gc * ld + gr;
                                    s0[m] = nw[j]; o0h[m] = hh[j]; o0l[m] = ll[j];
                                }
                            }
                        }
                    } else {
                        // D0 stop layer: FroErr0^2 = sum (S0 - X0)^2, S0 untouched (R4)
#pragma unroll
                        for (int j = 0; j < 32; ++j) {
                            const float x = __uint_as_float(v[j]) * unscale0;
                            const int gc = gc0 + j;
                            const float w = gr < gc ? 2.f : (gr == gc ? 1.f : 0.f);
                            const float dlt = old[j] - x;
                            f_f0 = fmaf(w * dlt, dlt, f_f0);
                        }
                    }
                }
                // ------------------------------------------------ order 1
                {
                    tmem_ld_32x32(trow + 128 + ch * 32, v);
                    float old[32];
                    const bool need_old1 = c.sigma < 0 || conv0;
                    if (need_old1) {
#pragma unroll
                        for (int j = 0; j < 32; j += 4) {
                            const float4 o = *reinterpret_cast<const float4*>(s1_old + (size_t)gr * ld + gc0 + j);
                            old[j] = o.x; old[j + 1] = o.y; old[j + 2] = o.z; old[j + 3] = o.w;
                        }
                    }
                    tmem_ld_wait();
                    __half hh[32], ll[32];
                    uint32_t ph[16], pl[16];
                    float nw[32];
#pragma unroll
                    for (int j = 0; j < 32; ++j) {
                        const float x = __uint_as_float(v[j]) * unscale1;
                        const float s = need_old1 ? fmaf(keep, old[j], sig * x) : x;
                        nw[j] = s;
                        split_scaled(s, scale1, hh[j], ll[j]);
                        if (j & 1) { ph[j >> 1] = pack2(hh[j - 1], hh[j]); pl[j >> 1] = pack2(ll[j - 1], ll[j]); }
                        const int gc = gc0 + j;
                        const bool in_upper = gr <= gc;
                        if (in_upper) r_mx1 = fmaxf(r_mx1, fabsf(s));
                        if (conv0) {
                            const float w = gr < gc ? 2.f : (gr == gc ? 1.f : 0.f);
                            const float dlt = old[j] - x;
                            f_f1 = fmaf(w * dlt, dlt, f_f1);
                        }
                    }
                    if (!diag) {
#pragma unroll
                        for (int j = 0; j < 32; j += 4)
                            st_f4(s1_new + (size_t)gr * ld + gc0 + j, nw[j], nw[j + 1], nw[j + 2], nw[j + 3]);
                        st_h32(o1h + (size_t)gr * ld + gc0, ph);
                        st_h32(o1l + (size_t)gr * ld + gc0, pl);
#pragma unroll
                        for (int j = 0; j < 32; ++j) {
                            const size_t m = (size_t)(gc0 + j) * ld + gr;
                            s1_new[m] = nw[j];
                            o1h[m] = hh[j];
                            o1l[m] = ll[j];
                        }
                    } else {
#pragma unroll
                        for (int j = 0; j < 32; ++j) {
                            const int gc = gc0 + j;
                            if (gr <= gc) {
                                const size_t dct = (size_t)gr * ld + gc;
                                s1_new[dct] = nw[j]; o1h[dct] = hh[j]; o1l[dct] = ll[j];
                            }
                            if (gr < gc) {
                                const size_t m = (size_t)gc * ld + gr;
                                s1_new[m] = nw[j]; o1h[m] = hh[j]; o1l[m] = ll[j];
                            }
                        }
                    }
                }
                r_tr += (double)f_tr;
                r_fs0 += (double)f_fs0;
                r_f0 += (double)f_f0;
                r_f1 += (double)f_f1;
            }
            // accumulators drained: hand the TMEM stage back to the MMA issuer
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(tempty_bar(acc));
            if (++acc == kAccStages) { acc = 0; acc_phase ^= 1; }
        }
        // per-warp partials, fixed slot per (CTA, warp): the finalizer sums them in a fixed order
        r_tr = warp_sum(r_tr);
        r_fs0 = warp_sum(r_fs0);
        r_f0 = warp_sum(r_f0);
        r_f1 = warp_sum(r_f1);
        const double mx1 = warp_max((double)r_mx1);
        if (lane == 0) {
            double* out = p.partials + ((size_t)blockIdx.x * kNumEpiWarps + (warp - kEpiWarp0)) * RED_COUNT;
            out[RED_TR_S0] = r_tr;
            out[RED_FRO_S0] = r_fs0;
            out[RED_FRO0] = r_f0;
            out[RED_FRO1] = r_f1;
            out[RED_MAX1] = mx1;
            out[RED_FRO2] = 0.0;
            out[RED_MAX2] = 0.0;
        }
    }

    // ---- teardown, then the last CTA of the launch runs Algorithms 2-3 for this layer
    tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        tmem_dealloc<1>(tmem_base, kTmemCols);
    }
    __shared__ int is_last;
    if (threadIdx.x == 0) {
        __threadfence();
        const unsigned int prev = atomicAdd(&p.ctl->ticket, 1u);
        is_last = (prev == gridDim.x - 1);
    }
    __syncthreads();
    if (is_last && warp == 0) {
        __threadfence();
        // fixed-order fp64 reduction: lane l sums slots l, l+32, ...; then a shuffle tree
        const int nslots = gridDim.x * kNumEpiWarps;
        double red[RED_COUNT];
#pragma unroll
        for (int k = 0; k < RED_COUNT; ++k) red[k] = 0.0;
        for (int s = lane; s < nslots; s += 32) {
            const volatile double* in = p.partials + (size_t)s * RED_COUNT;
#pragma unroll
            for (int k = 0; k < RED_COUNT; ++k) {
                if (k == RED_MAX1 || k == RED_MAX2) red[k] = fmax(red[k], in[k]);
                else red[k] += in[k];
            }
        }
#pragma unroll
        for (int k = 0; k < RED_COUNT; ++k) {
            if (k == RED_MAX1 || k == RED_MAX2) red[k] = warp_max(red[k]);
            else red[k] = warp_sum(red[k]);
        }
        if (lane == 0) {
            DmptCtl nc = *p.ctl;
            nc.ticket = 0;
            control_finalize(nc, p.logs, p.pb, red);
            *p.ctl = nc;
        }
    }
}

}  // namespace dmpt
