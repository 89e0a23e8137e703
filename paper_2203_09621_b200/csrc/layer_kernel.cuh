// One deep layer of DNN-SP2-PT in ONE launch (steps a4-a8 of DESIGN.md):
//
//   X0 = S0^2,  X1 = S0 S1 + S1 S0 in the dual half-precision representation,
//       each product = hi.hi + hi.lo + lo.hi, fp16 operands, fp32 accumulation
//                                                  PAPER.md:124-136 (Eqs. 14-16), 309-329 (Eqs. 44-46)
//   S0 <- sigma X0 + (1 - sigma) S0,  S1 <- sigma X1 + (1 - sigma) S1      PAPER.md:182, 193 (Eqs. 23, 25)
//   re-split of the new iterates to (hi, lo) fp16                          PAPER.md:120 (Eq. 13)
//   Tr S0, ||S0||_F^2, ||S0 - X0||_F^2, ||S1 - X1||_F^2, max|S1|
//   Algorithms 2 and 3 + the decision for the next layer (last CTA)
//
// Residual form.  With M = S0 - I/2 the two products are
// taken as  P0 = M.M  and  P1 = M.S1 + S1.M,  and
//       R = S0 - X0 = I/4 - P0,        V = X1 - S1 = P1,
//       S0 <- S0 - sigma R,            S1 <- S1 + sigma V,
// which is Eqs. 23/25 rewritten (S0^2 = S0 - R, 2 S0 - S0^2 = S0 + R; likewise for S1).  The same
// operand count and the same nine tensor-core products per tile; FroErr0 = ||R||_F and
// FroErr1 = ||V||_F fall out directly.  The operand matrices hold the split of M and of S1.
//
// Promoted accumulation.  tcgen05 accumulates in fp32 with TRUNCATION (measured: -0.9 ulp of the
// final sum per K=16 step, i.e. a relative bias of 4e-5 at K = 16384).  Every kChunkK columns of K
// the TMEM accumulators are therefore drained into fp32 registers of the epilogue warps with
// round-to-nearest adds and restarted from zero, which bounds the bias by that of kChunkK/16 steps.
//
// Design (sm_100a).  All iterates are exactly symmetric, so C[i,j] = sum_k A[i,k] B[j,k]: both
// operands of every product are K-major row panels of the same fp16 matrices ("TN" GEMM, the
// natural TMA/UMMA layout), and only output tiles on or above the diagonal are computed; each
// is stored twice (direct and mirrored), which keeps the iterates bit-symmetric.  A tile of P0
// and the matching tile of P1 are accumulated side by side in TMEM from the SAME eight operand
// tiles per k-block (Mhi, Mlo, S1hi, S1lo for row panel I and for row panel J): 9 MMAs per 8
// tiles loaded, against 1 per 2 for a plain GEMM.  Executed tensor work per layer is
// 4.5 N^3 FMA (3 N^3 once S0 froze) against the paper's 5 N^3 (3 N^3).
//
// CTA pairs: a cluster of two CTAs (one TPC) shares a 256 x 128 pair tile through
// tcgen05.mma.cta_group::2 (see the comment on the kernel).
//
// Warp roles (per CTA): warp 0 TMA producer, warp 1 MMA issuer (leader CTA, one elected lane) and TMEM owner, then the
// eight epilogue warps: epilogue warp e owns TMEM lane quadrant (its warp index) % 4 and column half e / 4 of both
// accumulators (64 + 64 fp32 registers per thread).  The order-2, order-3 and A.B^T passes have two more warps between
// them that only hand their registers over (setmaxnreg, three warpgroups); PASS 0 and PASS 2 measured faster without
// (Warps<PASS>).  TMEM holds two accumulator stages
// (2 x [P0 | P1] x 128 columns): the drain of chunk c overlaps the MMAs of chunk c + 1.
//
// Orders: PASS 0 of the kernel does orders 0 and 1 (order 0 alone when the context was created
// with order = 0: ground-state mode); PASS 1 is the order-2 pass of a layer (a9); PASS 4 the order-3 pass.
#pragma once
#include <cuda_fp16.h>

#include "control.cuh"
#include "kernels_hbm.cuh"
#include "ptx.cuh"

namespace dmpt {

constexpr int kTile = 128;                 // output tile edge (rows of panel I x rows of panel J)
constexpr int kBK = 32;                    // fp16 per k-block: 64-byte rows, SWIZZLE_64B
constexpr int kRowBytes = kBK * 2;
constexpr int kPair = 2 * kTile;           // rows of a CTA-pair tile (UMMA M = 256, cta_group::2)
constexpr int kBRows = kTile / 2;          // rows of the J panel each CTA of the pair stages (half of UMMA N)
constexpr int kABytes = kTile * kRowBytes;           // 8 KiB per A-side operand tile (this CTA's 128 rows of panel I)
constexpr int kBBytes = kBRows * kRowBytes;          // 4 KiB per B-side operand tile (this CTA's 64 rows of panel J)
// Per CTA and k-block: PASS 0 (orders 0 and 1) stages 4 A + 4 B tiles (48 KiB), 3 stages + 80 KiB of epilogue staging;
//                      PASS 1 (order 2) stages 6 A + 6 B tiles (72 KiB), 3 stages.
template <int PASS> struct PassCfg;
template <> struct PassCfg<0> { static constexpr int kOps = 4, kStages = 3; };
template <> struct PassCfg<1> { static constexpr int kOps = 6, kStages = 3; };
template <> struct PassCfg<2> { static constexpr int kOps = 6, kStages = 3; };
// PASS 3: a general product C = A.B^T on its own (A, B any n x n matrices; the congruence
// transforms Z^T H Z, Z D Z^T are two of these).  A tile is 256 rows x 256 columns: the A side stages A hi/lo
// (positions 0, 1), the B side B hi/lo of column block 2 JP (positions 2, 3) and of 2 JP + 1 (positions 4, 5);
// one accumulator per column block, six MMAs per 32 KiB staged.
template <> struct PassCfg<3> { static constexpr int kOps = 6, kStages = 3; };
// PASS 4: the order-3 pass of a layer (Eq. 26 at k = 3 with the symmetry saving of
// PAPER.md:325-329): X3 - S3 = (M.S3 + S3.M) + (S1.S2 + S2.S1).  Four operand pairs (M, S1, S2, S3) per side:
// 96 KiB per k-block and CTA, two stages; twelve MMAs per k-step into two accumulators.
template <> struct PassCfg<4> { static constexpr int kOps = 8, kStages = 2; };
constexpr int kChunkK = 128;               // promotion interval along K
constexpr int kKbPerChunk = kChunkK / kBK;
constexpr int kAccStages = 2;
constexpr int kRedStride = 2048;           // per-warp partials are stored [component][slot], slot < gridDim.x * 8 <= 2048
constexpr int kTmemCols = 512;
constexpr int kNumEpiWarps = 8;
// Registers: 384 threads x 168 at launch.  Where kSetMaxNReg says so, warpgroup 0 then gives registers back
// (setmaxnreg.dec) and the two epilogue warpgroups, which hold 2 x 64 fp32 accumulators per thread, grow to 176
// (152 + 2 x 176 = 504 <= 512 registers per lane of a scheduler)
constexpr int kRegsLight = 152, kRegsEpi = 176;
template <int PASS> struct kSetMaxNReg { static constexpr bool value = PASS == 1 || PASS == 3 || PASS == 4; };
// Warps of a CTA: TMA producer, MMA issuer, [two idle warps that only exist to hand their registers over: with setmaxnreg
// a warpgroup of four], then the eight epilogue warps.  PASS 0 and PASS 2: 10 warps (320 threads); the others: 12 (384).
template <int PASS> struct Warps {
    static constexpr int kEpi0 = kSetMaxNReg<PASS>::value ? 4 : 2;         // first epilogue warp
    static constexpr int kThreads = 32 * (kEpi0 + kNumEpiWarps);
};
constexpr int kHalfCols = kTile / 2;       // accumulator columns per epilogue thread and product
constexpr int kSub = 16;                   // columns per step of the final epilogue
// Final epilogue through shared memory and TMA (PASS 0).  Each epilogue warp owns 10 KiB:
//   ring[2]  32 x 16 fp32 (SWIZZLE_64B): the old iterate arrives here by TMA, the new one is written in place
//   dhi, dlo 32 x 32 fp16 (SWIZZLE_64B): the operand split of TWO consecutive steps, stored as one box of 64-byte rows
//   thi, tlo 16 x 32 fp16: the split of one step, transposed (mirrored copy)
// The fp32 iterates are only kept up to date on and above the diagonal (no product reads the rest); the lower triangle
// is restored when an iterate leaves the workspace (dmpt_symmetrize_kernel).
constexpr int kEpiWarpBytes = 10240;
constexpr int kEpiRing = 2048, kEpiDhi = 4096, kEpiDlo = 6144, kEpiThi = 8192, kEpiTlo = 9216;
template <int PASS> struct TmaEpilogue { static constexpr bool value = PASS == 0; };
template <int PASS>
constexpr int smem_bytes() {
    return PassCfg<PASS>::kStages * PassCfg<PASS>::kOps * (kABytes + kBBytes) +
           (TmaEpilogue<PASS>::value ? kNumEpiWarps * kEpiWarpBytes : 0) + 1024 /* alignment slack */ + 256 /* barriers */;
}

// operand matrices, in the order of LayerParams::maps / ::h; a stage holds the A tiles of the first kOps of
// them (rows of panel I), then the B tiles (rows of panel J)
enum Op : int { MH = 0, ML = 1, S1H = 2, S1L = 3, S2H = 4, S2L = 5, S3H = 6, S3L = 7 };
// positions inside a stage of PASS 1 / PASS 2 (M, then two more operand pairs)
enum Pos : int { PM_H = 0, PM_L = 1, PY_H = 2, PY_L = 3, PZ_H = 4, PZ_L = 5 };

struct LayerParams {
    CUtensorMap maps[2][8];     // [buffer][Mhi, Mlo, S1hi, S1lo, S2hi, S2lo, S3hi, S3lo], box = kBK x kBRows, SWIZZLE_64B
    // epilogue maps of the fp16 pairs: [..][0] direct 32 x 32 box (SWIZZLE_64B), [..][1] mirrored 32 x 16 box
    CUtensorMap emap32[3];      // fp32 iterates S0, S1[0], S1[1]: 16 x 32 box, SWIZZLE_64B
    CUtensorMap emap16[2][2][2];  // fp16 operand PAIRS [buffer][(Mhi, Mlo), (S1hi, S1lo)]: 3D maps, the hi and the lo matrix
                                // of a pair lie back to back in the workspace and are the two planes of one tensor, so
                                // that one TMA store writes a block of both
    float* s0;                  // fp32 S0, updated in place, ld = n_pad
    float* s1[2];               // fp32 S1, ping-pong
    float* s2[2];               // fp32 response slot 2, ping-pong (order 2: S2; multi-field: S1 of field 2)
    float* s3[2];               // fp32 response slot 3, ping-pong (multi-field: S1 of field 3)
    __half* h[2][8];            // fp16 operand matrices the epilogue writes, same order as maps
    const uint32_t* tiles;      // pair tiles (IP | J << 16): block rows 2 IP, 2 IP + 1 x block column J >= 2 IP
    int num_tiles;
    const uint32_t* tiles_full; // PASS 3: every (IP | J << 16) with J even: block rows 2 IP, 2 IP + 1 x block
                                // columns J, J + 1 (256 x 256); the output is not symmetric
    int num_tiles_full;
    int n_pad;
    int wave_sync;              // 1: producers of all CTAs re-align at every tile boundary (L2 reuse)
    int epilogue_direct;        // 1: row-per-thread final epilogue on every tile (dmpt_options::epilogue_direct)
    DmptCtl* ctl;
    DmptLogs logs;
    DmptProblem pb;
    double* partials;           // [gridDim.x][kNumEpiWarps][RED_COUNT], written by PASS 0
    double* partials2;          // same shape, written by PASS 1 / PASS 2 (RED_FRO2, RED_MAX2, RED_FRO3, RED_MAX3)
    double* partials3;          // same shape, written by PASS 4 (RED_FRO3, RED_MAX3)
    // order-parallel pair (DmptProblem::pair_side): per-layer records from the order-0 side; side 1 writes them in
    // its control step, side 2 reads its copies at the start of every launch.  NULL otherwise.
    DmptHandoff* handoff;
    // device-side loop (dmpt_options::loop_graph): the layer launches are the body of a CUDA-graph WHILE node; the
    // control step sets its condition (1: another layer, 0: done).  use_cond = 0: launches come from the host in chunks.
    cudaGraphConditionalHandle cond;
    int use_cond;
};

__device__ __forceinline__ uint32_t pack2(__half a, __half b) {
    return (uint32_t)__half_as_ushort(a) | ((uint32_t)__half_as_ushort(b) << 16);
}

// Final epilogue of one product for one thread: row `gr`, columns gc_base .. gc_base + 63 held in
// acc[].  ORDER 0: acc = (2^a M)(2^a M) sums;  ORDER 1: acc = P1 sums.
//   mode: 0 = update and store, 1 = measure only (D0 stop layer: FroErr0, S0 untouched).
struct EpiOut {
    float* dst;            // fp32 matrix to write (S0 in place, or the S1 ping-pong target)
    const float* old;      // fp32 matrix holding the previous iterate
    __half* hi;
    __half* lo;
    // TMA path: maps of the same matrices (direct box; the mirrored box is the next map); m_hl: the (hi, lo) pair
    const CUtensorMap* m_old;
    const CUtensorMap* m_dst;
    const CUtensorMap* m_hl;
};

struct EpiTma {            // shared-memory addresses of this warp's staging
    uint32_t ring[2], dhi, dlo, thi, tlo, bar[2];
};

template <int ORDER>
__device__ __forceinline__ void final_epilogue(float (&acc)[kHalfCols], const EpiOut& o, int ld, int gr,
                                               int gc_base, bool diag_tile, bool store, float sig,
                                               float unscale, float scale, bool want_fro, double& r_tr,
                                               double& r_fs, double& r_fro, float& r_max) {
#pragma unroll
    for (int sc = 0; sc < kHalfCols / kSub; ++sc) {
        const int gc0 = gc_base + sc * kSub;
        if (diag_tile && gc0 + kSub - 1 < gr) continue;          // strictly below the diagonal: mirrored by others
        float old[kSub];
#pragma unroll
        for (int j = 0; j < kSub; j += 4) {
            const float4 v = *reinterpret_cast<const float4*>(o.old + (size_t)gr * ld + gc0 + j);
            old[j] = v.x; old[j + 1] = v.y; old[j + 2] = v.z; old[j + 3] = v.w;
        }
        float f_tr = 0.f, f_fs = 0.f, f_fro = 0.f;
        uint32_t ph[kSub / 2], pl[kSub / 2];
        __half hprev = __float2half_rn(0.f), lprev = hprev;
#pragma unroll
        for (int j = 0; j < kSub; ++j) {
            const int gc = gc0 + j;
            const float w = gr < gc ? 2.f : (gr == gc ? 1.f : 0.f);
            const float dg = gr == gc ? 1.f : 0.f;
            float nw, delta;
            if (ORDER == 0) {
                delta = fmaf(-unscale, acc[sc * kSub + j], 0.25f * dg);      // R = I/4 - M.M
                nw = fmaf(-sig, delta, old[j]);                              // S0 - sigma R
            } else {
                delta = unscale * acc[sc * kSub + j];                        // V = M.S1 + S1.M
                nw = fmaf(sig, delta, old[j]);                               // S1 + sigma V
            }
            if (want_fro) f_fro = fmaf(w * delta, delta, f_fro);
            acc[sc * kSub + j] = nw;
            if (ORDER == 0) {
                f_fs = fmaf(w * nw, nw, f_fs);
                f_tr += dg * nw;
            } else if (w != 0.f) {
                r_max = fmaxf(r_max, fabsf(nw));
            }
            __half hh, ll;
            split_scaled(ORDER == 0 ? nw - 0.5f * dg : nw, scale, hh, ll);   // operands hold M = S0 - I/2
            if (j & 1) { ph[j >> 1] = pack2(hprev, hh); pl[j >> 1] = pack2(lprev, ll); }
            hprev = hh; lprev = ll;
        }
        r_tr += (double)f_tr;
        r_fs += (double)f_fs;
        r_fro += (double)f_fro;
        if (!store) continue;
        if (!diag_tile) {
            float* d = o.dst + (size_t)gr * ld + gc0;
#pragma unroll
            for (int j = 0; j < kSub; j += 4)
                *reinterpret_cast<float4*>(d + j) = make_float4(acc[sc * kSub + j], acc[sc * kSub + j + 1],
                                                                acc[sc * kSub + j + 2], acc[sc * kSub + j + 3]);
#pragma unroll
            for (int j = 0; j < kSub / 2; j += 4) {
                *reinterpret_cast<uint4*>(o.hi + (size_t)gr * ld + gc0 + 2 * j) = make_uint4(ph[j], ph[j + 1], ph[j + 2], ph[j + 3]);
                *reinterpret_cast<uint4*>(o.lo + (size_t)gr * ld + gc0 + 2 * j) = make_uint4(pl[j], pl[j + 1], pl[j + 2], pl[j + 3]);
            }
            // mirrored copy: for a fixed j the 32 lanes write 32 consecutive elements of row gc0 + j
#pragma unroll
            for (int j = 0; j < kSub; ++j) {
                const size_t m = (size_t)(gc0 + j) * ld + gr;
                const uint32_t hw = ph[j >> 1], lw = pl[j >> 1];
                o.dst[m] = acc[sc * kSub + j];
                o.hi[m] = __ushort_as_half((unsigned short)((j & 1) ? (hw >> 16) : (hw & 0xFFFF)));
                o.lo[m] = __ushort_as_half((unsigned short)((j & 1) ? (lw >> 16) : (lw & 0xFFFF)));
            }
        } else {
#pragma unroll
            for (int j = 0; j < kSub; ++j) {
                const int gc = gc0 + j;
                const uint32_t hw = ph[j >> 1], lw = pl[j >> 1];
                const __half hh = __ushort_as_half((unsigned short)((j & 1) ? (hw >> 16) : (hw & 0xFFFF)));
                const __half ll = __ushort_as_half((unsigned short)((j & 1) ? (lw >> 16) : (lw & 0xFFFF)));
                if (gr <= gc) {
                    const size_t dct = (size_t)gr * ld + gc;
                    o.dst[dct] = acc[sc * kSub + j]; o.hi[dct] = hh; o.lo[dct] = ll;
                }
                if (gr < gc) {
                    const size_t m = (size_t)gc * ld + gr;
                    o.dst[m] = acc[sc * kSub + j]; o.hi[m] = hh; o.lo[m] = ll;
                }
            }
        }
    }
}


// Final epilogue of one product on an OFF-DIAGONAL tile, through shared memory and TMA: the same arithmetic as
// final_epilogue with w = 2, dg = 0 (so delta = -+unscale acc exactly and S <- fmaf(+-unscale, acc, old)), but
//   * the old iterate comes by TMA into this warp's ring (issued one step ahead),
//   * the new iterate and its split are written to shared memory (the split also transposed) and leave by TMA stores:
//     per 32 x 16 block the fp32 values and the mirrored (hi, lo) pair, per two blocks the direct (hi, lo) pair as
//     one box of 64-byte rows - full lines instead of row-per-thread accesses, and as few, as wide TMA requests as
//     the staging allows (the stores are bound by the TMA unit's request rate),
//   * the split uses the packed conversions (cvt.rn.f16x2.f32).
// step s (0 .. ns-1) of the tile handles product s / 4 (0: P0, 1: P1; when only one is live it is steps 0-3) and
// columns (s & 3) * 16 of this thread's 64.
//
// Diagonal tiles (diag): the mirror of a diagonal block lies inside the block, so the box stores of one warp would
// overwrite what another warp owns.  Each 32 x 16 block of a step is then one of three kinds:
//   strictly above the diagonal - handled exactly as on an off-diagonal tile (its mirror lands strictly below the
//                                 diagonal, which no block writes directly);
//   strictly below              - nothing to do (written as the mirror of its transpose);
//   crossing the diagonal       - same staging, general arithmetic (diagonal terms I/4 and -I/2, weights 2 / 1 / 0),
//                                 and the warp stores the staged block itself with masked, coalesced accesses
//                                 (direct copy where row <= column, mirrored copy where row < column) instead of
//                                 one scalar store per lane and element.
template <int ORDER>
__device__ __forceinline__ void final_epilogue_tma(const float (&acc)[kHalfCols], const EpiOut& o, const EpiTma& et,
                                                   uint32_t& ring_phase, int s_base, int ns,
                                                   const CUtensorMap* next_old /* old map of step s_base + 4 */,
                                                   int gr0, int gcb, int lane, float su, float unscale, float scale,
                                                   bool want_fro, bool diag, float sig, int ld, double& r_tr,
                                                   double& r_fs, double& r_fro, float& r_max) {
    const uint32_t row64 = (uint32_t)lane * 64u, sw64 = ((uint32_t)lane >> 1) & 3u;
    const uint32_t row32 = (uint32_t)lane * 32u, sw32 = ((uint32_t)lane >> 2) & 1u;
#pragma unroll
    for (int sc = 0; sc < kHalfCols / kSub; ++sc) {
        const int s = s_base + sc;
        const int slot = s & 1;
        const int gc0 = gcb + sc * kSub;
        // the stores of the previous step must have read the staging before it is rewritten; the other ring slot
        // is then free for the old iterate of the next step
        if (lane == 0) {
            bulk_wait_read<0>();
            if (s >= 1 && s + 1 < ns) {
                const CUtensorMap* m = sc + 1 < kHalfCols / kSub ? o.m_old : next_old;
                const int gcn = sc + 1 < kHalfCols / kSub ? gc0 + kSub : gcb;
                mbar_arrive_expect_tx(et.bar[slot ^ 1], kSub * 32 * 4);
                tma_load_2d(et.ring[slot ^ 1], m, et.bar[slot ^ 1], gcn, gr0);
            }
        }
        __syncwarp();
        mbar_wait(et.bar[slot], (ring_phase >> slot) & 1u);
        ring_phase ^= 1u << slot;
        if (diag && gr0 > gc0 + kSub - 1) continue;       // strictly below the diagonal
        if (diag && !(gr0 + 31 < gc0)) {
            // ---- block crossing the diagonal: this thread's row is gr0 + lane
            const int gr = gr0 + lane;
            float f_fs = 0.f, f_fro = 0.f, f_tr = 0.f;
#pragma unroll
            for (int q2 = 0; q2 < 2; ++q2) {
                uint32_t ph[4], pl[4];
#pragma unroll
                for (int j4 = 2 * q2; j4 < 2 * q2 + 2; ++j4) {
                    const uint32_t a32 = et.ring[slot] + row64 + (((uint32_t)j4 ^ sw64) << 4);
                    const float4 x = lds128(a32);
                    float v[4] = {x.x, x.y, x.z, x.w};
#pragma unroll
                    for (int t = 0; t < 4; t += 2) {
                        const int j = 4 * j4 + t;
                        float nn[2], xs[2];
#pragma unroll
                        for (int u = 0; u < 2; ++u) {
                            const int gc = gc0 + j + u;
                            const float dg = gr == gc ? 1.f : 0.f;
                            const float w = gr < gc ? 2.f : dg;
                            const float a = acc[sc * kSub + j + u];
                            float delta, nw;
                            if (ORDER == 0) {
                                delta = fmaf(-unscale, a, 0.25f * dg);               // R = I/4 - M.M
                                nw = fmaf(-sig, delta, v[t + u]);                    // S0 - sigma R
                            } else {
                                delta = unscale * a;                                 // V = M.S1 + S1.M
                                nw = fmaf(sig, delta, v[t + u]);                     // S1 + sigma V
                            }
                            if (want_fro) f_fro = fmaf(w * delta, delta, f_fro);
                            if (ORDER == 0) {
                                f_fs = fmaf(w * nw, nw, f_fs);
                                f_tr += dg * nw;
                            } else if (w != 0.f) {
                                r_max = fmaxf(r_max, fabsf(nw));
                            }
                            nn[u] = nw;
                            xs[u] = (ORDER == 0 ? nw - 0.5f * dg : nw) * scale;      // operands hold M = S0 - I/2
                        }
                        v[t] = nn[0]; v[t + 1] = nn[1];
                        const __half2 h2 = __floats2half2_rn(xs[0], xs[1]);
                        const float2 hf = __half22float2(h2);
                        const __half2 l2 = __floats2half2_rn(xs[0] - hf.x, xs[1] - hf.y);
                        const uint32_t hw = *reinterpret_cast<const uint32_t*>(&h2);
                        const uint32_t lw = *reinterpret_cast<const uint32_t*>(&l2);
                        ph[(j >> 1) & 3] = hw;
                        pl[(j >> 1) & 3] = lw;
                        sts16(et.thi + (uint32_t)j * 64u + (uint32_t)lane * 2u, (uint16_t)(hw & 0xFFFF));
                        sts16(et.thi + (uint32_t)(j + 1) * 64u + (uint32_t)lane * 2u, (uint16_t)(hw >> 16));
                        sts16(et.tlo + (uint32_t)j * 64u + (uint32_t)lane * 2u, (uint16_t)(lw & 0xFFFF));
                        sts16(et.tlo + (uint32_t)(j + 1) * 64u + (uint32_t)lane * 2u, (uint16_t)(lw >> 16));
                    }
                    sts128(a32, __float_as_uint(v[0]), __float_as_uint(v[1]), __float_as_uint(v[2]), __float_as_uint(v[3]));
                }
                sts128(et.dhi + row32 + (((uint32_t)q2 ^ sw32) << 4), ph[0], ph[1], ph[2], ph[3]);
                sts128(et.dlo + row32 + (((uint32_t)q2 ^ sw32) << 4), pl[0], pl[1], pl[2], pl[3]);
            }
            r_tr += (double)f_tr;
            r_fs += (double)f_fs;
            r_fro += (double)f_fro;
            __syncwarp();
            // direct copy, two rows of 16 columns per instruction, where row <= column
            {
                const uint32_t c = (uint32_t)lane & 15u, rr = (uint32_t)lane >> 4;
#pragma unroll 4
                for (uint32_t i = 0; i < 16; ++i) {
                    const uint32_t r = 2 * i + rr;
                    const int grr = gr0 + (int)r, gcc = gc0 + (int)c;
                    if (grr <= gcc) {
                        const size_t g = (size_t)grr * ld + gcc;
                        o.dst[g] = lds32f(et.ring[slot] + r * 64u + ((((c >> 2) ^ ((r >> 1) & 3u))) << 4) + (c & 3u) * 4u);
                        const uint32_t b = r * 32u + ((((c >> 3) ^ ((r >> 2) & 1u))) << 4) + (c & 7u) * 2u;
                        o.hi[g] = __ushort_as_half(lds16(et.dhi + b));
                        o.lo[g] = __ushort_as_half(lds16(et.dlo + b));
                    }
                }
                // mirrored copy of the split (the fp32 iterate is kept on and above the diagonal only), one row of 32
                // columns per instruction, where row < column of the original
#pragma unroll 4
                for (uint32_t j = 0; j < 16; ++j) {
                    if (gr < gc0 + (int)j) {
                        const size_t g = (size_t)(gc0 + (int)j) * ld + gr;
                        o.hi[g] = __ushort_as_half(lds16(et.thi + j * 64u + (uint32_t)lane * 2u));
                        o.lo[g] = __ushort_as_half(lds16(et.tlo + j * 64u + (uint32_t)lane * 2u));
                    }
                }
            }
            __syncwarp();
            continue;
        }
        float f_fs = 0.f, f_fro = 0.f;
#pragma unroll
        for (int q2 = 0; q2 < 2; ++q2) {                  // eight columns: one 16-byte chunk of the fp16 rows
            uint32_t ph[4], pl[4];
#pragma unroll
            for (int j4 = 2 * q2; j4 < 2 * q2 + 2; ++j4) {
                const uint32_t a32 = et.ring[slot] + row64 + (((uint32_t)j4 ^ sw64) << 4);
                const float4 x = lds128(a32);
                float v[4] = {x.x, x.y, x.z, x.w};
#pragma unroll
                for (int t = 0; t < 4; t += 2) {
                    const int j = 4 * j4 + t;
                    const float a0 = acc[sc * kSub + j], a1 = acc[sc * kSub + j + 1];
                    const float n0 = fmaf(su, a0, v[t]), n1 = fmaf(su, a1, v[t + 1]);
                    if (want_fro) {
                        const float d0 = unscale * a0, d1 = unscale * a1;
                        f_fro = fmaf(d0, d0, f_fro);
                        f_fro = fmaf(d1, d1, f_fro);
                    }
                    if (ORDER == 0) {
                        f_fs = fmaf(n0, n0, f_fs);
                        f_fs = fmaf(n1, n1, f_fs);
                    } else {
                        r_max = fmaxf(r_max, fmaxf(fabsf(n0), fabsf(n1)));
                    }
                    v[t] = n0; v[t + 1] = n1;
                    const float t0 = n0 * scale, t1 = n1 * scale;
                    const __half2 h2 = __floats2half2_rn(t0, t1);
                    const float2 hf = __half22float2(h2);
                    const __half2 l2 = __floats2half2_rn(t0 - hf.x, t1 - hf.y);
                    const uint32_t hw = *reinterpret_cast<const uint32_t*>(&h2);
                    const uint32_t lw = *reinterpret_cast<const uint32_t*>(&l2);
                    ph[(j >> 1) & 3] = hw;
                    pl[(j >> 1) & 3] = lw;
                    // transposed: for a fixed column the 32 lanes write one row of the mirrored block
                    sts16(et.thi + (uint32_t)j * 64u + (uint32_t)lane * 2u, (uint16_t)(hw & 0xFFFF));
                    sts16(et.thi + (uint32_t)(j + 1) * 64u + (uint32_t)lane * 2u, (uint16_t)(hw >> 16));
                    sts16(et.tlo + (uint32_t)j * 64u + (uint32_t)lane * 2u, (uint16_t)(lw & 0xFFFF));
                    sts16(et.tlo + (uint32_t)(j + 1) * 64u + (uint32_t)lane * 2u, (uint16_t)(lw >> 16));
                }
                sts128(a32, __float_as_uint(v[0]), __float_as_uint(v[1]), __float_as_uint(v[2]), __float_as_uint(v[3]));   // in place
            }
            // chunk (2 (sc & 1) + q2) of this thread's 64-byte row of the two-step direct box
            const uint32_t ch = (((uint32_t)(2 * (sc & 1) + q2)) ^ sw64) << 4;
            sts128(et.dhi + row64 + ch, ph[0], ph[1], ph[2], ph[3]);
            sts128(et.dlo + row64 + ch, pl[0], pl[1], pl[2], pl[3]);
        }
        r_fs += (double)(2.f * f_fs);           // off-diagonal elements count twice
        r_fro += (double)(2.f * f_fro);
        fence_proxy_async_smem();
        __syncwarp();
        if (lane == 0) {
            tma_store_2d(o.m_dst, et.ring[slot], gc0, gr0);
            tma_store_3d(o.m_hl + 1, et.thi, gr0, gc0, 0);      // thi, tlo: the two planes of the mirrored box
            if (sc & 1) tma_store_3d(o.m_hl, et.dhi, gc0 - kSub, gr0, 0);      // dhi, dlo: 32 columns of two steps
            bulk_commit();
        }
    }
}

// One layer launch.  Clusters of two CTAs (one TPC) work on 256 x 128 pair tiles with
// tcgen05.mma.cta_group::2: CTA r of the pair owns block row 2 IP + r (its 128 rows of every A-side
// operand and its 128 TMEM lanes of both accumulators) and stages rows r*64 .. r*64+63 of the J panel
// (its half of UMMA N = 128).  Per MMA each SM reads 4 KiB (A) + 2 KiB (half of B) from shared memory
// instead of 8 KiB, and TMA brings 48 KiB instead of 64 KiB per k-block (profiles/: the 1-CTA kernel
// was bound by the shared-memory pipe).  Only the leader CTA (rank 0) issues MMAs; both run TMA and
// the epilogue.
//
// PASS 0: orders 0 and 1 of layer n (P0 = M.M, P1 = M.S1 + S1.M); its last CTA runs Algorithms 2-3.
// PASS 1: order 2 of layer n (a9, Eq. 25 third line, 201 Eq. 26):
//             V2 = X2 - S2 = (M.S2 + S2.M) + S1.S1,   S2 <- S2 + sigma V2,
//         two accumulators again: Q = S1.S1 (3 products, scale 2^(2 e1)) and P2 = M.S2 + S2.M (6 products,
//         scale 2^(a + e2)), combined in fp32 in the epilogue.  Launched BEFORE pass 0 of the same layer: it
//         reads the operands of S0_{n-1}, S1_{n-1}, S2_{n-1} and the decision pass 0 of layer n-1 left in
//         DmptCtl, writes S2_n into the other buffer and leaves ||V2||_F^2, max|S2_n| in partials2.
// WIDE (PASS 0 at order 0 only): the ground-state instantiation.  It stages the two operands of M.M only, in k-blocks
// of 64 columns - 128-byte operand rows, SWIZZLE_128B, through the tensor maps in slots S3H, S3L - so that its 48 KiB
// stages are full: twice the operand bytes in flight per CTA (3 x 40 KiB, as first order has) with half the TMA
// instructions.  The general instantiation at order 0 fills half of every stage (60 KiB in flight) while asking for
// 1.5 x first order's bytes per MMA, and the MMAs wait for the loads: tensor pipe 55 % against 89 % (DESIGN.md 12,
// item 6).  Same k16 steps in the same order: bit-identical results.
template <int PASS, bool WIDE = false>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(Warps<PASS>::kThreads, 1)
dmpt_layer_kernel(const __grid_constant__ LayerParams p) {
    static_assert(!WIDE || PASS == 0, "the wide k-block is the order-0 instantiation of pass 0");
    constexpr int kOps = WIDE ? 2 : PassCfg<PASS>::kOps;
    constexpr int kBK = WIDE ? 2 * dmpt::kBK : dmpt::kBK;          // these four shadow the namespace's
    constexpr int kRowBytes = kBK * 2;
    constexpr int kABytes = kTile * kRowBytes;
    constexpr int kBBytes = kBRows * kRowBytes;
    constexpr int kKbPerChunk = kChunkK / kBK;
    constexpr int kStages = PassCfg<PASS>::kStages;
    constexpr int kEpiWarp0 = Warps<PASS>::kEpi0;
    constexpr int kNumThreads = Warps<PASS>::kThreads;
    constexpr int kStageBytes = kOps * (kABytes + kBBytes);
    constexpr int kBOff = kOps * kABytes;          // B tiles follow the A tiles inside a stage
    // Layer launches that do not need the wave barrier are chained by programmatic dependent launch: the next launch
    // is released at once (its CTAs become resident as SMs free up - at N = 256 straight away - and park in
    // griddepcontrol.wait), so the stream's launch latency is off the critical path of a layer.
    griddep_launch_dependents();
    griddep_wait();
    // ---- the decision for this layer, taken by the previous launch (both CTAs of a pair read the same)
    DmptCtl c_in = *p.ctl;
    if (c_in.done) {
        // (a run that was over before its first layer, e.g. degenerate bounds: end the WHILE loop)
        if (PASS == 0 && p.use_cond && blockIdx.x == 0 && threadIdx.x == 0) cudaGraphSetConditional(p.cond, 0u);
        return;
    }
    if (PASS == 0 && p.pb.pair_side == 2) {
        handoff_merge(c_in, p.handoff[c_in.layer]);
        if (c_in.done) {            // the order-0 side stopped with an error: pass it on and stop
            if (blockIdx.x == 0 && threadIdx.x == 0) { p.ctl->status = c_in.status; p.ctl->done = 1; }
            return;
        }
    }
    if (PASS == 0 && threadIdx.x == 0) {
        // one stamp per SM and layer (dmpt_result.sm_clock_mhz): the clock the loop really runs at under the power cap.
        // Placed here, after the early exits: before them it changes the register allocation of the whole kernel
        // (PASS 0: 648 -> 1032 bytes of spills, 11 % slower at N = 16384).
        const unsigned int sm = sm_id() & (kMaxSmStamps - 1);
        long long* dst = &p.logs.clk->first[0][0] + (c_in.layer == 1 ? 0 : 2 * kMaxSmStamps) + 2 * sm;
        dst[0] = clock64();
        dst[1] = global_timer_ns();
    }
    const DmptCtl c = c_in;
    // order 2 after the D1 stop: S0 and S1 are frozen, pass 0 only runs the control step
    // (order 3 after the D2 stop: the order-2 pass has nothing left to do either)
    const bool idle = (PASS == 0 && c.conv1 != 0) || (PASS == 1 && c.conv2 != 0);

    extern __shared__ uint8_t smem_raw[];
    constexpr bool kTmaEpi = TmaEpilogue<PASS>::value;
    constexpr int kEpiBytes = kTmaEpi ? kNumEpiWarps * kEpiWarpBytes : 0;
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t epi_base = smem_base + kStages * kStageBytes;          // 1024-byte aligned: stages are multiples of 1 KiB
    const uint32_t bar_base = epi_base + kEpiBytes;
    auto full_bar = [&](int s) { return bar_base + 8u * s; };
    auto empty_bar = [&](int s) { return bar_base + 8u * (kStages + s); };
    auto tfull_bar = [&](int s) { return bar_base + 8u * (2 * kStages + s); };
    auto tempty_bar = [&](int s) { return bar_base + 8u * (2 * kStages + kAccStages + s); };
    auto ring_bar = [&](int w, int s) { return bar_base + 8u * (2 * kStages + 2 * kAccStages + 2 * w + s); };
    constexpr int kNumBars = 2 * kStages + 2 * kAccStages + 2 * kNumEpiWarps;
    const uint32_t tmem_slot = bar_base + 8u * kNumBars;
    uint8_t* smem_gen = smem_raw + (smem_base - smem_u32(smem_raw));
    volatile uint32_t* tmem_slot_ptr =
        reinterpret_cast<volatile uint32_t*>(smem_gen + kStages * kStageBytes + kEpiBytes + 8 * kNumBars);

    // warp index through a shuffle: the compiler then knows it is warp-uniform, and the single-thread
    // sections below are entered through elect.sync, so TMA / MMA operands stay in uniform registers
    // (with `lane == 0` every UTCHMMA / UTMALDG was wrapped in an ELECT + R2UR.BROADCAST + BRA.U.ANY loop)
    const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
    const int lane = threadIdx.x & 31;
    const uint32_t rank = cluster_ctarank();        // 0 = leader of the pair
    const int pair = blockIdx.x >> 1;
    const int num_pairs = gridDim.x >> 1;
    const int num_chunks = p.n_pad / kChunkK;
    const int num_tiles = PASS == 3 ? p.num_tiles_full : (idle ? 0 : p.num_tiles);
    const uint32_t* tile_list = PASS == 3 ? p.tiles_full : p.tiles;
    // accumulator 0 / 1 in use.  PASS 0: P0 until S0 froze / P1 unless order 0 (ground state only).
    // PASS 2: one accumulator per extra field, until that field's stopping test fired.
    // PASS 3: accumulator 0 only, fed by A hi/lo (positions 0, 1, A side) and B hi/lo (positions 2, 3, B side).
    const bool with_p0 = (PASS == 3 || PASS == 4) ? true : (PASS == 0 ? c.mode0 != MODE_FROZEN : (PASS == 1 || c.conv2 == 0));
    const bool with_p1 = (PASS == 3 || PASS == 4) ? true
                                   : (PASS == 0 ? p.pb.order >= 1 : (PASS == 1 || (p.pb.nfields >= 3 && c.conv3 == 0)));
    const int nops = WIDE ? 2 : ((with_p1 || PASS == 3) ? kOps : kOps - 2);    // the last operand pair only feeds accumulator 1
    unsigned int* wave_ctr = PASS == 0 ? &p.ctl->wave : (PASS == 4 ? &p.ctl->wave3 : &p.ctl->wave2);

    if (warp == 0 && lane == 0) {
        for (int m = 0; m < 2; ++m) {
            prefetch_tensormap(&p.maps[c.s0_buf][m]);
            prefetch_tensormap(&p.maps[c.s1_buf][2 + m]);
            if (PASS == 1 || PASS == 2 || PASS == 4) prefetch_tensormap(&p.maps[c.s2_buf][S2H + m]);       // only maps that were encoded
            if ((PASS == 2 && p.pb.nfields >= 3) || PASS == 4) prefetch_tensormap(&p.maps[c.s3_buf][S3H + m]);
        }
        for (int s = 0; s < kStages; ++s) {
            mbar_init(full_bar(s), 1);                       // leader's: its producer's arrive + both CTAs' bytes
            mbar_init(empty_bar(s), 1);                      // MMA commit, multicast to both CTAs
        }
        for (int s = 0; s < kAccStages; ++s) {
            mbar_init(tfull_bar(s), 1);                      // MMA commit, multicast to both CTAs
            mbar_init(tempty_bar(s), 2 * kNumEpiWarps);      // leader's: epilogue warps of both CTAs
        }
        for (int w = 0; w < kNumEpiWarps; ++w) {
            mbar_init(ring_bar(w, 0), 1);                    // old-iterate ring of epilogue warp w (TMA epilogue)
            mbar_init(ring_bar(w, 1), 1);
        }
        fence_mbar_init();
    }
    if (warp == 1) {
        tmem_alloc<2>(tmem_slot, kTmemCols);
        tmem_relinquish<2>();
    }
    tc_fence_before();
    cluster_sync_all();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_ptr;
    // Register re-allocation between the warpgroups (setmaxnreg 152 / 176 / 176) only where it measured faster: the
    // order-2, order-3 and A.B^T passes.  PASS 0 and PASS 2 run with the launch bound's 168 registers for every warp:
    // 30.6 instead of 31.1 ms per layer at N = 16384, and the drain loop no longer spills.
    if (kSetMaxNReg<PASS>::value) {
        if (warp < kEpiWarp0) setmaxnreg_dec<kRegsLight>(); else setmaxnreg_inc<kRegsEpi>();
    }

    if (warp == 0) {
        // =========================== TMA producer (both CTAs) ===========================
        {
            // staged operand pairs: PASS 0: M, S1;  PASS 1: M, S1, S2;  PASS 2: M, slot 2, slot 3;  PASS 4: M, S1, S2, S3
            const CUtensorMap* maps[8] = {
                &p.maps[c.s0_buf][WIDE ? S3H : MH], &p.maps[c.s0_buf][WIDE ? S3L : ML],
                PASS == 2 ? &p.maps[c.s2_buf][S2H] : &p.maps[c.s1_buf][S1H],
                PASS == 2 ? &p.maps[c.s2_buf][S2L] : &p.maps[c.s1_buf][S1L],
                PASS == 2 ? &p.maps[c.s3_buf][S3H] : &p.maps[c.s2_buf][S2H],
                PASS == 2 ? &p.maps[c.s3_buf][S3L] : &p.maps[c.s2_buf][S2L],
                &p.maps[c.s3_buf][S3H], &p.maps[c.s3_buf][S3L]};
            const int num_kb = p.n_pad / kBK;
            int stage = 0;
            uint32_t phase = 0;
            unsigned int wave = 0;
            const unsigned int num_waves = (num_tiles + num_pairs - 1) / num_pairs;
            for (int t = pair; t < num_tiles; t += num_pairs, ++wave) {
                if (p.wave_sync && wave > 0) {
                    // re-align the K phase of all CTAs: tiles in flight then stream the same k-blocks of
                    // few row panels at the same time and share them through L2
                    if (lane == 0) {
                        __threadfence();
                        atomicAdd(wave_ctr, 1u);
                        const unsigned int target = gridDim.x * wave;
                        unsigned int spins = 0;
                        while (ld_acquire_u32(wave_ctr) < target) {
                            __nanosleep(64);
                            if (++spins > (1u << 26)) __trap();
                        }
                    }
                    __syncwarp();
                }
                const uint32_t tl = tile_list[t];
                const int row_a = (2 * (int)(tl & 0xFFFF) + (int)rank) * kTile;
                const int row_b = (int)(tl >> 16) * kTile + (int)rank * kBRows;
                for (int kb = 0; kb < num_kb; ++kb) {
                    mbar_wait(empty_bar(stage), phase ^ 1);
                    const uint32_t fb = full_bar(stage);      // completion is counted on the LEADER's barrier
                    const uint32_t base = smem_base + stage * kStageBytes;
                    if (elect_one()) {
                        if (rank == 0)
                            mbar_arrive_expect_tx(fb, PASS == 3 ? 2 * (2 * kABytes + 4 * kBBytes) : 2 * nops * (kABytes + kBBytes));
                        const int k0 = kb * kBK;
#pragma unroll
                        for (int o = 0; o < kOps; ++o) {
                            if (o < nops && !(PASS == 3 && o >= 2)) {        // A side (PASS 3: A hi/lo only)
                                tma_load_2d_2sm(base + o * kABytes, maps[o], fb, k0, row_a);
                                tma_load_2d_2sm(base + o * kABytes + kBBytes, maps[o], fb, k0, row_a + kBRows);
                            }
                            if (o < nops && !(PASS == 3 && o < 2))           // B side (PASS 3: B hi/lo of two column blocks)
                                tma_load_2d_2sm(base + kBOff + o * kBBytes, maps[PASS == 3 && o >= 4 ? o - 2 : o], fb, k0,
                                                PASS == 3 && o >= 4 ? row_b + kTile : row_b);
                        }
                    }
                    __syncwarp();
                    if (++stage == kStages) { stage = 0; phase ^= 1; }
                }
            }
            // CTAs with fewer tiles still owe their arrivals to the later waves
            if (p.wave_sync && wave < num_waves && wave > 0 && lane == 0) atomicAdd(wave_ctr, num_waves - wave);
        }
    } else if (warp == 1) {
        // =========================== MMA issuer (leader CTA only) ===========================
        if (rank == 0) {
            constexpr uint32_t idesc = make_idesc_f16(kPair, kTile);     // M = 256 over the pair, N = 128
            int stage = 0;
            uint32_t phase = 0;
            int acc = 0;
            uint32_t acc_phase = 0;
            for (int t = pair; t < num_tiles; t += num_pairs) {
                for (int ch = 0; ch < num_chunks; ++ch) {
                    mbar_wait(tempty_bar(acc), acc_phase ^ 1);
                    tc_fence_after();
                    const uint32_t d0 = tmem_base + acc * 256;        // P0 (pass 1: Q) accumulator columns
                    const uint32_t d1 = d0 + 128;                     // P1 (pass 1: P2) accumulator columns
                    for (int kb = 0; kb < kKbPerChunk; ++kb) {
                        mbar_wait(full_bar(stage), phase);
                        tc_fence_after();
                        const uint32_t base = smem_base + stage * kStageBytes;
                        if (elect_one()) {
                            uint64_t a[kOps < 6 ? 6 : kOps], b[kOps < 6 ? 6 : kOps];
#pragma unroll
                            for (int o = 0; o < kOps; ++o) {
                                a[o] = make_smem_desc<kRowBytes>(base + o * kABytes);
                                b[o] = make_smem_desc<kRowBytes>(base + kBOff + o * kBBytes);
                            }
#pragma unroll
                            for (int ks = 0; ks < kBK / 16; ++ks) {
                                const uint64_t adv = (uint64_t)(ks * 32 >> 4);     // 16 fp16 = 32 bytes along K
                                const uint32_t accum = (kb | ks) != 0;             // 0: start the chunk from zero
                                // SQUARE(X): X.X = Xhi.Xhi + Xhi.Xlo + Xlo.Xhi              (Eqs. 14-16)
                                auto square = [&](uint32_t d, int xh, int xl) {
                                    umma_f16<2>(d, a[xh] + adv, b[xh] + adv, idesc, accum);
                                    umma_f16<2>(d, a[xh] + adv, b[xl] + adv, idesc, 1);
                                    umma_f16<2>(d, a[xl] + adv, b[xh] + adv, idesc, 1);
                                };
                                // CROSS(X, Y): X.Y + Y.X, three partial products each        (Eqs. 44-46)
                                auto cross2 = [&](uint32_t d, int xh, int xl, int yh, int yl) {
                                    umma_f16<2>(d, a[xh] + adv, b[yh] + adv, idesc, accum);     // Xhi.Yhi
                                    umma_f16<2>(d, a[yh] + adv, b[xh] + adv, idesc, 1);         // Yhi.Xhi
                                    umma_f16<2>(d, a[xh] + adv, b[yl] + adv, idesc, 1);         // Xhi.Ylo
                                    umma_f16<2>(d, a[xl] + adv, b[yh] + adv, idesc, 1);         // Xlo.Yhi
                                    umma_f16<2>(d, a[yh] + adv, b[xl] + adv, idesc, 1);         // Yhi.Xlo
                                    umma_f16<2>(d, a[yl] + adv, b[xh] + adv, idesc, 1);         // Ylo.Xhi
                                };
                                auto cross = [&](uint32_t d, int yh, int yl) { cross2(d, PM_H, PM_L, yh, yl); };
                                if (PASS == 0) {            // P0 = M.M, P1 = M.S1 + S1.M
                                    if (with_p0) square(d0, PM_H, PM_L);
                                    if (!WIDE && with_p1) cross(d1, PY_H, PY_L);
                                } else if (PASS == 3) {     // C = A.B^T: Ahi.Bhi + Ahi.Blo + Alo.Bhi, two column blocks
                                    umma_f16<2>(d0, a[PM_H] + adv, b[PY_H] + adv, idesc, accum);
                                    umma_f16<2>(d0, a[PM_H] + adv, b[PY_L] + adv, idesc, 1);
                                    umma_f16<2>(d0, a[PM_L] + adv, b[PY_H] + adv, idesc, 1);
                                    umma_f16<2>(d1, a[PM_H] + adv, b[PZ_H] + adv, idesc, accum);
                                    umma_f16<2>(d1, a[PM_H] + adv, b[PZ_L] + adv, idesc, 1);
                                    umma_f16<2>(d1, a[PM_L] + adv, b[PZ_H] + adv, idesc, 1);
                                } else if (PASS == 1) {     // Q = S1.S1, P2 = M.S2 + S2.M
                                    square(d0, PY_H, PY_L);
                                    cross(d1, PZ_H, PZ_L);
                                } else if (PASS == 4) {     // Q3 = S1.S2 + S2.S1, P3 = M.S3 + S3.M
                                    cross2(d0, PY_H, PY_L, PZ_H, PZ_L);
                                    cross(d1, kOps > 6 ? 6 : 0, kOps > 6 ? 7 : 1);
                                } else {                    // two more first-order fields: M.Y + Y.M, M.Z + Z.M
                                    if (with_p0) cross(d0, PY_H, PY_L);
                                    if (with_p1) cross(d1, PZ_H, PZ_L);
                                }
                            }
                            umma_commit_2sm(empty_bar(stage), 0b11);       // frees the smem stage in both CTAs
                            if (kb == kKbPerChunk - 1)
                                umma_commit_2sm(tfull_bar(acc), 0b11);     // chunk accumulators complete, both CTAs
                        }
                        __syncwarp();
                        if (++stage == kStages) { stage = 0; phase ^= 1; }
                    }
                    if (++acc == kAccStages) { acc = 0; acc_phase ^= 1; }
                }
            }
        }
    } else if (warp >= kEpiWarp0) {
        // =========================== epilogue (both CTAs) ===========================
        const int q = warp & 3;                         // TMEM lane quadrant this warp may read
        const int half = (warp - kEpiWarp0) >> 2;       // which 64 accumulator columns
        const int ld = p.n_pad;
        const float sig = (float)c.sigma;
        const float unscale0 = exp2f(-2.f * (float)p.pb.s0_shift);
        const float unscale1 = exp2f(-(float)(p.pb.s0_shift + c.e1_in));
        const float scale0 = exp2f((float)p.pb.s0_shift);
        const float scale1 = exp2f((float)c.e1_out);
        const float unscale_q = exp2f(-2.f * (float)c.e1_in);                     // S1.S1 sums
        const float unscale2 = exp2f(-(float)(p.pb.s0_shift + c.e2_in));          // M.S2 + S2.M sums
        const float scale2 = exp2f((float)c.e2_out);
        const float unscale3 = exp2f(-(float)(p.pb.s0_shift + c.e3_in));          // PASS 2: M.Z + Z.M sums
        const float unscale_ab = exp2f(-(float)(c.e2_in + c.e1_in));              // PASS 3: A scaled by 2^e2, B by 2^e1; PASS 4: S1.S2 + S2.S1 sums
        const float scale3 = exp2f((float)c.e3_out);
        const bool upd0 = c.mode0 == MODE_ACTIVE;
        const bool conv0 = c.conv0 != 0;                // FroErr1 wanted (stop layer or frozen)
        EpiOut o0, o1;
        if (PASS == 0) {
            o0.dst = p.s0; o0.old = p.s0;
            o0.hi = p.h[c.s0_buf ^ 1][MH]; o0.lo = p.h[c.s0_buf ^ 1][ML];
            o1.dst = p.s1[c.s1_buf ^ 1]; o1.old = p.s1[c.s1_buf];
            o1.hi = p.h[c.s1_buf ^ 1][S1H]; o1.lo = p.h[c.s1_buf ^ 1][S1L];
            o0.m_old = o0.m_dst = &p.emap32[0];
            o0.m_hl = &p.emap16[c.s0_buf ^ 1][0][0];
            o1.m_old = &p.emap32[1 + c.s1_buf]; o1.m_dst = &p.emap32[1 + (c.s1_buf ^ 1)];
            o1.m_hl = &p.emap16[c.s1_buf ^ 1][1][0];
        } else if (PASS == 1) {
            o0.dst = nullptr; o0.old = nullptr; o0.hi = nullptr; o0.lo = nullptr;
            o1.dst = p.s2[c.s2_buf ^ 1]; o1.old = p.s2[c.s2_buf];
            o1.hi = p.h[c.s2_buf ^ 1][S2H]; o1.lo = p.h[c.s2_buf ^ 1][S2L];
        } else if (PASS == 4) {
            o0.dst = nullptr; o0.old = nullptr; o0.hi = nullptr; o0.lo = nullptr;
            o1.dst = p.s3[c.s3_buf ^ 1]; o1.old = p.s3[c.s3_buf];
            o1.hi = p.h[c.s3_buf ^ 1][S3H]; o1.lo = p.h[c.s3_buf ^ 1][S3L];
        } else {
            o0.dst = p.s2[c.s2_buf ^ 1]; o0.old = p.s2[c.s2_buf];
            o0.hi = p.h[c.s2_buf ^ 1][S2H]; o0.lo = p.h[c.s2_buf ^ 1][S2L];
            o1.dst = p.s3[c.s3_buf ^ 1]; o1.old = p.s3[c.s3_buf];
            o1.hi = p.h[c.s3_buf ^ 1][S3H]; o1.lo = p.h[c.s3_buf ^ 1][S3L];
        }

        double r_tr = 0.0, r_fs0 = 0.0, r_f0 = 0.0, r_f1 = 0.0, r_dummy = 0.0;
        float r_mx1 = 0.f, r_mx0 = 0.f, r_mx_dummy = 0.f;
        int acc = 0;
        uint32_t acc_phase = 0;
        // TMA epilogue (PASS 0): this warp's staging, and the steps of a tile: 4 per live product
        EpiTma et;
        uint32_t ring_phase = 0;
        {
            const uint32_t eb = epi_base + (uint32_t)(warp - kEpiWarp0) * kEpiWarpBytes;
            et.ring[0] = eb; et.ring[1] = eb + kEpiRing;
            et.dhi = eb + kEpiDhi; et.dlo = eb + kEpiDlo; et.thi = eb + kEpiThi; et.tlo = eb + kEpiTlo;
            et.bar[0] = ring_bar(warp - kEpiWarp0, 0); et.bar[1] = ring_bar(warp - kEpiWarp0, 1);
        }
        const bool tma_on = kTmaEpi && !p.epilogue_direct;
        const bool do0 = tma_on && with_p0 && upd0, do1 = tma_on && with_p1;
        const int ns = 4 * (int)do0 + 4 * (int)do1;
        const int pre_ch = num_chunks > 4 ? num_chunks - 4 : 0;       // where the first old blocks are requested
        for (int t = pair; t < num_tiles; t += num_pairs) {
            const uint32_t tl = tile_list[t];
            const int ti = 2 * (int)(tl & 0xFFFF) + (int)rank, tj = (int)(tl >> 16);
            const int gr = ti * kTile + q * 32 + lane;  // global row of this thread's TMEM lane
            const int gc_base = tj * kTile + half * kHalfCols;
            // the pair tile (IP, J = 2 IP) holds block (2 IP + 1, 2 IP) below the diagonal: its mirror is
            // computed by the pair tile (IP, 2 IP + 1), so the peer CTA only drains it
            const bool live = PASS == 3 || ti <= tj;
            const bool tma_tile = kTmaEpi && live && ns > 0;      // diagonal tiles too (see final_epilogue_tma)
            const int gr0 = ti * kTile + q * 32;          // first row of this warp's 32 x 64 block
            float a0[kHalfCols], a1[kHalfCols];
#pragma unroll
            for (int j = 0; j < kHalfCols; ++j) { a0[j] = 0.f; a1[j] = 0.f; }
            // ---- promoted accumulation: drain every chunk with round-to-nearest adds
            for (int ch = 0; ch < num_chunks; ++ch) {
                if (kTmaEpi && tma_tile && ch == pre_ch && lane == 0) {
                    // old iterate of steps 0 and 1 into the ring (the previous tile's stores have long been read),
                    // the rest of this warp's block into L2
                    bulk_wait_read<0>();
                    for (int s = 0; s < ns; ++s) {
                        const CUtensorMap* m = (do0 && s < 4) ? o0.m_old : o1.m_old;
                        const int gc = gc_base + (s & 3) * kSub;
                        if (s < 2) {
                            mbar_arrive_expect_tx(et.bar[s], kSub * 32 * 4);
                            tma_load_2d(et.ring[s], m, et.bar[s], gc, gr0);
                        } else {
                            tma_prefetch_l2_2d(m, gc, gr0);
                        }
                    }
                }
                mbar_wait(tfull_bar(acc), acc_phase);
                tc_fence_after();
                const uint32_t trow = tmem_base + ((uint32_t)(q * 32) << 16) + acc * 256 + half * kHalfCols;
                uint32_t v[16];
                if (live) {
                    if (with_p0) {
#pragma unroll
                        for (int g = 0; g < kHalfCols / 16; ++g) {
                            tmem_ld_32x16(trow + g * 16, v);
                            tmem_ld_wait();
#pragma unroll
                            for (int j = 0; j < 16; ++j) a0[g * 16 + j] += __uint_as_float(v[j]);
                        }
                    }
                    if (with_p1) {
#pragma unroll
                        for (int g = 0; g < kHalfCols / 16; ++g) {
                            tmem_ld_32x16(trow + 128 + g * 16, v);
                            tmem_ld_wait();
#pragma unroll
                            for (int j = 0; j < 16; ++j) a1[g * 16 + j] += __uint_as_float(v[j]);
                        }
                    }
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive_cluster(tempty_bar(acc), 0);      // on the leader's barrier
                if (++acc == kAccStages) { acc = 0; acc_phase ^= 1; }
            }
            if (!live) continue;
            // ---- branch, update, re-split, reductions
            const bool diag = ti == tj;
            if (PASS == 0) {
                if (with_p0 && !(tma_tile && upd0))       // diagonal tiles, and the measure-only D0 stop layer
                    final_epilogue<0>(a0, o0, ld, gr, gc_base, diag, upd0, sig, unscale0, scale0, !upd0, r_tr, r_fs0,
                                      r_f0, r_mx_dummy);
                if (with_p1 && !tma_tile)
                    final_epilogue<1>(a1, o1, ld, gr, gc_base, diag, true, sig, unscale1, scale1, conv0, r_dummy,
                                      r_dummy, r_f1, r_mx1);
                if (kTmaEpi && tma_tile) {
                    if (do0)
                        final_epilogue_tma<0>(a0, o0, et, ring_phase, 0, ns, o1.m_old, gr0, gc_base, lane, sig * unscale0,
                                              unscale0, scale0, false, diag, sig, ld, r_tr, r_fs0, r_dummy, r_mx_dummy);
                    if (do1)
                        final_epilogue_tma<1>(a1, o1, et, ring_phase, do0 ? 4 : 0, ns, nullptr, gr0, gc_base, lane,
                                              sig * unscale1, unscale1, scale1, conv0, diag, sig, ld, r_dummy, r_dummy,
                                              r_f1, r_mx1);
                }
            } else if (PASS == 3) {
                // C = 2^-(eA+eB) (A.B^T sums): plain fp32 output, no update, no split, no mirror
                float* d = p.s1[1] + (size_t)gr * ld + gc_base;
#pragma unroll
                for (int j = 0; j < kHalfCols; j += 4) {
                    *reinterpret_cast<float4*>(d + j) = make_float4(unscale_ab * a0[j], unscale_ab * a0[j + 1],
                                                                    unscale_ab * a0[j + 2], unscale_ab * a0[j + 3]);
                    *reinterpret_cast<float4*>(d + kTile + j) = make_float4(unscale_ab * a1[j], unscale_ab * a1[j + 1],
                                                                            unscale_ab * a1[j + 2], unscale_ab * a1[j + 3]);
                }
            } else if (PASS == 2) {
                // two more first-order fields, each exactly as P1 of pass 0
                if (with_p0)
                    final_epilogue<1>(a0, o0, ld, gr, gc_base, diag, true, sig, unscale2, scale2, conv0, r_dummy,
                                      r_dummy, r_f0, r_mx0);
                if (with_p1)
                    final_epilogue<1>(a1, o1, ld, gr, gc_base, diag, true, sig, unscale3, scale3, conv0, r_dummy,
                                      r_dummy, r_f1, r_mx1);
            } else if (PASS == 4) {
                // V3 = 2^-(a+e3) P3 + 2^-(e1+e2) Q3: both factors are powers of two, one fp32 rounding per element
#pragma unroll
                for (int j = 0; j < kHalfCols; ++j) a1[j] = fmaf(unscale_ab, a0[j], unscale3 * a1[j]);
                final_epilogue<1>(a1, o1, ld, gr, gc_base, diag, true, sig, 1.f, scale3, true, r_dummy, r_dummy,
                                  r_f1, r_mx1);
            } else {
                // V2 = 2^-(a+e2) P2 + 2^-(2 e1) Q: both factors are powers of two, one fp32 rounding per element
#pragma unroll
                for (int j = 0; j < kHalfCols; ++j) a1[j] = fmaf(unscale_q, a0[j], unscale2 * a1[j]);
                final_epilogue<1>(a1, o1, ld, gr, gc_base, diag, true, sig, 1.f, scale2, true, r_dummy, r_dummy,
                                  r_f1, r_mx1);
            }
        }
        if (kTmaEpi && lane == 0) bulk_wait<0>();      // this warp's TMA stores have been performed
        // per-warp partials, fixed slot per (CTA, warp): the finalizer sums them in a fixed order
        r_tr = warp_sum(r_tr);
        r_fs0 = warp_sum(r_fs0);
        r_f0 = warp_sum(r_f0);
        r_f1 = warp_sum(r_f1);
        const double mx1 = warp_max((double)r_mx1);
        const double mx0 = warp_max((double)r_mx0);
        if (lane == 0) {
            // component-major: [RED_x][slot], so that the control step reads consecutive doubles
            double* out = (PASS == 0 ? p.partials : (PASS == 4 ? p.partials3 : p.partials2)) +
                          ((size_t)blockIdx.x * kNumEpiWarps + (warp - kEpiWarp0));
            out[RED_TR_S0 * kRedStride] = r_tr;
            out[RED_FRO_S0 * kRedStride] = r_fs0;
            out[RED_FRO0 * kRedStride] = PASS == 0 ? r_f0 : 0.0;
            out[RED_FRO1 * kRedStride] = PASS == 0 ? r_f1 : 0.0;
            out[RED_MAX1 * kRedStride] = PASS == 0 ? mx1 : 0.0;
            out[RED_FRO2 * kRedStride] = PASS == 1 ? r_f1 : (PASS == 2 ? r_f0 : 0.0);      // slot 2: S2, or field 2
            out[RED_MAX2 * kRedStride] = PASS == 1 ? mx1 : (PASS == 2 ? mx0 : 0.0);
            out[RED_FRO3 * kRedStride] = (PASS == 2 || PASS == 4) ? r_f1 : 0.0;             // slot 3: field 3, or S3
            out[RED_MAX3 * kRedStride] = (PASS == 2 || PASS == 4) ? mx1 : 0.0;
        }
    }

    // ---- teardown: neither CTA may leave while its peer can still read its smem or signal its barriers
    tc_fence_before();
    cluster_sync_all();
    if (warp == 1) {
        tc_fence_after();
        tmem_dealloc<2>(tmem_base, kTmemCols);
    }
    if (PASS != 0) return;          // pass 0 of the same layer follows on the stream and takes the decisions

    // ---- the last CTA of the launch runs Algorithms 2-3 for this layer
    __shared__ int is_last;
    if (threadIdx.x == 0) {
        __threadfence();
        const unsigned int prev = atomicAdd(&p.ctl->ticket, 1u);
        is_last = (prev == gridDim.x - 1);
    }
    __syncthreads();
    if (is_last) {
        __threadfence();
        // fixed-order fp64 reduction by the whole CTA: thread t sums slots t, t + 384, ...; a shuffle tree per warp;
        // the twelve warp sums are added in warp order
        __shared__ double s_red[kNumThreads / 32][RED_COUNT];
        const int nslots = gridDim.x * kNumEpiWarps;
        const bool second = p.pb.order >= 2 || p.pb.nfields >= 2;       // slots 2, 3 come from the other passes
        const bool third = p.pb.order == 3;                             // slot 3 from the order-3 pass
        double red[RED_COUNT];
#pragma unroll
        for (int k = 0; k < RED_COUNT; ++k) red[k] = 0.0;
        for (int s = (int)threadIdx.x; s < nslots; s += kNumThreads) {
            const double* in = p.partials + s;          // written by other CTAs: read past L1
            const double* in2 = p.partials2 + s;
            const double* in3 = p.partials3 + s;
#pragma unroll
            for (int k = 0; k < RED_COUNT; ++k) {
                if (k == RED_MAX1) red[k] = fmax(red[k], __ldcg(in + k * kRedStride));
                else if (k == RED_MAX2) { if (second) red[k] = fmax(red[k], __ldcg(in2 + k * kRedStride)); }
                else if (k == RED_MAX3) { if (second) red[k] = fmax(red[k], __ldcg((third ? in3 : in2) + k * kRedStride)); }
                else if (k == RED_FRO2) { if (second) red[k] += __ldcg(in2 + k * kRedStride); }
                else if (k == RED_FRO3) { if (second) red[k] += __ldcg((third ? in3 : in2) + k * kRedStride); }
                else if (k < RED_FRO2) red[k] += __ldcg(in + k * kRedStride);
            }
        }
#pragma unroll
        for (int k = 0; k < RED_COUNT; ++k) {
            if (k == RED_MAX1 || k == RED_MAX2 || k == RED_MAX3) red[k] = warp_max(red[k]);
            else red[k] = warp_sum(red[k]);
            if (lane == 0) s_red[warp][k] = red[k];
        }
        __syncthreads();
        // the twelve warp sums of component k are added by lane k (fp64 adds are slow: not one thread for all)
        if (warp == 0) {
            double v = 0.0;
            if (lane < RED_COUNT) {
                const bool is_max = lane == RED_MAX1 || lane == RED_MAX2 || lane == RED_MAX3;
                v = s_red[0][lane];
                for (int w = 1; w < kNumThreads / 32; ++w) v = is_max ? fmax(v, s_red[w][lane]) : v + s_red[w][lane];
            }
#pragma unroll
            for (int k = 0; k < RED_COUNT; ++k) red[k] = __shfl_sync(0xffffffffu, v, k);
        }
        if (threadIdx.x == 0) {
            DmptCtl nc = *p.ctl;
            nc.ticket = 0;
            nc.wave = 0;
            nc.wave2 = 0;
            nc.wave3 = 0;
            if (p.pb.pair_side == 2) handoff_merge(nc, p.handoff[nc.layer]);      // what this launch ran with
            control_finalize(nc, p.logs, p.pb, red, p.handoff);
            *p.ctl = nc;
            if (p.use_cond) cudaGraphSetConditional(p.cond, nc.done ? 0u : 1u);
        }
    }
}

}  // namespace dmpt
