// C ABI of the DNN-SP2-PT hot path (include/dmpt.h): context, workspace carve-up, TMA tensor
// maps, and the host driver that enqueues bounds -> transform -> split -> layers on one stream.
// No device memory is allocated here and there is no CPU fallback.
#include <cuda.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <vector>

#include "../../include/dmpt.h"
#include "control.cuh"
#include "kernels_hbm.cuh"
#include "layer_kernel.cuh"

using namespace dmpt;

namespace {

constexpr int kMaxLayersCap = 1024;
constexpr int kPartialDoubles = 8192 * RED_COUNT;   // >= max(transform grid * 3, layer grid * 4 * RED_COUNT)
constexpr int kNumEvents = 4;
constexpr int kFlagSlots = 64;

size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

struct Carve {
    size_t off = 0;
    size_t take(size_t bytes) {
        size_t o = off;
        off = align_up(off + bytes, 256);
        return o;
    }
};

struct Layout {
    int n, n_pad, order, nfields, num_tiles;
    size_t ctl, bounds, h1max, s2_est, sigma, tr_s, tr_x, id_err, fro1, fro2, fro3, partials, partials2, partials3, handoff,
        tiles, tiles_full;
    size_t s0, s1[2], s2[2], s3[2];
    size_t h[2][8];          // [buffer][S0hi, S0lo, S1hi, S1lo, slot-2 hi, lo, slot-3 hi, lo]
    size_t stage_h0, stage_h1, stage_hx[2], lanczos, clk;
    size_t total;
};

// pair tiles (IP, J): block rows 2 IP, 2 IP + 1 x block column J >= 2 IP, nb even
int num_tiles_for(int nb) {
    int t = 0;
    for (int ip = 0; ip < nb / 2; ++ip) t += nb - 2 * ip;
    return t;
}

// response slots in use: 1 (order 1), 2 (order 2, or two fields), 3 (order 3, or three fields); 0 at order 0
int num_slots(int order, int nfields) { return order >= 2 ? order : (order == 1 ? nfields : 0); }

Layout make_layout(int n, int order, int nfields) {
    Layout L{};
    L.n = n;
    L.order = order;
    L.nfields = nfields;
    L.n_pad = (int)align_up((size_t)n, kPair);
    const int nb = L.n_pad / kTile;
    L.num_tiles = num_tiles_for(nb);
    const size_t np2 = (size_t)L.n_pad * L.n_pad;
    Carve c;
    L.ctl = c.take(sizeof(DmptCtl));
    L.bounds = c.take(2 * sizeof(long long));
    L.h1max = c.take(4 * sizeof(unsigned int));
    L.s2_est = c.take(4 * sizeof(unsigned long long));
    L.sigma = c.take(kMaxLayersCap * sizeof(int));
    L.tr_s = c.take(kMaxLayersCap * sizeof(double));
    L.tr_x = c.take(kMaxLayersCap * sizeof(double));
    L.id_err = c.take(kMaxLayersCap * sizeof(double));
    L.fro1 = c.take(kMaxLayersCap * sizeof(double));
    L.fro2 = c.take(kMaxLayersCap * sizeof(double));
    L.fro3 = c.take(kMaxLayersCap * sizeof(double));
    L.partials = c.take(kPartialDoubles * sizeof(double));
    L.partials2 = c.take(kPartialDoubles * sizeof(double));
    L.partials3 = c.take(kPartialDoubles * sizeof(double));
    L.handoff = c.take((kMaxLayersCap + 2) * sizeof(DmptHandoff));
    L.lanczos = c.take(sizeof(LanczosState) + 3 * (size_t)L.n_pad * sizeof(double));
    L.clk = c.take(sizeof(DmptClockStamps));
    L.tiles = c.take((size_t)L.num_tiles * sizeof(uint32_t));
    L.tiles_full = c.take((size_t)(nb / 2) * nb * sizeof(uint32_t));
    L.s0 = c.take(np2 * 4);
    L.s1[0] = c.take(np2 * 4);
    L.s1[1] = c.take(np2 * 4);
    const int slots = num_slots(order, nfields);
    if (slots >= 2) {
        L.s2[0] = c.take(np2 * 4);
        L.s2[1] = c.take(np2 * 4);
    }
    if (slots >= 3) {
        L.s3[0] = c.take(np2 * 4);
        L.s3[1] = c.take(np2 * 4);
    }
    const int nh = 2 + 2 * (slots < 1 ? 1 : slots);
    for (int b = 0; b < 2; ++b)
        for (int m = 0; m < nh; ++m) L.h[b][m] = c.take(np2 * 2);
    L.stage_h0 = c.take((size_t)n * n * 4);
    L.stage_h1 = c.take((size_t)n * n * 4);
    for (int f = 0; f < 2; ++f) L.stage_hx[f] = (order == 1 && nfields >= f + 2) ? c.take((size_t)n * n * 4) : 0;
    L.total = c.off;
    return L;
}

// Launch order of the upper-triangular pair tiles: bands of `band` pair rows, column by column inside
// a band, so that the ~#SM/2 pair tiles in flight share few row panels (L2 reuse of the operand panels).
// The pair tiles that hold a diagonal block ((IP, 2 IP) and (IP, 2 IP + 1)) come last, together: their final
// epilogue is the element-wise one (the mirror of a diagonal block lies inside the block), several times slower
// than the TMA epilogue of the other tiles, and with wave-aligned producers every CTA of a wave waits for the
// slowest tile in it - spread over the bands, one such tile per wave held all 74 pairs back on every wave.
std::vector<uint32_t> make_tile_order(int nb, int band) {
    std::vector<uint32_t> t, diag;
    t.reserve(num_tiles_for(nb));
    const int nbp = nb / 2;
    for (int b0 = 0; b0 < nbp; b0 += band) {
        const int b1 = b0 + band < nbp ? b0 + band : nbp;
        for (int j = 2 * b0; j < nb; ++j)
            for (int ip = b0; ip < b1 && 2 * ip <= j; ++ip)
                (j <= 2 * ip + 1 ? diag : t).push_back((uint32_t)ip | ((uint32_t)j << 16));
    }
    t.insert(t.end(), diag.begin(), diag.end());
    return t;
}

// Every 256 x 256 tile (IP, J even), same band order: the general product C = A.B^T has no symmetry to exploit.
std::vector<uint32_t> make_tile_order_full(int nb, int band) {
    std::vector<uint32_t> t;
    const int nbp = nb / 2;
    t.reserve((size_t)nbp * nbp);
    for (int b0 = 0; b0 < nbp; b0 += band) {
        const int b1 = b0 + band < nbp ? b0 + band : nbp;
        for (int j = 0; j < nb; j += 2)                      // block columns j, j + 1 together
            for (int ip = b0; ip < b1; ++ip) t.push_back((uint32_t)ip | ((uint32_t)j << 16));
    }
    return t;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*,
                                  CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                  CUtensorMapFloatOOBfill);

}  // namespace

struct dmpt_ctx {
    int n = 0, n_occ = 0, ld_in = 0;
    dmpt_options opt{};
    Layout L{};
    uint8_t* ws = nullptr;
    cudaStream_t stream = nullptr;
    const float* d_h0 = nullptr;
    const float* d_h1 = nullptr;          // field 1
    const float* d_h1x[2] = {nullptr, nullptr};   // fields 2, 3 (multi-field contexts)
    int num_sms = 0;
    int grid_layer = 0;
    int s0_shift = 14;
    LayerParams lp{};
    cudaEvent_t ev[kNumEvents]{};
    cudaEvent_t ev_t[6]{};       // 0 start, 1 loop start, 2 loop end, 3 end, 4 after bounds, 5 after transform
    int* h_flags = nullptr;      // pinned: ctl.done after every chunk of launches
    int* h_flags0 = nullptr;     // pinned: ctl.conv0 after every chunk (dmpt_run_host: early copy of D0)
    cudaStream_t side = nullptr; // copy stream of dmpt_run_host's early D0 read-back
    cudaEvent_t ev_side = nullptr;
    DmptCtl* h_ctl = nullptr;    // pinned
    // device-side loop (dmpt_options::loop_graph): one WHILE node whose body is the launches of a layer
    cudaGraph_t loop_graph = nullptr;
    cudaGraphExec_t loop_exec = nullptr;
    cudaStream_t capture = nullptr;
    int loop_n_occ = -1;         // the graph's kernel nodes hold a copy of LayerParams: rebuilt when n_occ changes
    bool loop_used = false;      // the current run went through the graph
    char err[256] = {0};

    template <typename T>
    T* at(size_t off) const { return reinterpret_cast<T*>(ws + off); }
};

#define CK(call)                                                                             \
    do {                                                                                     \
        cudaError_t e_ = (call);                                                             \
        if (e_ != cudaSuccess) {                                                             \
            snprintf(ctx->err, sizeof ctx->err, "%s: %s (%s:%d)", #call, cudaGetErrorString(e_), \
                     __FILE__, __LINE__);                                                    \
            return DMPT_ECUDA;                                                               \
        }                                                                                    \
    } while (0)

extern "C" void dmpt_default_options(dmpt_options* opt) {
    if (!opt) return;
    memset(opt, 0, sizeof *opt);
    opt->max_layers = 200;
    opt->order = 1;
    opt->s0_shift = -1;
    opt->s1_autoscale = 1;
    opt->bounds = 0;
    opt->wave_sync = 1;
    opt->num_fields = 1;
}

extern "C" size_t dmpt_workspace_bytes(int n, int order) {
    if (n <= 0 || order < 0 || order > 3 || n > 65535 * kTile) return 0;
    return make_layout(n, order, 1).total;
}

extern "C" size_t dmpt_workspace_bytes_fields(int n, int num_fields) {
    if (n <= 0 || num_fields < 1 || num_fields > 3 || n > 65535 * kTile) return 0;
    return make_layout(n, 1, num_fields).total;
}

extern "C" const char* dmpt_strerror(int code) {
    switch (code) {
        case DMPT_OK: return "ok";
        case DMPT_EINVAL: return "invalid argument";
        case DMPT_ESTATE: return "dmpt_run called before dmpt_set_hamiltonian";
        case DMPT_ECUDA: return "CUDA error (see dmpt_last_cuda_error)";
        case DMPT_EDEGENERATE: return "spectral bounds degenerate: eps_max - eps_min not positive and finite";
        case DMPT_ENOCONV: return "max_layers reached before the stopping tests fired";
        case DMPT_ENUMERIC: return "NaN/Inf in the scalar state";
        case DMPT_EWORKSPACE: return "workspace too small or not 256-byte aligned";
        case DMPT_ELIMIT: return "size beyond a compiled-in limit (n > DMPT_NOALLOC_MAX_N of the no-allocation entry point)";
        default: return "unknown error code";
    }
}

extern "C" const char* dmpt_last_cuda_error(const dmpt_ctx* ctx) { return ctx ? ctx->err : ""; }

static int build_tensor_maps(dmpt_ctx* ctx) {
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    CK(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres));
    if (!fn || qres != cudaDriverEntryPointSuccess) {
        snprintf(ctx->err, sizeof ctx->err, "cuTensorMapEncodeTiled not available from the driver");
        return DMPT_ECUDA;
    }
    EncodeTiledFn encode = reinterpret_cast<EncodeTiledFn>(fn);
    const Layout& L = ctx->L;
    const cuuint64_t dims[2] = {(cuuint64_t)L.n_pad, (cuuint64_t)L.n_pad};
    const cuuint64_t strides[1] = {(cuuint64_t)L.n_pad * 2};
    const cuuint32_t box[2] = {(cuuint32_t)kBK, (cuuint32_t)kBRows};
    const cuuint32_t estr[2] = {1, 1};
    const int slots = num_slots(L.order, L.nfields);
    const int nh = 2 + 2 * (slots < 1 ? 1 : slots);
    for (int b = 0; b < 2; ++b)
        for (int m = 0; m < nh; ++m) {
            CUresult r = encode(&ctx->lp.maps[b][m], CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 2,
                                ctx->at<void>(L.h[b][m]), dims, strides, box, estr,
                                CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_64B,
                                // 256-byte promotion: measured 30.73 -> 30.58 ms per layer at N = 16384 against 128 B
                                CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
            if (r != CUDA_SUCCESS) {
                snprintf(ctx->err, sizeof ctx->err, "cuTensorMapEncodeTiled failed with CUresult %d", (int)r);
                return DMPT_ECUDA;
            }
        }
    // order-0 contexts: the same two operand matrices again as 128-byte rows (64 columns, SWIZZLE_128B) in the unused
    // slots S3H, S3L, for the ground-state instantiation of pass 0 (dmpt_layer_kernel<0, true>)
    if (L.order == 0)
        for (int b = 0; b < 2; ++b)
            for (int m = 0; m < 2; ++m) {
                const cuuint32_t wbox[2] = {(cuuint32_t)(2 * kBK), (cuuint32_t)kBRows};
                CUresult r = encode(&ctx->lp.maps[b][S3H + m], CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 2,
                                    ctx->at<void>(L.h[b][m]), dims, strides, wbox, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                    CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
                if (r != CUDA_SUCCESS) {
                    snprintf(ctx->err, sizeof ctx->err, "cuTensorMapEncodeTiled (wide map) failed with CUresult %d", (int)r);
                    return DMPT_ECUDA;
                }
            }
    // epilogue maps of the layer kernel's TMA path (layer_kernel.cuh, final_epilogue_tma).  fp32 iterates: a 16 x 32 box,
    // swizzled so that one thread per row reads and writes it without bank conflicts
    void* f32[3] = {ctx->at<void>(L.s0), ctx->at<void>(L.s1[0]), ctx->at<void>(L.s1[1])};
    for (int i = 0; i < 3; ++i) {
        const cuuint64_t est1[1] = {(cuuint64_t)L.n_pad * 4};
        const cuuint32_t ebox[2] = {(cuuint32_t)kSub, 32};
        CUresult r = encode(&ctx->lp.emap32[i], CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, f32[i], dims, est1, ebox, estr,
                            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_64B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) {
            snprintf(ctx->err, sizeof ctx->err, "cuTensorMapEncodeTiled (epilogue map) failed with CUresult %d", (int)r);
            return DMPT_ECUDA;
        }
    }
    // (hi, lo) pairs as 3D tensors: dimension 2 = the word (hi: plane 0, lo: plane 1); the two matrices of a pair are
    // consecutive blocks of the workspace (make_layout), n_pad^2 fp16 apart
    for (int b = 0; b < 2; ++b)
        for (int pr = 0; pr < 2; ++pr)
            for (int t = 0; t < 2; ++t) {
                const bool mirrored = t == 1;
                if (L.h[b][2 * pr + 1] - L.h[b][2 * pr] != (size_t)L.n_pad * L.n_pad * 2) {
                    snprintf(ctx->err, sizeof ctx->err, "workspace layout: hi and lo of an operand pair are not adjacent");
                    return DMPT_ECUDA;
                }
                const cuuint64_t dims3[3] = {(cuuint64_t)L.n_pad, (cuuint64_t)L.n_pad, 2};
                const cuuint64_t str3[2] = {(cuuint64_t)L.n_pad * 2, (cuuint64_t)L.n_pad * L.n_pad * 2};
                // direct: 32 columns (two epilogue steps) x 32 rows, 64-byte rows; mirrored: 32 columns x 16 rows
                const cuuint32_t box3[3] = {32, (cuuint32_t)(mirrored ? kSub : 32), 2};
                const cuuint32_t es3[3] = {1, 1, 1};
                CUresult r = encode(&ctx->lp.emap16[b][pr][t], CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 3,
                                    ctx->at<void>(L.h[b][2 * pr]), dims3, str3, box3, es3, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                    mirrored ? CU_TENSOR_MAP_SWIZZLE_NONE : CU_TENSOR_MAP_SWIZZLE_64B,
                                    CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
                if (r != CUDA_SUCCESS) {
                    snprintf(ctx->err, sizeof ctx->err, "cuTensorMapEncodeTiled (operand-pair map) failed with CUresult %d", (int)r);
                    return DMPT_ECUDA;
                }
            }
    return DMPT_OK;
}

static int create_impl(dmpt_ctx** out, int n, const dmpt_options* opt, void* d_workspace, size_t workspace_bytes,
                       void* cuda_stream, int pair_side);

extern "C" int dmpt_create(dmpt_ctx** out, int n, const dmpt_options* opt, void* d_workspace,
                           size_t workspace_bytes, void* cuda_stream) {
    return create_impl(out, n, opt, d_workspace, workspace_bytes, cuda_stream, 0);
}

// pair_side: 0 = a context of its own; 1, 2 = the two sides of an order-parallel pair (dmpt_pair_create)
static int create_impl(dmpt_ctx** out, int n, const dmpt_options* opt, void* d_workspace, size_t workspace_bytes,
                       void* cuda_stream, int pair_side) {
    if (!out) return DMPT_EINVAL;
    *out = nullptr;
    dmpt_options o;
    if (opt) o = *opt; else dmpt_default_options(&o);
    if (n <= 0 || o.order < 0 || o.order > 3 || !d_workspace) return DMPT_EINVAL;
    if (o.max_layers <= 0) o.max_layers = 200;
    if (o.max_layers > kMaxLayersCap) o.max_layers = kMaxLayersCap;
    if (o.s0_shift > 15 || o.bounds < 0 || o.bounds > 2 || o.lanczos_steps < 0) return DMPT_EINVAL;
    if (pair_side) o.loop_graph = 0;
    if (o.num_fields == 0) o.num_fields = 1;
    if (o.num_fields < 1 || o.num_fields > 3 || (o.num_fields > 1 && o.order != 1)) return DMPT_EINVAL;
    const size_t need = o.num_fields > 1 ? dmpt_workspace_bytes_fields(n, o.num_fields) : dmpt_workspace_bytes(n, o.order);
    if (need == 0) return DMPT_EINVAL;
    if (workspace_bytes < need || (reinterpret_cast<uintptr_t>(d_workspace) & 255)) return DMPT_EWORKSPACE;

    dmpt_ctx* ctx = new dmpt_ctx();
    ctx->n = n;
    ctx->opt = o;
    ctx->s0_shift = o.s0_shift < 0 ? 14 : o.s0_shift;
    ctx->L = make_layout(n, o.order, o.num_fields);
    ctx->ws = static_cast<uint8_t*>(d_workspace);
    ctx->stream = static_cast<cudaStream_t>(cuda_stream);
    auto fail = [&](int code) {
        // keep the message reachable: the caller has no ctx on failure, so print it
        fprintf(stderr, "dmpt_create: %s\n", ctx->err);
        for (auto& e : ctx->ev) if (e) cudaEventDestroy(e);
        for (auto& e : ctx->ev_t) if (e) cudaEventDestroy(e);
        if (ctx->h_flags) cudaFreeHost(ctx->h_flags);
        if (ctx->h_flags0) cudaFreeHost(ctx->h_flags0);
        if (ctx->h_ctl) cudaFreeHost(ctx->h_ctl);
        if (ctx->side) cudaStreamDestroy(ctx->side);
        if (ctx->ev_side) cudaEventDestroy(ctx->ev_side);
        delete ctx;
        return code;
    };
#define CKC(call)                                                                              \
    do {                                                                                       \
        cudaError_t e_ = (call);                                                               \
        if (e_ != cudaSuccess) {                                                               \
            snprintf(ctx->err, sizeof ctx->err, "%s: %s", #call, cudaGetErrorString(e_));      \
            return fail(DMPT_ECUDA);                                                           \
        }                                                                                      \
    } while (0)
    int dev = 0;
    CKC(cudaGetDevice(&dev));
    CKC(cudaDeviceGetAttribute(&ctx->num_sms, cudaDevAttrMultiProcessorCount, dev));
    int cc_major = 0;
    CKC(cudaDeviceGetAttribute(&cc_major, cudaDevAttrComputeCapabilityMajor, dev));
    if (cc_major != 10) {
        snprintf(ctx->err, sizeof ctx->err, "device compute capability %d.x: this library is sm_100a only", cc_major);
        return fail(DMPT_ECUDA);
    }
    for (auto& e : ctx->ev) CKC(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    for (auto& e : ctx->ev_t) CKC(cudaEventCreate(&e));
    CKC(cudaHostAlloc(&ctx->h_flags, kFlagSlots * sizeof(int), cudaHostAllocDefault));
    CKC(cudaHostAlloc(&ctx->h_flags0, kFlagSlots * sizeof(int), cudaHostAllocDefault));
    CKC(cudaStreamCreateWithFlags(&ctx->side, cudaStreamNonBlocking));
    CKC(cudaEventCreateWithFlags(&ctx->ev_side, cudaEventDisableTiming));
    CKC(cudaHostAlloc(&ctx->h_ctl, sizeof(DmptCtl), cudaHostAllocDefault));
    CKC(cudaFuncSetAttribute(dmpt_layer_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes<0>()));
    CKC(cudaFuncSetAttribute(dmpt_layer_kernel<0, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes<0>()));
    CKC(cudaFuncSetAttribute(dmpt_layer_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes<1>()));
    CKC(cudaFuncSetAttribute(dmpt_layer_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes<2>()));
    CKC(cudaFuncSetAttribute(dmpt_layer_kernel<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes<3>()));
    CKC(cudaFuncSetAttribute(dmpt_layer_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes<4>()));

    const Layout& L = ctx->L;
    const int nb = L.n_pad / kTile;
    int band = 1;
    while ((band + 1) * (band + 1) <= ctx->num_sms) ++band;      // ~sqrt(#SM) block rows per band
    band = band / 2 > 0 ? band / 2 : 1;                          // ... in pair rows
    std::vector<uint32_t> tiles = make_tile_order(nb, band);
    CKC(cudaMemcpyAsync(ctx->at<void>(L.tiles), tiles.data(), tiles.size() * sizeof(uint32_t),
                        cudaMemcpyHostToDevice, ctx->stream));
    std::vector<uint32_t> tiles_full = make_tile_order_full(nb, band);
    CKC(cudaMemcpyAsync(ctx->at<void>(L.tiles_full), tiles_full.data(), tiles_full.size() * sizeof(uint32_t),
                        cudaMemcpyHostToDevice, ctx->stream));
    CKC(cudaStreamSynchronize(ctx->stream));
    // one CTA pair (cluster of 2, one TPC) per pair tile in flight
    int max_clusters = 0;
    {
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3(ctx->num_sms & ~1);
        cfg.blockDim = dim3(Warps<1>::kThreads);
        cfg.dynamicSmemBytes = smem_bytes<1>();
        CKC(cudaOccupancyMaxActiveClusters(&max_clusters, dmpt_layer_kernel<1>, &cfg));
    }
    if (max_clusters < 1) {
        snprintf(ctx->err, sizeof ctx->err, "no CTA pair of the layer kernel fits this device");
        return fail(DMPT_ECUDA);
    }
    if (max_clusters > ctx->num_sms / 2) max_clusters = ctx->num_sms / 2;
    if (max_clusters > kRedStride / (2 * kNumEpiWarps)) max_clusters = kRedStride / (2 * kNumEpiWarps);   // partials: [component][slot]
    ctx->grid_layer = 2 * (L.num_tiles < max_clusters ? L.num_tiles : max_clusters);

    LayerParams& lp = ctx->lp;
    lp.s0 = ctx->at<float>(L.s0);
    lp.s1[0] = ctx->at<float>(L.s1[0]);
    lp.s1[1] = ctx->at<float>(L.s1[1]);
    const int slots = num_slots(o.order, o.num_fields);
    const int nh = 2 + 2 * (slots < 1 ? 1 : slots);
    for (int b = 0; b < 2; ++b) {
        lp.s2[b] = slots >= 2 ? ctx->at<float>(L.s2[b]) : nullptr;
        lp.s3[b] = slots >= 3 ? ctx->at<float>(L.s3[b]) : nullptr;
        for (int m = 0; m < 8; ++m) lp.h[b][m] = m < nh ? ctx->at<__half>(L.h[b][m]) : nullptr;
    }
    lp.tiles = ctx->at<uint32_t>(L.tiles);
    lp.num_tiles = L.num_tiles;
    lp.tiles_full = ctx->at<uint32_t>(L.tiles_full);
    lp.num_tiles_full = (nb / 2) * (nb / 2);
    lp.n_pad = L.n_pad;
    lp.wave_sync = (o.wave_sync && L.num_tiles > ctx->grid_layer / 2) ? 1 : 0;
    lp.epilogue_direct = o.epilogue_direct ? 1 : 0;
    lp.ctl = ctx->at<DmptCtl>(L.ctl);
    lp.logs.sigma = ctx->at<int>(L.sigma);
    lp.logs.tr_s = ctx->at<double>(L.tr_s);
    lp.logs.tr_x = ctx->at<double>(L.tr_x);
    lp.logs.id_err = ctx->at<double>(L.id_err);
    lp.logs.fro1 = ctx->at<double>(L.fro1);
    lp.logs.fro2 = ctx->at<double>(L.fro2);
    lp.logs.fro3 = ctx->at<double>(L.fro3);
    lp.logs.clk = ctx->at<DmptClockStamps>(L.clk);
    lp.partials = ctx->at<double>(L.partials);
    lp.partials2 = ctx->at<double>(L.partials2);
    lp.partials3 = ctx->at<double>(L.partials3);
    lp.handoff = pair_side ? ctx->at<DmptHandoff>(L.handoff) : nullptr;
    lp.pb.pair_side = pair_side;
    lp.pb.n = n;
    lp.pb.n_pad = L.n_pad;
    lp.pb.n_occ = 0;
    lp.pb.order = o.order;
    lp.pb.max_layers = o.max_layers;
    lp.pb.s0_shift = ctx->s0_shift;
    lp.pb.s1_autoscale = o.s1_autoscale ? 1 : 0;
    lp.pb.nfields = o.num_fields;
    if (build_tensor_maps(ctx) != DMPT_OK) return fail(DMPT_ECUDA);
#undef CKC
    *out = ctx;
    return DMPT_OK;
}

extern "C" int dmpt_destroy(dmpt_ctx* ctx) {
    if (!ctx) return DMPT_EINVAL;
    cudaStreamSynchronize(ctx->stream);
    for (auto& e : ctx->ev) if (e) cudaEventDestroy(e);
    for (auto& e : ctx->ev_t) if (e) cudaEventDestroy(e);
    if (ctx->h_flags) cudaFreeHost(ctx->h_flags);
    if (ctx->h_flags0) cudaFreeHost(ctx->h_flags0);
    if (ctx->h_ctl) cudaFreeHost(ctx->h_ctl);
    if (ctx->side) cudaStreamDestroy(ctx->side);
    if (ctx->ev_side) cudaEventDestroy(ctx->ev_side);
    if (ctx->loop_exec) cudaGraphExecDestroy(ctx->loop_exec);
    if (ctx->loop_graph) cudaGraphDestroy(ctx->loop_graph);
    if (ctx->capture) cudaStreamDestroy(ctx->capture);
    delete ctx;
    return DMPT_OK;
}

extern "C" int dmpt_set_hamiltonian(dmpt_ctx* ctx, const float* d_h0, const float* d_h1, int ld, int n_occ) {
    if (!ctx || !d_h0 || (!d_h1 && ctx->opt.order != 0)) return DMPT_EINVAL;     // order 0 takes no perturbation
    if (ld < ctx->n || n_occ <= 0 || n_occ >= ctx->n) return DMPT_EINVAL;
    ctx->d_h0 = d_h0;
    ctx->d_h1 = d_h1;
    ctx->ld_in = ld;
    ctx->n_occ = n_occ;
    ctx->lp.pb.n_occ = n_occ;
    return DMPT_OK;
}

template <int PASS>
static int launch_pass(dmpt_ctx* ctx, cudaStream_t capture = nullptr) {
    // clusters of 2 come from the kernel's __cluster_dims__; the wave barrier needs every CTA resident:
    // a cooperative launch guarantees it or fails
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(ctx->grid_layer);
    cfg.blockDim = dim3(Warps<PASS>::kThreads);
    cfg.dynamicSmemBytes = smem_bytes<PASS>();
    cfg.stream = capture ? capture : ctx->stream;
    cudaLaunchAttribute attr[2];
    attr[0].id = cudaLaunchAttributeCooperative;
    attr[0].val.cooperative = ctx->lp.wave_sync ? 1 : 0;
    // without the wave barrier (at most one tile per CTA pair): programmatic dependent launch, see the kernel's first lines
    attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[1].val.programmaticStreamSerializationAllowed = (ctx->lp.wave_sync || ctx->opt.no_pdl || capture) ? 0 : 1;
    cfg.attrs = attr;
    cfg.numAttrs = 2;
    if (PASS == 0 && ctx->opt.order == 0 && ctx->lp.pb.pair_side == 0 && !ctx->opt.order0_narrow)
        CK(cudaLaunchKernelEx(&cfg, dmpt_layer_kernel<0, true>, ctx->lp));      // ground state: 128-byte operand rows
    else
        CK(cudaLaunchKernelEx(&cfg, dmpt_layer_kernel<PASS>, ctx->lp));
    return DMPT_OK;
}

// One layer: at order 2 the S2 pass goes first (it reads the iterates pass 0 is about to replace and
// leaves its reductions for pass 0's control step).
extern "C" int dmpt_set_hamiltonian_fields(dmpt_ctx* ctx, const float* d_h0, const float* const* d_h1, int ld,
                                           int n_occ) {
    if (!ctx || !d_h0 || !d_h1 || ctx->opt.order != 1) return DMPT_EINVAL;
    for (int f = 0; f < ctx->opt.num_fields; ++f)
        if (!d_h1[f]) return DMPT_EINVAL;
    int rc = dmpt_set_hamiltonian(ctx, d_h0, d_h1[0], ld, n_occ);
    if (rc) return rc;
    for (int f = 1; f < ctx->opt.num_fields; ++f) ctx->d_h1x[f - 1] = d_h1[f];
    return DMPT_OK;
}

static int launch_layer(dmpt_ctx* ctx, int* launches, cudaStream_t capture = nullptr) {
    if (ctx->opt.order >= 2) {
        // highest order first: every pass reads the iterates the lower-order passes of this layer are about to replace
        if (ctx->opt.order == 3) {
            int rc = launch_pass<4>(ctx, capture);
            if (rc) return rc;
            ++*launches;
        }
        int rc = launch_pass<1>(ctx, capture);
        if (rc) return rc;
        ++*launches;
    } else if (ctx->opt.num_fields > 1) {       // fields 2 (and 3): same ordering argument as the order-2 pass
        int rc = launch_pass<2>(ctx, capture);
        if (rc) return rc;
        ++*launches;
    }
    ++*launches;
    return launch_pass<0>(ctx, capture);
}

static int passes_per_layer(const dmpt_ctx* ctx) {
    return ctx->opt.order >= 2 ? ctx->opt.order : (ctx->opt.num_fields > 1 ? 2 : 1);
}

// Device-side layer loop: a CUDA graph with ONE conditional WHILE node; its body is the launches of a layer, captured
// from launch_layer; the control step of pass 0 sets the condition (layer_kernel.cuh).  The host launches the graph
// once per run and never looks at a flag.  The kernel nodes hold a copy of LayerParams, so the graph is rebuilt when
// the problem (n_occ) changes.
static int build_loop_graph(dmpt_ctx* ctx) {
    if (ctx->loop_exec && ctx->loop_n_occ == ctx->lp.pb.n_occ) return DMPT_OK;
    if (ctx->loop_exec) { cudaGraphExecDestroy(ctx->loop_exec); ctx->loop_exec = nullptr; }
    if (ctx->loop_graph) { cudaGraphDestroy(ctx->loop_graph); ctx->loop_graph = nullptr; }
    if (!ctx->capture) CK(cudaStreamCreateWithFlags(&ctx->capture, cudaStreamNonBlocking));
    CK(cudaGraphCreate(&ctx->loop_graph, 0));
    cudaGraphConditionalHandle handle;
    CK(cudaGraphConditionalHandleCreate(&handle, ctx->loop_graph, 1, cudaGraphCondAssignDefault));
    cudaGraphNodeParams np = {cudaGraphNodeTypeConditional};
    np.type = cudaGraphNodeTypeConditional;
    np.conditional.handle = handle;
    np.conditional.type = cudaGraphCondTypeWhile;
    np.conditional.size = 1;
    cudaGraphNode_t node;
    CK(cudaGraphAddNode(&node, ctx->loop_graph, nullptr, 0, &np));
    cudaGraph_t body = np.conditional.phGraph_out[0];
    ctx->lp.cond = handle;
    ctx->lp.use_cond = 1;
    CK(cudaStreamBeginCaptureToGraph(ctx->capture, body, nullptr, nullptr, 0, cudaStreamCaptureModeThreadLocal));
    int dummy = 0;
    const int rc = launch_layer(ctx, &dummy, ctx->capture);
    cudaGraph_t out = nullptr;
    const cudaError_t e = cudaStreamEndCapture(ctx->capture, &out);
    ctx->lp.use_cond = 0;
    if (rc) return rc;
    CK(e);
    CK(cudaGraphInstantiate(&ctx->loop_exec, ctx->loop_graph, 0));
    ctx->loop_n_occ = ctx->lp.pb.n_occ;
    return DMPT_OK;
}

static int elementwise_grid(const dmpt_ctx* ctx, long long work_items, int threads) {
    long long blocks = (work_items + threads - 1) / threads;
    const long long cap = (long long)ctx->num_sms * 8;
    if (blocks > cap) blocks = cap;
    if (blocks < 1) blocks = 1;
    return (int)blocks;
}

// Lower triangle of an fp32 workspace iterate <- its upper triangle (the layer kernel's TMA epilogue keeps only the
// blocks on or above the diagonal up to date): before the iterate is copied out or read row by row.
static int symmetrize(dmpt_ctx* ctx, float* m, cudaStream_t st, int* launches = nullptr) {
    const long long tiles = (long long)(ctx->L.n_pad / 32) * (ctx->L.n_pad / 32);
    dmpt_symmetrize_kernel<<<elementwise_grid(ctx, tiles * 256, 256), 256, 0, st>>>(m, ctx->L.n_pad);
    CK(cudaGetLastError());
    if (launches) ++*launches;
    return DMPT_OK;
}

// a2 + a3 fused (dmpt_transform_split_kernel): S0, S1_f and their first operand splits in one pass over H0, H1_f.
static int launch_transform_split(dmpt_ctx* ctx, const float* d_h0, const H1Ptrs& h1p, int ld, int nf, int* grid_out) {
    const Layout& L = ctx->L;
    const int np = L.n_pad;
    TransformArgs ta{};
    ta.h0 = d_h0;
    ta.n = ctx->n;
    ta.ld = ld;
    ta.n_pad = np;
    ta.s0_shift = ctx->s0_shift;
    ta.s0 = ctx->lp.s0;
    ta.mh = ctx->lp.h[0][0];
    ta.ml = ctx->lp.h[0][1];
    float* s1dst[3] = {ctx->lp.s1[0], ctx->lp.s2[0], ctx->lp.s3[0]};
    for (int f = 0; f < nf; ++f) {
        ta.h1[f] = h1p.p[f];
        ta.s1[f] = s1dst[f];
        ta.yh[f] = ctx->lp.h[0][2 + 2 * f];
        ta.yl[f] = ctx->lp.h[0][3 + 2 * f];
    }
    ta.ctl = ctx->at<DmptCtl>(L.ctl);
    ta.partials = ctx->at<double>(L.partials);
    const int grid = elementwise_grid(ctx, (long long)np * 256, 256);       // block per row, 8 blocks per SM at most
    *grid_out = grid;
    cudaStream_t st = ctx->stream;
    switch (nf) {
        case 0: dmpt_transform_split_kernel<0><<<grid, 256, 0, st>>>(ta); break;
        case 1: dmpt_transform_split_kernel<1><<<grid, 256, 0, st>>>(ta); break;
        case 2: dmpt_transform_split_kernel<2><<<grid, 256, 0, st>>>(ta); break;
        default: dmpt_transform_split_kernel<3><<<grid, 256, 0, st>>>(ta); break;
    }
    CK(cudaGetLastError());
    return DMPT_OK;
}

// a1: spectral bounds of H0 into `bounds` (and max|H1_f| into h1max in the same pass), then into ctl.
//   bounds == 0: Gershgorin discs;  1: the caller's numbers;  2: Gershgorin, then tightened by Lanczos steps.
static int launch_bounds(dmpt_ctx* ctx, const float* d_h0, const H1Ptrs& h1p, int ld, int nf, int* launches) {
    const Layout& L = ctx->L;
    const int n = ctx->n;
    cudaStream_t st = ctx->stream;
    DmptCtl* ctl = ctx->at<DmptCtl>(L.ctl);
    long long* bounds = ctx->at<long long>(L.bounds);
    unsigned int* h1max = ctx->at<unsigned int>(L.h1max);
    const int mode = ctx->opt.bounds;
    if (mode != 1 || nf > 0) {
        const int grid = elementwise_grid(ctx, (long long)n * 32, 256);
        dmpt_gershgorin_kernel<<<grid, 256, 0, st>>>(mode == 1 ? nullptr : d_h0, h1p, n, ld, bounds, h1max);
        CK(cudaGetLastError());
        ++*launches;
    }
    if (mode == 2) {
        LanczosState* ls = ctx->at<LanczosState>(L.lanczos);
        double* vec = reinterpret_cast<double*>(ctx->ws + L.lanczos + sizeof(LanczosState));
        double* v[3] = {vec, vec + L.n_pad, vec + 2 * (size_t)L.n_pad};
        int steps = ctx->opt.lanczos_steps > 0 ? ctx->opt.lanczos_steps : 20;
        if (steps > kLanczosMaxSteps) steps = kLanczosMaxSteps;
        if (steps > n) steps = n;
        const int grid = elementwise_grid(ctx, (long long)n * 32, 256);
        if (n <= 1024) {        // one block does the whole recursion
            dmpt_lanczos_small_kernel<<<1, 1024, 0, st>>>(d_h0, n, ld, steps, ls);
            CK(cudaGetLastError());
            steps = 0;
            *launches += 1;
        } else {
            dmpt_lanczos_init_kernel<<<1, 1024, 0, st>>>(v[0], v[1], n, ls);
            CK(cudaGetLastError());
            *launches += 1;
        }
        for (int j = 1; j <= steps; ++j) {
            // v_{j-1} = v[(j-1) % 3], v_j = v[j % 3], w -> v[(j+1) % 3], which the update turns into v_{j+1}
            dmpt_lanczos_matvec_kernel<<<grid, 256, 0, st>>>(d_h0, n, ld, v[j % 3], v[(j - 1) % 3], v[(j + 1) % 3], ls, j);
            CK(cudaGetLastError());
            dmpt_lanczos_update_kernel<<<1, 1024, 0, st>>>(v[j % 3], v[(j + 1) % 3], n, ls, j);
            CK(cudaGetLastError());
        }
        dmpt_lanczos_bounds_kernel<<<1, 32, 0, st>>>(ls, bounds);
        CK(cudaGetLastError());
        *launches += 1 + 2 * steps;
    }
    dmpt_bounds_to_ctl_kernel<<<1, 32, 0, st>>>(bounds, h1max, ctl, ctx->lp.pb, mode == 1 ? 1 : 0, ctx->opt.eps_min,
                                                ctx->opt.eps_max);
    CK(cudaGetLastError());
    ++*launches;
    return DMPT_OK;
}

// Everything from the spectral bounds to the last layer; leaves the result in the workspace.
// `h_d0_early` (dmpt_run_host only): S0 is final once Algorithm 2 fired, two to four layers before the run
// ends, so its read-back to the host is started on a side stream as soon as the host sees ctl.conv0 and
// overlaps the remaining layers.  *early_issued tells the caller whether that happened.
static int run_core(dmpt_ctx* ctx, const float* d_h0, const float* d_h1, int ld, int* launches,
                    float* h_d0_early = nullptr, int ld_early = 0, bool* early_issued = nullptr) {
    const Layout& L = ctx->L;
    const int n = ctx->n, np = L.n_pad;
    cudaStream_t st = ctx->stream;
    DmptCtl* ctl = ctx->at<DmptCtl>(L.ctl);
    long long* bounds = ctx->at<long long>(L.bounds);
    double* partials = ctx->at<double>(L.partials);

    unsigned int* h1max = ctx->at<unsigned int>(L.h1max);
    const int nf = ctx->opt.order == 0 ? 0 : ctx->opt.num_fields;
    H1Ptrs h1p{{nf >= 1 ? d_h1 : nullptr, nf >= 2 ? ctx->d_h1x[0] : nullptr, nf >= 3 ? ctx->d_h1x[1] : nullptr}};

    dmpt_reset_state_kernel<<<1, 32, 0, st>>>(ctl, bounds, h1max);
    CK(cudaGetLastError());
    // a1: Gershgorin discs of H0 and, in the same pass, max|H1_f| (the scale of the first split of S1_0)
    int rcb = launch_bounds(ctx, d_h0, h1p, ld, nf, launches);
    if (rcb) return rcb;
    CK(cudaEventRecord(ctx->ev_t[4], st));
    // a2 + a3: one pass writes S0, S1_f (fp32) and their first operand splits
    int tgrid = 0;
    int rc0 = launch_transform_split(ctx, d_h0, h1p, ld, nf, &tgrid);
    if (rc0) return rc0;
    dmpt_control_init_kernel<<<1, 32, 0, st>>>(ctl, ctx->lp.logs, ctx->lp.pb, partials, tgrid, ctx->lp.handoff);
    CK(cudaGetLastError());
    CK(cudaEventRecord(ctx->ev_t[5], st));
    *launches += 3;
    if (ctx->opt.order >= 2) {      // S2_0 = 0 (H2 = 0): fp32 iterate and its operands
        const size_t np2 = (size_t)np * np;
        CK(cudaMemsetAsync(ctx->lp.s2[0], 0, np2 * 4, st));
        CK(cudaMemsetAsync(ctx->lp.h[0][4], 0, np2 * 2, st));
        CK(cudaMemsetAsync(ctx->lp.h[0][5], 0, np2 * 2, st));
        if (ctx->opt.order == 3) {  // S3_0 = 0 likewise
            CK(cudaMemsetAsync(ctx->lp.s3[0], 0, np2 * 4, st));
            CK(cudaMemsetAsync(ctx->lp.h[0][6], 0, np2 * 2, st));
            CK(cudaMemsetAsync(ctx->lp.h[0][7], 0, np2 * 2, st));
        }
        unsigned long long* est = ctx->at<unsigned long long>(L.s2_est);
        CK(cudaMemsetAsync(est, 0, 4 * sizeof *est, st));
        dmpt_rowsq_max_kernel<<<elementwise_grid(ctx, (long long)np * 32, 256), 256, 0, st>>>(ctx->lp.s1[0], np, est);
        CK(cudaGetLastError());
        dmpt_s2_scale_init_kernel<<<1, 32, 0, st>>>(ctl, ctx->lp.pb, est);
        CK(cudaGetLastError());
        *launches += 2;
    }
    CK(cudaEventRecord(ctx->ev_t[1], st));

    if (ctx->opt.loop_graph && !h_d0_early && ctx->opt.order != 3) {
        // device-side loop: one graph launch, no flag for the host to look at (order 3 sets the first scale of S3
        // between layers 1 and 2 and keeps the chunked launches)
        int rcg = build_loop_graph(ctx);
        if (rcg) return rcg;
        CK(cudaGraphLaunch(ctx->loop_exec, st));
        CK(cudaEventRecord(ctx->ev_t[2], st));
        ctx->loop_used = true;       // finish() adds layers x passes per layer to the launch count
        return DMPT_OK;
    }
    // Layer loop.  Launches are enqueued in chunks, two chunks ahead of the GPU; after each chunk a
    // 4-byte copy of ctl.done lands in pinned memory.  Launches after convergence exit at once.
    const int max_layers = ctx->opt.max_layers;
    const int chunk_len = np <= 1024 ? 8 : (np <= 4096 ? 4 : 2);
    int launched = 0, chunks = 0;
    auto launch_chunk = [&]() -> int {
        for (int i = 0; i < chunk_len && launched < max_layers; ++i, ++launched) {
            int rc = launch_layer(ctx, launches);
            if (rc) return rc;
            if (ctx->opt.order == 3 && launched == 0) {
                // S3_0 = S3_1 = 0: the first non-zero iterate is S3_2 = sigma_2 (S1_1 S2_1 + S2_1 S1_1), written by
                // layer 2, and the scale of its split has no predecessor to go by.  Cauchy-Schwarz on the rows:
                // max|S3_2| <= 2 max_i ||row_i S1_1|| max_j ||row_j S2_1||; two HBM passes (reading R12 at order 3).
                unsigned long long* est = ctx->at<unsigned long long>(L.s2_est);
                const int rg = elementwise_grid(ctx, (long long)np * 32, 256);
                { int rs = symmetrize(ctx, ctx->lp.s1[1], st, launches); if (rs) return rs; }      // whole rows are read
                dmpt_rowsq_max_kernel<<<rg, 256, 0, st>>>(ctx->lp.s1[1], np, est + 1);
                CK(cudaGetLastError());
                dmpt_rowsq_max_kernel<<<rg, 256, 0, st>>>(ctx->lp.s2[1], np, est + 2);
                CK(cudaGetLastError());
                dmpt_s3_scale_init_kernel<<<1, 32, 0, st>>>(ctl, ctx->lp.pb, est + 1, est + 2);
                CK(cudaGetLastError());
                *launches += 3;
            }
        }
        CK(cudaMemcpyAsync(&ctx->h_flags[chunks % kFlagSlots], &ctl->done, sizeof(int), cudaMemcpyDeviceToHost, st));
        if (h_d0_early)
            CK(cudaMemcpyAsync(&ctx->h_flags0[chunks % kFlagSlots], &ctl->conv0, sizeof(int), cudaMemcpyDeviceToHost, st));
        CK(cudaEventRecord(ctx->ev[chunks % kNumEvents], st));
        ++chunks;
        return DMPT_OK;
    };
    int rc = launch_chunk();
    if (rc) return rc;
    if (launched < max_layers && (rc = launch_chunk())) return rc;
    for (int w = 0; w < chunks; ++w) {
        CK(cudaEventSynchronize(ctx->ev[w % kNumEvents]));
        if (h_d0_early && !*early_issued && ctx->h_flags0[w % kFlagSlots] && !ctx->h_flags[w % kFlagSlots]) {
            // the launch that set conv0 has completed: S0 will not change any more
            { int rs = symmetrize(ctx, ctx->lp.s0, ctx->side, launches); if (rs) return rs; }
            CK(cudaMemcpy2DAsync(h_d0_early, (size_t)ld_early * 4, ctx->lp.s0, (size_t)np * 4, (size_t)n * 4, n,
                                 cudaMemcpyDeviceToHost, ctx->side));
            CK(cudaEventRecord(ctx->ev_side, ctx->side));
            *early_issued = true;
        }
        if (ctx->h_flags[w % kFlagSlots]) break;
        if (launched < max_layers && (rc = launch_chunk())) return rc;
    }
    CK(cudaEventRecord(ctx->ev_t[2], st));
    return DMPT_OK;
}

static int finish(dmpt_ctx* ctx, dmpt_result* res, int launches) {
    cudaStream_t st = ctx->stream;
    const Layout& L = ctx->L;
    CK(cudaEventRecord(ctx->ev_t[3], st));
    CK(cudaStreamSynchronize(st));
    const DmptCtl& c = *ctx->h_ctl;
    int status = c.status;
    if (status == 0 && !c.done) status = DMPT_ENOCONV;
    if (ctx->loop_used) launches += c.layers * passes_per_layer(ctx);      // device-side loop: count from the layers
    ctx->loop_used = false;
    if (res) {
        res->status = status;
        res->layers = c.layers;
        res->layers_d0 = c.n_c;
        res->layers_d1 = c.n_c1;
        res->layers_d2 = c.n_c2;
        res->layers_d3 = c.n_c3;
        res->launches = launches;
        res->eps_min = c.eps_min;
        res->eps_max = c.eps_max;
        res->fro_err0 = c.fro0;
        float ms = 0.f;
        CK(cudaEventElapsedTime(&ms, ctx->ev_t[0], ctx->ev_t[3]));
        res->ms_total = ms;
        CK(cudaEventElapsedTime(&ms, ctx->ev_t[1], ctx->ev_t[2]));
        res->ms_loop = ms;
        CK(cudaEventElapsedTime(&ms, ctx->ev_t[0], ctx->ev_t[4]));
        res->ms_bounds = ms;
        CK(cudaEventElapsedTime(&ms, ctx->ev_t[4], ctx->ev_t[5]));
        res->ms_transform = ms;
        CK(cudaEventElapsedTime(&ms, ctx->ev_t[5], ctx->ev_t[1]));
        res->ms_split = ms;
        res->sm_clock_mhz = 0.0;
        const int nl = c.layers;
        if (nl > 1) {       // SM cycles over device nanoseconds between the first and the last layer launch, all SMs
            std::vector<DmptClockStamps> cs(1);
            CK(cudaMemcpy(cs.data(), ctx->at<DmptClockStamps>(L.clk), sizeof(DmptClockStamps), cudaMemcpyDeviceToHost));
            double cyc = 0.0, ns = 0.0;
            for (int i = 0; i < kMaxSmStamps; ++i)
                if (cs[0].first[i][1] > 0 && cs[0].last[i][1] > cs[0].first[i][1]) {
                    cyc += (double)(cs[0].last[i][0] - cs[0].first[i][0]);
                    ns += (double)(cs[0].last[i][1] - cs[0].first[i][1]);
                }
            if (ns > 0.0) res->sm_clock_mhz = 1e3 * cyc / ns;
        }
        if (nl > 0) {
            std::vector<int> sg(nl);
            if (res->sigma) {
                CK(cudaMemcpy(sg.data(), ctx->at<int>(L.sigma), nl * sizeof(int), cudaMemcpyDeviceToHost));
                for (int i = 0; i < nl; ++i) res->sigma[i] = (int8_t)sg[i];
            }
            if (res->tr_s) CK(cudaMemcpy(res->tr_s, ctx->at<double>(L.tr_s), nl * sizeof(double), cudaMemcpyDeviceToHost));
            if (res->tr_x) CK(cudaMemcpy(res->tr_x, ctx->at<double>(L.tr_x), nl * sizeof(double), cudaMemcpyDeviceToHost));
            if (res->id_err) CK(cudaMemcpy(res->id_err, ctx->at<double>(L.id_err), nl * sizeof(double), cudaMemcpyDeviceToHost));
            if (res->fro_err1) CK(cudaMemcpy(res->fro_err1, ctx->at<double>(L.fro1), nl * sizeof(double), cudaMemcpyDeviceToHost));
            if (res->fro_err2 && (ctx->opt.order >= 2 || ctx->opt.num_fields > 1))
                CK(cudaMemcpy(res->fro_err2, ctx->at<double>(L.fro2), nl * sizeof(double), cudaMemcpyDeviceToHost));
            if (res->fro_err3 && (ctx->opt.num_fields > 2 || ctx->opt.order == 3))
                CK(cudaMemcpy(res->fro_err3, ctx->at<double>(L.fro3), nl * sizeof(double), cudaMemcpyDeviceToHost));
            // the norms were taken on the prescaled iterates (DmptCtl::p1..p3; 0 in all but extreme cases)
            const int pw[3] = {c.p1, ctx->opt.order >= 2 ? 2 * c.p1 : c.p2, ctx->opt.order == 3 ? 3 * c.p1 : c.p3};
            double* logs[3] = {res->fro_err1, res->fro_err2, res->fro_err3};
            for (int k = 0; k < 3; ++k)
                if (logs[k] && pw[k] != 0 && (k == 0 || ctx->opt.order > k || ctx->opt.num_fields > k))
                    for (int i = 0; i < nl; ++i) logs[k][i] = ldexp(logs[k][i], -pw[k]);
        }
    }
    return status;
}

// after run_core: fetch ctl (which buffer holds the accepted S1), then enqueue the output copies
static int fetch_ctl(dmpt_ctx* ctx) {
    CK(cudaMemcpyAsync(ctx->h_ctl, ctx->at<DmptCtl>(ctx->L.ctl), sizeof(DmptCtl), cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    return DMPT_OK;
}

// Undo the prescale of the response iterates (DmptCtl::p1..p3, nonzero only for a perturbation far outside
// fp16's reach) on the accepted buffers, before they are copied out.  Needs ctx->h_ctl (fetch_ctl).
static int unscale_outputs(dmpt_ctx* ctx, int* launches) {
    const DmptCtl& c = *ctx->h_ctl;
    const int np = ctx->L.n_pad;
    const int order = ctx->opt.order, nf = ctx->opt.num_fields;
    float* buf[3] = {order >= 1 ? ctx->lp.s1[c.s1_buf & 1] : nullptr,
                     (order >= 2 || nf >= 2) ? ctx->lp.s2[c.s2_buf & 1] : nullptr,
                     (order == 3 || nf >= 3) ? ctx->lp.s3[c.s3_buf & 1] : nullptr};
    const int pw[3] = {c.p1, order >= 2 ? 2 * c.p1 : c.p2, order == 3 ? 3 * c.p1 : c.p3};
    for (int k = 0; k < 3; ++k)
        if (buf[k] && pw[k] != 0) {
            dmpt_unscale_kernel<<<elementwise_grid(ctx, (long long)np * np, 256), 256, 0, ctx->stream>>>(buf[k], np, -pw[k]);
            CK(cudaGetLastError());
            ++*launches;
        }
    return DMPT_OK;
}

static int run_orders_impl(dmpt_ctx* ctx, float* d_d0, float* d_d1, float* d_d2, float* d_d3, int ld, dmpt_result* res) {
    const int order = ctx->opt.order;
    if (!d_d0 || (!d_d1 && order >= 1) || (!d_d2 && order >= 2) || (!d_d3 && order >= 3)) return DMPT_EINVAL;
    if (!ctx->d_h0) return DMPT_ESTATE;
    if (ld < ctx->n || ctx->opt.num_fields > 1) return DMPT_EINVAL;
    const Layout& L = ctx->L;
    const size_t n = ctx->n, np = L.n_pad;
    int launches = 0;
    CK(cudaEventRecord(ctx->ev_t[0], ctx->stream));
    int rc = run_core(ctx, ctx->d_h0, ctx->d_h1, ctx->ld_in, &launches);
    if (rc) return rc;
    if ((rc = fetch_ctl(ctx))) return rc;
    if ((rc = unscale_outputs(ctx, &launches))) return rc;
    if ((rc = symmetrize(ctx, ctx->lp.s0, ctx->stream, &launches))) return rc;
    if (order >= 1 && (rc = symmetrize(ctx, ctx->lp.s1[ctx->h_ctl->s1_buf & 1], ctx->stream, &launches))) return rc;
    CK(cudaMemcpy2DAsync(d_d0, (size_t)ld * 4, ctx->lp.s0, np * 4, n * 4, n, cudaMemcpyDeviceToDevice, ctx->stream));
    if (order >= 1)
        CK(cudaMemcpy2DAsync(d_d1, (size_t)ld * 4, ctx->lp.s1[ctx->h_ctl->s1_buf & 1], np * 4, n * 4, n,
                             cudaMemcpyDeviceToDevice, ctx->stream));
    if (order >= 2)
        CK(cudaMemcpy2DAsync(d_d2, (size_t)ld * 4, ctx->lp.s2[ctx->h_ctl->s2_buf & 1], np * 4, n * 4, n,
                             cudaMemcpyDeviceToDevice, ctx->stream));
    if (order >= 3)
        CK(cudaMemcpy2DAsync(d_d3, (size_t)ld * 4, ctx->lp.s3[ctx->h_ctl->s3_buf & 1], np * 4, n * 4, n,
                             cudaMemcpyDeviceToDevice, ctx->stream));
    return finish(ctx, res, launches);
}

extern "C" int dmpt_run(dmpt_ctx* ctx, float* d_d0, float* d_d1, float* d_d2, int ld, dmpt_result* res) {
    if (!ctx || ctx->opt.order > 2) return DMPT_EINVAL;          // order 3 has one more output: dmpt_run_orders
    return run_orders_impl(ctx, d_d0, d_d1, d_d2, nullptr, ld, res);
}

extern "C" int dmpt_run_orders(dmpt_ctx* ctx, float* const* d_d, int ld, dmpt_result* res) {
    if (!ctx || !d_d) return DMPT_EINVAL;
    const int order = ctx->opt.order;
    return run_orders_impl(ctx, d_d[0], order >= 1 ? d_d[1] : nullptr, order >= 2 ? d_d[2] : nullptr,
                           order >= 3 ? d_d[3] : nullptr, ld, res);
}

extern "C" int dmpt_run_fields(dmpt_ctx* ctx, float* d_d0, float* const* d_d1, int ld, dmpt_result* res) {
    if (!ctx || !d_d0 || !d_d1 || ctx->opt.order != 1) return DMPT_EINVAL;
    const int nf = ctx->opt.num_fields;
    for (int f = 0; f < nf; ++f)
        if (!d_d1[f]) return DMPT_EINVAL;
    if (!ctx->d_h0 || (nf > 1 && !ctx->d_h1x[0]) || (nf > 2 && !ctx->d_h1x[1])) return DMPT_ESTATE;
    if (ld < ctx->n) return DMPT_EINVAL;
    const Layout& L = ctx->L;
    const size_t n = ctx->n, np = L.n_pad;
    int launches = 0;
    CK(cudaEventRecord(ctx->ev_t[0], ctx->stream));
    int rc = run_core(ctx, ctx->d_h0, ctx->d_h1, ctx->ld_in, &launches);
    if (rc) return rc;
    if ((rc = fetch_ctl(ctx))) return rc;
    if ((rc = unscale_outputs(ctx, &launches))) return rc;
    const DmptCtl& c = *ctx->h_ctl;
    const float* src[3] = {ctx->lp.s1[c.s1_buf & 1], nf > 1 ? ctx->lp.s2[c.s2_buf & 1] : nullptr,
                           nf > 2 ? ctx->lp.s3[c.s3_buf & 1] : nullptr};
    if ((rc = symmetrize(ctx, ctx->lp.s0, ctx->stream, &launches))) return rc;
    if ((rc = symmetrize(ctx, ctx->lp.s1[c.s1_buf & 1], ctx->stream, &launches))) return rc;
    CK(cudaMemcpy2DAsync(d_d0, (size_t)ld * 4, ctx->lp.s0, np * 4, n * 4, n, cudaMemcpyDeviceToDevice, ctx->stream));
    for (int f = 0; f < nf; ++f)
        CK(cudaMemcpy2DAsync(d_d1[f], (size_t)ld * 4, src[f], np * 4, n * 4, n, cudaMemcpyDeviceToDevice, ctx->stream));
    return finish(ctx, res, launches);
}

extern "C" int dmpt_run_fields_host(dmpt_ctx* ctx, const float* h_h0, const float* const* h_h1, int ld_in, int n_occ,
                                    float* h_d0, float* const* h_d1, int ld_out, dmpt_result* res) {
    if (!ctx || !h_h0 || !h_h1 || !h_d0 || !h_d1 || ctx->opt.order != 1) return DMPT_EINVAL;
    const int nf = ctx->opt.num_fields;
    for (int f = 0; f < nf; ++f)
        if (!h_h1[f] || !h_d1[f]) return DMPT_EINVAL;
    if (ld_in < ctx->n || ld_out < ctx->n || n_occ <= 0 || n_occ >= ctx->n) return DMPT_EINVAL;
    const Layout& L = ctx->L;
    const size_t n = ctx->n, np = L.n_pad;
    cudaStream_t st = ctx->stream;
    float* s_h0 = ctx->at<float>(L.stage_h0);
    float* s_h1[3] = {ctx->at<float>(L.stage_h1), nf > 1 ? ctx->at<float>(L.stage_hx[0]) : nullptr,
                      nf > 2 ? ctx->at<float>(L.stage_hx[1]) : nullptr};
    ctx->n_occ = n_occ;
    ctx->lp.pb.n_occ = n_occ;
    int launches = 0;
    CK(cudaEventRecord(ctx->ev_t[0], st));
    CK(cudaMemcpy2DAsync(s_h0, n * 4, h_h0, (size_t)ld_in * 4, n * 4, n, cudaMemcpyHostToDevice, st));
    for (int f = 0; f < nf; ++f)
        CK(cudaMemcpy2DAsync(s_h1[f], n * 4, h_h1[f], (size_t)ld_in * 4, n * 4, n, cudaMemcpyHostToDevice, st));
    // run_core reads fields 2, 3 through the context: point it at the staged copies for this call
    const float* keep[2] = {ctx->d_h1x[0], ctx->d_h1x[1]};
    ctx->d_h1x[0] = s_h1[1];
    ctx->d_h1x[1] = s_h1[2];
    bool early = false;
    int rc = run_core(ctx, s_h0, s_h1[0], (int)n, &launches, h_d0, ld_out, &early);
    ctx->d_h1x[0] = keep[0];
    ctx->d_h1x[1] = keep[1];
    if (rc) return rc;
    if ((rc = fetch_ctl(ctx))) return rc;
    if ((rc = unscale_outputs(ctx, &launches))) return rc;
    const DmptCtl& c = *ctx->h_ctl;
    const float* src[3] = {ctx->lp.s1[c.s1_buf & 1], nf > 1 ? ctx->lp.s2[c.s2_buf & 1] : nullptr,
                           nf > 2 ? ctx->lp.s3[c.s3_buf & 1] : nullptr};
    if ((rc = symmetrize(ctx, ctx->lp.s1[c.s1_buf & 1], st, &launches))) return rc;
    if (early) {
        CK(cudaStreamWaitEvent(st, ctx->ev_side, 0));
    } else {
        if ((rc = symmetrize(ctx, ctx->lp.s0, st, &launches))) return rc;
        CK(cudaMemcpy2DAsync(h_d0, (size_t)ld_out * 4, ctx->lp.s0, np * 4, n * 4, n, cudaMemcpyDeviceToHost, st));
    }
    for (int f = 0; f < nf; ++f)
        CK(cudaMemcpy2DAsync(h_d1[f], (size_t)ld_out * 4, src[f], np * 4, n * 4, n, cudaMemcpyDeviceToHost, st));
    return finish(ctx, res, launches);
}

extern "C" int dmpt_run_host(dmpt_ctx* ctx, const float* h_h0, const float* h_h1, int ld_in, int n_occ,
                             float* h_d0, float* h_d1, float* h_d2, int ld_out, dmpt_result* res) {
    if (!ctx || !h_h0 || !h_d0) return DMPT_EINVAL;
    if (ctx->opt.order != 0 && (!h_h1 || !h_d1)) return DMPT_EINVAL;
    if (ld_in < ctx->n || ld_out < ctx->n || n_occ <= 0 || n_occ >= ctx->n) return DMPT_EINVAL;
    if ((ctx->opt.order == 2 && !h_d2) || ctx->opt.num_fields > 1 || ctx->opt.order > 2) return DMPT_EINVAL;
    const Layout& L = ctx->L;
    const size_t n = ctx->n, np = L.n_pad;
    float* s_h0 = ctx->at<float>(L.stage_h0);
    float* s_h1 = ctx->at<float>(L.stage_h1);
    ctx->n_occ = n_occ;
    ctx->lp.pb.n_occ = n_occ;
    int launches = 0;
    CK(cudaEventRecord(ctx->ev_t[0], ctx->stream));
    CK(cudaMemcpy2DAsync(s_h0, n * 4, h_h0, (size_t)ld_in * 4, n * 4, n, cudaMemcpyHostToDevice, ctx->stream));
    if (ctx->opt.order >= 1)
        CK(cudaMemcpy2DAsync(s_h1, n * 4, h_h1, (size_t)ld_in * 4, n * 4, n, cudaMemcpyHostToDevice, ctx->stream));
    bool early = false;
    int rc = run_core(ctx, s_h0, ctx->opt.order >= 1 ? s_h1 : nullptr, (int)n, &launches, h_d0, ld_out, &early);
    if (rc) return rc;
    if ((rc = fetch_ctl(ctx))) return rc;
    if ((rc = unscale_outputs(ctx, &launches))) return rc;
    if (ctx->opt.order >= 1 && (rc = symmetrize(ctx, ctx->lp.s1[ctx->h_ctl->s1_buf & 1], ctx->stream, &launches))) return rc;
    if (early) {
        CK(cudaStreamWaitEvent(ctx->stream, ctx->ev_side, 0));       // D0 went out while the last layers ran
    } else {
        if ((rc = symmetrize(ctx, ctx->lp.s0, ctx->stream, &launches))) return rc;
        CK(cudaMemcpy2DAsync(h_d0, (size_t)ld_out * 4, ctx->lp.s0, np * 4, n * 4, n, cudaMemcpyDeviceToHost, ctx->stream));
    }
    if (ctx->opt.order >= 1)
        CK(cudaMemcpy2DAsync(h_d1, (size_t)ld_out * 4, ctx->lp.s1[ctx->h_ctl->s1_buf & 1], np * 4, n * 4, n,
                             cudaMemcpyDeviceToHost, ctx->stream));
    if (ctx->opt.order == 2)
        CK(cudaMemcpy2DAsync(h_d2, (size_t)ld_out * 4, ctx->lp.s2[ctx->h_ctl->s2_buf & 1], np * 4, n * 4, n,
                             cudaMemcpyDeviceToHost, ctx->stream));
    return finish(ctx, res, launches);
}

// ---------------------------------------------------------------------------------------------
// dmpt_layer_products: one layer launch on caller-provided S0, S1 (sigma = +1, no decisions)
// ---------------------------------------------------------------------------------------------
namespace {
__global__ void single_shot_init_kernel(DmptCtl* ctl, DmptProblem pb, const double* __restrict__ partials,
                                        const double* __restrict__ partials2 /* max|S2| or NULL */,
                                        const double* __restrict__ partials3 /* max|S3| or NULL */, int nblocks) {
    if (threadIdx.x | blockIdx.x) return;
    double m = 0.0, m2 = 0.0, m3 = 0.0;
    for (int b = 0; b < nblocks; ++b) m = fmax(m, partials[b]);
    if (partials2)
        for (int b = 0; b < nblocks; ++b) m2 = fmax(m2, partials2[b]);
    if (partials3)
        for (int b = 0; b < nblocks; ++b) m3 = fmax(m3, partials3[b]);
    DmptCtl c;
    memset(&c, 0, sizeof c);
    c.layer = 1;
    c.mode0 = MODE_ACTIVE;
    c.sigma = 1;
    c.single_shot = 1;
    c.s1_max = m;
    c.e1_in = c.e1_out = pb.s1_autoscale ? scale_exponent(m) : 0;
    c.s2_max = m2;
    c.e2_in = c.e2_out = pb.s1_autoscale ? scale_exponent(m2) : 0;
    c.s3_max = m3;
    c.e3_in = c.e3_out = pb.s1_autoscale ? scale_exponent(m3) : 0;
    *ctl = c;
}
}  // namespace

extern "C" int dmpt_layer_products(dmpt_ctx* ctx, const float* d_s0, const float* d_s1, int ld,
                                   float* d_x0, float* d_x1, int ld_out) {
    if (!ctx || !d_s0 || !d_s1 || !d_x0 || !d_x1) return DMPT_EINVAL;
    if (ld < ctx->n || ld_out < ctx->n || ctx->opt.order < 1) return DMPT_EINVAL;      // order 0 forms no X1
    const Layout& L = ctx->L;
    const size_t n = ctx->n, np = L.n_pad;
    cudaStream_t st = ctx->stream;
    DmptCtl* ctl = ctx->at<DmptCtl>(L.ctl);
    double* partials = ctx->at<double>(L.partials);
    const int grid = elementwise_grid(ctx, (long long)np * np, 256);
    dmpt_pad_copy_kernel<<<grid, 256, 0, st>>>(d_s0, (int)n, ld, (int)np, ctx->lp.s0, partials);
    CK(cudaGetLastError());
    dmpt_pad_copy_kernel<<<grid, 256, 0, st>>>(d_s1, (int)n, ld, (int)np, ctx->lp.s1[0], partials);
    CK(cudaGetLastError());
    single_shot_init_kernel<<<1, 32, 0, st>>>(ctl, ctx->lp.pb, partials, nullptr, nullptr, grid);
    CK(cudaGetLastError());
    const long long c8 = (long long)np * np / 8;
    const int sgrid = elementwise_grid(ctx, c8, 256);
    dmpt_split_kernel<<<sgrid, 256, 0, st>>>(ctx->lp.s0, (int)np, ctx->lp.h[0][0], ctx->lp.h[0][1], ctl, 0, ctx->s0_shift, 1);
    CK(cudaGetLastError());
    dmpt_split_kernel<<<sgrid, 256, 0, st>>>(ctx->lp.s1[0], (int)np, ctx->lp.h[0][2], ctx->lp.h[0][3], ctl, 1, ctx->s0_shift, 0);
    CK(cudaGetLastError());
    int rc = launch_pass<0>(ctx);
    if (rc) return rc;
    if ((rc = symmetrize(ctx, ctx->lp.s0, st))) return rc;
    if ((rc = symmetrize(ctx, ctx->lp.s1[1], st))) return rc;
    CK(cudaMemcpy2DAsync(d_x0, (size_t)ld_out * 4, ctx->lp.s0, np * 4, n * 4, n, cudaMemcpyDeviceToDevice, st));
    CK(cudaMemcpy2DAsync(d_x1, (size_t)ld_out * 4, ctx->lp.s1[1], np * 4, n * 4, n, cudaMemcpyDeviceToDevice, st));
    CK(cudaStreamSynchronize(st));
    return DMPT_OK;
}

extern "C" int dmpt_layer_products2(dmpt_ctx* ctx, const float* d_s0, const float* d_s1, const float* d_s2, int ld,
                                    float* d_x2, int ld_out) {
    if (!ctx || !d_s0 || !d_s1 || !d_s2 || !d_x2) return DMPT_EINVAL;
    if (ld < ctx->n || ld_out < ctx->n || ctx->opt.order < 2) return DMPT_EINVAL;
    const Layout& L = ctx->L;
    const size_t n = ctx->n, np = L.n_pad;
    cudaStream_t st = ctx->stream;
    DmptCtl* ctl = ctx->at<DmptCtl>(L.ctl);
    double* partials = ctx->at<double>(L.partials);
    double* partials2 = ctx->at<double>(L.partials2);
    const int grid = elementwise_grid(ctx, (long long)np * np, 256);
    dmpt_pad_copy_kernel<<<grid, 256, 0, st>>>(d_s0, (int)n, ld, (int)np, ctx->lp.s0, partials);
    CK(cudaGetLastError());
    dmpt_pad_copy_kernel<<<grid, 256, 0, st>>>(d_s1, (int)n, ld, (int)np, ctx->lp.s1[0], partials);
    CK(cudaGetLastError());
    dmpt_pad_copy_kernel<<<grid, 256, 0, st>>>(d_s2, (int)n, ld, (int)np, ctx->lp.s2[0], partials2);
    CK(cudaGetLastError());
    single_shot_init_kernel<<<1, 32, 0, st>>>(ctl, ctx->lp.pb, partials, partials2, nullptr, grid);
    CK(cudaGetLastError());
    const long long c8 = (long long)np * np / 8;
    const int sgrid = elementwise_grid(ctx, c8, 256);
    dmpt_split_kernel<<<sgrid, 256, 0, st>>>(ctx->lp.s0, (int)np, ctx->lp.h[0][0], ctx->lp.h[0][1], ctl, 0, ctx->s0_shift, 1);
    CK(cudaGetLastError());
    dmpt_split_kernel<<<sgrid, 256, 0, st>>>(ctx->lp.s1[0], (int)np, ctx->lp.h[0][2], ctx->lp.h[0][3], ctl, 1, ctx->s0_shift, 0);
    CK(cudaGetLastError());
    dmpt_split_kernel<<<sgrid, 256, 0, st>>>(ctx->lp.s2[0], (int)np, ctx->lp.h[0][4], ctx->lp.h[0][5], ctl, 2, ctx->s0_shift, 0);
    CK(cudaGetLastError());
    int rc = launch_pass<1>(ctx);
    if (rc) return rc;
    CK(cudaMemcpy2DAsync(d_x2, (size_t)ld_out * 4, ctx->lp.s2[1], np * 4, n * 4, n, cudaMemcpyDeviceToDevice, st));
    CK(cudaStreamSynchronize(st));
    return DMPT_OK;
}

extern "C" int dmpt_layer_products3(dmpt_ctx* ctx, const float* d_s0, const float* d_s1, const float* d_s2,
                                    const float* d_s3, int ld, float* d_x3, int ld_out) {
    if (!ctx || !d_s0 || !d_s1 || !d_s2 || !d_s3 || !d_x3) return DMPT_EINVAL;
    if (ld < ctx->n || ld_out < ctx->n || ctx->opt.order != 3) return DMPT_EINVAL;
    const Layout& L = ctx->L;
    const size_t n = ctx->n, np = L.n_pad;
    cudaStream_t st = ctx->stream;
    DmptCtl* ctl = ctx->at<DmptCtl>(L.ctl);
    double* partials = ctx->at<double>(L.partials);
    double* partials2 = ctx->at<double>(L.partials2);
    double* partials3 = ctx->at<double>(L.partials3);
    const int grid = elementwise_grid(ctx, (long long)np * np, 256);
    dmpt_pad_copy_kernel<<<grid, 256, 0, st>>>(d_s0, (int)n, ld, (int)np, ctx->lp.s0, partials);
    CK(cudaGetLastError());
    dmpt_pad_copy_kernel<<<grid, 256, 0, st>>>(d_s1, (int)n, ld, (int)np, ctx->lp.s1[0], partials);
    CK(cudaGetLastError());
    dmpt_pad_copy_kernel<<<grid, 256, 0, st>>>(d_s2, (int)n, ld, (int)np, ctx->lp.s2[0], partials2);
    CK(cudaGetLastError());
    dmpt_pad_copy_kernel<<<grid, 256, 0, st>>>(d_s3, (int)n, ld, (int)np, ctx->lp.s3[0], partials3);
    CK(cudaGetLastError());
    single_shot_init_kernel<<<1, 32, 0, st>>>(ctl, ctx->lp.pb, partials, partials2, partials3, grid);
    CK(cudaGetLastError());
    const long long c8 = (long long)np * np / 8;
    const int sgrid = elementwise_grid(ctx, c8, 256);
    dmpt_split_kernel<<<sgrid, 256, 0, st>>>(ctx->lp.s0, (int)np, ctx->lp.h[0][0], ctx->lp.h[0][1], ctl, 0, ctx->s0_shift, 1);
    CK(cudaGetLastError());
    dmpt_split_kernel<<<sgrid, 256, 0, st>>>(ctx->lp.s1[0], (int)np, ctx->lp.h[0][2], ctx->lp.h[0][3], ctl, 1, ctx->s0_shift, 0);
    CK(cudaGetLastError());
    dmpt_split_kernel<<<sgrid, 256, 0, st>>>(ctx->lp.s2[0], (int)np, ctx->lp.h[0][4], ctx->lp.h[0][5], ctl, 2, ctx->s0_shift, 0);
    CK(cudaGetLastError());
    dmpt_split_kernel<<<sgrid, 256, 0, st>>>(ctx->lp.s3[0], (int)np, ctx->lp.h[0][6], ctx->lp.h[0][7], ctl, 3, ctx->s0_shift, 0);
    CK(cudaGetLastError());
    int rc = launch_pass<4>(ctx);
    if (rc) return rc;
    CK(cudaMemcpy2DAsync(d_x3, (size_t)ld_out * 4, ctx->lp.s3[1], np * 4, n * 4, n, cudaMemcpyDeviceToDevice, st));
    CK(cudaStreamSynchronize(st));
    return DMPT_OK;
}

// ---------------------------------------------------------------------------------------------
// dmpt_product_nt: C = A.B^T for general n x n matrices in the dual half-precision representation
// (the congruence transforms either side of the hot path are two of these)
// ---------------------------------------------------------------------------------------------
static int product_nt_impl(dmpt_ctx* ctx, const float* d_a, int lda, const float* d_b, int ldb, float* d_c, int ld_out,
                           bool sync, bool trans_a = false, bool trans_b = false);

extern "C" int dmpt_product_nt(dmpt_ctx* ctx, const float* d_a, const float* d_b, int ld, float* d_c, int ld_out) {
    if (!ctx || !d_a || !d_b || !d_c) return DMPT_EINVAL;
    if (ld < ctx->n || ld_out < ctx->n || ctx->opt.order < 1) return DMPT_EINVAL;      // needs the S1 buffers
    return product_nt_impl(ctx, d_a, ld, d_b, ld, d_c, ld_out, true);
}

// C may alias A or B here: both are copied into the workspace before the product and C is written afterwards.
// trans_a / trans_b: the operand is the TRANSPOSE of the caller's matrix (transposed while it is copied in).
static int product_nt_impl(dmpt_ctx* ctx, const float* d_a, int lda, const float* d_b, int ldb, float* d_c, int ld_out,
                           bool sync, bool trans_a, bool trans_b) {
    const Layout& L = ctx->L;
    const size_t n = ctx->n, np = L.n_pad;
    cudaStream_t st = ctx->stream;
    DmptCtl* ctl = ctx->at<DmptCtl>(L.ctl);
    double* partials = ctx->at<double>(L.partials);
    double* partials2 = ctx->at<double>(L.partials2);
    const int grid = elementwise_grid(ctx, (long long)np * np, 256);
    // A -> the S0 buffers (operand pair 0, scale 2^e2), B -> the S1 buffers (operand pair 1, scale 2^e1)
    if (trans_a) dmpt_pad_copy_t_kernel<<<grid, 256, 0, st>>>(d_a, (int)n, lda, (int)np, ctx->lp.s0, partials2);
    else dmpt_pad_copy_kernel<<<grid, 256, 0, st>>>(d_a, (int)n, lda, (int)np, ctx->lp.s0, partials2);
    CK(cudaGetLastError());
    if (trans_b) dmpt_pad_copy_t_kernel<<<grid, 256, 0, st>>>(d_b, (int)n, ldb, (int)np, ctx->lp.s1[0], partials);
    else dmpt_pad_copy_kernel<<<grid, 256, 0, st>>>(d_b, (int)n, ldb, (int)np, ctx->lp.s1[0], partials);
    CK(cudaGetLastError());
    single_shot_init_kernel<<<1, 32, 0, st>>>(ctl, ctx->lp.pb, partials, partials2, nullptr, grid);
    CK(cudaGetLastError());
    const long long c8 = (long long)np * np / 8;
    const int sgrid = elementwise_grid(ctx, c8, 256);
    dmpt_split_kernel<<<sgrid, 256, 0, st>>>(ctx->lp.s0, (int)np, ctx->lp.h[0][0], ctx->lp.h[0][1], ctl, 2, ctx->s0_shift, 0);
    CK(cudaGetLastError());
    dmpt_split_kernel<<<sgrid, 256, 0, st>>>(ctx->lp.s1[0], (int)np, ctx->lp.h[0][2], ctx->lp.h[0][3], ctl, 1, ctx->s0_shift, 0);
    CK(cudaGetLastError());
    int rc = launch_pass<3>(ctx);
    if (rc) return rc;
    CK(cudaMemcpy2DAsync(d_c, (size_t)ld_out * 4, ctx->lp.s1[1], np * 4, n * 4, n, cudaMemcpyDeviceToDevice, st));
    if (sync) CK(cudaStreamSynchronize(st));
    return DMPT_OK;
}

// Congruence transforms either side of the hot path (Eq. 81, A17-A18), two products each:
//   transpose_z != 0:  C = Z^T X Z   (H_orth = Z^T H Z):  T = Z^T X^T (A = Z transposed on the way in, B = X), C = T (Z^T)^T
//   transpose_z == 0:  C = Z X Z^T   (D = Z D_orth Z^T):  T = Z X^T,  C = T Z^T
// X symmetric (X^T = X).  T lives in the workspace's staging buffer.
extern "C" int dmpt_congruence(dmpt_ctx* ctx, const float* d_z, const float* d_x, int ld, int transpose_z, float* d_c,
                               int ld_out) {
    if (!ctx || !d_z || !d_x || !d_c) return DMPT_EINVAL;
    if (ld < ctx->n || ld_out < ctx->n || ctx->opt.order < 1) return DMPT_EINVAL;
    const int n = ctx->n;
    float* t = ctx->at<float>(ctx->L.stage_h0);
    int rc = product_nt_impl(ctx, d_z, ld, d_x, ld, t, n, false, transpose_z != 0, false);
    if (rc) return rc;
    return product_nt_impl(ctx, t, n, d_z, ld, d_c, ld_out, true, false, transpose_z != 0);
}

// ---------------------------------------------------------------------------------------------
// dmpt_fd_response: D1 by finite differences of ground-state runs (Eqs. 83-84)
// ---------------------------------------------------------------------------------------------
extern "C" int dmpt_fd_response(dmpt_ctx* ctx, const float* d_h0, const float* d_h1, int ld, int n_occ, double h,
                                int points, float* d_d1, int ld_out, int* h_layers, double* h_ms) {
    if (!ctx || !d_h0 || !d_h1 || !d_d1 || ctx->opt.order != 0) return DMPT_EINVAL;
    if (ld < ctx->n || ld_out < ctx->n || n_occ <= 0 || n_occ >= ctx->n || !(h > 0.0) || !isfinite(h)) return DMPT_EINVAL;
    if (points != 2 && points != 4) return DMPT_EINVAL;
    const Layout& L = ctx->L;
    const int n = ctx->n, np = L.n_pad;
    cudaStream_t st = ctx->stream;
    float* hp = ctx->at<float>(L.stage_h0);          // H0 + t H1
    // Eq. 83: (D(+h) - D(-h)) / 2h;   Eq. 84: (-D(+2h) + 8 D(+h) - 8 D(-h) + D(-2h)) / 12h
    const double t2[2] = {1.0, -1.0}, w2[2] = {0.5, -0.5};
    const double t4[4] = {2.0, 1.0, -1.0, -2.0}, w4[4] = {-1.0 / 12.0, 8.0 / 12.0, -8.0 / 12.0, 1.0 / 12.0};
    const double* ts = points == 2 ? t2 : t4;
    const double* ws = points == 2 ? w2 : w4;
    ctx->n_occ = n_occ;
    ctx->lp.pb.n_occ = n_occ;
    const int egrid = elementwise_grid(ctx, (long long)n * n, 256);
    double ms_sum = 0.0;
    int status = DMPT_OK;
    for (int k = 0; k < points; ++k) {
        int launches = 0;
        CK(cudaEventRecord(ctx->ev_t[0], st));
        dmpt_axpy_kernel<<<egrid, 256, 0, st>>>(d_h0, d_h1, n, ld, ts[k] * h, hp);
        CK(cudaGetLastError());
        int rc = run_core(ctx, hp, nullptr, n, &launches);
        if (rc) return rc;
        if ((rc = fetch_ctl(ctx))) return rc;
        if ((rc = symmetrize(ctx, ctx->lp.s0, st))) return rc;
        dmpt_fd_accum_kernel<<<egrid, 256, 0, st>>>(ctx->lp.s0, n, np, ws[k] / h, k == 0, d_d1, ld_out);
        CK(cudaGetLastError());
        CK(cudaEventRecord(ctx->ev_t[3], st));
        CK(cudaStreamSynchronize(st));
        float ms = 0.f;
        CK(cudaEventElapsedTime(&ms, ctx->ev_t[0], ctx->ev_t[3]));
        ms_sum += ms;
        const DmptCtl& c = *ctx->h_ctl;
        if (h_layers) h_layers[k] = c.layers;
        if (c.status != 0) status = c.status;
        else if (!c.done && status == DMPT_OK) status = DMPT_ENOCONV;
    }
    if (h_ms) *h_ms = ms_sum;
    return status;
}

// ---------------------------------------------------------------------------------------------
// dmpt_inverse_factor: Z with Z^T S Z = I by the third-order recursion of PAPER.md:693-703 (A19-A21)
// ---------------------------------------------------------------------------------------------
extern "C" int dmpt_inverse_factor(dmpt_ctx* ctx, const float* d_s, int ld, float* d_z, int ld_z, int max_iter,
                                   double tol, int* h_iters, double* h_err) {
    if (!ctx || !d_s || !d_z || ld < ctx->n || ld_z < ctx->n || ctx->opt.order < 1) return DMPT_EINVAL;
    if (max_iter <= 0) max_iter = 30;
    const Layout& L = ctx->L;
    const int n = ctx->n;
    cudaStream_t st = ctx->stream;
    DmptCtl* ctl = ctx->at<DmptCtl>(L.ctl);
    long long* bounds = ctx->at<long long>(L.bounds);
    double* partials = ctx->at<double>(L.partials);
    float* x = ctx->at<float>(L.stage_h0);       // n x n scratch (the staging buffers of dmpt_run_host)
    float* t = ctx->at<float>(L.stage_h1);
    // Z_0 = I / sqrt(eps_max): S is positive definite, so X_0 = S / eps_max has its spectrum in (0, 1]
    dmpt_reset_state_kernel<<<1, 32, 0, st>>>(ctl, bounds, ctx->at<unsigned int>(L.h1max));
    CK(cudaGetLastError());
    dmpt_gershgorin_kernel<<<elementwise_grid(ctx, (long long)n * 32, 256), 256, 0, st>>>(
        d_s, H1Ptrs{{nullptr, nullptr, nullptr}}, n, ld, bounds, ctx->at<unsigned int>(L.h1max));
    CK(cudaGetLastError());
    long long hb[2];
    CK(cudaMemcpyAsync(hb, bounds, sizeof hb, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    const double emax = ordered_to_dbl(hb[1]);
    if (!(emax > 0.0) || !isfinite(emax)) return DMPT_EDEGENERATE;
    const int egrid = elementwise_grid(ctx, (long long)n * n, 256);
    dmpt_scaled_identity_kernel<<<egrid, 256, 0, st>>>(d_z, n, ld_z, bounds);
    CK(cudaGetLastError());
    std::vector<double> hp(egrid);
    double err = INFINITY, prev = INFINITY;
    int it = 0, rc = DMPT_OK;
    for (; it < max_iter; ++it) {
        // X_n = Z_n^T S Z_n (A19); every Z_n is a polynomial in S, hence symmetric: Z^T = Z
        if ((rc = product_nt_impl(ctx, d_z, ld_z, d_s, ld, t, n, false))) return rc;      // T = Z S
        if ((rc = product_nt_impl(ctx, t, n, d_z, ld_z, x, n, false))) return rc;         // X = T Z
        if ((rc = product_nt_impl(ctx, x, n, x, n, t, n, false))) return rc;              // X^2
        dmpt_zpoly_kernel<<<egrid, 256, 0, st>>>(x, t, n, partials);                       // W = sum a_k X^k, ||X - I||_F^2
        CK(cudaGetLastError());
        CK(cudaMemcpyAsync(hp.data(), partials, egrid * sizeof(double), cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        prev = err;
        err = 0.0;
        for (int b = 0; b < egrid; ++b) err += hp[b];
        err = sqrt(err);
        if (!isfinite(err)) { rc = DMPT_ENUMERIC; break; }
        // stop at the requested error, or at the noise floor of the arithmetic (no further decrease)
        if (err <= tol || (it > 0 && err >= 0.5 * prev && err < 1e-2)) break;
        if ((rc = product_nt_impl(ctx, d_z, ld_z, t, n, d_z, ld_z, false))) return rc;    // Z_{n+1} = Z_n W (A20)
    }
    CK(cudaStreamSynchronize(st));
    if (h_iters) *h_iters = it;
    if (h_err) *h_err = err;
    if (rc == DMPT_OK && it >= max_iter) rc = DMPT_ENOCONV;
    return rc;
}

// ---------------------------------------------------------------------------------------------
// a1-a3 on their own: the same kernels dmpt_run launches, on caller matrices
// ---------------------------------------------------------------------------------------------
extern "C" int dmpt_spectral_bounds(dmpt_ctx* ctx, const float* d_h0, int ld, double* h_eps_min,
                                    double* h_eps_max) {
    if (!ctx || !d_h0 || !h_eps_min || !h_eps_max || ld < ctx->n) return DMPT_EINVAL;
    const int n = ctx->n;
    cudaStream_t st = ctx->stream;
    DmptCtl* ctl = ctx->at<DmptCtl>(ctx->L.ctl);
    long long* bounds = ctx->at<long long>(ctx->L.bounds);
    unsigned int* h1max = ctx->at<unsigned int>(ctx->L.h1max);
    dmpt_reset_state_kernel<<<1, 32, 0, st>>>(ctl, bounds, h1max);
    CK(cudaGetLastError());
    const int grid = elementwise_grid(ctx, (long long)n * 32, 256);
    dmpt_gershgorin_kernel<<<grid, 256, 0, st>>>(d_h0, H1Ptrs{{nullptr, nullptr, nullptr}}, n, ld, bounds, h1max);
    CK(cudaGetLastError());
    long long hb[2];
    CK(cudaMemcpyAsync(hb, bounds, sizeof hb, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    *h_eps_min = ordered_to_dbl(hb[0]);
    *h_eps_max = ordered_to_dbl(hb[1]);
    return DMPT_OK;
}

extern "C" int dmpt_initial_transform(dmpt_ctx* ctx, const float* d_h0, const float* d_h1, int ld,
                                      double eps_min, double eps_max, float* d_s0, float* d_s1, int ld_out,
                                      double* h_tr_s0) {
    if (!ctx || !d_h0 || !d_h1 || !d_s0 || !d_s1 || ld < ctx->n || ld_out < ctx->n) return DMPT_EINVAL;
    const double w = eps_max - eps_min;
    if (!(w > 0.0) || !isfinite(w)) return DMPT_EDEGENERATE;
    const Layout& L = ctx->L;
    const size_t n = ctx->n, np = L.n_pad;
    cudaStream_t st = ctx->stream;
    DmptCtl* ctl = ctx->at<DmptCtl>(L.ctl);
    long long* bounds = ctx->at<long long>(L.bounds);
    double* partials = ctx->at<double>(L.partials);
    // the same two launches dmpt_run makes: max|H1| (scale of the first split), then the fused a2 + a3 kernel
    unsigned int* h1max = ctx->at<unsigned int>(L.h1max);
    const H1Ptrs h1p{{d_h1, nullptr, nullptr}};
    dmpt_reset_state_kernel<<<1, 32, 0, st>>>(ctl, bounds, h1max);
    CK(cudaGetLastError());
    dmpt_gershgorin_kernel<<<elementwise_grid(ctx, (long long)n * 32, 256), 256, 0, st>>>(nullptr, h1p, (int)n, ld, bounds,
                                                                                         h1max);
    CK(cudaGetLastError());
    DmptProblem pb1 = ctx->lp.pb;
    pb1.order = 1;
    pb1.nfields = 1;
    dmpt_bounds_to_ctl_kernel<<<1, 32, 0, st>>>(bounds, h1max, ctl, pb1, 1, eps_min, eps_max);
    CK(cudaGetLastError());
    int tgrid = 0;
    int rc = launch_transform_split(ctx, d_h0, h1p, ld, 1, &tgrid);
    if (rc) return rc;
    if ((rc = fetch_ctl(ctx))) return rc;
    if (ctx->h_ctl->p1 != 0) {       // hand back S1 itself, not the prescaled iterate
        dmpt_unscale_kernel<<<elementwise_grid(ctx, (long long)np * np, 256), 256, 0, st>>>(ctx->lp.s1[0], (int)np,
                                                                                           -ctx->h_ctl->p1);
        CK(cudaGetLastError());
    }
    CK(cudaMemcpy2DAsync(d_s0, (size_t)ld_out * 4, ctx->lp.s0, np * 4, n * 4, n, cudaMemcpyDeviceToDevice, st));
    CK(cudaMemcpy2DAsync(d_s1, (size_t)ld_out * 4, ctx->lp.s1[0], np * 4, n * 4, n, cudaMemcpyDeviceToDevice, st));
    std::vector<double> hp((size_t)tgrid * 3);
    CK(cudaMemcpyAsync(hp.data(), partials, hp.size() * sizeof(double), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    if (h_tr_s0) {
        double t = 0.0;
        for (int b = 0; b < tgrid; ++b) t += hp[(size_t)b * 3];
        *h_tr_s0 = t;
    }
    return DMPT_OK;
}

extern "C" int dmpt_split(dmpt_ctx* ctx, const float* d_x, int ld, int shift, int diag_half, uint16_t* d_hi,
                          uint16_t* d_lo, int ld_out) {
    if (!ctx || !d_x || !d_hi || !d_lo || ld < ctx->n || ld_out < ctx->n || shift < 0 || shift > 15) return DMPT_EINVAL;
    const Layout& L = ctx->L;
    const size_t n = ctx->n, np = L.n_pad;
    cudaStream_t st = ctx->stream;
    DmptCtl* ctl = ctx->at<DmptCtl>(L.ctl);
    double* partials = ctx->at<double>(L.partials);
    const int grid = elementwise_grid(ctx, (long long)np * np, 256);
    dmpt_pad_copy_kernel<<<grid, 256, 0, st>>>(d_x, (int)n, ld, (int)np, ctx->lp.s0, partials);
    CK(cudaGetLastError());
    const long long c8 = (long long)np * np / 8;
    const int sgrid = elementwise_grid(ctx, c8, 256);
    dmpt_split_kernel<<<sgrid, 256, 0, st>>>(ctx->lp.s0, (int)np, ctx->lp.h[0][0], ctx->lp.h[0][1], ctl, 0, shift,
                                             diag_half ? 1 : 0);
    CK(cudaGetLastError());
    CK(cudaMemcpy2DAsync(d_hi, (size_t)ld_out * 2, ctx->lp.h[0][0], np * 2, n * 2, n, cudaMemcpyDeviceToDevice, st));
    CK(cudaMemcpy2DAsync(d_lo, (size_t)ld_out * 2, ctx->lp.h[0][1], np * 2, n * 2, n, cudaMemcpyDeviceToDevice, st));
    CK(cudaStreamSynchronize(st));
    return DMPT_OK;
}

// ---------------------------------------------------------------------------------------------
// Order-parallel pair (Sec. III.C, 548-550): the order-0 side computes
// f^(0) = S0^2 (sigma_n, Algorithm 2), the order-1 side f^(1) = S0.S1 + S1.S0 (Algorithm 3).  Per layer one one-way
// hand-off: the operand pair (Mhi, Mlo) of S0_{n-1}, 4 N^2 bytes, and a DmptHandoff record, by cudaMemcpyPeerAsync on
// a copy stream, so that it overlaps the products of both sides.  With both sides on one device the copies are
// device-local and the two launches of a layer take turns on the SMs; the results are bit-identical to dmpt_run
// either way (same kernels, same operands, same decisions).
//
//   events:  A_n  order-0 side finished layer n          (A_0: its initial transform)
//            C_n  hand-off for layer n has landed        (operands of S0_{n-1}: written by the order-0 side's layer n-1)
//            B_n  order-1 side finished layer n
//   copy(n)  waits A_{n-1}, B_{n-2} (it overwrites the operand buffer layer n-2 of the order-1 side read; B_0 = that
//            side's set-up)
//   side 0, layer n  waits C_{n-1} (it overwrites the operand buffer copy(n-1) read)
//   side 1, layer n  waits C_n
// The host stays two layers ahead of either side (events A_{n-2}, B_{n-2}), so that no copy is issued once the
// order-0 side has finished: a later copy would target the buffer the order-1 side keeps reading.
// ---------------------------------------------------------------------------------------------
namespace {
constexpr int kPairRing = 4;
}

struct dmpt_pair {
    dmpt_ctx* side[2] = {nullptr, nullptr};
    int dev[2] = {0, 0};
    int n = 0;
    cudaStream_t st[2] = {nullptr, nullptr};
    cudaStream_t copy = nullptr;                 // on dev[0]
    cudaEvent_t evA[kPairRing]{}, evC[kPairRing]{}, evB[kPairRing]{};
    cudaEvent_t ev_bounds = nullptr;
    int* h_done[2] = {nullptr, nullptr};         // pinned, kPairRing entries each
    char err[256] = {0};
};

#define PK(call)                                                                                     \
    do {                                                                                             \
        cudaError_t e_ = (call);                                                                     \
        if (e_ != cudaSuccess) {                                                                     \
            snprintf(pr->err, sizeof pr->err, "%s: %s (%s:%d)", #call, cudaGetErrorString(e_),       \
                     __FILE__, __LINE__);                                                            \
            return DMPT_ECUDA;                                                                       \
        }                                                                                            \
    } while (0)

extern "C" size_t dmpt_pair_workspace_bytes(int n, int side) {
    if (n <= 0 || side < 0 || side > 1 || n > 65535 * kTile) return 0;
    return make_layout(n, side, 1).total;
}

extern "C" const char* dmpt_pair_last_cuda_error(const dmpt_pair* pr) {
    if (!pr) return "";
    if (pr->err[0]) return pr->err;
    for (int s = 0; s < 2; ++s)
        if (pr->side[s] && pr->side[s]->err[0]) return pr->side[s]->err;
    return "";
}

extern "C" int dmpt_pair_destroy(dmpt_pair* pr) {
    if (!pr) return DMPT_EINVAL;
    int cur = 0;
    cudaGetDevice(&cur);
    for (int s = 0; s < 2; ++s) {
        cudaSetDevice(pr->dev[s]);
        if (pr->st[s]) cudaStreamSynchronize(pr->st[s]);
        if (s == 0 && pr->copy) cudaStreamSynchronize(pr->copy);
        if (pr->side[s]) dmpt_destroy(pr->side[s]);
        if (pr->h_done[s]) cudaFreeHost(pr->h_done[s]);
    }
    cudaSetDevice(pr->dev[0]);
    for (auto& e : pr->evA) if (e) cudaEventDestroy(e);
    for (auto& e : pr->evC) if (e) cudaEventDestroy(e);
    if (pr->ev_bounds) cudaEventDestroy(pr->ev_bounds);
    if (pr->copy) cudaStreamDestroy(pr->copy);
    if (pr->st[0]) cudaStreamDestroy(pr->st[0]);
    cudaSetDevice(pr->dev[1]);
    for (auto& e : pr->evB) if (e) cudaEventDestroy(e);
    if (pr->st[1]) cudaStreamDestroy(pr->st[1]);
    cudaSetDevice(cur);
    delete pr;
    return DMPT_OK;
}

extern "C" int dmpt_pair_create(dmpt_pair** out, int n, const dmpt_options* opt, int device0, void* d_workspace0,
                                size_t workspace0_bytes, int device1, void* d_workspace1, size_t workspace1_bytes) {
    if (!out) return DMPT_EINVAL;
    *out = nullptr;
    dmpt_options o;
    if (opt) o = *opt; else dmpt_default_options(&o);
    if (n <= 0 || o.order != 1 || o.num_fields > 1 || !d_workspace0 || !d_workspace1) return DMPT_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device0 < 0 || device1 < 0 || device0 >= ndev || device1 >= ndev)
        return ndev == 0 ? DMPT_ECUDA : DMPT_EINVAL;
    int cur = 0;
    cudaGetDevice(&cur);
    dmpt_pair* pr = new dmpt_pair();
    pr->n = n;
    pr->dev[0] = device0;
    pr->dev[1] = device1;
    auto fail = [&](int code) {
        fprintf(stderr, "dmpt_pair_create: %s\n", dmpt_pair_last_cuda_error(pr));
        dmpt_pair_destroy(pr);
        cudaSetDevice(cur);
        return code;
    };
#define PKC(call)                                                                          \
    do {                                                                                   \
        cudaError_t e_ = (call);                                                           \
        if (e_ != cudaSuccess) {                                                           \
            snprintf(pr->err, sizeof pr->err, "%s: %s", #call, cudaGetErrorString(e_));    \
            return fail(DMPT_ECUDA);                                                       \
        }                                                                                  \
    } while (0)
    void* ws[2] = {d_workspace0, d_workspace1};
    const size_t wsb[2] = {workspace0_bytes, workspace1_bytes};
    for (int s = 0; s < 2; ++s) {
        PKC(cudaSetDevice(pr->dev[s]));
        PKC(cudaStreamCreateWithFlags(&pr->st[s], cudaStreamNonBlocking));
        PKC(cudaHostAlloc(&pr->h_done[s], kPairRing * sizeof(int), cudaHostAllocDefault));
        if (s == 0) {
            PKC(cudaStreamCreateWithFlags(&pr->copy, cudaStreamNonBlocking));
            for (auto& e : pr->evA) PKC(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
            for (auto& e : pr->evC) PKC(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
            PKC(cudaEventCreateWithFlags(&pr->ev_bounds, cudaEventDisableTiming));
        } else {
            for (auto& e : pr->evB) PKC(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        }
        dmpt_options os = o;
        os.order = s;                      // side 0: S0 alone; side 1: the response product alone
        os.num_fields = 1;
        const int rc = create_impl(&pr->side[s], n, &os, ws[s], wsb[s], pr->st[s], s + 1);
        if (rc != DMPT_OK) {
            snprintf(pr->err, sizeof pr->err, "side %d: %s", s, dmpt_strerror(rc));
            return fail(rc);
        }
    }
    if (device0 != device1) {
        // direct NVLink path for the hand-off when the devices are peers (the copies work without it, staged)
        for (int s = 0; s < 2; ++s) {
            int can = 0;
            PKC(cudaDeviceCanAccessPeer(&can, pr->dev[s], pr->dev[s ^ 1]));
            if (can) {
                PKC(cudaSetDevice(pr->dev[s]));
                const cudaError_t e = cudaDeviceEnablePeerAccess(pr->dev[s ^ 1], 0);
                if (e != cudaSuccess && e != cudaErrorPeerAccessAlreadyEnabled) {
                    snprintf(pr->err, sizeof pr->err, "cudaDeviceEnablePeerAccess: %s", cudaGetErrorString(e));
                    return fail(DMPT_ECUDA);
                }
                cudaGetLastError();
            }
        }
    }
#undef PKC
    cudaSetDevice(cur);
    *out = pr;
    return DMPT_OK;
}

extern "C" int dmpt_pair_set_hamiltonian(dmpt_pair* pr, const float* d_h0, const float* d_h1, int ld, int n_occ) {
    if (!pr || !d_h0 || !d_h1 || ld < pr->n || n_occ <= 0 || n_occ >= pr->n) return DMPT_EINVAL;
    for (int s = 0; s < 2; ++s) {
        dmpt_ctx* c = pr->side[s];
        c->d_h0 = s == 0 ? d_h0 : nullptr;
        c->d_h1 = s == 1 ? d_h1 : nullptr;
        c->ld_in = ld;
        c->n_occ = n_occ;
        c->lp.pb.n_occ = n_occ;
    }
    return DMPT_OK;
}

extern "C" int dmpt_pair_run(dmpt_pair* pr, float* d_d0, float* d_d1, int ld, dmpt_result* res) {
    if (!pr || !d_d0 || !d_d1 || ld < pr->n) return DMPT_EINVAL;
    dmpt_ctx* c0 = pr->side[0];
    dmpt_ctx* c1 = pr->side[1];
    if (!c0->d_h0 || !c1->d_h1) return DMPT_ESTATE;
    const Layout& L0 = c0->L;
    const Layout& L1 = c1->L;
    const size_t n = pr->n, np = L0.n_pad;
    const size_t op_bytes = np * np * 2;
    int cur = 0;
    cudaGetDevice(&cur);
    struct Restore { int d; ~Restore() { cudaSetDevice(d); } } restore{cur};
    int launches = 0;
    DmptCtl* ctl0 = c0->at<DmptCtl>(L0.ctl);
    DmptCtl* ctl1 = c1->at<DmptCtl>(L1.ctl);
    const H1Ptrs none{{nullptr, nullptr, nullptr}};

    // ---- order-0 side: a1, then a2 + a3 for S0 alone, then the decision for layer 1 (handoff[1])
    PK(cudaSetDevice(pr->dev[0]));
    {
        cudaStream_t st = pr->st[0];
        PK(cudaEventRecord(c0->ev_t[0], st));
        dmpt_reset_state_kernel<<<1, 32, 0, st>>>(ctl0, c0->at<long long>(L0.bounds), c0->at<unsigned int>(L0.h1max));
        PK(cudaGetLastError());
        PK(cudaMemsetAsync(c0->lp.handoff, 0, (kMaxLayersCap + 2) * sizeof(DmptHandoff), st));
        if (launch_bounds(c0, c0->d_h0, none, c0->ld_in, 0, &launches)) {
            snprintf(pr->err, sizeof pr->err, "%s", c0->err);
            return DMPT_ECUDA;
        }
        PK(cudaEventRecord(pr->ev_bounds, st));
        PK(cudaEventRecord(c0->ev_t[4], st));
        int tgrid = 0;
        if (launch_transform_split(c0, c0->d_h0, none, c0->ld_in, 0, &tgrid)) {
            snprintf(pr->err, sizeof pr->err, "%s", c0->err);
            return DMPT_ECUDA;
        }
        dmpt_control_init_kernel<<<1, 32, 0, st>>>(ctl0, c0->lp.logs, c0->lp.pb, c0->at<double>(L0.partials), tgrid,
                                                   c0->lp.handoff);
        PK(cudaGetLastError());
        PK(cudaEventRecord(c0->ev_t[5], st));
        PK(cudaEventRecord(c0->ev_t[1], st));
        PK(cudaEventRecord(pr->evA[0], st));
        launches += 3;
    }
    // ---- order-1 side: max|H1|, the bounds of the other side (16 bytes), a2 + a3 for S1 alone
    PK(cudaSetDevice(pr->dev[1]));
    {
        cudaStream_t st = pr->st[1];
        const H1Ptrs h1p{{c1->d_h1, nullptr, nullptr}};
        PK(cudaEventRecord(c1->ev_t[0], st));
        dmpt_reset_state_kernel<<<1, 32, 0, st>>>(ctl1, c1->at<long long>(L1.bounds), c1->at<unsigned int>(L1.h1max));
        PK(cudaGetLastError());
        PK(cudaMemsetAsync(c1->lp.handoff, 0, (kMaxLayersCap + 2) * sizeof(DmptHandoff), st));
        dmpt_gershgorin_kernel<<<elementwise_grid(c1, (long long)n * 32, 256), 256, 0, st>>>(
            nullptr, h1p, (int)n, c1->ld_in, c1->at<long long>(L1.bounds), c1->at<unsigned int>(L1.h1max));
        PK(cudaGetLastError());
        PK(cudaStreamWaitEvent(st, pr->ev_bounds, 0));
        // eps_min, eps_max as the order-0 side settled them (Gershgorin or caller-supplied)
        PK(cudaMemcpyPeerAsync(&ctl1->eps_min, pr->dev[1], &ctl0->eps_min, pr->dev[0], 2 * sizeof(double), st));
        dmpt_bounds_to_ctl_kernel<<<1, 32, 0, st>>>(c1->at<long long>(L1.bounds), c1->at<unsigned int>(L1.h1max), ctl1,
                                                    c1->lp.pb, 2, 0.0, 0.0);
        PK(cudaGetLastError());
        PK(cudaEventRecord(c1->ev_t[4], st));
        int tgrid = 0;
        if (launch_transform_split(c1, nullptr, h1p, c1->ld_in, 1, &tgrid)) {
            snprintf(pr->err, sizeof pr->err, "%s", c1->err);
            return DMPT_ECUDA;
        }
        dmpt_control_init_kernel<<<1, 32, 0, st>>>(ctl1, c1->lp.logs, c1->lp.pb, c1->at<double>(L1.partials), tgrid,
                                                   c1->lp.handoff);
        PK(cudaGetLastError());
        PK(cudaEventRecord(c1->ev_t[5], st));
        PK(cudaEventRecord(c1->ev_t[1], st));
        PK(cudaEventRecord(pr->evB[0], st));          // B_0: this side's set-up is done (its handoff array is cleared)
        launches += 5;
    }

    // ---- layers
    const int max_layers = c1->opt.max_layers;
    bool side0_live = true;
    for (int l = 1; l <= max_layers; ++l) {
        bool copied = false;
        if (side0_live && l >= 3) {
            PK(cudaEventSynchronize(pr->evA[(l - 2) % kPairRing]));
            if (pr->h_done[0][(l - 2) % kPairRing]) side0_live = false;
        }
        if (side0_live) {
            PK(cudaSetDevice(pr->dev[0]));
            const int b = (l - 1) & 1;                  // operand buffer of S0_{l-1} while S0 is being updated
            PK(cudaStreamWaitEvent(pr->copy, pr->evA[(l - 1) % kPairRing], 0));
            PK(cudaStreamWaitEvent(pr->copy, pr->evB[l >= 3 ? (l - 2) % kPairRing : 0], 0));
            PK(cudaMemcpyPeerAsync(c1->lp.h[b][MH], pr->dev[1], c0->lp.h[b][MH], pr->dev[0], op_bytes, pr->copy));
            PK(cudaMemcpyPeerAsync(c1->lp.h[b][ML], pr->dev[1], c0->lp.h[b][ML], pr->dev[0], op_bytes, pr->copy));
            PK(cudaMemcpyPeerAsync(c1->lp.handoff + l, pr->dev[1], c0->lp.handoff + l, pr->dev[0], sizeof(DmptHandoff),
                                   pr->copy));
            PK(cudaEventRecord(pr->evC[l % kPairRing], pr->copy));
            copied = true;
            if (l >= 2) PK(cudaStreamWaitEvent(pr->st[0], pr->evC[(l - 1) % kPairRing], 0));
            if (launch_pass<0>(c0)) {
                snprintf(pr->err, sizeof pr->err, "%s", c0->err);
                return DMPT_ECUDA;
            }
            ++launches;
            PK(cudaMemcpyAsync(&pr->h_done[0][l % kPairRing], &ctl0->done, sizeof(int), cudaMemcpyDeviceToHost, pr->st[0]));
            PK(cudaEventRecord(pr->evA[l % kPairRing], pr->st[0]));
        }
        PK(cudaSetDevice(pr->dev[1]));
        if (copied) PK(cudaStreamWaitEvent(pr->st[1], pr->evC[l % kPairRing], 0));
        if (launch_pass<0>(c1)) {
            snprintf(pr->err, sizeof pr->err, "%s", c1->err);
            return DMPT_ECUDA;
        }
        ++launches;
        PK(cudaMemcpyAsync(&pr->h_done[1][l % kPairRing], &ctl1->done, sizeof(int), cudaMemcpyDeviceToHost, pr->st[1]));
        PK(cudaEventRecord(pr->evB[l % kPairRing], pr->st[1]));
        if (l >= 3) {
            PK(cudaEventSynchronize(pr->evB[(l - 2) % kPairRing]));
            if (pr->h_done[1][(l - 2) % kPairRing]) break;
        }
    }

    // ---- results: D0 from the order-0 side, D1 (the last ACCEPTED iterate) from the order-1 side
    PK(cudaSetDevice(pr->dev[1]));
    PK(cudaEventRecord(c1->ev_t[2], pr->st[1]));
    if (fetch_ctl(c1)) { snprintf(pr->err, sizeof pr->err, "%s", c1->err); return DMPT_ECUDA; }
    if (unscale_outputs(c1, &launches)) { snprintf(pr->err, sizeof pr->err, "%s", c1->err); return DMPT_ECUDA; }
    if (symmetrize(c1, c1->lp.s1[c1->h_ctl->s1_buf & 1], pr->st[1], &launches)) { snprintf(pr->err, sizeof pr->err, "%s", c1->err); return DMPT_ECUDA; }
    PK(cudaMemcpy2DAsync(d_d1, (size_t)ld * 4, c1->lp.s1[c1->h_ctl->s1_buf & 1], np * 4, n * 4, n,
                         cudaMemcpyDeviceToDevice, pr->st[1]));
    PK(cudaEventRecord(c1->ev_t[3], pr->st[1]));
    PK(cudaSetDevice(pr->dev[0]));
    PK(cudaStreamSynchronize(pr->copy));
    if (fetch_ctl(c0)) { snprintf(pr->err, sizeof pr->err, "%s", c0->err); return DMPT_ECUDA; }
    if (symmetrize(c0, c0->lp.s0, pr->st[0], &launches)) { snprintf(pr->err, sizeof pr->err, "%s", c0->err); return DMPT_ECUDA; }
    PK(cudaMemcpy2DAsync(d_d0, (size_t)ld * 4, c0->lp.s0, np * 4, n * 4, n, cudaMemcpyDeviceToDevice, pr->st[0]));
    PK(cudaStreamSynchronize(pr->st[0]));
    PK(cudaSetDevice(pr->dev[1]));
    PK(cudaStreamSynchronize(pr->st[1]));

    const DmptCtl& k0 = *c0->h_ctl;
    const DmptCtl& k1 = *c1->h_ctl;
    int status = k1.status != 0 ? k1.status : k0.status;
    if (status == 0 && !k1.done) status = DMPT_ENOCONV;
    if (res) {
        res->status = status;
        res->layers = k1.layers;
        res->layers_d0 = k0.n_c;
        res->layers_d1 = k1.n_c1;
        res->layers_d2 = res->layers_d3 = 0;
        res->launches = launches;
        res->eps_min = k0.eps_min;
        res->eps_max = k0.eps_max;
        res->fro_err0 = k0.fro0;
        float ms = 0.f;
        PK(cudaEventElapsedTime(&ms, c1->ev_t[0], c1->ev_t[3]));
        res->ms_total = ms;
        PK(cudaEventElapsedTime(&ms, c1->ev_t[1], c1->ev_t[2]));
        res->ms_loop = ms;
        PK(cudaEventElapsedTime(&ms, c1->ev_t[0], c1->ev_t[4]));
        res->ms_bounds = ms;
        PK(cudaEventElapsedTime(&ms, c1->ev_t[4], c1->ev_t[5]));
        res->ms_transform = ms;
        res->ms_split = 0.0;
        res->sm_clock_mhz = 0.0;      // two devices, two clocks: not reported for the pair
        const int nl = k1.layers, nl0 = k0.layers < nl ? k0.layers : nl;
        if (nl > 0) {
            std::vector<int> sg(nl);
            std::vector<double> tmp(nl);
            if (res->sigma) {
                PK(cudaMemcpy(sg.data(), c1->at<int>(L1.sigma), nl * sizeof(int), cudaMemcpyDeviceToHost));
                for (int i = 0; i < nl; ++i) res->sigma[i] = (int8_t)sg[i];
            }
            if (res->fro_err1) {
                PK(cudaMemcpy(res->fro_err1, c1->at<double>(L1.fro1), nl * sizeof(double), cudaMemcpyDeviceToHost));
                if (k1.p1 != 0)
                    for (int i = 0; i < nl; ++i) res->fro_err1[i] = ldexp(res->fro_err1[i], -k1.p1);
            }
            PK(cudaSetDevice(pr->dev[0]));
            double* dst[3] = {res->tr_s, res->tr_x, res->id_err};
            const size_t src[3] = {L0.tr_s, L0.tr_x, L0.id_err};
            for (int k = 0; k < 3; ++k) {
                if (!dst[k]) continue;
                for (int i = 0; i < nl; ++i) dst[k][i] = NAN;
                if (nl0 > 0) PK(cudaMemcpy(dst[k], c0->at<double>(src[k]), nl0 * sizeof(double), cudaMemcpyDeviceToHost));
            }
            // N_S is constant once S0 froze
            if (res->tr_s && nl0 > 0)
                for (int i = nl0; i < nl; ++i) res->tr_s[i] = res->tr_s[nl0 - 1];
        }
    }
    return status;
}
