// dmpt_spectral_bounds_noalloc: step a1 (Gershgorin discs) for callers that cannot allocate.
//
// The entry point needs no dmpt_ctx (dmpt_create pins host memory) and calls no cudaMalloc, cudaFree, cudaHostAlloc
// or allocating library routine: the scratch of its kernel is the file-scope device array below, which every GPU
// that loads libdmpt.so holds until the process exits.  The array's name is a device symbol: host code must not pass
// it to a kernel.  The device address is asked for once per device with cudaGetSymbolAddress (scratch_for_device) and
// that pointer is what the launches receive.
//
// Scratch contents: [0, 256) a header (one counter of finished blocks, which must be zero when the first kernel
// starts: cleared on the stream at every call), then the two disc ends of every row, 16 bytes per row.  All calls on
// one device share the array: two calls that overlap on the GPU (different streams, no ordering between them) race on
// it and both results are undefined; calls ordered on one stream, or by events, are safe.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdint>
#include <mutex>

#include "../../include/dmpt.h"

namespace {

constexpr int kMaxN = DMPT_NOALLOC_MAX_N;
constexpr size_t kHeaderBytes = 256;
constexpr size_t kScratchBytes = kHeaderBytes + (size_t)kMaxN * 2 * sizeof(double);      // 256 B + 1 MiB
constexpr int kMaxDevices = 64;

static __device__ __align__(256) unsigned char g_noalloc_scratch[kScratchBytes];

struct ScratchView {
    unsigned int* blocks_done;      // header: blocks of the rows kernel that have written their rows
    double* ends;                   // ends[2 i] = H0_ii - r_i, ends[2 i + 1] = H0_ii + r_i
};

__device__ __host__ inline ScratchView view_of(unsigned char* base) {
    return ScratchView{reinterpret_cast<unsigned int*>(base), reinterpret_cast<double*>(base + kHeaderBytes)};
}

__device__ __forceinline__ double warp_sum_f64(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// One warp per row: r_i = sum_{j != i} |H0_ij| with fp32 partial sums per lane (four accumulators on the vector
// path), fp64 across the lanes: the arithmetic of dmpt_gershgorin_kernel (kernels_hbm.cuh), so that the two entry
// points agree.  Each row's disc ends go to the scratch; the last block to finish (header counter) takes the minimum
// and maximum over all rows and writes d_eps[0] = eps_min, d_eps[1] = eps_max.
__global__ void __launch_bounds__(256) dmpt_gershgorin_noalloc_kernel(const float* __restrict__ h0, int n, int ld,
                                                                      unsigned char* scratch, double* __restrict__ d_eps) {
    const ScratchView sv = view_of(scratch);
    const int warps_per_block = blockDim.x >> 5;
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const bool vec = (ld & 3) == 0 && (reinterpret_cast<uintptr_t>(h0) & 15) == 0;
    for (int row = blockIdx.x * warps_per_block + warp; row < n; row += gridDim.x * warps_per_block) {
        const size_t off = (size_t)row * ld;
        float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f;
        int j = 0;
        if (vec) {
            const int n4 = n & ~3;
            for (j = lane * 4; j < n4; j += 128) {
                const float4 v = __ldg(reinterpret_cast<const float4*>(h0 + off + j));
                a0 += fabsf(v.x); a1 += fabsf(v.y); a2 += fabsf(v.z); a3 += fabsf(v.w);
            }
            j = n4;
        }
        for (j += lane; j < n; j += 32) a0 += fabsf(h0[off + j]);
        const double s = warp_sum_f64((double)a0 + (double)a1 + (double)a2 + (double)a3);
        if (lane == 0) {
            const double d = (double)h0[off + row];
            const double r = s - fabs(d);
            sv.ends[2 * row] = d - r;
            sv.ends[2 * row + 1] = d + r;
        }
    }
    // last block: every other block's rows are visible after its fence + counter increment
    __shared__ bool s_last;
    __shared__ double s_lo[8], s_hi[8];
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        s_last = atomicAdd(sv.blocks_done, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    double lo = INFINITY, hi = -INFINITY;
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
        lo = fmin(lo, __ldcg(sv.ends + 2 * i));
        hi = fmax(hi, __ldcg(sv.ends + 2 * i + 1));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        lo = fmin(lo, __shfl_xor_sync(0xffffffffu, lo, o));
        hi = fmax(hi, __shfl_xor_sync(0xffffffffu, hi, o));
    }
    if (lane == 0) { s_lo[warp] = lo; s_hi[warp] = hi; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < warps_per_block; ++w) { lo = fmin(lo, s_lo[w]); hi = fmax(hi, s_hi[w]); }
        d_eps[0] = lo;
        d_eps[1] = hi;
        *sv.blocks_done = 0;        // leave the header clean (the entry point clears it again anyway)
    }
}

// device address of g_noalloc_scratch, asked for once per device with that device current
std::mutex g_mu;
unsigned char* g_scratch_ptr[kMaxDevices] = {};
int g_sm_count[kMaxDevices] = {};

int scratch_for_device(int dev, unsigned char** out, int* sms) {
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_scratch_ptr[dev]) {
        void* p = nullptr;
        if (cudaGetSymbolAddress(&p, g_noalloc_scratch) != cudaSuccess || !p) return DMPT_ECUDA;
        int n_sm = 0;
        if (cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n_sm <= 0)
            return DMPT_ECUDA;
        g_scratch_ptr[dev] = static_cast<unsigned char*>(p);
        g_sm_count[dev] = n_sm;
    }
    *out = g_scratch_ptr[dev];
    *sms = g_sm_count[dev];
    return DMPT_OK;
}

}  // namespace

extern "C" int dmpt_spectral_bounds_noalloc(const float* d_h0, int n, int ld, double* d_eps, void* cuda_stream) {
    if (!d_h0 || !d_eps || n <= 0 || ld < n) return DMPT_EINVAL;
    if (n > kMaxN) return DMPT_ELIMIT;
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return DMPT_ECUDA; }
    if (dev < 0 || dev >= kMaxDevices) return DMPT_ELIMIT;
    unsigned char* scratch = nullptr;
    int sms = 0;
    if (int rc = scratch_for_device(dev, &scratch, &sms)) { cudaGetLastError(); return rc; }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    if (cudaMemsetAsync(scratch, 0, kHeaderBytes, st) != cudaSuccess) { cudaGetLastError(); return DMPT_ECUDA; }
    const int blocks_needed = (n + 7) / 8;                       // 8 rows (warps) per block and pass
    const int grid = blocks_needed < 8 * sms ? blocks_needed : 8 * sms;
    dmpt_gershgorin_noalloc_kernel<<<grid, 256, 0, st>>>(d_h0, n, ld, scratch, d_eps);
    if (cudaGetLastError() != cudaSuccess) return DMPT_ECUDA;
    return DMPT_OK;
}
