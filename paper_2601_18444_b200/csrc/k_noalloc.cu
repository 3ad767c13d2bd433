// k_noalloc.cu -- nms_azimuthal_average_noalloc: the |q|-histogram average of a-4 (Eq. 30, reading 8) for callers that
// cannot allocate device memory (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).
//
// The existing path (k_post.cu: k_bin_index, k_bin_accumulate, k_bin_finish) keeps three scratch arrays in the context,
// grown with cudaMalloc on demand: the bin index of every detector point, the per-bin counts and the per-(map, bin) fp64
// sums.  This variant needs no per-point scratch -- one kernel derives the bin of a point and accumulates all maps at it --
// and keeps counts and sums in ONE file-scope device array of fixed size:
//
//     g_hist_scratch: NOALLOC_MAX_SUMS doubles (sums, [n_maps][n_bins]) followed by NOALLOC_MAX_BINS int32 (counts)
//                     = 65536 x 8 B + 16384 x 4 B = 576 KB, held by every GPU that loads libnms.so until the process exits.
//
// In host code the array's name is a host-side stand-in, not a device address; the address is resolved once per device,
// with that device current, by cudaGetSymbolAddress (scratch_address below) and passed to the kernels as a pointer.
// Every call, from every context on the device, shares the array, and it keeps the last call's contents: each call clears
// the part it uses on its own stream first.  Two calls that overlap on the GPU (different streams, or contexts of two host
// threads on one device) race on it -- serialise them.
//
// The entry point calls no cudaMalloc, cudaFree or allocating library routine and records no timing events; the bin
// arithmetic is that of k_bin_index, operation by operation, so counts are identical to the existing path's and the
// averages differ only by the order of the fp64 additions.
#include "nms_internal.h"

#include <mutex>

namespace nms {

constexpr int NOALLOC_MAX_BINS = 16384;      // n_bins
constexpr int NOALLOC_MAX_SUMS = 65536;      // n_maps * n_bins
constexpr int NOALLOC_MAX_DEVICES = 64;

static __device__ __align__(256) double g_hist_scratch[NOALLOC_MAX_SUMS + NOALLOC_MAX_BINS / 2];

// One thread per detector point: its bin (fp64, individually rounded operations, exactly as k_bin_index), one count, and
// for every map the warp-aggregated sum of the lanes that share the bin -- one fp64 atomic per distinct bin, map and warp.
__global__ void __launch_bounds__(256) k_hist_fused(const float* __restrict__ maps, const double2* __restrict__ qc, int64_t n_q,
                                                    int n_maps, int n_bins, double q_lo, double q_hi,
                                                    double* __restrict__ bin_sum, int32_t* __restrict__ bin_cnt)
{
    const int64_t f = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
    int b = -1;
    if (f < n_q) {
        const double2 q = qc[f];
        const double qq = sqrt(__dadd_rn(__dmul_rn(q.x, q.x), __dmul_rn(q.y, q.y)));
        if (!(qq < q_lo)) {
            const double fb = floor(__dmul_rn(__ddiv_rn(__dsub_rn(qq, q_lo), __dsub_rn(q_hi, q_lo)), (double)n_bins));
            if (fb < (double)n_bins) b = (int)fb;
        }
    }
    const unsigned peers = __match_any_sync(0xffffffffu, b);
    const bool leader = b >= 0 && lane == (__ffs(peers) - 1);
    if (leader) atomicAdd(bin_cnt + b, __popc(peers));
    for (int map = 0; map < n_maps; ++map) {
        const double v = b >= 0 ? (double)maps[(int64_t)map * n_q + f] : 0.0;
        double s = 0.0;
#pragma unroll
        for (int src = 0; src < 32; ++src) {
            const double o = __shfl_sync(0xffffffffu, v, src);
            if ((peers >> src) & 1u) s += o;
        }
        if (leader) atomicAdd(bin_sum + (int64_t)map * n_bins + b, s);
    }
}

__global__ void __launch_bounds__(256) k_hist_finish(const double* __restrict__ bin_sum, const int32_t* __restrict__ bin_cnt,
                                                     int n_maps, int n_bins, double q_lo, double q_hi, float* __restrict__ out_I,
                                                     float* __restrict__ out_q, int32_t* __restrict__ out_count)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (int64_t)n_maps * n_bins) return;
    const int b = (int)(i % n_bins);
    const int cnt = bin_cnt[b];
    out_I[i] = cnt > 0 ? (float)(bin_sum[i] / (double)cnt) : 0.f;
    if (i < n_bins) {
        if (out_q) out_q[b] = (float)(q_lo + ((double)b + 0.5) * (q_hi - q_lo) / (double)n_bins);   // bin centre
        if (out_count) out_count[b] = cnt;
    }
}

// Device address of g_hist_scratch on the context's device, resolved once per device with that device current.
static nms_status scratch_address(nms_ctx* c, double** out)
{
    static std::mutex mu;
    static double* table[NOALLOC_MAX_DEVICES] = {};
    if (c->device < 0 || c->device >= NOALLOC_MAX_DEVICES)
        return fail(c, NMS_E_UNSUPPORTED, "device ordinal %d outside 0..%d", c->device, NOALLOC_MAX_DEVICES - 1);
    std::lock_guard<std::mutex> lock(mu);
    if (!table[c->device]) {
        double* p = nullptr;
        NMS_CUDA(c, cudaSetDevice(c->device));
        NMS_CUDA(c, cudaGetSymbolAddress((void**)&p, g_hist_scratch));
        if (!p) return fail(c, NMS_E_CUDA, "cudaGetSymbolAddress returned a NULL address for the histogram scratch");
        table[c->device] = p;
    }
    *out = table[c->device];
    return NMS_OK;
}

}  // namespace nms

using namespace nms;

extern "C" nms_status nms_azimuthal_average_noalloc(nms_ctx* c, const float* maps, int n_maps, int n_bins, double q_lo,
                                                    double q_hi, float* out_I, float* out_q, int32_t* out_count)
{
    if (!c) return NMS_E_ARG;
    c->err[0] = 0;
    NMS_CUDA(c, cudaSetDevice(c->device));
    if (!c->grid_valid)
        return fail(c, NMS_E_STATE, "nms_azimuthal_average_noalloc needs a current grid (nms_amplitudes / nms_compute)");
    if (!maps || !out_I || n_maps <= 0 || n_bins <= 0) return fail(c, NMS_E_ARG, "maps/out_I NULL or non-positive sizes");
    if (!(q_hi > q_lo))
        return fail(c, NMS_E_ARG, "nms_azimuthal_average_noalloc is the |q| histogram (q_hi > q_lo); the ring mode of "
                                  "nms_azimuthal_average uses no scratch memory");
    if (n_bins > NOALLOC_MAX_BINS || (int64_t)n_maps * n_bins > NOALLOC_MAX_SUMS)
        return fail(c, NMS_E_UNSUPPORTED, "n_bins = %d, n_maps * n_bins = %lld exceed the static scratch (n_bins <= %d, "
                                          "n_maps * n_bins <= %d): use nms_azimuthal_average",
                    n_bins, (long long)n_maps * n_bins, NOALLOC_MAX_BINS, NOALLOC_MAX_SUMS);
    double* scratch = nullptr;
    if (nms_status st = scratch_address(c, &scratch)) return st;
    double* bin_sum = scratch;
    int32_t* bin_cnt = reinterpret_cast<int32_t*>(scratch + NOALLOC_MAX_SUMS);
    // the array keeps the last call's contents: clear what this call uses (stream-ordered, nothing is allocated)
    NMS_CUDA(c, cudaMemsetAsync(bin_sum, 0, sizeof(double) * (size_t)n_maps * n_bins, c->stream));
    NMS_CUDA(c, cudaMemsetAsync(bin_cnt, 0, sizeof(int32_t) * (size_t)n_bins, c->stream));
    const unsigned qb = (unsigned)((c->n_q + 255) / 256);
    k_hist_fused<<<qb, 256, 0, c->stream>>>(maps, (const double2*)c->qc.p, c->n_q, n_maps, n_bins, q_lo, q_hi, bin_sum, bin_cnt);
    const unsigned fb = (unsigned)(((int64_t)n_maps * n_bins + 255) / 256);
    k_hist_finish<<<fb, 256, 0, c->stream>>>(bin_sum, bin_cnt, n_maps, n_bins, q_lo, q_hi, out_I, out_q, out_count);
    c->launches += 2;
    NMS_CUDA(c, cudaGetLastError());
    return NMS_OK;
}
