// k_post.cu -- a-4 azimuthal average (Eq. 30, trapezoidal rule L183) and a-5 correlation function
// c(r), p(r) (Eq. 34-35).  Both passes move at most a few MB: they are bounded by HBM traffic
// in principle and by launch latency in practice.
#include "nms_internal.h"

namespace nms {

// ---- polar rings: periodic trapezoid == arithmetic mean over theta (reading 7) --------------------
// one warp per (map, ring); lanes stride over theta, fp64 partial sums combined by warp shuffles.
__global__ void __launch_bounds__(256) k_ring_mean(const float* __restrict__ maps, int n_maps, int n0, int n1,
                                                   const float* __restrict__ u0, float* __restrict__ out_I,
                                                   float* __restrict__ out_q, int32_t* __restrict__ out_count)
{
    const int64_t w = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (w >= (int64_t)n_maps * n0) return;
    const float* row = maps + w * n1;
    double s = 0.0;
    for (int j = lane; j < n1; j += 32) s += (double)row[j];
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane == 0) {
        out_I[w] = (float)(s / (double)n1);
        if (w < n0) {
            if (out_q) out_q[w] = u0[w];
            if (out_count) out_count[w] = n1;
        }
    }
}

// ---- |q| histogram (reading 8) ---------------------------------------------------------------------
// bin = floor((|q| - q_lo) / (q_hi - q_lo) * n_bins), |q| = sqrt(q_y^2 + q_z^2), in fp64 in exactly this
// order with individually rounded operations (no FMA contraction): the bin is an integer decision.
__global__ void __launch_bounds__(256) k_bin_index(const double2* __restrict__ qc, int64_t n_q, int n_bins, double q_lo,
                                                   double q_hi, int32_t* __restrict__ bin_idx,
                                                   int32_t* __restrict__ bin_cnt)
{
    const int64_t f = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (f >= n_q) return;
    const double2 q = qc[f];
    const double qq = sqrt(__dadd_rn(__dmul_rn(q.x, q.x), __dmul_rn(q.y, q.y)));
    int b = -1;
    if (!(qq < q_lo)) {
        const double fb = floor(__dmul_rn(__ddiv_rn(__dsub_rn(qq, q_lo), __dsub_rn(q_hi, q_lo)), (double)n_bins));
        if (fb < (double)n_bins) b = (int)fb;
    }
    bin_idx[f] = b;
    if (b >= 0) atomicAdd(bin_cnt + b, 1);
}

// warp-aggregated accumulation: lanes that hit the same bin are combined by shuffles, one fp64 atomic per
// distinct bin and warp.
__global__ void __launch_bounds__(256) k_bin_accumulate(const float* __restrict__ maps, int64_t n_q, int n_bins,
                                                        const int32_t* __restrict__ bin_idx, double* __restrict__ bin_sum)
{
    const int64_t f = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int map = blockIdx.y;
    const int lane = threadIdx.x & 31;
    int b = -1;
    double v = 0.0;
    if (f < n_q) { b = bin_idx[f]; v = (double)maps[(int64_t)map * n_q + f]; }
    const unsigned peers = __match_any_sync(0xffffffffu, b);
    double s = 0.0;
#pragma unroll
    for (int src = 0; src < 32; ++src) {
        const double o = __shfl_sync(0xffffffffu, v, src);
        if ((peers >> src) & 1u) s += o;
    }
    if (b >= 0 && lane == (__ffs(peers) - 1)) atomicAdd(bin_sum + (int64_t)map * n_bins + b, s);
}

__global__ void __launch_bounds__(256) k_bin_finish(const double* __restrict__ bin_sum, const int32_t* __restrict__ bin_cnt,
                                                    int n_maps, int n_bins, double q_lo, double q_hi,
                                                    float* __restrict__ out_I, float* __restrict__ out_q,
                                                    int32_t* __restrict__ out_count)
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

nms_status launch_azimuthal(nms_ctx* c, const float* maps, int n_maps, int n_bins, double q_lo, double q_hi,
                            float* out_I, float* out_q, int32_t* out_count)
{
    timer_begin(c, NMS_T_AZIMUTHAL);
    if (c->g_type == 0 && !(q_hi > q_lo)) {
        const int64_t warps = (int64_t)n_maps * c->g_n0;
        const unsigned blocks = (unsigned)((warps * 32 + 255) / 256);
        k_ring_mean<<<blocks, 256, 0, c->stream>>>(maps, n_maps, c->g_n0, c->g_n1, (const float*)c->u0.p, out_I, out_q,
                                                   out_count);
        c->launches += 1;
    } else {
        if (nms_status st = ensure(c, c->bin_idx, sizeof(int32_t) * (size_t)c->n_q)) return st;
        if (nms_status st = ensure(c, c->bin_cnt, sizeof(int32_t) * (size_t)n_bins)) return st;
        if (nms_status st = ensure(c, c->bin_sum, sizeof(double) * (size_t)n_bins * n_maps)) return st;
        NMS_CUDA(c, cudaMemsetAsync(c->bin_cnt.p, 0, sizeof(int32_t) * (size_t)n_bins, c->stream));
        NMS_CUDA(c, cudaMemsetAsync(c->bin_sum.p, 0, sizeof(double) * (size_t)n_bins * n_maps, c->stream));
        const unsigned qb = (unsigned)((c->n_q + 255) / 256);
        k_bin_index<<<qb, 256, 0, c->stream>>>((const double2*)c->qc.p, c->n_q, n_bins, q_lo, q_hi,
                                               (int32_t*)c->bin_idx.p, (int32_t*)c->bin_cnt.p);
        k_bin_accumulate<<<dim3(qb, (unsigned)n_maps), 256, 0, c->stream>>>(maps, c->n_q, n_bins,
                                                                           (const int32_t*)c->bin_idx.p,
                                                                           (double*)c->bin_sum.p);
        const unsigned fb = (unsigned)(((int64_t)n_maps * n_bins + 255) / 256);
        k_bin_finish<<<fb, 256, 0, c->stream>>>((const double*)c->bin_sum.p, (const int32_t*)c->bin_cnt.p, n_maps,
                                                n_bins, q_lo, q_hi, out_I, out_q, out_count);
        c->launches += 3;
    }
    timer_end(c, NMS_T_AZIMUTHAL);
    NMS_CUDA(c, cudaGetLastError());
    return NMS_OK;
}

// ---- correlation function (Eq. 34-35) ----------------------------------------------------------------
// c(r) = (1/2 pi^2) trapz_q [ I(q) j0(q r) q^2 ] over the non-empty bins only (reading 9).  The trapezoid
// is rewritten as a weighted sum, sum_t g_t j0(q_t r) with g_t = I_t q_t^2 * (half the sum of the two
// neighbouring gaps); pass 1 compacts the non-empty bins and forms g, pass 2 is one thread per (curve, r).
__global__ void k_corr_compact(const float* __restrict__ I, const float* __restrict__ q, const int32_t* __restrict__ count,
                               int n_maps, int n_bins, double* __restrict__ qv, double* __restrict__ gv,
                               int32_t* __restrict__ n_valid)
{
    // single block; thread 0 compacts (n_bins is a few thousand at most), then all threads form g
    __shared__ int n_sh;
    extern __shared__ int idx[];
    if (threadIdx.x == 0) {
        int n = 0;
        for (int b = 0; b < n_bins; ++b)
            if (!count || count[b] > 0) idx[n++] = b;
        n_sh = n;
        *n_valid = n;
    }
    __syncthreads();
    const int n = n_sh;
    for (int t = threadIdx.x; t < n; t += blockDim.x) {
        const double qt = (double)q[idx[t]];
        double w = 0.0;
        if (t + 1 < n) w += (double)q[idx[t + 1]] - qt;
        if (t > 0) w += qt - (double)q[idx[t - 1]];
        w *= 0.5;
        qv[t] = qt;
        for (int a = 0; a < n_maps; ++a) gv[(int64_t)a * n_bins + t] = (double)I[(int64_t)a * n_bins + idx[t]] * qt * qt * w;
    }
}

__global__ void __launch_bounds__(128) k_corr(const double* __restrict__ qv, const double* __restrict__ gv,
                                              const int32_t* __restrict__ n_valid, int n_bins,
                                              const float* __restrict__ r, int n_r, float* __restrict__ out_c,
                                              float* __restrict__ out_p)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    const int a = blockIdx.y;
    if (k >= n_r) return;
    const int n = *n_valid;
    const double rk = (double)r[k];
    const double* g = gv + (int64_t)a * n_bins;
    double s = 0.0;
    for (int t = 0; t < n; ++t) {
        const double x = qv[t] * rk;
        const double j0 = fabs(x) < 1e-4 ? 1.0 - x * x / 6.0 : sin(x) / x;
        s += g[t] * j0;
    }
    const double cc = s / (2.0 * 3.14159265358979323846 * 3.14159265358979323846);
    out_c[(int64_t)a * n_r + k] = (float)cc;
    out_p[(int64_t)a * n_r + k] = (float)(rk * rk * cc);
}

nms_status launch_correlation(nms_ctx* c, const float* I, const float* q_of_bin, const int32_t* count, int n_maps,
                              int n_bins, const float* r, int n_r, float* out_c, float* out_p)
{
    // scratch: qv [n_bins] | gv [n_maps][n_bins] | n_valid
    const size_t need = sizeof(double) * (size_t)n_bins * (1 + (size_t)n_maps) + 16;
    if (nms_status st = ensure(c, c->bin_sum, need)) return st;
    double* qv = (double*)c->bin_sum.p;
    double* gv = qv + n_bins;
    int32_t* n_valid = (int32_t*)(gv + (size_t)n_maps * n_bins);
    timer_begin(c, NMS_T_CORRELATION);
    k_corr_compact<<<1, 256, sizeof(int) * (size_t)n_bins, c->stream>>>(I, q_of_bin, count, n_maps, n_bins, qv, gv, n_valid);
    k_corr<<<dim3((unsigned)((n_r + 127) / 128), (unsigned)n_maps), 128, 0, c->stream>>>(qv, gv, n_valid, n_bins, r, n_r,
                                                                                        out_c, out_p);
    timer_end(c, NMS_T_CORRELATION);
    c->launches += 2;
    NMS_CUDA(c, cudaGetLastError());
    return NMS_OK;
}

}  // namespace nms
