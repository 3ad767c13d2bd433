// k_epilogue.cu -- a-3: sum the fp64 chunk partials of the amplitude kernel and form the requested
// response functions (Eq. 3-29) in the same pass; the amplitudes are only written out when
// the caller asks for them (nms_amplitudes) -- the fused nms_compute path goes partials -> responses.
#include "nms_internal.h"
#include "nms_response.cuh"

namespace nms {

struct EpiArgs {
    const double* part;     // [n_chunks][8][n_q]
    const double* formpart; // split: [n_chunks][n_kinds][n_q]
    const double2* sc;      // (sin th, cos th)
    const int32_t* kinds;
    int n_kinds, n_chunks;
    int64_t n_q;
    int64_t n_q_part;       // detector points of the partials (= n_q, or n_q / 2 under Friedel halving)
    int friedel_n1;         // 0, or n1 of the polar grid whose second half of every ring is the conjugate of the first
    float* out_maps;        // [n_kinds][n_q] or NULL
    float* out_form;        // split: [n_kinds][n_q] or NULL
    float* out_amp;         // [8][n_q] or NULL
    double* amp64;          // [8][n_q] or NULL
    RespParams rp;
};

__global__ void __launch_bounds__(256) k_epilogue(const EpiArgs a)
{
    const int64_t f = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (f >= a.n_q) return;
    double A[8];
#pragma unroll
    for (int r = 0; r < 8; ++r) A[r] = 0.0;
    if (a.part) {
        // Friedel halving (f-4): real weights give A(-q) = A(q)^* (Eq. 42-43), and on a ring theta -> theta + pi is -q
        int64_t fs = f;
        bool conj = false;
        if (a.friedel_n1) {
            const int64_t i = f / a.friedel_n1, j = f % a.friedel_n1, hn = a.friedel_n1 / 2;
            conj = j >= hn;
            fs = i * hn + (conj ? j - hn : j);
        }
        for (int ch = 0; ch < a.n_chunks; ++ch)
#pragma unroll
            for (int r = 0; r < 8; ++r) A[r] += a.part[((int64_t)ch * 8 + r) * a.n_q_part + fs];
        if (conj) { A[1] = -A[1]; A[3] = -A[3]; A[5] = -A[5]; A[7] = -A[7]; }
    } else {
#pragma unroll
        for (int r = 0; r < 8; ++r) A[r] = a.amp64[(int64_t)r * a.n_q + f];
    }
    if (a.part && a.amp64) {
#pragma unroll
        for (int r = 0; r < 8; ++r) a.amp64[(int64_t)r * a.n_q + f] = A[r];
    }
    if (a.out_amp) {
#pragma unroll
        for (int r = 0; r < 8; ++r) a.out_amp[(int64_t)r * a.n_q + f] = (float)A[r];
    }
    if (a.out_maps && a.n_kinds > 0) {
        const double2 d = a.sc[f];
        double val[NMS_KIND_COUNT];
        responses_at_point(A, d.x, d.y, a.rp, val);
        for (int i = 0; i < a.n_kinds; ++i) a.out_maps[(int64_t)i * a.n_q + f] = (float)val[a.kinds[i]];
    }
    if (a.out_form && a.formpart) {
        for (int i = 0; i < a.n_kinds; ++i) {
            double s = 0.0;
            for (int ch = 0; ch < a.n_chunks; ++ch) s += a.formpart[((int64_t)ch * a.n_kinds + i) * a.n_q + f];
            a.out_form[(int64_t)i * a.n_q + f] = (float)s;
        }
    }
}

// Fourier cross-correlation components (Eq. 51-52): G_ab = invV sM^2 M~_a M~_b^*, a, b in (x, y, z),
// from the stored fp64 amplitudes; rows 3 a + b of G^R and G^I.
__global__ void __launch_bounds__(256) k_cross_spectra(const double* __restrict__ amp64, int64_t n_q, double scale,
                                                       float* __restrict__ out_GR, float* __restrict__ out_GI)
{
    const int64_t f = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (f >= n_q) return;
    double re[3], im[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        re[c] = amp64[(int64_t)(2 + 2 * c) * n_q + f];
        im[c] = amp64[(int64_t)(3 + 2 * c) * n_q + f];
    }
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            // (ra + i ia)(rb - i ib) = (ra rb + ia ib) + i (ia rb - ra ib)
            if (out_GR) out_GR[(int64_t)(3 * a + b) * n_q + f] = (float)(scale * (re[a] * re[b] + im[a] * im[b]));
            if (out_GI) out_GI[(int64_t)(3 * a + b) * n_q + f] = (float)(scale * (im[a] * re[b] - re[a] * im[b]));
        }
}

nms_status launch_cross_spectra(nms_ctx* c, float* out_GR, float* out_GI)
{
    const unsigned blocks = (unsigned)((c->n_q + 255) / 256);
    if (nms_status ts_ = timer_begin(c, NMS_T_EPILOGUE)) return ts_;
    k_cross_spectra<<<blocks, 256, 0, c->stream>>>((const double*)c->amp64.p, c->n_q, c->invV * c->sM * c->sM, out_GR, out_GI);
    if (nms_status ts_ = timer_end(c, NMS_T_EPILOGUE)) return ts_;
    c->launches += 1;
    NMS_CUDA(c, cudaGetLastError());
    return NMS_OK;
}

static void fill_rp(const nms_ctx* c, RespParams& rp)
{
    rp.Px = c->P[0]; rp.Py = c->P[1]; rp.Pz = c->P[2];
    rp.sN = c->sN; rp.sM = c->sM; rp.invV = c->invV;
}

static nms_status run(nms_ctx* c, const EpiArgs& a)
{
    const int threads = 256;
    const unsigned blocks = (unsigned)((c->n_q + threads - 1) / threads);
    if (nms_status ts_ = timer_begin(c, NMS_T_EPILOGUE)) return ts_;
    k_epilogue<<<blocks, threads, 0, c->stream>>>(a);
    if (nms_status ts_ = timer_end(c, NMS_T_EPILOGUE)) return ts_;
    c->launches += 1;
    NMS_CUDA(c, cudaGetLastError());
    return NMS_OK;
}

nms_status launch_epilogue(nms_ctx* c, int n_chunks, const int32_t* kinds_dev, int n_kinds, float* out_maps,
                           float* out_amp, bool keep_amp64)
{
    EpiArgs a = {};
    a.part = (const double*)c->part.p; a.sc = (const double2*)c->sc.p; a.kinds = kinds_dev;
    a.n_kinds = n_kinds; a.n_chunks = n_chunks; a.n_q = c->n_q;
    a.n_q_part = c->friedel_active ? c->n_q / 2 : c->n_q; a.friedel_n1 = c->friedel_active ? c->g_n1 : 0;
    a.out_maps = out_maps; a.out_amp = out_amp;
    if (keep_amp64) {
        if (nms_status st = ensure(c, c->amp64, sizeof(double) * 8 * (size_t)c->n_q)) return st;
        a.amp64 = (double*)c->amp64.p;
    }
    fill_rp(c, a.rp);
    return run(c, a);
}

nms_status launch_response_from_amp(nms_ctx* c, const int32_t* kinds_dev, int n_kinds, float* out_maps)
{
    EpiArgs a = {};
    a.amp64 = (double*)c->amp64.p; a.sc = (const double2*)c->sc.p; a.kinds = kinds_dev;
    a.n_kinds = n_kinds; a.n_q = c->n_q; a.out_maps = out_maps;
    fill_rp(c, a.rp);
    return run(c, a);
}

nms_status launch_split_epilogue(nms_ctx* c, int n_chunks, const int32_t* kinds_dev, int n_kinds, float* out_total,
                                 float* out_form)
{
    EpiArgs a = {};
    a.part = (const double*)c->part.p; a.formpart = (const double*)c->formpart.p; a.sc = (const double2*)c->sc.p;
    a.kinds = kinds_dev; a.n_kinds = n_kinds; a.n_chunks = n_chunks; a.n_q = c->n_q; a.n_q_part = c->n_q;
    a.out_maps = out_total; a.out_form = out_form;
    fill_rp(c, a.rp);
    return run(c, a);
}

}  // namespace nms
