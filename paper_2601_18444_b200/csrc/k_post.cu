// k_post.cu -- a-4 azimuthal average (Eq. 30, trapezoidal rule L183) and a-5 correlation function
// c(r), p(r) (Eq. 34-35).  Both passes move at most a few MB: they are bounded by HBM traffic
// in principle and by launch latency in practice.
#include <utility>
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

// ---- angular modal decomposition (Eq. 31-33) -------------------------------
// I_k^{s,c}(q_i) = (2 - delta_k0) / n_theta * sum_j f(q_i, theta_j) {sin, cos}(k theta_j): the trapezoidal rule
// of L183 on the periodic theta grid (reading 7).  Pass 1 tabulates (sin, cos)(k theta_j) in fp64 from the
// grid's own float angles; pass 2 is one warp per (map, k, ring) with fp64 partial sums and warp shuffles;
// pass 3 (one block per map, one warp per k) forms a_k = sum_i I_k(q_i) (Eq. 32) from the fp64 ring values
// and A_k = a_k / sum_j sqrt(a_j^s^2 + a_j^c^2) (Eq. 33).
__global__ void k_modal_table(const float* __restrict__ theta, int n1, int nk, double2* __restrict__ tab)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= nk * n1) return;
    const int k = t / n1, j = t % n1;
    double s, c;
    sincos((double)k * (double)theta[j], &s, &c);
    tab[t] = make_double2(s, c);
}

__global__ void __launch_bounds__(256) k_modal_rings(const float* __restrict__ maps, int n_maps, int n0, int n1, int nk,
                                                     const double2* __restrict__ tab, double2* __restrict__ ring,
                                                     float* __restrict__ out_Is, float* __restrict__ out_Ic)
{
    const int64_t w = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;   // (map, k, ring)
    const int lane = threadIdx.x & 31;
    if (w >= (int64_t)n_maps * nk * n0) return;
    const int i = (int)(w % n0), k = (int)((w / n0) % nk), a = (int)(w / ((int64_t)n0 * nk));
    const float* row = maps + ((int64_t)a * n0 + i) * n1;
    const double2* tk = tab + (int64_t)k * n1;
    double ss = 0.0, cc = 0.0;
    for (int j = lane; j < n1; j += 32) {
        const double f = (double)row[j];
        const double2 sc = tk[j];
        ss = fma(f, sc.x, ss);
        cc = fma(f, sc.y, cc);
    }
    for (int o = 16; o > 0; o >>= 1) {
        ss += __shfl_xor_sync(0xffffffffu, ss, o);
        cc += __shfl_xor_sync(0xffffffffu, cc, o);
    }
    if (lane == 0) {
        const double pref = (k == 0 ? 1.0 : 2.0) / (double)n1;
        ss *= pref; cc *= pref;
        ring[w] = make_double2(ss, cc);
        if (out_Is) out_Is[w] = (float)ss;
        if (out_Ic) out_Ic[w] = (float)cc;
    }
}

constexpr int MODAL_KMAX = 63;

__global__ void __launch_bounds__(1024) k_modal_amplitudes(const double2* __restrict__ ring, int n0, int nk,
                                                           float* __restrict__ out_a, float* __restrict__ out_A)
{
    __shared__ double as_[MODAL_KMAX + 1], ac_[MODAL_KMAX + 1];
    __shared__ double norm;
    const int a = blockIdx.x, lane = threadIdx.x & 31, warp = threadIdx.x >> 5, n_warps = blockDim.x >> 5;
    for (int k = warp; k < nk; k += n_warps) {
        const double2* r = ring + ((int64_t)a * nk + k) * n0;
        double ss = 0.0, cc = 0.0;
        for (int i = lane; i < n0; i += 32) { ss += r[i].x; cc += r[i].y; }
        for (int o = 16; o > 0; o >>= 1) {
            ss += __shfl_xor_sync(0xffffffffu, ss, o);
            cc += __shfl_xor_sync(0xffffffffu, cc, o);
        }
        if (lane == 0) { as_[k] = ss; ac_[k] = cc; }
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double n = 0.0;
        for (int k = 0; k < nk; ++k) n += sqrt(as_[k] * as_[k] + ac_[k] * ac_[k]);
        norm = n;
    }
    __syncthreads();
    for (int k = threadIdx.x; k < nk; k += blockDim.x) {
        const int64_t o = (int64_t)a * 2 * nk;
        if (out_a) { out_a[o + k] = (float)as_[k]; out_a[o + nk + k] = (float)ac_[k]; }
        if (out_A) {
            out_A[o + k] = norm > 0.0 ? (float)(as_[k] / norm) : 0.f;
            out_A[o + nk + k] = norm > 0.0 ? (float)(ac_[k] / norm) : 0.f;
        }
    }
}

nms_status launch_modal(nms_ctx* c, const float* maps, int n_maps, int k_max, float* out_Is, float* out_Ic, float* out_a,
                        float* out_A)
{
    const int nk = k_max + 1, n0 = c->g_n0, n1 = c->g_n1;
    if (nms_status st = ensure(c, c->modal_tab, sizeof(double2) * (size_t)nk * n1)) return st;
    if (nms_status st = ensure(c, c->modal_ring, sizeof(double2) * (size_t)n_maps * nk * n0)) return st;
    if (nms_status ts_ = timer_begin(c, NMS_T_MODAL)) return ts_;
    k_modal_table<<<(unsigned)((nk * n1 + 255) / 256), 256, 0, c->stream>>>((const float*)c->u1.p, n1, nk,
                                                                           (double2*)c->modal_tab.p);
    const int64_t warps = (int64_t)n_maps * nk * n0;
    k_modal_rings<<<(unsigned)((warps * 32 + 255) / 256), 256, 0, c->stream>>>(maps, n_maps, n0, n1, nk,
                                                                              (const double2*)c->modal_tab.p,
                                                                              (double2*)c->modal_ring.p, out_Is, out_Ic);
    c->launches += 2;
    if (out_a || out_A) {
        k_modal_amplitudes<<<(unsigned)n_maps, 1024, 0, c->stream>>>((const double2*)c->modal_ring.p, n0, nk, out_a, out_A);
        c->launches += 1;
    }
    if (nms_status ts_ = timer_end(c, NMS_T_MODAL)) return ts_;
    NMS_CUDA(c, cudaGetLastError());
    return NMS_OK;
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
    if (nms_status ts_ = timer_begin(c, NMS_T_AZIMUTHAL)) return ts_;
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
    if (nms_status ts_ = timer_end(c, NMS_T_AZIMUTHAL)) return ts_;
    NMS_CUDA(c, cudaGetLastError());
    return NMS_OK;
}

// ---- two-dimensional correlation function (Eq. 36) -----------------------------
// C(rho, alpha) = sum_pixels w_p exp(+i (Y_p rho_y + Z_p rho_z)),  (Y_p, Z_p) = (q sin th, q cos th),
// w_p = f_p q wq dtheta: the direct Fourier sum of k_amplitude.cu with the detector pixels as cells and the
// (rho, alpha) points as detector.  Pass 1 writes the pixels as Cell records (weight in the nuclear channel);
// the amplitude kernel then runs unchanged on them; pass 3 sums the chunk partials: C = conj(N~).
__global__ void __launch_bounds__(256) k_pixel_cells(const float* __restrict__ map, const double2* __restrict__ qc,
                                                     const float* __restrict__ u0, int n0, int n1,
                                                     Cell* __restrict__ cells, TileMeta* __restrict__ meta)
{
    const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t n = (int64_t)n0 * n1;
    if (p < n) {
        const int i = (int)(p / n1);
        const double q = (double)u0[i];
        double wq = 1.0;                                   // non-uniform trapezoid in q, no extrapolation
        if (n0 > 1)
            wq = i == 0 ? 0.5 * ((double)u0[1] - q)
                        : (i == n0 - 1 ? 0.5 * (q - (double)u0[n0 - 2]) : 0.5 * ((double)u0[i + 1] - (double)u0[i - 1]));
        const double2 yz = qc[p];                           // (q sin th, q cos th) in fp64 (k_qsetup)
        Cell ce;
        ce.Y = yz.x; ce.Z = yz.y;
        ce.wN = (float)((double)map[p] * q * wq * (6.283185307179586476925 / (double)n1));
        ce.wx = 0.f; ce.wy = 0.f; ce.wz = 0.f;
        cells[p] = ce;
    }
    if (p % TILE == 0 && p < n) {
        TileMeta tm;
        tm.Y0 = 0.0; tm.Z0 = 0.0; tm.first_slot = p; tm.n_slots = (int32_t)((n - p) < TILE ? (n - p) : TILE);
        tm.flags = 3;
        meta[p / TILE] = tm;
    }
}

__global__ void __launch_bounds__(256) k_corr2d_finish(const double* __restrict__ part, int n_chunks, int64_t n_r,
                                                       float* __restrict__ out_re, float* __restrict__ out_im)
{
    const int64_t f = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (f >= n_r) return;
    double re = 0.0, im = 0.0;
    for (int ch = 0; ch < n_chunks; ++ch) {
        re += part[((int64_t)ch * 8 + 0) * n_r + f];
        im += part[((int64_t)ch * 8 + 1) * n_r + f];
    }
    if (out_re) out_re[f] = (float)re;
    if (out_im) out_im[f] = (float)(-im);      // the kernel sums exp(-i Psi): C = conj
}

nms_status launch_correlation_2d(nms_ctx* c, const float* map, const nms_qgrid* rgrid, float* out_re, float* out_im)
{
    const int64_t n_pix = c->n_q;
    const int64_t n_tiles = (n_pix + TILE - 1) / TILE;
    if (nms_status st = ensure(c, c->pix_cells, sizeof(Cell) * (size_t)n_pix)) return st;
    if (nms_status st = ensure(c, c->pix_meta, sizeof(TileMeta) * (size_t)n_tiles)) return st;
    k_pixel_cells<<<(unsigned)((n_pix + 255) / 256), 256, 0, c->stream>>>(map, (const double2*)c->qc.p, (const float*)c->u0.p,
                                                                          c->g_n0, c->g_n1, (Cell*)c->pix_cells.p,
                                                                          (TileMeta*)c->pix_meta.p);
    c->launches += 1;
    NMS_CUDA(c, cudaGetLastError());

    // run the amplitude path on (pixels, r-grid): exchange the context's sample and grid state, restore afterwards
    struct Saved {
        DevBuf cells, tile_meta, u0, u1, qc, sc;
        int64_t n_tiles, n_slots, W, K, n_q;
        bool grid_valid, g_uniform, has_N, has_M, amp_valid;
        int g_type, g_n0, g_n1, opt_qt, opt_bases, amp_timer;
        int variant_used, n_chunks_used, blocks_per_sm_used, qt_used, npoly_used, nb_used, rec3_used, interp_used;
        double g_dq, g_dev, g_qmax, geo_rmax, geo_ext, geo_extz;
        bool geo_pending;
        std::vector<float> h_u0, h_u1;
    } sv;
    auto exchange = [&]() {
        std::swap(sv.cells, c->cells); std::swap(sv.tile_meta, c->tile_meta);
        std::swap(sv.u0, c->u0); std::swap(sv.u1, c->u1); std::swap(sv.qc, c->qc); std::swap(sv.sc, c->sc);
        std::swap(sv.n_tiles, c->n_tiles); std::swap(sv.n_slots, c->n_slots); std::swap(sv.W, c->W); std::swap(sv.K, c->K);
        std::swap(sv.n_q, c->n_q); std::swap(sv.grid_valid, c->grid_valid); std::swap(sv.g_uniform, c->g_uniform);
        std::swap(sv.has_N, c->has_N); std::swap(sv.has_M, c->has_M);
        std::swap(sv.g_type, c->g_type); std::swap(sv.g_n0, c->g_n0); std::swap(sv.g_n1, c->g_n1); std::swap(sv.g_dq, c->g_dq);
        std::swap(sv.h_u0, c->h_u0); std::swap(sv.h_u1, c->h_u1);
        // the caller's stored amplitudes, tuning options and "used" records survive the exchanged run; the inner
        // amplitude launch is timed under NMS_T_CORR2D only
        std::swap(sv.amp_valid, c->amp_valid); std::swap(sv.opt_qt, c->opt_qt); std::swap(sv.opt_bases, c->opt_bases);
        std::swap(sv.amp_timer, c->amp_timer);
        std::swap(sv.g_dev, c->g_dev); std::swap(sv.g_qmax, c->g_qmax); std::swap(sv.geo_rmax, c->geo_rmax);
        std::swap(sv.geo_ext, c->geo_ext); std::swap(sv.geo_extz, c->geo_extz); std::swap(sv.geo_pending, c->geo_pending);
    };
    auto keep_used = [&](bool save) {
        int* u[] = {&c->variant_used, &c->n_chunks_used, &c->blocks_per_sm_used, &c->qt_used, &c->npoly_used, &c->nb_used, &c->rec3_used, &c->interp_used};
        int* s[] = {&sv.variant_used, &sv.n_chunks_used, &sv.blocks_per_sm_used, &sv.qt_used, &sv.npoly_used, &sv.nb_used, &sv.rec3_used, &sv.interp_used};
        for (int i = 0; i < 8; ++i) { if (save) *s[i] = *u[i]; else *u[i] = *s[i]; }
    };
    sv.cells = c->pix_cells; sv.tile_meta = c->pix_meta; sv.u0 = c->pix_u0; sv.u1 = c->pix_u1; sv.qc = c->pix_qc; sv.sc = c->pix_sc;
    sv.n_tiles = n_tiles; sv.n_slots = n_pix; sv.W = n_pix; sv.K = 0; sv.n_q = 0;
    sv.grid_valid = false; sv.g_uniform = false; sv.has_N = true; sv.has_M = false;
    sv.g_type = 0; sv.g_n0 = 0; sv.g_n1 = 0; sv.g_dq = 0.0;
    // the pixel sample: radius = largest |q| of the detector; a tile is an arc of a ring (centre left at 0: no correction)
    sv.g_dev = 0.0; sv.g_qmax = 0.0; sv.geo_rmax = c->g_qmax; sv.geo_ext = 0.0; sv.geo_extz = 0.0; sv.geo_pending = false;
    sv.amp_valid = false; sv.opt_qt = 0; sv.opt_bases = 0; sv.amp_timer = -1;
    keep_used(true);
    exchange();                                   // the context now describes the pixel sample, no grid yet
    nms_status st = set_grid(c, rgrid);
    AmpPlan plan;
    if (!st) st = plan_amplitude(c, false, false, &plan);
    if (!st) {
        st = timer_begin(c, NMS_T_CORR2D);
        if (!st) st = launch_amplitude(c, plan, nullptr, 0);
        if (!st) {
            const int64_t n_r = c->n_q;
            k_corr2d_finish<<<(unsigned)((n_r + 255) / 256), 256, 0, c->stream>>>((const double*)c->part.p, c->n_chunks_used,
                                                                                   n_r, out_re, out_im);
            c->launches += 1;
            st = timer_end(c, NMS_T_CORR2D);
        }
        c->corr2d_variant = c->variant_used;
    }
    exchange();                                   // back: sv holds the pixel / r-grid buffers again (possibly regrown)
    keep_used(false);
    c->pix_cells = sv.cells; c->pix_meta = sv.tile_meta; c->pix_u0 = sv.u0; c->pix_u1 = sv.u1; c->pix_qc = sv.qc; c->pix_sc = sv.sc;
    if (st) return st;
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
    if (nms_status ts_ = timer_begin(c, NMS_T_CORRELATION)) return ts_;
    k_corr_compact<<<1, 256, sizeof(int) * (size_t)n_bins, c->stream>>>(I, q_of_bin, count, n_maps, n_bins, qv, gv, n_valid);
    k_corr<<<dim3((unsigned)((n_r + 127) / 128), (unsigned)n_maps), 128, 0, c->stream>>>(qv, gv, n_valid, n_bins, r, n_r,
                                                                                        out_c, out_p);
    if (nms_status ts_ = timer_end(c, NMS_T_CORRELATION)) return ts_;
    c->launches += 2;
    NMS_CUDA(c, cudaGetLastError());
    return NMS_OK;
}

}  // namespace nms
