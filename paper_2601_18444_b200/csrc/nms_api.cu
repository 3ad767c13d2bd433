// nms_api.cu -- the C ABI of include/nms.h: context, argument checks, host-side planning.  Every
// numerical step runs in the kernels of k_prep.cu / k_amplitude.cu / k_epilogue.cu / k_post.cu.
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <string.h>
#include <new>
#include "nms_internal.h"

namespace nms {

nms_status fail(nms_ctx* c, nms_status st, const char* fmt, ...)
{
    if (c) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(c->err, sizeof(c->err), fmt, ap);
        va_end(ap);
    }
    return st;
}

nms_status cuda_fail(nms_ctx* c, cudaError_t e, const char* where)
{
    return fail(c, e == cudaErrorMemoryAllocation ? NMS_E_NOMEM : NMS_E_CUDA, "CUDA error '%s' in %s", cudaGetErrorString(e), where);
}

nms_status ensure(nms_ctx* c, DevBuf& b, size_t bytes)
{
    if (bytes == 0) bytes = 16;
    if (b.cap >= bytes) return NMS_OK;
    if (b.p) {
        // the stream may still use the old buffer
        cudaError_t e = cudaStreamSynchronize(c->stream);
        if (e != cudaSuccess) return cuda_fail(c, e, "cudaStreamSynchronize");
        cudaFree(b.p);
        b.p = nullptr; b.cap = 0;
    }
    cudaError_t e = cudaMalloc(&b.p, bytes);
    if (e != cudaSuccess) { b.p = nullptr; return cuda_fail(c, e, "cudaMalloc"); }
    b.cap = bytes;
    return NMS_OK;
}

nms_status timer_begin(nms_ctx* c, int which)
{
    if (!c->opt_timing || which < 0) return NMS_OK;
    Timer& t = c->timers[which];
    if (t.used == t.beg.size()) {
        cudaEvent_t b = nullptr, e = nullptr;
        NMS_CUDA(c, cudaEventCreate(&b));
        if (cudaError_t err = cudaEventCreate(&e)) { cudaEventDestroy(b); return cuda_fail(c, err, "cudaEventCreate"); }
        t.beg.push_back(b); t.end.push_back(e);
    }
    NMS_CUDA(c, cudaEventRecord(t.beg[t.used], c->stream));
    return NMS_OK;
}
nms_status timer_end(nms_ctx* c, int which)
{
    if (!c->opt_timing || which < 0) return NMS_OK;
    Timer& t = c->timers[which];
    NMS_CUDA(c, cudaEventRecord(t.end[t.used], c->stream));
    t.used += 1;
    return NMS_OK;
}

static void free_buf(DevBuf& b)
{
    if (b.p) cudaFree(b.p);
    b.p = nullptr; b.cap = 0;
}

static bool orthonormal(const double* R)
{
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
            double d = 0.0;
            for (int k = 0; k < 3; ++k) d += R[3 * i + k] * R[3 * j + k];
            if (!(fabs(d - (i == j ? 1.0 : 0.0)) <= 1e-6)) return false;
        }
    return true;
}

// Tile table: tiles of <= TILE consecutive cells that never straddle an object (L310-L317).
static nms_status build_tiles(nms_ctx* c)
{
    c->h_tile_src.clear(); c->h_tile_flags.clear(); c->h_tile_first_slot.clear();
    int64_t slot = 0;
    auto add_range = [&](int64_t b, int64_t e, int32_t particle) {
        if (e <= b) return;
        const size_t first_index = c->h_tile_src.size();
        for (int64_t s = b; s < e; s += TILE) {
            TileSrc ts; ts.src_first = s; ts.n_src = (int32_t)((e - s) < TILE ? (e - s) : TILE); ts.particle = particle;
            c->h_tile_src.push_back(ts);
            c->h_tile_flags.push_back(0);
            c->h_tile_first_slot.push_back(slot);
            slot += (ts.n_src + SLOT_PAD - 1) / SLOT_PAD * SLOT_PAD;
        }
        c->h_tile_flags[first_index] |= 2;      // first tile of the object
        c->h_tile_flags.back() |= 1;            // last tile of the object
    };
    if (c->K > 0) for (int64_t k = 0; k < c->K; ++k) add_range(c->offsets[k], c->offsets[k + 1], (int32_t)k);
    else add_range(0, c->W, -1);
    c->n_tiles = (int64_t)c->h_tile_src.size();
    c->n_slots = slot;
    if (c->n_tiles > 0x7fffffff / 2) return fail(c, NMS_E_UNSUPPORTED, "too many tiles");
    const size_t n = (size_t)c->n_tiles;
    const size_t bytes = n * (sizeof(TileSrc) + sizeof(int64_t) + sizeof(int32_t));
    if (nms_status st = ensure(c, c->tile_src, bytes)) return st;
    if (nms_status st = ensure(c, c->tile_meta, n * sizeof(TileMeta))) return st;
    if (nms_status st = ensure(c, c->cells, (size_t)slot * sizeof(Cell))) return st;
    if (nms_status st = ensure(c, c->wsum, 7 * sizeof(double))) return st;
    char* base = (char*)c->tile_src.p;
    NMS_CUDA(c, cudaMemcpyAsync(base, c->h_tile_src.data(), n * sizeof(TileSrc), cudaMemcpyHostToDevice, c->stream));
    NMS_CUDA(c, cudaMemcpyAsync(base + n * sizeof(TileSrc), c->h_tile_first_slot.data(), n * sizeof(int64_t),
                                cudaMemcpyHostToDevice, c->stream));
    NMS_CUDA(c, cudaMemcpyAsync(base + n * (sizeof(TileSrc) + sizeof(int64_t)), c->h_tile_flags.data(), n * sizeof(int32_t),
                                cudaMemcpyHostToDevice, c->stream));
    c->h_chunk_begin.clear();
    return NMS_OK;
}

static nms_status repack(nms_ctx* c)
{
    c->amp_valid = false;
    c->packed_valid = false;
    if (nms_status st = launch_prep(c)) return st;
    c->packed_valid = true;
    return NMS_OK;
}

// pos/N/m may be host or device pointers (cudaMemcpyDefault resolves the direction through UVA)
static nms_status set_sample_impl(nms_ctx* c, const float* pos, const float* N, const float* m, int64_t W, const double* R)
{
    if (!pos) return fail(c, NMS_E_ARG, "nms_set_sample: pos is NULL");
    if (W <= 0) return fail(c, NMS_E_ARG, "nms_set_sample: W = %lld must be positive", (long long)W);
    if (!N && !m) return fail(c, NMS_E_ARG, "nms_set_sample: both N and m are NULL");
    if (R && !orthonormal(R)) return fail(c, NMS_E_ARG, "nms_set_sample: R is not orthonormal within 1e-6");
    if (nms_status st = ensure(c, c->raw_pos, sizeof(float) * 3 * (size_t)W)) return st;
    NMS_CUDA(c, cudaMemcpyAsync(c->raw_pos.p, pos, sizeof(float) * 3 * (size_t)W, cudaMemcpyDefault, c->stream));
    if (N) {
        if (nms_status st = ensure(c, c->raw_N, sizeof(float) * (size_t)W)) return st;
        NMS_CUDA(c, cudaMemcpyAsync(c->raw_N.p, N, sizeof(float) * (size_t)W, cudaMemcpyDefault, c->stream));
    }
    if (m) {
        if (nms_status st = ensure(c, c->raw_m, sizeof(float) * 3 * (size_t)W)) return st;
        NMS_CUDA(c, cudaMemcpyAsync(c->raw_m.p, m, sizeof(float) * 3 * (size_t)W, cudaMemcpyDefault, c->stream));
    }
    c->W = W; c->has_N = N != nullptr; c->has_M = m != nullptr;
    c->K = 0; c->offsets.clear(); c->has_centres = false;
    static const double I3[9] = {1, 0, 0, 0, 1, 0, 0, 0, 1};
    memcpy(c->R, R ? R : I3, sizeof(c->R));
    if (nms_status st = build_tiles(c)) return st;
    return repack(c);
}

nms_status set_grid(nms_ctx* c, const nms_qgrid* g)
{
    if (!g) return fail(c, NMS_E_ARG, "grid is NULL");
    if (g->type < 0 || g->type > 2) return fail(c, NMS_E_ARG, "grid type %d unknown", g->type);
    if (g->n0 <= 0 || g->n1 <= 0 || !g->u0 || !g->u1) return fail(c, NMS_E_ARG, "grid sizes must be positive and abscissae non-NULL");
    if (g->type == 2 && g->n1 != 1) return fail(c, NMS_E_ARG, "list grid needs n1 == 1");
    const int len1 = g->type == 2 ? g->n0 : g->n1;
    const bool same = c->grid_valid && c->g_type == g->type && c->g_n0 == g->n0 && c->g_n1 == g->n1 &&
                      memcmp(c->h_u0.data(), g->u0, sizeof(float) * g->n0) == 0 &&
                      memcmp(c->h_u1.data(), g->u1, sizeof(float) * len1) == 0;
    if (same) return NMS_OK;
    for (int i = 0; i < g->n0; ++i) if (!isfinite(g->u0[i])) return fail(c, NMS_E_ARG, "grid abscissa u0[%d] is not finite", i);
    for (int i = 0; i < len1; ++i) if (!isfinite(g->u1[i])) return fail(c, NMS_E_ARG, "grid abscissa u1[%d] is not finite", i);
    c->grid_valid = false; c->amp_valid = false;
    c->g_type = g->type; c->g_n0 = g->n0; c->g_n1 = g->n1; c->n_q = (int64_t)g->n0 * g->n1;
    c->h_u0.assign(g->u0, g->u0 + g->n0);
    c->h_u1.assign(g->u1, g->u1 + len1);
    // equally spaced along the thread line (u0)?  (decides whether the recurrence kernels may be used: every
    // abscissa must lie within one fp32 ulp of the largest one from the progression u0[0] + i d)
    bool uni = g->type != 2 && g->n0 >= 2;
    double dq = 0.0, devq = 0.0;
    {
        double m0 = 0.0, m1 = 0.0;
        for (int i = 0; i < g->n0; ++i) m0 = fmax(m0, fabs((double)g->u0[i]));
        for (int i = 0; i < len1; ++i) m1 = fmax(m1, fabs((double)g->u1[i]));
        c->g_qmax = g->type == 0 ? m0 : sqrt(m0 * m0 + m1 * m1);
    }
    if (uni) {
        const double a0 = g->u0[0];
        dq = ((double)g->u0[g->n0 - 1] - a0) / (double)(g->n0 - 1);
        double amax = 0.0, dev = 0.0;
        for (int i = 0; i < g->n0; ++i) {
            amax = fmax(amax, fabs((double)g->u0[i]));
            dev = fmax(dev, fabs((double)g->u0[i] - (a0 + dq * i)));
        }
        uni = dq != 0.0 && dev <= 1.2e-7 * amax;
        devq = dev;
    }
    c->g_dq = dq;
    c->g_dev = devq;
    c->g_uniform = uni;
    if (nms_status st = ensure(c, c->u0, sizeof(float) * (size_t)g->n0)) return st;
    if (nms_status st = ensure(c, c->u1, sizeof(float) * (size_t)len1)) return st;
    if (nms_status st = ensure(c, c->qc, sizeof(double2) * (size_t)c->n_q)) return st;
    if (nms_status st = ensure(c, c->sc, sizeof(double2) * (size_t)c->n_q)) return st;
    NMS_CUDA(c, cudaMemcpyAsync(c->u0.p, c->h_u0.data(), sizeof(float) * (size_t)g->n0, cudaMemcpyHostToDevice, c->stream));
    NMS_CUDA(c, cudaMemcpyAsync(c->u1.p, c->h_u1.data(), sizeof(float) * (size_t)len1, cudaMemcpyHostToDevice, c->stream));
    if (nms_status st = launch_qsetup(c)) return st;
    c->grid_valid = true;
    return NMS_OK;
}

static nms_status upload_kinds(nms_ctx* c, const nms_kind* kinds, int n_kinds, const int32_t** dev)
{
    if (n_kinds < 0 || n_kinds > 4 * NMS_KIND_COUNT) return fail(c, NMS_E_ARG, "n_kinds = %d out of range", n_kinds);
    if (n_kinds > 0 && !kinds) return fail(c, NMS_E_ARG, "kinds is NULL");
    int32_t tmp[4 * NMS_KIND_COUNT + 1];
    for (int i = 0; i < n_kinds; ++i) {
        if ((int)kinds[i] < 0 || (int)kinds[i] >= NMS_KIND_COUNT) return fail(c, NMS_E_ARG, "unknown response kind %d", (int)kinds[i]);
        tmp[i] = (int32_t)kinds[i];
    }
    if (nms_status st = ensure(c, c->kinds_dev, sizeof(tmp))) return st;
    // the copy below reads a stack buffer: pageable H2D copies are staged before the call returns
    NMS_CUDA(c, cudaMemcpyAsync(c->kinds_dev.p, tmp, sizeof(int32_t) * (size_t)(n_kinds > 0 ? n_kinds : 1), cudaMemcpyHostToDevice, c->stream));
    *dev = (const int32_t*)c->kinds_dev.p;
    return NMS_OK;
}

}  // namespace nms

using namespace nms;

#define CHECK_CTX(c) do { if (!(c)) return NMS_E_ARG; (c)->err[0] = 0; cudaSetDevice((c)->device); } while (0)

extern "C" {

nms_status nms_create(nms_ctx** out, int device, void* cuda_stream)
{
    if (!out) return NMS_E_ARG;
    *out = nullptr;
    int n = 0;
    if (cudaGetDeviceCount(&n) != cudaSuccess || n <= 0 || device < 0 || device >= n) { cudaGetLastError(); return NMS_E_CUDA; }
    cudaDeviceProp pr;
    if (cudaGetDeviceProperties(&pr, device) != cudaSuccess) { cudaGetLastError(); return NMS_E_CUDA; }
    if (pr.major != 10) return NMS_E_CUDA;   // built for sm_100a only
    if (cudaSetDevice(device) != cudaSuccess) { cudaGetLastError(); return NMS_E_CUDA; }
    nms_ctx* c = new (std::nothrow) nms_ctx();
    if (!c) return NMS_E_NOMEM;
    c->device = device;
    c->stream = (cudaStream_t)cuda_stream;
    c->sm_count = pr.multiProcessorCount;
    if (cudaMallocHost((void**)&c->h_geo, 3 * sizeof(double)) != cudaSuccess ||
        cudaEventCreateWithFlags(&c->geo_event, cudaEventDisableTiming) != cudaSuccess) {
        cudaGetLastError();
        if (c->h_geo) cudaFreeHost(c->h_geo);
        delete c;
        return NMS_E_NOMEM;
    }
    c->h_geo[0] = c->h_geo[1] = c->h_geo[2] = 0.0;
    *out = c;
    return NMS_OK;
}

void nms_destroy(nms_ctx* c)
{
    if (!c) return;
    cudaSetDevice(c->device);
    cudaStreamSynchronize(c->stream);
    DevBuf* bufs[] = {&c->raw_pos, &c->raw_N, &c->raw_m, &c->centres, &c->tile_src, &c->tile_meta, &c->cells,
                      &c->wsum, &c->u0, &c->u1, &c->qc, &c->sc, &c->amp64, &c->part, &c->formpart,
                      &c->chunk_begin, &c->kinds_dev, &c->bin_idx, &c->bin_sum, &c->bin_cnt, &c->modal_tab, &c->modal_ring,
                      &c->tile_wsum, &c->interp_sb, &c->interp_spb, &c->qc_half, &c->sc_half, &c->diag, &c->batch_cells, &c->batch_ampN, &c->pix_cells, &c->pix_meta, &c->pix_u0, &c->pix_u1, &c->pix_qc, &c->pix_sc};
    for (DevBuf* b : bufs) free_buf(*b);
    for (DevBuf& b : c->host_stage) free_buf(b);
    if (c->h_geo) cudaFreeHost(c->h_geo);
    if (c->geo_event) cudaEventDestroy(c->geo_event);
    for (Timer& t : c->timers) {
        for (cudaEvent_t e : t.beg) cudaEventDestroy(e);
        for (cudaEvent_t e : t.end) cudaEventDestroy(e);
    }
    delete c;
}

const char* nms_last_error(const nms_ctx* c) { return c ? c->err : "NULL context"; }

nms_status nms_synchronize(nms_ctx* c)
{
    CHECK_CTX(c);
    NMS_CUDA(c, cudaStreamSynchronize(c->stream));
    return NMS_OK;
}

nms_status nms_set_sample(nms_ctx* c, const float* pos, const float* N, const float* m, int64_t W, const double* R)
{
    CHECK_CTX(c);
    return set_sample_impl(c, pos, N, m, W, R);
}

nms_status nms_set_particles(nms_ctx* c, const int64_t* offsets, int64_t K, const float* centres)
{
    CHECK_CTX(c);
    if (c->W <= 0) return fail(c, NMS_E_STATE, "nms_set_particles before nms_set_sample");
    if (K < 0) return fail(c, NMS_E_ARG, "K = %lld is negative", (long long)K);
    if (K == 0) {
        c->K = 0; c->offsets.clear(); c->has_centres = false;
    } else {
        if (!offsets) return fail(c, NMS_E_ARG, "offsets is NULL");
        if (offsets[0] != 0 || offsets[K] != c->W) return fail(c, NMS_E_ARG, "offsets[0] must be 0 and offsets[K] must equal W");
        for (int64_t k = 0; k < K; ++k)
            if (offsets[k + 1] < offsets[k]) return fail(c, NMS_E_ARG, "offsets decrease at object %lld", (long long)k);
        if (centres) {
            if (nms_status st = ensure(c, c->centres, sizeof(float) * 3 * (size_t)K)) return st;
            NMS_CUDA(c, cudaMemcpyAsync(c->centres.p, centres, sizeof(float) * 3 * (size_t)K, cudaMemcpyDefault, c->stream));
        }
        c->K = K; c->offsets.assign(offsets, offsets + K + 1); c->has_centres = centres != nullptr;
    }
    if (nms_status st = build_tiles(c)) return st;
    return repack(c);
}

nms_status nms_set_rotation(nms_ctx* c, const double* R)
{
    CHECK_CTX(c);
    if (c->W <= 0) return fail(c, NMS_E_STATE, "nms_set_rotation before nms_set_sample");
    static const double I3[9] = {1, 0, 0, 0, 1, 0, 0, 0, 1};
    if (R && !orthonormal(R)) return fail(c, NMS_E_ARG, "nms_set_rotation: R is not orthonormal within 1e-6");
    memcpy(c->R, R ? R : I3, sizeof(c->R));
    return repack(c);
}

nms_status nms_set_polarization(nms_ctx* c, const double* P)
{
    CHECK_CTX(c);
    if (!P) return fail(c, NMS_E_ARG, "P is NULL");
    const double n = sqrt(P[0] * P[0] + P[1] * P[1] + P[2] * P[2]);
    if (!(n > 0.0) || !isfinite(n)) return fail(c, NMS_E_ARG, "P must be a non-zero finite vector");
    for (int i = 0; i < 3; ++i) c->P[i] = P[i] / n;
    return NMS_OK;
}

nms_status nms_set_scales(nms_ctx* c, double sN, double sM, double invV)
{
    CHECK_CTX(c);
    if (!isfinite(sN) || !isfinite(sM) || !isfinite(invV)) return fail(c, NMS_E_ARG, "scales must be finite");
    c->sN = sN; c->sM = sM; c->invV = invV;
    return NMS_OK;
}

// Friedel halving (f-4; Eq. 42-43 L353-L356 with real weights: A(-q) = A(q)^*; L183: the theta grid closes under
// theta -> theta + pi): the rings' second halves are the point reflections of the first.  Admitted on a polar grid with an
// even number of angles whose float values satisfy theta[j + n1/2] = theta[j] + pi within one ulp of 2 pi; the second half
// then carries the direction of its float angle rotated by that deviation (<= 2.4e-7 rad).
static bool friedel_admissible(const nms_ctx* c)
{
    if (c->g_type != 0 || c->g_n1 < 2 || (c->g_n1 & 1)) return false;
    const int hn = c->g_n1 / 2;
    for (int j = 0; j < hn; ++j)
        if (fabs((double)c->h_u1[j + hn] - (double)c->h_u1[j] - 3.14159265358979323846) > 4.8e-7) return false;
    return true;
}

__global__ void k_half_rings(const double2* __restrict__ qc, const double2* __restrict__ sc, int n0, int n1,
                             double2* __restrict__ qc_h, double2* __restrict__ sc_h)
{
    const int hn = n1 / 2;
    const int64_t f = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (f >= (int64_t)n0 * hn) return;
    const int64_t src = (f / hn) * n1 + (f % hn);
    qc_h[f] = qc[src];
    sc_h[f] = sc[src];
}

// The signed difference kinds NM = (PP - MM)/2 and CHI = (PM - MP)/2 cross zero; the north-star criterion (1e-3 relative
// above 1e-6 of the map's own maximum) then asks the amplitudes for ~5e-10 sum|w|: they get the
// accurate variant of the fp32 kernels unless the caller says otherwise.
static bool wants_signed(const nms_kind* kinds, int n_kinds)
{
    for (int i = 0; i < n_kinds; ++i)
        if (kinds[i] == NMS_NM || kinds[i] == NMS_CHI) return true;
    return false;
}

static nms_status amplitudes_common(nms_ctx* c, const nms_qgrid* grid, bool split, bool want_accurate, const int32_t* kinds_dev,
                                    int n_kinds, int* n_chunks)
{
    if (!c->packed_valid) return fail(c, NMS_E_STATE, "no sample: call nms_set_sample first");
    if (nms_status st = set_grid(c, grid)) return st;
    c->friedel_active = false;
    if (c->opt_friedel) {
        if (split) return fail(c, NMS_E_UNSUPPORTED, "Friedel halving does not cover the form-factor split");
        if (!friedel_admissible(c))
            return fail(c, NMS_E_UNSUPPORTED, "Friedel halving needs a polar grid with an even number of angles closed under theta -> theta + pi");
    }
    AmpPlan plan;
    if (!c->opt_friedel) {
        if (nms_status st = plan_amplitude(c, split, want_accurate, &plan)) return st;
        if (nms_status st = launch_amplitude(c, plan, kinds_dev, n_kinds)) return st;
    } else {
        // run the amplitude kernels on the first half of every ring: the context describes the half grid for the launch
        const int n1 = c->g_n1, hn = n1 / 2;
        const int64_t nq = c->n_q;
        if (nms_status st = ensure(c, c->qc_half, sizeof(double2) * (size_t)c->g_n0 * hn)) return st;
        if (nms_status st = ensure(c, c->sc_half, sizeof(double2) * (size_t)c->g_n0 * hn)) return st;
        k_half_rings<<<(unsigned)(((int64_t)c->g_n0 * hn + 255) / 256), 256, 0, c->stream>>>(
            (const double2*)c->qc.p, (const double2*)c->sc.p, c->g_n0, n1, (double2*)c->qc_half.p, (double2*)c->sc_half.p);
        c->launches += 1;
        std::swap(c->qc, c->qc_half); std::swap(c->sc, c->sc_half);
        c->g_n1 = hn; c->n_q = (int64_t)c->g_n0 * hn;
        nms_status st = plan_amplitude(c, false, want_accurate, &plan);
        if (!st) st = launch_amplitude(c, plan, kinds_dev, n_kinds);
        std::swap(c->qc, c->qc_half); std::swap(c->sc, c->sc_half);
        c->g_n1 = n1; c->n_q = nq;
        if (st) return st;
        c->friedel_active = true;
    }
    *n_chunks = c->n_chunks_used;
    return NMS_OK;
}

nms_status nms_amplitudes(nms_ctx* c, const nms_qgrid* grid, float* out_amp)
{
    CHECK_CTX(c);
    int n_chunks = 0;
    c->amp_valid = false;
    if (nms_status st = amplitudes_common(c, grid, false, true, nullptr, 0, &n_chunks)) return st;
    if (nms_status st = launch_epilogue(c, n_chunks, nullptr, 0, nullptr, out_amp, true)) return st;
    c->amp_valid = true;
    return NMS_OK;
}

nms_status nms_response(nms_ctx* c, const nms_kind* kinds, int n_kinds, float* out)
{
    CHECK_CTX(c);
    if (!c->amp_valid) return fail(c, NMS_E_STATE, "nms_response needs a preceding nms_amplitudes on the current sample");
    if (n_kinds <= 0 || !out) return fail(c, NMS_E_ARG, "n_kinds must be positive and out non-NULL");
    const int32_t* kd = nullptr;
    if (nms_status st = upload_kinds(c, kinds, n_kinds, &kd)) return st;
    return launch_response_from_amp(c, kd, n_kinds, out);
}

nms_status nms_cross_spectra(nms_ctx* c, float* out_GR, float* out_GI)
{
    CHECK_CTX(c);
    if (!c->amp_valid) return fail(c, NMS_E_STATE, "nms_cross_spectra needs a preceding nms_amplitudes on the current sample");
    if (!out_GR && !out_GI) return fail(c, NMS_E_ARG, "no output requested");
    return launch_cross_spectra(c, out_GR, out_GI);
}

nms_status nms_compute(nms_ctx* c, const nms_qgrid* grid, const nms_kind* kinds, int n_kinds, float* out)
{
    CHECK_CTX(c);
    if (n_kinds <= 0 || !out) return fail(c, NMS_E_ARG, "n_kinds must be positive and out non-NULL");
    const int32_t* kd = nullptr;
    if (nms_status st = upload_kinds(c, kinds, n_kinds, &kd)) return st;
    int n_chunks = 0;
    c->amp_valid = false;
    if (nms_status st = amplitudes_common(c, grid, false, wants_signed(kinds, n_kinds), kd, n_kinds, &n_chunks)) return st;
    return launch_epilogue(c, n_chunks, kd, n_kinds, out, nullptr, false);
}

nms_status nms_compute_batch(nms_ctx* c, const nms_qgrid* grid, const float* m_batch, int n_fields, const nms_kind* kinds,
                             int n_kinds, float* out_maps, float* out_amp)
{
    CHECK_CTX(c);
    if (!c->packed_valid) return fail(c, NMS_E_STATE, "no sample: call nms_set_sample first (its positions, N, particles and rotation are the fixed geometry)");
    if (!m_batch || n_fields <= 0) return fail(c, NMS_E_ARG, "m_batch NULL or n_fields <= 0");
    if (!out_maps && !out_amp) return fail(c, NMS_E_ARG, "no output requested");
    if (out_maps && n_kinds <= 0) return fail(c, NMS_E_ARG, "out_maps needs n_kinds > 0");
    const int32_t* kd = nullptr;
    if (nms_status st = upload_kinds(c, kinds, out_maps ? n_kinds : 0, &kd)) return st;
    if (nms_status st = set_grid(c, grid)) return st;
    c->amp_valid = false;
    const bool accurate = c->opt_precision == 2 || (c->opt_precision == 0 && (out_amp != nullptr || wants_signed(kinds, out_maps ? n_kinds : 0)));
    return launch_batch(c, m_batch, n_fields, kd, n_kinds, out_maps, out_amp, accurate);
}

nms_status nms_form_factor_split(nms_ctx* c, const nms_qgrid* grid, const nms_kind* kinds, int n_kinds, float* out_total,
                                 float* out_form)
{
    CHECK_CTX(c);
    if (c->K <= 0) return fail(c, NMS_E_STATE, "nms_form_factor_split needs nms_set_particles");
    if (n_kinds <= 0 || (!out_total && !out_form)) return fail(c, NMS_E_ARG, "n_kinds must be positive and an output non-NULL");
    const int32_t* kd = nullptr;
    if (nms_status st = upload_kinds(c, kinds, n_kinds, &kd)) return st;
    int n_chunks = 0;
    c->amp_valid = false;
    if (nms_status st = amplitudes_common(c, grid, true, wants_signed(kinds, n_kinds), kd, n_kinds, &n_chunks)) return st;
    return launch_split_epilogue(c, n_chunks, kd, n_kinds, out_total, out_form);
}

nms_status nms_azimuthal_average(nms_ctx* c, const float* maps, int n_maps, int n_bins, double q_lo, double q_hi,
                                 float* out_I, float* out_q, int32_t* out_count)
{
    CHECK_CTX(c);
    if (!c->grid_valid) return fail(c, NMS_E_STATE, "nms_azimuthal_average needs a current grid (nms_amplitudes / nms_compute)");
    if (!maps || !out_I || n_maps <= 0 || n_bins <= 0) return fail(c, NMS_E_ARG, "maps/out_I NULL or non-positive sizes");
    if (!(q_hi > q_lo)) {
        if (c->g_type != 0) return fail(c, NMS_E_ARG, "q_hi <= q_lo (ring mode) needs a polar grid");
        if (n_bins != c->g_n0) return fail(c, NMS_E_ARG, "ring mode needs n_bins == n0 (%d)", c->g_n0);
    }
    return launch_azimuthal(c, maps, n_maps, n_bins, q_lo, q_hi, out_I, out_q, out_count);
}

nms_status nms_modal_decomposition(nms_ctx* c, const float* maps, int n_maps, int k_max, float* out_Is, float* out_Ic,
                                   float* out_a, float* out_A)
{
    CHECK_CTX(c);
    if (!c->grid_valid) return fail(c, NMS_E_STATE, "nms_modal_decomposition needs a current grid (nms_amplitudes / nms_compute)");
    if (c->g_type != 0) return fail(c, NMS_E_UNSUPPORTED, "nms_modal_decomposition needs a polar grid");
    if (!maps || n_maps <= 0) return fail(c, NMS_E_ARG, "maps NULL or n_maps <= 0");
    if (k_max < 0 || k_max > 63) return fail(c, NMS_E_ARG, "k_max = %d outside 0..63", k_max);
    if (!out_Is && !out_Ic && !out_a && !out_A) return fail(c, NMS_E_ARG, "no output requested");
    return launch_modal(c, maps, n_maps, k_max, out_Is, out_Ic, out_a, out_A);
}

nms_status nms_correlation_2d(nms_ctx* c, const float* map, const nms_qgrid* rgrid, float* out_re, float* out_im)
{
    CHECK_CTX(c);
    if (!c->grid_valid) return fail(c, NMS_E_STATE, "nms_correlation_2d needs a current grid (nms_amplitudes / nms_compute)");
    if (c->g_type != 0) return fail(c, NMS_E_UNSUPPORTED, "nms_correlation_2d needs a polar detector grid");
    if (!map || !rgrid || (!out_re && !out_im)) return fail(c, NMS_E_ARG, "NULL argument");
    if (rgrid->type != 0 || rgrid->n0 <= 0 || rgrid->n1 <= 0 || !rgrid->u0 || !rgrid->u1)
        return fail(c, NMS_E_ARG, "the (rho, alpha) grid must be polar with positive sizes");
    return launch_correlation_2d(c, map, rgrid, out_re, out_im);
}

nms_status nms_correlation(nms_ctx* c, const float* I, const float* q_of_bin, const int32_t* count, int n_maps, int n_bins,
                           const float* r, int n_r, float* out_c, float* out_p)
{
    CHECK_CTX(c);
    if (!I || !q_of_bin || !r || !out_c || !out_p) return fail(c, NMS_E_ARG, "NULL argument");
    if (n_maps <= 0 || n_bins <= 0 || n_r <= 0) return fail(c, NMS_E_ARG, "non-positive size");
    if (n_bins > 12000) return fail(c, NMS_E_UNSUPPORTED, "n_bins = %d exceeds 12000", n_bins);
    return launch_correlation(c, I, q_of_bin, count, n_maps, n_bins, r, n_r, out_c, out_p);
}

nms_status nms_run_host(nms_ctx* c, const float* pos, const float* N, const float* m, int64_t W, const double* R,
                        const nms_qgrid* grid, const nms_kind* kinds, int n_kinds, float* out_maps, int n_bins, double q_lo,
                        double q_hi, float* out_I, const float* r, int n_r, float* out_c, float* out_p)
{
    CHECK_CTX(c);
    if (!grid || n_kinds <= 0) return fail(c, NMS_E_ARG, "grid NULL or n_kinds <= 0");
    if (n_bins > 0 && !out_I) return fail(c, NMS_E_ARG, "n_bins > 0 needs out_I");
    if (n_r > 0 && (n_bins <= 0 || !r || !out_c || !out_p)) return fail(c, NMS_E_ARG, "n_r > 0 needs n_bins > 0, r, out_c, out_p");
    if (nms_status st = set_sample_impl(c, pos, N, m, W, R)) return st;
    const size_t nq = (size_t)grid->n0 * grid->n1;
    DevBuf& d_maps = c->host_stage[0]; DevBuf& d_I = c->host_stage[1]; DevBuf& d_q = c->host_stage[2];
    DevBuf& d_cnt = c->host_stage[3]; DevBuf& d_r = c->host_stage[4]; DevBuf& d_c = c->host_stage[5]; DevBuf& d_p = c->host_stage[6];
    if (nms_status st = ensure(c, d_maps, sizeof(float) * nq * n_kinds)) return st;
    if (nms_status st = nms_compute(c, grid, kinds, n_kinds, (float*)d_maps.p)) return st;
    if (out_maps) NMS_CUDA(c, cudaMemcpyAsync(out_maps, d_maps.p, sizeof(float) * nq * n_kinds, cudaMemcpyDeviceToHost, c->stream));
    if (n_bins > 0) {
        if (nms_status st = ensure(c, d_I, sizeof(float) * (size_t)n_bins * n_kinds)) return st;
        if (nms_status st = ensure(c, d_q, sizeof(float) * (size_t)n_bins)) return st;
        if (nms_status st = ensure(c, d_cnt, sizeof(int32_t) * (size_t)n_bins)) return st;
        if (nms_status st = nms_azimuthal_average(c, (const float*)d_maps.p, n_kinds, n_bins, q_lo, q_hi, (float*)d_I.p,
                                                  (float*)d_q.p, (int32_t*)d_cnt.p)) return st;
        NMS_CUDA(c, cudaMemcpyAsync(out_I, d_I.p, sizeof(float) * (size_t)n_bins * n_kinds, cudaMemcpyDeviceToHost, c->stream));
        if (n_r > 0) {
            if (nms_status st = ensure(c, d_r, sizeof(float) * (size_t)n_r)) return st;
            if (nms_status st = ensure(c, d_c, sizeof(float) * (size_t)n_r * n_kinds)) return st;
            if (nms_status st = ensure(c, d_p, sizeof(float) * (size_t)n_r * n_kinds)) return st;
            NMS_CUDA(c, cudaMemcpyAsync(d_r.p, r, sizeof(float) * (size_t)n_r, cudaMemcpyHostToDevice, c->stream));
            if (nms_status st = nms_correlation(c, (const float*)d_I.p, (const float*)d_q.p, (const int32_t*)d_cnt.p, n_kinds,
                                                n_bins, (const float*)d_r.p, n_r, (float*)d_c.p, (float*)d_p.p)) return st;
            NMS_CUDA(c, cudaMemcpyAsync(out_c, d_c.p, sizeof(float) * (size_t)n_r * n_kinds, cudaMemcpyDeviceToHost, c->stream));
            NMS_CUDA(c, cudaMemcpyAsync(out_p, d_p.p, sizeof(float) * (size_t)n_r * n_kinds, cudaMemcpyDeviceToHost, c->stream));
        }
    }
    NMS_CUDA(c, cudaStreamSynchronize(c->stream));
    return NMS_OK;
}

nms_status nms_run_host_split(nms_ctx* c, const float* pos, const float* N, const float* m, int64_t W, const int64_t* offsets,
                              int64_t K, const float* centres, const double* R, const nms_qgrid* grid, const nms_kind* kinds,
                              int n_kinds, float* out_total, float* out_form)
{
    CHECK_CTX(c);
    if (!grid || n_kinds <= 0 || (!out_total && !out_form)) return fail(c, NMS_E_ARG, "grid NULL, n_kinds <= 0 or no output");
    if (nms_status st = set_sample_impl(c, pos, N, m, W, R)) return st;
    if (nms_status st = nms_set_particles(c, offsets, K, centres)) return st;
    const size_t bytes = sizeof(float) * (size_t)grid->n0 * grid->n1 * n_kinds;
    DevBuf& d_tot = c->host_stage[0]; DevBuf& d_form = c->host_stage[7];
    if (nms_status st = ensure(c, d_tot, bytes)) return st;
    if (nms_status st = ensure(c, d_form, bytes)) return st;
    if (nms_status st = nms_form_factor_split(c, grid, kinds, n_kinds, (float*)d_tot.p, (float*)d_form.p)) return st;
    if (out_total) NMS_CUDA(c, cudaMemcpyAsync(out_total, d_tot.p, bytes, cudaMemcpyDeviceToHost, c->stream));
    if (out_form) NMS_CUDA(c, cudaMemcpyAsync(out_form, d_form.p, bytes, cudaMemcpyDeviceToHost, c->stream));
    NMS_CUDA(c, cudaStreamSynchronize(c->stream));
    return NMS_OK;
}

nms_status nms_run_host_scan(nms_ctx* c, const float* pos, const float* N, const float* m, int64_t W, const double* R,
                             int n_rot, const nms_qgrid* grid, const nms_kind* kinds, int n_kinds, float* out_maps)
{
    CHECK_CTX(c);
    if (!grid || n_kinds <= 0 || n_rot <= 0 || !R || !out_maps) return fail(c, NMS_E_ARG, "NULL argument or non-positive count");
    const size_t count = (size_t)grid->n0 * grid->n1 * n_kinds;
    DevBuf& d_maps = c->host_stage[0];
    if (nms_status st = ensure(c, d_maps, sizeof(float) * count * 2)) return st;      // two buffers: copy out while the next rotation runs
    for (int i = 0; i < n_rot; ++i) {
        if (nms_status st = (i == 0 ? set_sample_impl(c, pos, N, m, W, R) : nms_set_rotation(c, R + 9 * (size_t)i))) return st;
        float* dst = (float*)d_maps.p + (size_t)(i & 1) * count;
        if (nms_status st = nms_compute(c, grid, kinds, n_kinds, dst)) return st;
        NMS_CUDA(c, cudaMemcpyAsync(out_maps + (size_t)i * count, dst, sizeof(float) * count, cudaMemcpyDeviceToHost, c->stream));
    }
    NMS_CUDA(c, cudaStreamSynchronize(c->stream));
    return NMS_OK;
}

nms_status nms_get_weight_sums(nms_ctx* c, double* out)
{
    CHECK_CTX(c);
    if (!out) return fail(c, NMS_E_ARG, "out is NULL");
    if (!c->packed_valid) return fail(c, NMS_E_STATE, "no sample");
    NMS_CUDA(c, cudaMemcpyAsync(out, c->wsum.p, 4 * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    NMS_CUDA(c, cudaStreamSynchronize(c->stream));
    return NMS_OK;
}

nms_status nms_set_option(nms_ctx* c, const char* key, int64_t value)
{
    CHECK_CTX(c);
    if (!key) return fail(c, NMS_E_ARG, "key is NULL");
    if (!strcmp(key, "variant")) { if (value < 0 || value > 3) return fail(c, NMS_E_ARG, "variant must be 0, 1, 2 or 3"); c->opt_variant = (int)value; }
    else if (!strcmp(key, "timing")) { c->opt_timing = value != 0; for (Timer& t : c->timers) t.used = 0; }
    else if (!strcmp(key, "chunks")) { if (value < 0) return fail(c, NMS_E_ARG, "chunks must be >= 0"); c->opt_chunks = (int)value; }
    else if (!strcmp(key, "bases")) { if (value < 0 || value > 4) return fail(c, NMS_E_ARG, "bases must be 0..4"); c->opt_bases = (int)value; }
    else if (!strcmp(key, "precision")) { if (value < 0 || value > 2) return fail(c, NMS_E_ARG, "precision must be 0, 1 or 2"); c->opt_precision = (int)value; }
    else if (!strcmp(key, "friedel")) { if (value < 0 || value > 1) return fail(c, NMS_E_ARG, "friedel must be 0 or 1"); c->opt_friedel = (int)value; }
    else if (!strcmp(key, "uniform")) { c->opt_uniform = (int)value; }
    else if (!strcmp(key, "recurrence")) { if (value < 0 || value > 2) return fail(c, NMS_E_ARG, "recurrence must be 0, 1 or 2"); c->opt_rec3 = (int)value; }
    else if (!strcmp(key, "interp")) { if (value < 0 || value > 2) return fail(c, NMS_E_ARG, "interp must be 0, 1 or 2"); c->opt_interp = (int)value; }
    else if (!strcmp(key, "qt")) { if (value != 0 && value != 4 && value != 8 && value != 16) return fail(c, NMS_E_ARG, "qt must be 0, 4, 8 or 16"); c->opt_qt = (int)value; }
    else return fail(c, NMS_E_ARG, "unknown option '%s'", key);
    return NMS_OK;
}

nms_status nms_get_info(nms_ctx* c, const char* key, int64_t* value)
{
    CHECK_CTX(c);
    if (!key || !value) return fail(c, NMS_E_ARG, "NULL argument");
    if (!strcmp(key, "launches")) *value = c->launches;
    else if (!strcmp(key, "variant_used")) *value = c->variant_used;
    else if (!strcmp(key, "n_chunks")) *value = c->n_chunks_used;
    else if (!strcmp(key, "n_tiles")) *value = c->n_tiles;
    else if (!strcmp(key, "n_slots")) *value = c->n_slots;
    else if (!strcmp(key, "sm_count")) *value = c->sm_count;
    else if (!strcmp(key, "blocks_per_sm")) *value = c->blocks_per_sm_used;
    else if (!strcmp(key, "qt")) *value = c->qt_used;
    else if (!strcmp(key, "poly_phasors")) *value = c->npoly_used;
    else if (!strcmp(key, "bases")) *value = c->nb_used;
    else if (!strcmp(key, "three_term")) *value = c->rec3_used;
    else if (!strcmp(key, "interp")) *value = c->interp_used;
    else if (!strcmp(key, "corr2d_variant")) *value = c->corr2d_variant;
    else return fail(c, NMS_E_ARG, "unknown info key '%s'", key);
    return NMS_OK;
}

nms_status nms_kernel_time_ms(nms_ctx* c, nms_timer which, float* ms)
{
    CHECK_CTX(c);
    if ((int)which < 0 || (int)which >= NMS_T_COUNT || !ms) return fail(c, NMS_E_ARG, "bad timer index or NULL");
    Timer& t = c->timers[which];
    if (t.used == 0) return fail(c, NMS_E_STATE, "that kernel has not run with timing enabled");
    NMS_CUDA(c, cudaEventSynchronize(t.end[t.used - 1]));
    NMS_CUDA(c, cudaEventElapsedTime(ms, t.beg[t.used - 1], t.end[t.used - 1]));
    return NMS_OK;
}

nms_status nms_kernel_time_total(nms_ctx* c, nms_timer which, double* total_ms, int64_t* count)
{
    CHECK_CTX(c);
    if ((int)which < 0 || (int)which >= NMS_T_COUNT || !total_ms || !count) return fail(c, NMS_E_ARG, "bad timer index or NULL");
    Timer& t = c->timers[which];
    double sum = 0.0;
    for (size_t i = 0; i < t.used; ++i) {
        float ms = 0.f;
        NMS_CUDA(c, cudaEventSynchronize(t.end[i]));
        NMS_CUDA(c, cudaEventElapsedTime(&ms, t.beg[i], t.end[i]));
        sum += (double)ms;
    }
    *total_ms = sum; *count = (int64_t)t.used;
    return NMS_OK;
}

}  // extern "C"
