// k_amplitude.cu -- a-2 (and a-6): the direct sums of Eq. 42-47 (L353-L368) on the FP32 + XU pipes.
//
//   A_c(q) = sum_j w_cj exp(-i Psi_j(q)),  Psi_j = q_y Y_j + q_z Z_j  (Eq. 41),  c in {N, x, y, z}.
//
// Work decomposition: grid = (detector blocks) x (cell chunks).  A block owns 128*QT detector points
// (thread = one position along the fast detector index i1 and QT consecutive positions along i0) and
// walks the tiles of its chunk.  Tiles (<= 1024 cells, 24 B each) are brought into shared memory by one
// elected thread with cp.async.bulk + mbarrier, double buffered; every lane of a warp reads the same
// cell (LDS broadcast, no bank conflicts) and updates 8 fp32 accumulators per detector point.
//
// Numerics: cells are stored relative to a tile origin r0, so the in-tile phase is small and its fp32
// rounding negligible; because the sum is linear,  sum_j w_j e^{-i q.(r0+d_j)} = e^{-i q.r0} sum_j w_j
// e^{-i q.d_j}:  at the end of a tile the thread rotates its 8 fp32 tile sums by the tile phasor
// (phase in fp64, reduced exactly to [-1/2,1/2] cycles) and adds them to fp64 chunk partials in global
// memory (block-private slots, plain read-modify-write, deterministic).  The epilogue kernel sums the
// chunks and forms the responses.
//
// Phasor variants (MODE):
//   1  general direct : t = q_y dY + q_z dZ per pair, sin/cos by MUFU                     (list grids)
//   2  polar direct   : p = s dY + c dZ per (cell,thread), t_k = q_k p, MUFU              (any |q| spacing)
//   4  cart. direct   : u = q_y dY per (cell,thread), t_k = u + q_z,k dZ, MUFU
//   3  line recurrence: the thread's QT points are equally spaced on a line q_k = b + k s; base and step
//                       phasors by MUFU once per (cell,thread), then a complex rotation per point
//                       (4 FP32 ops, no MUFU), resynchronised at every cell.
#include "nms_internal.h"
#include "nms_response.cuh"

namespace nms {

constexpr int AMP_THREADS = 128;

struct AmpArgs {
    const float4* A;
    const float2* B;
    const TileMeta* tiles;
    const int32_t* chunk_begin;   // [n_chunks+1] or NULL (equal parts of n_tiles)
    int n_tiles;
    int type, n0, n1;
    int64_t n_q;
    const float* u0;
    const double2* qc;   // (q_y, q_z) [rad/nm] fp64
    const double2* sc;   // (sin th, cos th)
    double* part;        // [n_chunks][8][n_q]
    double* ppart;       // split: [n_chunks][8][n_q] running amplitudes of the current object
    double* form;        // split: [n_chunks][n_kinds][n_q]
    const int32_t* kinds;
    int n_kinds;
    RespParams rp;
};

// ---- mbarrier / bulk-copy primitives (sm_90+ PTX) ----------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

__device__ __forceinline__ void issue_tile(const AmpArgs& a, int tile, float4* dA, float2* dB, uint64_t* bar)
{
    const TileMeta tm = a.tiles[tile];
    const uint32_t n = (uint32_t)tm.n_slots;
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    mbar_expect_tx(bar, n * 24u);
    bulk_g2s(dA, a.A + tm.first_slot, n * 16u, bar);
    bulk_g2s(dB, a.B + tm.first_slot, n * 8u, bar);
}

// 8 accumulate FFMAs of one (cell, detector point) pair: sums of w cos and w sin.
__device__ __forceinline__ void accumulate(float (&acc)[8], const float4& ca, const float2& cb, float c, float s)
{
    acc[0] = fmaf(ca.z, c, acc[0]); acc[1] = fmaf(ca.z, s, acc[1]);
    acc[2] = fmaf(ca.w, c, acc[2]); acc[3] = fmaf(ca.w, s, acc[3]);
    acc[4] = fmaf(cb.x, c, acc[4]); acc[5] = fmaf(cb.x, s, acc[5]);
    acc[6] = fmaf(cb.y, c, acc[6]); acc[7] = fmaf(cb.y, s, acc[7]);
}

template <int MODE, int QT, bool SPLIT, int UNR, int MINB>
__global__ void __launch_bounds__(AMP_THREADS, MINB) k_amp(const AmpArgs a)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float4* sA = reinterpret_cast<float4*>(smem_raw);                               // [2][TILE]
    float2* sB = reinterpret_cast<float2*>(smem_raw + 2 * TILE * sizeof(float4));    // [2][TILE]
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw + 2 * TILE * (sizeof(float4) + sizeof(float2)));

    const int tid = threadIdx.x;
    const int chunk = blockIdx.y;
    int tile_beg, tile_end;   // chunk boundaries: a table in split mode (object boundaries), else equal parts
    if (a.chunk_begin) { tile_beg = a.chunk_begin[chunk]; tile_end = a.chunk_begin[chunk + 1]; }
    else {
        tile_beg = (int)(((int64_t)a.n_tiles * chunk) / gridDim.y);
        tile_end = (int)(((int64_t)a.n_tiles * (chunk + 1)) / gridDim.y);
    }

    // ---- this thread's detector points ---------------------------------------------------------
    const int n_groups = (a.n0 + QT - 1) / QT;
    const int64_t n_slots_q = (int64_t)n_groups * a.n1;
    int64_t slot = (int64_t)blockIdx.x * AMP_THREADS + tid;
    const bool valid = slot < n_slots_q;
    if (!valid) slot = 0;
    const int grp = (int)(slot / a.n1), i1 = (int)(slot % a.n1);
    const int i0 = grp * QT;
    const int kmax = valid ? min(QT, a.n0 - i0) : 0;
    const int kclamp = max(min(QT, a.n0 - i0), 1);
    const int64_t flat0 = (int64_t)i0 * a.n1 + i1;

    float c0 = 0.f, c1 = 0.f, c2 = 0.f, c3 = 0.f;   // mode-dependent per-thread constants
    float g[QT], h[QT];                              // per-point constants (modes 1, 2, 4)
    if (MODE == 1) {
#pragma unroll
        for (int k = 0; k < QT; ++k) {
            const double2 q = a.qc[flat0 + (int64_t)min(k, kclamp - 1) * a.n1];
            g[k] = (float)q.x; h[k] = (float)q.y;
        }
    } else if (MODE == 2) {
        const double2 d = a.sc[flat0];
        c0 = (float)d.x; c1 = (float)d.y;
#pragma unroll
        for (int k = 0; k < QT; ++k) g[k] = a.u0[i0 + min(k, kclamp - 1)];
    } else if (MODE == 4) {
        c0 = (float)a.qc[flat0].x;
#pragma unroll
        for (int k = 0; k < QT; ++k) g[k] = a.u0[i0 + min(k, kclamp - 1)];
    } else {   // MODE 3
        const double2 qb = a.qc[flat0];
        const double2 qe = a.qc[flat0 + (int64_t)(kclamp - 1) * a.n1];
        const double inv = kclamp > 1 ? 1.0 / (double)(kclamp - 1) : 0.0;
        c0 = (float)qb.x; c1 = (float)qb.y;
        c2 = (float)((qe.x - qb.x) * inv); c3 = (float)((qe.y - qb.y) * inv);
    }
    (void)h;

    if (tid == 0) {
        mbar_init(&bar[0], 1);
        mbar_init(&bar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (tid == 0) {
        if (tile_beg < tile_end) issue_tile(a, tile_beg, sA, sB, &bar[0]);
        if (tile_beg + 1 < tile_end) issue_tile(a, tile_beg + 1, sA + TILE, sB + TILE, &bar[1]);
    }

    float acc[QT][8];
    bool first_total = true;   // SPLIT: no object of this chunk has been completed yet

    for (int t = tile_beg; t < tile_end; ++t) {
        const int it = t - tile_beg;
        const int stage = it & 1;
        const TileMeta tm = a.tiles[t];
        const float4* __restrict__ tA = sA + stage * TILE;
        const float2* __restrict__ tB = sB + stage * TILE;
#pragma unroll
        for (int k = 0; k < QT; ++k)
#pragma unroll
            for (int r = 0; r < 8; ++r) acc[k][r] = 0.f;
        mbar_wait(&bar[stage], (uint32_t)((it >> 1) & 1));

        const int n = tm.n_slots;
#pragma unroll UNR
        for (int j = 0; j < n; ++j) {
            const float4 ca = tA[j];
            const float2 cb = tB[j];
            if (MODE == 1) {
#pragma unroll
                for (int k = 0; k < QT; ++k) {
                    const float ph = fmaf(h[k], ca.y, g[k] * ca.x);
                    accumulate(acc[k], ca, cb, __cosf(ph), __sinf(ph));
                }
            } else if (MODE == 2) {
                const float p = fmaf(c1, ca.y, c0 * ca.x);
#pragma unroll
                for (int k = 0; k < QT; ++k) {
                    const float ph = g[k] * p;
                    accumulate(acc[k], ca, cb, __cosf(ph), __sinf(ph));
                }
            } else if (MODE == 4) {
                const float u = c0 * ca.x;
#pragma unroll
                for (int k = 0; k < QT; ++k) {
                    const float ph = fmaf(g[k], ca.y, u);
                    accumulate(acc[k], ca, cb, __cosf(ph), __sinf(ph));
                }
            } else {
                const float t0 = fmaf(c1, ca.y, c0 * ca.x);
                const float dt = fmaf(c3, ca.y, c2 * ca.x);
                float pc = __cosf(t0), ps = __sinf(t0);
                const float dc = __cosf(dt), ds = __sinf(dt);
#pragma unroll
                for (int k = 0; k < QT; ++k) {
                    accumulate(acc[k], ca, cb, pc, ps);
                    if (k < QT - 1) {
                        const float nc = fmaf(pc, dc, -(ps * ds));
                        const float ns = fmaf(ps, dc, pc * ds);
                        pc = nc; ps = ns;
                    }
                }
            }
        }

        __syncthreads();   // every thread is done with this stage: refill it while the flush runs
        if (tid == 0 && t + 2 < tile_end) issue_tile(a, t + 2, sA + stage * TILE, sB + stage * TILE, &bar[stage]);

        // ---- flush: rotate the tile sums by exp(-i q.r0) and add them to the fp64 chunk partials --
        const bool first = (t == tile_beg);
        const bool p_first = SPLIT ? ((tm.flags & 2) != 0) : false;
        const bool p_last = SPLIT ? ((tm.flags & 1) != 0) : false;
#pragma unroll
        for (int k = 0; k < QT; ++k) {
            if (k < kmax) {
                const int64_t f = flat0 + (int64_t)k * a.n1;
                const double2 q = a.qc[f];
                double ph = (q.x * tm.Y0 + q.y * tm.Z0) * 0.15915494309189533577;   // cycles
                ph -= rint(ph);
                const float rh = (float)ph;
                const float rl = (float)(ph - (double)rh);
                float s0f, c0f;
                sincospif(2.0f * rh, &s0f, &c0f);
                const double e = 6.283185307179586 * (double)rl;
                const double cd = (double)c0f - e * (double)s0f;
                const double sd = (double)s0f + e * (double)c0f;
                double Ap[8];
#pragma unroll
                for (int w = 0; w < 4; ++w) {
                    const double C = (double)acc[k][2 * w], S = (double)acc[k][2 * w + 1];
                    Ap[2 * w] = C * cd - S * sd;          // Re: + sum w cos(Psi)   (Eq. 44, 46)
                    Ap[2 * w + 1] = -(S * cd + C * sd);   // Im: - sum w sin(Psi)   (Eq. 45, 47)
                }
                if (!SPLIT) {
#pragma unroll
                    for (int r = 0; r < 8; ++r) {
                        double* dst = a.part + ((int64_t)chunk * 8 + r) * a.n_q + f;
                        *dst = first ? Ap[r] : (*dst + Ap[r]);
                    }
                } else {
#pragma unroll
                    for (int r = 0; r < 8; ++r) {
                        double* pp = a.ppart + ((int64_t)chunk * 8 + r) * a.n_q + f;
                        if (!p_first) Ap[r] += *pp;
                        if (!p_last) *pp = Ap[r];
                    }
                    if (p_last) {   // object complete: form += B(A_p, A_p), total amplitude += A_p  (Eq. 49-50)
                        const double2 d = a.sc[f];
                        double val[NMS_KIND_COUNT];
                        responses_at_point(Ap, d.x, d.y, a.rp, val);
                        for (int i = 0; i < a.n_kinds; ++i) {
                            double* dst = a.form + ((int64_t)chunk * a.n_kinds + i) * a.n_q + f;
                            const double v = val[a.kinds[i]];
                            *dst = first_total ? v : (*dst + v);
                        }
#pragma unroll
                        for (int r = 0; r < 8; ++r) {
                            double* dst = a.part + ((int64_t)chunk * 8 + r) * a.n_q + f;
                            *dst = first_total ? Ap[r] : (*dst + Ap[r]);
                        }
                    }
                }
            }
        }
        if (SPLIT && p_last) first_total = false;
    }
}

// ---- host side: planning and dispatch ------------------------------------------------------------
constexpr size_t AMP_SMEM = 2 * TILE * (sizeof(float4) + sizeof(float2)) + 2 * sizeof(uint64_t);

typedef void (*amp_kernel_t)(const AmpArgs);

template <int MODE, int QT, int UNR, int MINB>
static amp_kernel_t pick_split(bool split)
{
    return split ? (amp_kernel_t)k_amp<MODE, QT, true, UNR, MINB> : (amp_kernel_t)k_amp<MODE, QT, false, UNR, MINB>;
}

static amp_kernel_t pick_kernel(int variant, int qt, bool split)
{
    switch (variant) {
    case 1: return pick_split<1, 4, 2, 4>(split);
    case 2:
        if (qt == 4) return pick_split<2, 4, 2, 4>(split);
        return pick_split<2, 8, 2, 4>(split);
    case 4:
        if (qt == 4) return pick_split<4, 4, 2, 4>(split);
        return pick_split<4, 8, 2, 4>(split);
    default:
        if (qt == 4) return pick_split<3, 4, 2, 4>(split);
        if (qt == 8) return pick_split<3, 8, 2, 4>(split);
        return pick_split<3, 16, 1, 2>(split);
    }
}

static int64_t ceil_div(int64_t a, int64_t b) { return (a + b - 1) / b; }

nms_status plan_amplitude(nms_ctx* c, bool split, AmpPlan* plan)
{
    // variant: list grids are general; equally spaced lines allow the recurrence; otherwise line-direct
    int variant;
    if (c->g_type == 2) variant = 1;
    else if (c->g_uniform && c->opt_variant != 1) variant = 3;
    else variant = (c->g_type == 0) ? 2 : 4;
    if (c->opt_variant == 2 && variant != 3 && c->g_type != 2)
        return fail(c, NMS_E_UNSUPPORTED, "recurrence variant forced but the detector lines are not equally spaced");

    // units of work along the cell dimension: tiles, or whole objects in split mode
    const int64_t units = split ? c->K : c->n_tiles;
    int dev_slots_guess = c->sm_count * 4;
    // q points per thread: the largest that still yields enough blocks to fill the device
    int qt_opts[3]; int n_opts = 0;
    if (variant == 1) { qt_opts[n_opts++] = 4; }
    else if (variant == 3) { qt_opts[n_opts++] = 16; qt_opts[n_opts++] = 8; qt_opts[n_opts++] = 4; }
    else { qt_opts[n_opts++] = 8; qt_opts[n_opts++] = 4; }
    int qt = qt_opts[n_opts - 1];
    if (c->opt_qt) {
        bool ok = false;
        for (int i = 0; i < n_opts; ++i) ok |= (qt_opts[i] == c->opt_qt);
        if (!ok) return fail(c, NMS_E_ARG, "option qt=%d is not available for kernel variant %d", c->opt_qt, variant);
        qt = c->opt_qt;
    } else {
        for (int i = 0; i < n_opts; ++i) {
            const int64_t qb = ceil_div(ceil_div(c->g_n0, qt_opts[i]) * c->g_n1, AMP_THREADS);
            if (qb * units >= dev_slots_guess || i == n_opts - 1) { qt = qt_opts[i]; break; }
        }
    }
    amp_kernel_t kern = pick_kernel(variant, qt, split);
    NMS_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)AMP_SMEM));
    int occ = 0;
    NMS_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, AMP_THREADS, AMP_SMEM));
    if (occ < 1) return fail(c, NMS_E_CUDA, "amplitude kernel does not fit on an SM");
    const int64_t slots = (int64_t)c->sm_count * occ;
    const int64_t n_qb = ceil_div(ceil_div(c->g_n0, qt) * c->g_n1, AMP_THREADS);

    // number of cell chunks: smallest count whose last wave is >= 97 % full (equal-sized blocks)
    int64_t max_chunks = units;
    const int64_t mem_cap = (int64_t)(1.5e9 / (64.0 * (double)c->n_q * (split ? 2.5 : 1.0)));
    if (max_chunks > mem_cap) max_chunks = mem_cap < 1 ? 1 : mem_cap;
    if (max_chunks > 4096) max_chunks = 4096;
    int64_t best_c = 1; double best_eff = -1.0;
    if (c->opt_chunks > 0) best_c = c->opt_chunks < max_chunks ? c->opt_chunks : max_chunks;
    else {
        for (int64_t nc = 1; nc <= max_chunks; ++nc) {
            const int64_t blocks = n_qb * nc;
            const double wave_eff = (double)blocks / (double)(ceil_div(blocks, slots) * slots);
            const double bal_eff = (double)units / (double)(ceil_div(units, nc) * nc);
            const double eff = wave_eff * bal_eff;
            if (eff > best_eff + 1e-9) { best_eff = eff; best_c = nc; }
            if (eff >= 0.97) { best_c = nc; break; }
        }
    }
    plan->variant = variant; plan->qt = qt; plan->n_chunks = (int)best_c; plan->n_qblocks = (int)n_qb;
    plan->blocks_per_sm = occ; plan->split = split;
    return NMS_OK;
}

nms_status launch_amplitude(nms_ctx* c, const AmpPlan& plan, const int32_t* kinds_dev, int n_kinds)
{
    // chunk boundaries (in tiles): equal parts computed in the kernel, except in split mode where they
    // must fall on object boundaries (table, uploaded only when it changes)
    int n_chunks = plan.n_chunks;
    if (plan.split) {
        std::vector<int32_t> cb;
        cb.reserve(plan.n_chunks + 1);
        cb.push_back(0);
        int64_t t = 0;
        for (int i = 1; i < plan.n_chunks; ++i) {
            const int64_t target = (c->n_tiles * (int64_t)i) / plan.n_chunks;
            while (t < c->n_tiles && !(t >= target && t > 0 && (c->h_tile_flags[t - 1] & 1))) ++t;
            if (t > cb.back() && t < c->n_tiles) cb.push_back((int32_t)t);
        }
        cb.push_back((int32_t)c->n_tiles);
        n_chunks = (int)cb.size() - 1;
        if (cb != c->h_chunk_begin) {
            if (nms_status st = ensure(c, c->chunk_begin, sizeof(int32_t) * cb.size())) return st;
            c->h_chunk_begin = cb;
            NMS_CUDA(c, cudaMemcpyAsync(c->chunk_begin.p, c->h_chunk_begin.data(), sizeof(int32_t) * cb.size(),
                                        cudaMemcpyHostToDevice, c->stream));
        }
    }
    if (nms_status st = ensure(c, c->part, sizeof(double) * 8 * (size_t)c->n_q * n_chunks)) return st;
    if (plan.split) {
        if (nms_status st = ensure(c, c->ppart, sizeof(double) * 8 * (size_t)c->n_q * n_chunks)) return st;
        if (nms_status st = ensure(c, c->formpart, sizeof(double) * (size_t)n_kinds * (size_t)c->n_q * n_chunks)) return st;
    }
    AmpArgs a;
    a.A = (const float4*)c->cellA.p; a.B = (const float2*)c->cellB.p;
    a.tiles = (const TileMeta*)c->tile_meta.p;
    a.chunk_begin = plan.split ? (const int32_t*)c->chunk_begin.p : nullptr;
    a.n_tiles = (int)c->n_tiles;
    a.type = c->g_type; a.n0 = c->g_n0; a.n1 = c->g_n1; a.n_q = c->n_q;
    a.u0 = (const float*)c->u0.p; a.qc = (const double2*)c->qc.p; a.sc = (const double2*)c->sc.p;
    a.part = (double*)c->part.p; a.ppart = (double*)c->ppart.p; a.form = (double*)c->formpart.p;
    a.kinds = kinds_dev; a.n_kinds = n_kinds;
    a.rp.Px = c->P[0]; a.rp.Py = c->P[1]; a.rp.Pz = c->P[2]; a.rp.sN = c->sN; a.rp.sM = c->sM; a.rp.invV = c->invV;

    amp_kernel_t kern = pick_kernel(plan.variant, plan.qt, plan.split);
    NMS_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)AMP_SMEM));
    dim3 grid((unsigned)plan.n_qblocks, (unsigned)n_chunks);
    timer_begin(c, NMS_T_AMPLITUDE);
    kern<<<grid, AMP_THREADS, AMP_SMEM, c->stream>>>(a);
    timer_end(c, NMS_T_AMPLITUDE);
    c->launches += 1;
    NMS_CUDA(c, cudaGetLastError());
    c->variant_used = plan.variant; c->n_chunks_used = n_chunks; c->blocks_per_sm_used = plan.blocks_per_sm;
    c->qt_used = plan.qt;
    return NMS_OK;
}

}  // namespace nms
