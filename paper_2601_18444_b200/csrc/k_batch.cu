// k_batch.cu -- f-3: batched magnetisation fields on a fixed geometry (the paper's loop mode: one magnetisation file m_i
// per field / temperature / time step on the same NucData and StructData, L254, L323, L391; "~1000 applied-field values"
// per hysteresis loop, L686).
//
// For B fields the phasor exp(-i Psi_j(q)) and the nuclear sum N~ are the same; only the three magnetic sums differ.
// The fields are processed in groups of BF = 3: a pass packs the group into 64-byte records {Y, Z (fp64), N, 3 x (m'x, m'y,
// m'z)} (k_prep_batch: rotation in fp64, one rounding, as a-1), and k_amp_batch evaluates ONE phasor per (cell, detector
// point) and feeds it to 10 packed accumulations (1 nuclear + 9 magnetic) instead of 4: 20 FMA-pipe cycles + ~6 issue slots
// for the phasor per 3 pair-fields against 3 x (8 + ~6) -- 8.7 instead of 14 cycles per pair-field.  With 10 complex
// accumulators per point a thread owns QT = 4 points (80 registers, 3 blocks per SM) in the DIRECT kernel (any detector
// grid: the 2 MUFU per pair need 16 XU cycles against 20 FMA cycles, so it is not XU-bound), and QT = 8 points (160
// registers, 2 blocks per SM) in the LINE-RECURRENCE kernel that the accurate variant runs on equally spaced lines: one
// exactly evaluated point per 8, the others by rotations (accurate) or rotation + three-term recurrence (fast, on request
// only), as in k_amplitude.cuh.
// k_epilogue_batch sums the chunk partials and forms the requested responses of every field of the group with the shared N~.
#include "k_amplitude.cuh"

namespace nms {

constexpr int BF = 3;              // fields per pass
constexpr int BQT = 4;             // detector points per thread, direct kernel
constexpr int BQT_REC = 8;         // detector points per thread, line-recurrence kernel
constexpr int BCH = 1 + 3 * BF;    // weight channels per record

struct BCell {                     // 64 B
    double Y, Z;
    float w[12];                   // N, field 0 (x, y, z), field 1, field 2, 2 x padding
};

struct BatchArgs {
    const BCell* cells;
    const TileMeta* tiles;
    int n_tiles;
    int type, n0, n1;
    int64_t n_q;
    const float* u0;
    double dq;                     // recurrence: spacing of u0
    int sh;                        // recurrence, accurate: the step phase stays within a quarter cycle
    const double2* qc;
    const double2* sc;
    double* part;                  // [n_chunks][2 * BCH][n_q]
};

struct PrepBatchArgs {
    const float* pos;
    const float* N;
    const float* m;                // [B][W][3]
    const float* centres;
    const TileSrc* src;
    const int64_t* first_slot;
    BCell* cells;
    int64_t W;
    int field0, n_fields;          // fields field0 ... field0 + n_fields - 1 of this pass (n_fields <= BF)
    double R[9];
};

__global__ void __launch_bounds__(256) k_prep_batch(const PrepBatchArgs a)
{
    const TileSrc ts = a.src[blockIdx.x];
    const int64_t first_slot = a.first_slot[blockIdx.x];
    const int i = threadIdx.x;
    if (i >= ts.n_src) return;
    const int64_t j = ts.src_first + i;
    double cx = 0.0, cy = 0.0, cz = 0.0;
    if (a.centres && ts.particle >= 0) {
        cx = (double)a.centres[3 * (int64_t)ts.particle + 0];
        cy = (double)a.centres[3 * (int64_t)ts.particle + 1];
        cz = (double)a.centres[3 * (int64_t)ts.particle + 2];
    }
    const double x = (double)a.pos[3 * j + 0] + cx, y = (double)a.pos[3 * j + 1] + cy, z = (double)a.pos[3 * j + 2] + cz;
    BCell ce;
    ce.Y = a.R[3] * x + a.R[4] * y + a.R[5] * z;   // Eq. 39
    ce.Z = a.R[6] * x + a.R[7] * y + a.R[8] * z;   // Eq. 40
#pragma unroll
    for (int k = 0; k < 12; ++k) ce.w[k] = 0.f;
    if (a.N && a.field0 == 0) ce.w[0] = a.N[j];    // the nuclear sum is formed in the first pass only
    for (int f = 0; f < a.n_fields; ++f) {
        const float* mp = a.m + ((int64_t)(a.field0 + f) * a.W + j) * 3;
        const double mx = (double)mp[0], my = (double)mp[1], mz = (double)mp[2];
        ce.w[1 + 3 * f + 0] = (float)(a.R[0] * mx + a.R[1] * my + a.R[2] * mz);   // m' = R m (reading 2)
        ce.w[1 + 3 * f + 1] = (float)(a.R[3] * mx + a.R[4] * my + a.R[5] * mz);
        ce.w[1 + 3 * f + 2] = (float)(a.R[6] * mx + a.R[7] * my + a.R[8] * mz);
    }
    float4* dst = reinterpret_cast<float4*>(a.cells + first_slot + i);
    const float4* srcv = reinterpret_cast<const float4*>(&ce);
#pragma unroll
    for (int k = 0; k < 4; ++k) dst[k] = srcv[k];
}

constexpr size_t BATCH_SMEM = 2 * TILE * sizeof(BCell) + 2 * sizeof(uint64_t);

// MODE as in k_amplitude.cuh (0 polar, 1 Cartesian, 2 list).  Same tile pipeline (cp.async.bulk + mbarrier, double
// buffered), same exact phase reduction and MUFU phasor; 10 packed accumulations per pair.
// 3 blocks per SM: 80 accumulator registers + phase constants need ~150 registers (at 128 the kernel spills and was
// measured 20 % slower: C5 2578 against 3084 Gpair-field/s).
// ACC: the accurate variant (polynomial phasor, fp64 sub-accumulation of the shared nuclear channel every NSUB_CELLS cells).
// REC: line recurrence over the thread's BQT = 8 points (MODE 0 / 1 with equally spaced u0; 2 blocks per SM): the point
//      KB is evaluated exactly, fast variant: its upper neighbour by one rotation and the others by the three-term
//      recurrence (runs of <= 3 steps); accurate variant: rotations both ways (<= 4 steps).  The deviation of the float
//      abscissae from the progression is corrected at the flush, to first order, at the tile centre (as k_amp).
template <int MODE, bool ACC, int BQT, bool REC>
__global__ void __launch_bounds__(AMP_THREADS, REC ? 2 : 3) k_amp_batch(const BatchArgs a)
{
    static_assert(!REC || MODE != 2, "the recurrence needs a line of equally spaced abscissae");
    constexpr int KB = ACC ? BQT / 2 : (BQT - 1) / 2;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    BCell* sC = reinterpret_cast<BCell*>(smem_raw);
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw + 2 * TILE * sizeof(BCell));
    double* nacc = reinterpret_cast<double*>(smem_raw + BATCH_SMEM);                       // ACC: [BQT * 2][128]
    const int tid = threadIdx.x, chunk = blockIdx.y;
    const int tile_beg = (int)(((int64_t)a.n_tiles * chunk) / gridDim.y);
    const int tile_end = (int)(((int64_t)a.n_tiles * (chunk + 1)) / gridDim.y);

    const int n_groups = (a.n0 + BQT - 1) / BQT;
    int64_t slot = (int64_t)blockIdx.x * AMP_THREADS + tid;
    const bool valid = slot < (int64_t)n_groups * a.n1;
    if (!valid) slot = 0;
    const int grp = (int)(slot / a.n1), i1 = (int)(slot % a.n1);
    const int i0 = grp * BQT;
    const int kmax = valid ? min(BQT, a.n0 - i0) : 0;
    const int kclamp = max(min(BQT, a.n0 - i0), 1);
    const int64_t flat0 = (int64_t)i0 * a.n1 + i1;
    double c0 = 0.0, c1 = 0.0, g[BQT], h[BQT];
#pragma unroll
    for (int k = 0; k < BQT; ++k) {
        const int kk = min(k, kclamp - 1);
        if (MODE == 0) { g[k] = (double)a.u0[i0 + kk] * INV_2PI; h[k] = 0.0; }
        else { const double2 q = a.qc[flat0 + (int64_t)kk * a.n1]; g[k] = q.y * INV_2PI; h[k] = q.x * INV_2PI; }
        asm volatile("" : "+d"(g[k]));
        if (MODE == 2) asm volatile("" : "+d"(h[k]));
    }
    if (MODE == 0) { const double2 d = a.sc[flat0]; c0 = d.x; c1 = d.y; }
    if (MODE == 1) c0 = h[0];
    const double dq = a.dq * INV_2PI;
    double gb = g[KB < BQT ? KB : 0];   // abscissa of the exactly evaluated point; beyond the edge it continues the progression
    if (REC && KB >= kclamp) gb += (double)(KB - (kclamp - 1)) * dq;

    auto issue = [&](int tile, BCell* dst, uint64_t* b) {
        const TileMeta tm = a.tiles[tile];
        const uint32_t bytes = (uint32_t)tm.n_slots * (uint32_t)sizeof(BCell);
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        mbar_expect_tx(b, bytes);
        bulk_g2s(dst, a.cells + tm.first_slot, bytes, b);
    };
    if (tid == 0) {
        mbar_init(&bar[0], 1);
        mbar_init(&bar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (tid == 0) {
        if (tile_beg < tile_end) issue(tile_beg, sC, &bar[0]);
        if (tile_beg + 1 < tile_end) issue(tile_beg + 1, sC + TILE, &bar[1]);
    }

    u64 acc[BQT][BCH];
    for (int t = tile_beg; t < tile_end; ++t) {
        const int it = t - tile_beg, stage = it & 1;
        const TileMeta tm = a.tiles[t];
        const int nc = tm.n_slots;
        const BCell* __restrict__ tC = sC + stage * TILE;
#pragma unroll
        for (int k = 0; k < BQT; ++k)
#pragma unroll
            for (int r = 0; r < BCH; ++r) acc[k][r] = 0ull;
        mbar_wait(&bar[stage], (uint32_t)((it >> 1) & 1));
        auto cell = [&](int j) {
            const double2 YZ = *reinterpret_cast<const double2*>(&tC[j].Y);
            const float4 w0 = *reinterpret_cast<const float4*>(&tC[j].w[0]);
            const float4 w1 = *reinterpret_cast<const float4*>(&tC[j].w[4]);
            const float2 w2 = *reinterpret_cast<const float2*>(&tC[j].w[8]);
            double p = 0.0;
            if (MODE == 0) p = fma(c1, YZ.y, c0 * YZ.x);
            if (MODE == 1) p = c0 * YZ.x;
            u64 phs[BQT];
            if (REC) {
                float cd, sd;
                const int kd = __double2loint(fma(dq, MODE == 0 ? p : YZ.y, MAGIC));
                if (!ACC) sincos_mufu(kd, cd, sd);
                else if (a.sh) sincos_poly_half(kd, cd, sd);
                else sincos_poly(kd, cd, sd);
                phs[KB] = phasor<ACC>(MODE == 0 ? fma(gb, p, MAGIC) : fma(gb, YZ.y, p) + MAGIC);
                if (!ACC) {
                    const float two_cd = cd + cd;
                    phs[KB + 1] = rotate(phs[KB], cd, sd);
#pragma unroll
                    for (int k = KB + 2; k < BQT; ++k) phs[k] = three_term(phs[k - 1], phs[k - 2], two_cd);
#pragma unroll
                    for (int k = KB - 1; k >= 0; --k) phs[k] = three_term(phs[k + 1], phs[k + 2], two_cd);
                } else {
#pragma unroll
                    for (int k = KB + 1; k < BQT; ++k) phs[k] = rotate(phs[k - 1], cd, sd);
#pragma unroll
                    for (int k = KB - 1; k >= 0; --k) phs[k] = rotate(phs[k + 1], cd, -sd);
                }
            }
#pragma unroll
            for (int k = 0; k < BQT; ++k) {
                u64 ph;
                if (REC) ph = phs[k];
                else {
                    double m;
                    if (MODE == 0) m = fma(g[k], p, MAGIC);
                    else if (MODE == 1) m = fma(g[k], YZ.y, p) + MAGIC;
                    else m = fma(g[k], YZ.y, h[k] * YZ.x) + MAGIC;
                    ph = phasor<ACC>(m);
                }
                acc[k][0] = ffma2(pack2(w0.x, w0.x), ph, acc[k][0]);
                acc[k][1] = ffma2(pack2(w0.y, w0.y), ph, acc[k][1]);
                acc[k][2] = ffma2(pack2(w0.z, w0.z), ph, acc[k][2]);
                acc[k][3] = ffma2(pack2(w0.w, w0.w), ph, acc[k][3]);
                acc[k][4] = ffma2(pack2(w1.x, w1.x), ph, acc[k][4]);
                acc[k][5] = ffma2(pack2(w1.y, w1.y), ph, acc[k][5]);
                acc[k][6] = ffma2(pack2(w1.z, w1.z), ph, acc[k][6]);
                acc[k][7] = ffma2(pack2(w1.w, w1.w), ph, acc[k][7]);
                acc[k][8] = ffma2(pack2(w2.x, w2.x), ph, acc[k][8]);
                acc[k][9] = ffma2(pack2(w2.y, w2.y), ph, acc[k][9]);
            }
        };
        if (!ACC) {
#pragma unroll (REC ? 2 : 4)
            for (int j = 0; j < nc; ++j) cell(j);
        } else {
#pragma unroll
            for (int r = 0; r < 2 * BQT; ++r) nacc[r * AMP_THREADS + tid] = 0.0;
            for (int j0 = 0; j0 < nc; j0 += NSUB_CELLS) {
                const int j1 = min(nc, j0 + NSUB_CELLS);
#pragma unroll (REC ? 2 : 4)
                for (int j = j0; j < j1; ++j) cell(j);
#pragma unroll
                for (int k = 0; k < BQT; ++k) {
                    float cs, sn;
                    unpack2(acc[k][0], cs, sn);
                    nacc[(2 * k) * AMP_THREADS + tid] += (double)cs;
                    nacc[(2 * k + 1) * AMP_THREADS + tid] += (double)sn;
                    acc[k][0] = 0ull;
                }
            }
        }
        __syncthreads();
        if (tid == 0 && t + 2 < tile_end) issue(t + 2, sC + stage * TILE, &bar[stage]);
        double p0 = 0.0;                                   // projection of the tile centre (recurrence correction)
        if (REC) p0 = MODE == 0 ? fma(c1, tm.Z0, c0 * tm.Y0) : tm.Z0;
#pragma unroll
        for (int k = 0; k < BQT; ++k) {
            if (k < kmax) {
                const int64_t f = flat0 + (int64_t)k * a.n1;
                float eps = 0.f;
                if (REC && k != KB) {
                    const double gk = MODE == 0 ? (double)a.u0[i0 + k] * INV_2PI : a.qc[f].y * INV_2PI;
                    eps = (float)(6.283185307179586 * (gk - (gb + (double)(k - KB) * dq)) * p0);
                }
#pragma unroll
                for (int r = 0; r < BCH; ++r) {
                    float cs, sn;
                    unpack2(acc[k][r], cs, sn);
                    double dc = (double)cs, ds = (double)sn;
                    if (ACC && r == 0) { dc = nacc[(2 * k) * AMP_THREADS + tid]; ds = nacc[(2 * k + 1) * AMP_THREADS + tid]; }
                    if (REC) {                             // cos(psi + eps), sin(psi + eps) to first order
                        const double d2 = fma(-(double)eps, ds, dc);
                        ds = fma((double)eps, dc, ds);
                        dc = d2;
                    }
                    atomicAdd(a.part + ((int64_t)chunk * 2 * BCH + 2 * r) * a.n_q + f, dc);        // Re: + sum w cos
                    atomicAdd(a.part + ((int64_t)chunk * 2 * BCH + 2 * r + 1) * a.n_q + f, -ds);   // Im: - sum w sin
                }
            }
        }
    }
}

// Sum the chunk partials of one pass; the nuclear amplitude of the first pass is kept (fp64) for the later ones; write
// the requested responses of the pass's fields (and optionally their amplitudes).
__global__ void __launch_bounds__(256) k_epilogue_batch(const double* __restrict__ part, int n_chunks, int64_t n_q,
                                                        double* __restrict__ ampN, int field0, int n_fields, int B,
                                                        const double2* __restrict__ sc, const int32_t* __restrict__ kinds,
                                                        int n_kinds, RespParams rp, float* __restrict__ out_maps,
                                                        float* __restrict__ out_amp)
{
    const int64_t f = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (f >= n_q) return;
    double S[2 * BCH];
#pragma unroll
    for (int r = 0; r < 2 * BCH; ++r) S[r] = 0.0;
    for (int ch = 0; ch < n_chunks; ++ch)
#pragma unroll
        for (int r = 0; r < 2 * BCH; ++r) S[r] += part[((int64_t)ch * 2 * BCH + r) * n_q + f];
    if (field0 == 0) { ampN[f] = S[0]; ampN[n_q + f] = S[1]; }
    else { S[0] = ampN[f]; S[1] = ampN[n_q + f]; }
    const double2 d = sc[f];
    for (int b = 0; b < n_fields; ++b) {
        double A[8];
        A[0] = S[0]; A[1] = S[1];
        for (int r = 0; r < 6; ++r) A[2 + r] = S[2 + 6 * b + r];
        if (out_amp)
            for (int r = 0; r < 8; ++r) out_amp[((int64_t)(field0 + b) * 8 + r) * n_q + f] = (float)A[r];
        if (out_maps) {
            double val[NMS_KIND_COUNT];
            responses_at_point(A, d.x, d.y, rp, val);
            for (int i = 0; i < n_kinds; ++i) out_maps[((int64_t)(field0 + b) * n_kinds + i) * n_q + f] = (float)val[kinds[i]];
        }
    }
    (void)B;
}

nms_status launch_batch(nms_ctx* c, const float* m_batch, int B, const int32_t* kinds_dev, int n_kinds, float* out_maps,
                        float* out_amp, bool accurate)
{
    if (nms_status st = wait_geometry(c)) return st;
    typedef void (*kern_t)(const BatchArgs);
    // line recurrence: the ACCURATE variant where the lines are equally spaced and the cell order is spatially coherent (the
    // criterion of plan_amplitude) -- its polynomial phasors cost FMA-pipe cycles, so one per 8 points pays (measured, 6
    // fields: C5 2.12 -> 2.51, C4 geometry 2.19 -> 2.77 T pair-fields/s); the FAST variant stays direct (MUFU phasors run on
    // the otherwise idle XU pipe: 2.99 direct against 2.81 with the recurrence on C5).  "variant" 1 forces the direct
    // kernel, 2 the recurrence
    const bool line_ok = c->g_type != 2 && c->g_uniform && c->g_n0 >= 2;
    if (c->opt_variant == 2 && !line_ok)
        return fail(c, NMS_E_UNSUPPORTED, "the line-recurrence variant needs a polar or Cartesian detector with equally spaced u0");
    const bool rec = line_ok && (c->opt_variant == 2 || (c->opt_variant == 0 && accurate &&
                                                         c->g_dev * (c->g_type == 0 ? c->geo_ext : c->geo_extz) <= 1e-4));
    const int qt = rec ? BQT_REC : BQT;
    kern_t kern;
    if (rec) {
        if (accurate) kern = c->g_type == 0 ? (kern_t)k_amp_batch<0, true, BQT_REC, true> : (kern_t)k_amp_batch<1, true, BQT_REC, true>;
        else kern = c->g_type == 0 ? (kern_t)k_amp_batch<0, false, BQT_REC, true> : (kern_t)k_amp_batch<1, false, BQT_REC, true>;
    } else if (accurate) {
        kern = c->g_type == 0 ? (kern_t)k_amp_batch<0, true, BQT, false>
                              : (c->g_type == 1 ? (kern_t)k_amp_batch<1, true, BQT, false> : (kern_t)k_amp_batch<2, true, BQT, false>);
    } else {
        kern = c->g_type == 0 ? (kern_t)k_amp_batch<0, false, BQT, false>
                              : (c->g_type == 1 ? (kern_t)k_amp_batch<1, false, BQT, false> : (kern_t)k_amp_batch<2, false, BQT, false>);
    }
    const size_t smem = BATCH_SMEM + (accurate ? (size_t)qt * 2 * AMP_THREADS * sizeof(double) : 0);
    NMS_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int occ = 0;
    NMS_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, AMP_THREADS, smem));
    if (occ < 1) return fail(c, NMS_E_CUDA, "batch amplitude kernel does not fit on an SM");
    const int64_t n_qb = (((int64_t)(c->g_n0 + qt - 1) / qt) * c->g_n1 + AMP_THREADS - 1) / AMP_THREADS;
    const int n_chunks = choose_chunks(c, n_qb, (int64_t)c->sm_count * occ, c->n_tiles, 8.0 * 2 * BCH * (double)c->n_q, 8, 2.0e9);
    const size_t part_bytes = sizeof(double) * 2 * BCH * (size_t)c->n_q * n_chunks;
    if (nms_status st = ensure(c, c->part, part_bytes)) return st;
    if (nms_status st = ensure(c, c->batch_cells, sizeof(BCell) * (size_t)c->n_slots)) return st;
    if (nms_status st = ensure(c, c->batch_ampN, sizeof(double) * 2 * (size_t)c->n_q)) return st;

    PrepBatchArgs pa;
    pa.pos = (const float*)c->raw_pos.p;
    pa.N = c->has_N ? (const float*)c->raw_N.p : nullptr;
    pa.m = m_batch;
    pa.centres = c->has_centres ? (const float*)c->centres.p : nullptr;
    pa.src = (const TileSrc*)c->tile_src.p;
    pa.first_slot = (const int64_t*)((const char*)c->tile_src.p + sizeof(TileSrc) * (size_t)c->n_tiles);
    pa.cells = (BCell*)c->batch_cells.p;
    pa.W = c->W;
    for (int i = 0; i < 9; ++i) pa.R[i] = c->R[i];
    BatchArgs a;
    a.cells = (const BCell*)c->batch_cells.p;
    a.tiles = (const TileMeta*)c->tile_meta.p;
    a.n_tiles = (int)c->n_tiles;
    a.type = c->g_type; a.n0 = c->g_n0; a.n1 = c->g_n1; a.n_q = c->n_q;
    a.u0 = (const float*)c->u0.p; a.qc = (const double2*)c->qc.p; a.sc = (const double2*)c->sc.p;
    a.dq = c->g_dq; a.sh = fabs(c->g_dq) * c->geo_rmax < 0.24 * 6.283185307179586 ? 1 : 0;
    a.part = (double*)c->part.p;
    RespParams rp;
    rp.Px = c->P[0]; rp.Py = c->P[1]; rp.Pz = c->P[2]; rp.sN = c->sN; rp.sM = c->sM; rp.invV = c->invV;

    for (int f0 = 0; f0 < B; f0 += BF) {
        pa.field0 = f0; pa.n_fields = B - f0 < BF ? B - f0 : BF;
        if (nms_status st = timer_begin(c, NMS_T_PREP)) return st;
        k_prep_batch<<<(unsigned)c->n_tiles, 256, 0, c->stream>>>(pa);
        if (nms_status st = timer_end(c, NMS_T_PREP)) return st;
        NMS_CUDA(c, cudaMemsetAsync(c->part.p, 0, part_bytes, c->stream));
        if (nms_status st = timer_begin(c, NMS_T_BATCH)) return st;
        kern<<<dim3((unsigned)n_qb, (unsigned)n_chunks), AMP_THREADS, smem, c->stream>>>(a);
        if (nms_status st = timer_end(c, NMS_T_BATCH)) return st;
        if (nms_status st = timer_begin(c, NMS_T_EPILOGUE)) return st;
        k_epilogue_batch<<<(unsigned)((c->n_q + 255) / 256), 256, 0, c->stream>>>(
            (const double*)c->part.p, n_chunks, c->n_q, (double*)c->batch_ampN.p, f0, pa.n_fields, B, (const double2*)c->sc.p,
            kinds_dev, n_kinds, rp, out_maps, out_amp);
        if (nms_status st = timer_end(c, NMS_T_EPILOGUE)) return st;
        c->launches += 3;
        NMS_CUDA(c, cudaGetLastError());
    }
    c->n_chunks_used = n_chunks; c->blocks_per_sm_used = occ; c->qt_used = qt; c->variant_used = rec ? 17 : 16;
    c->npoly_used = accurate ? (rec ? 1 : qt) : 0; c->nb_used = rec ? 1 : 0; c->rec3_used = rec && !accurate ? 1 : 0;
    return NMS_OK;
}

}  // namespace nms
