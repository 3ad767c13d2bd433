// k_amplitude.cu -- a-2 (and a-6): the exact fp64 amplitude kernel, and the host side of all amplitude kernels
// (planning and dispatch).  The fp32 kernel templates live in k_amplitude.cuh.
#include "k_amplitude.cuh"

namespace nms {

// ---- exact variant: everything in fp64 -----------------------------------------------------------
// One thread per detector point, cells read straight from global memory (every lane of a block reads the
// same record: L1 broadcast).  Phase t = (q/2pi).r in fp64, reduced exactly to [-1/2, 1/2] cycle, sincospi
// and the 8 accumulations in fp64.  ~50 fp64 operations per pair: 7x slower than the fp32 kernels, chosen
// automatically only for small problems (launch-bound anyway), where it makes the result exact to the
// fp32 rounding of the rotated weights.  See DESIGN.md section 7 (precision policy).
// SPLIT (a-6, Eq. 49-50): the running amplitudes of the current object stay in registers; when the
// object is complete its responses go to the form accumulators and its amplitudes to the totals.
template <bool SPLIT>
__global__ void __launch_bounds__(AMP_THREADS) k_amp_f64(const AmpArgs a)
{
    const int chunk = blockIdx.y;
    int tile_beg, tile_end;
    chunk_range(a, tile_beg, tile_end);
    const int64_t f = (int64_t)blockIdx.x * AMP_THREADS + threadIdx.x;
    if (f >= a.n_q) return;
    const double2 q = a.qc[f];
    const double qy = q.x * INV_2PI, qz = q.y * INV_2PI;
    double Ap[8];
#pragma unroll
    for (int r = 0; r < 8; ++r) Ap[r] = 0.0;
    for (int t = tile_beg; t < tile_end; ++t) {
        const TileMeta tm = a.tiles[t];
        const Cell* __restrict__ tC = a.cells + tm.first_slot;
        for (int j = 0; j < tm.n_slots; ++j) {
            const Cell ce = tC[j];
            double ph = fma(qz, ce.Z, qy * ce.Y);          // Eq. 41, in cycles
            ph -= rint(ph);
            double sn, cs;
            sincospi(2.0 * ph, &sn, &cs);
            const double w[4] = {(double)ce.wN, (double)ce.wx, (double)ce.wy, (double)ce.wz};
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                Ap[2 * c] = fma(w[c], cs, Ap[2 * c]);            // Re: + sum w cos(Psi)   (Eq. 44, 46)
                Ap[2 * c + 1] = fma(-w[c], sn, Ap[2 * c + 1]);   // Im: - sum w sin(Psi)   (Eq. 45, 47)
            }
        }
        if (SPLIT && (tm.flags & 1)) {                           // the object is complete
            flush_object(a, chunk, f, Ap);
#pragma unroll
            for (int r = 0; r < 8; ++r) Ap[r] = 0.0;
        }
    }
    if (!SPLIT)
#pragma unroll
        for (int r = 0; r < 8; ++r) atomicAdd(a.part + ((int64_t)chunk * 8 + r) * a.n_q + f, Ap[r]);
}

// ---- host side: planning and dispatch ------------------------------------------------------------
// variant: 1 list direct, 2 polar direct, 4 cartesian direct, 3 polar recurrence, 5 cartesian recurrence
// (all with fp32 accumulation over a tile), 8 exact (fp64)
static amp_kernel_t pick_kernel(const AmpPlan& p)
{
    if (p.interp) return amp_kernel_interp(p.variant == 3 ? 0 : 1);
    switch (p.variant) {
    case 1: return amp_kernel_direct(2, p.qt, p.split, p.nch, p.npoly, false);
    case 2: return amp_kernel_direct(0, p.qt, p.split, p.nch, p.npoly, p.uni);
    case 4: return amp_kernel_direct(1, p.qt, p.split, p.nch, p.npoly, p.uni);
    case 3: return amp_kernel_rec_polar(p.qt, p.nb, p.split, p.nch, p.npoly != 0, p.rec3 != 0, p.uni, p.sh);
    case 5: return amp_kernel_rec_cart(p.qt, p.nb, p.split, p.nch, p.npoly != 0, p.rec3 != 0, p.uni, p.sh);
    default: return p.split ? (amp_kernel_t)k_amp_f64<true> : (amp_kernel_t)k_amp_f64<false>;
    }
}

static int64_t ceil_div(int64_t a, int64_t b) { return (a + b - 1) / b; }

// Number of cell chunks.  Measured on B200 (C3, C4, C5): many short blocks beat one long wave (C5 0.759 -> 0.785,
// C4 0.763 -> 0.813, C3 0.587 -> 0.630 of the roofline from 9 chunks to 16+ waves) -- the blocks are equal-sized, so
// what counts is that blocks / (SMs x resident blocks) comes out close to a whole number and that there are enough
// waves for the dynamic scheduler to even out.  Search 16 ... 48 waves for the best product of wave fill and unit
// balance; the fp64 partials (chunk_bytes per chunk) cap it at mem_bytes; at least min_units units of work per chunk.
int choose_chunks(nms_ctx* c, int64_t n_qb, int64_t slots, int64_t units, double chunk_bytes, int64_t min_units, double mem_bytes)
{
    int64_t max_chunks = units;
    const int64_t mem_cap = (int64_t)(mem_bytes / chunk_bytes);
    if (max_chunks > mem_cap) max_chunks = mem_cap < 1 ? 1 : mem_cap;
    if (max_chunks > 4096) max_chunks = 4096;
    if (n_qb * (units / min_units) < 2 * slots) min_units = 1;   // small problem: filling the device comes first
    if (max_chunks > units / min_units) max_chunks = units / min_units < 1 ? 1 : units / min_units;
    int64_t best_c = 1; double best_eff = -1.0;
    if (c->opt_chunks > 0) return (int)(c->opt_chunks < units ? c->opt_chunks : units);
    int64_t lo = ceil_div(16 * slots, n_qb), hi = ceil_div(48 * slots, n_qb);
    if (lo > max_chunks) lo = 1;                    // small problem: take the best there is
    if (hi > max_chunks) hi = max_chunks;
    for (int64_t nc = lo; nc <= hi; ++nc) {
        const int64_t blocks = n_qb * nc;
        const double wave_eff = (double)blocks / (double)(ceil_div(blocks, slots) * slots);
        const double bal_eff = (double)units / (double)(ceil_div(units, nc) * nc);
        const double eff = wave_eff * bal_eff;
        if (eff > best_eff + 1e-9) { best_eff = eff; best_c = nc; }
        if (eff >= 0.995) break;
    }
    return (int)best_c;
}

// Geometry of the packed sample (k_prep) on the host -- waits for the prep pass only -- and the range check of the fp32
// kernels: the adder-rounding reduction of the phase holds for |t| < 2^19 cycles (nms_phasor.cuh).
nms_status wait_geometry(nms_ctx* c)
{
    if (c->geo_pending) {
        NMS_CUDA(c, cudaEventSynchronize(c->geo_event));
        c->geo_rmax = c->h_geo[0]; c->geo_ext = c->h_geo[1]; c->geo_extz = c->h_geo[2];
        c->geo_pending = false;
    }
    if (c->g_qmax * c->geo_rmax * INV_2PI >= 524288.0 * 0.99)
        return fail(c, NMS_E_UNSUPPORTED, "q_max r_max / 2 pi = %.3g cycles exceeds 2^19: use the exact kernel (variant 3)",
                    c->g_qmax * c->geo_rmax * INV_2PI);
    return NMS_OK;
}

nms_status plan_amplitude(nms_ctx* c, bool split, bool want_accurate, AmpPlan* plan)
{
    // precision policy: small problems run the exact fp64 kernel; otherwise the line
    // recurrence where the thread lines are equally spaced, else the direct kernel.  The accurate variant (polynomial
    // phasors, rotations, fp64 sub-accumulation of the nuclear channel) runs when the caller needs the signed kinds NM /
    // CHI at the north-star criterion (want_accurate: they were requested, or the amplitudes are kept for later requests),
    // the fast one (MUFU phasors, three-term recurrence) otherwise; the "precision" option overrides: 1 fast, 2 accurate
    AmpPlan p = {};
    p.split = split;
    const bool small = (double)c->W * (double)c->n_q <= 1073741824.0;
    const bool line_ok = c->g_type != 2 && c->g_uniform && c->g_n0 >= 2;
    if (c->opt_variant == 2 && !line_ok)
        return fail(c, NMS_E_UNSUPPORTED, "the line-recurrence variant needs a polar or Cartesian detector with equally spaced u0");
    const bool accurate = c->opt_precision == 2 || (c->opt_precision == 0 && want_accurate);
    if (c->opt_variant == 3 || (c->opt_variant == 0 && small)) p.variant = 8;
    else if (c->g_type == 2) p.variant = 1;
    else if (c->opt_variant == 2 || (c->opt_variant == 0 && line_ok)) p.variant = (c->g_type == 0) ? 3 : 5;
    else p.variant = (c->g_type == 0) ? 2 : 4;
    if (p.variant != 8) {
        if (nms_status st = wait_geometry(c)) return st;
        // automatic choice: after its first-order correction at the tile centres the recurrence leaves a phase error
        // <= (deviation of the float abscissae from the progression) x (half extent of a tile along the line's
        // direction: any direction of the detector plane for a polar grid, Z for a Cartesian one); beyond 1e-4 rad
        // (spatially incoherent cell order) use the direct kernel
        if (c->opt_variant == 0 && (p.variant == 3 || p.variant == 5) &&
            c->g_dev * (c->g_type == 0 ? c->geo_ext : c->geo_extz) > 1e-4)
            p.variant = (c->g_type == 0) ? 2 : 4;
    }
    const bool rec = p.variant == 3 || p.variant == 5;
    p.nch = (c->has_M || split) ? 4 : 1;

    // units of work along the cell dimension: tiles, or whole objects in split mode
    const int64_t units = split ? c->K : c->n_tiles;
    const int dev_slots_guess = c->sm_count * 3;
    // q points per thread: the largest that still yields enough blocks to fill the device
    int qt_opts[3]; int n_opts = 0;
    if (p.variant == 8) { qt_opts[n_opts++] = 1; }
    else if (p.variant == 1) { qt_opts[n_opts++] = 4; }
    else if (rec) {   // 16 points per thread: one channel, or four channels (2 blocks per SM) in the default arrangements
        const bool defaults = c->opt_bases == 0 && c->opt_rec3 == 0;
        if (defaults && (p.nch == 1 || !split)) qt_opts[n_opts++] = 16;
        qt_opts[n_opts++] = 8;
    }
    else { qt_opts[n_opts++] = 8; qt_opts[n_opts++] = 4; }
    p.qt = qt_opts[n_opts - 1];
    if (c->opt_qt && p.variant != 8) {
        bool ok = false;
        for (int i = 0; i < n_opts; ++i) ok |= (qt_opts[i] == c->opt_qt);
        if (!ok) return fail(c, NMS_E_ARG, "option qt=%d is not available for kernel variant %d", c->opt_qt, p.variant);
        p.qt = c->opt_qt;
    } else {
        for (int i = 0; i < n_opts; ++i) {
            const int64_t qb = ceil_div(ceil_div(c->g_n0, qt_opts[i]) * c->g_n1, AMP_THREADS);
            if (qb * units >= dev_slots_guess || i == n_opts - 1) { p.qt = qt_opts[i]; break; }
        }
    }
    // recurrence: one exactly evaluated point per 8 and the three-term recurrence (measured fastest: C5 0.69 -> 0.785 of
    // the roofline against 2 bases + rotations, errors of the same size); the accurate variant keeps the rotations
    if (rec) {
        p.nb = c->opt_bases ? c->opt_bases : (p.nch == 1 ? (p.qt == 16 ? 4 : 2) : (p.qt == 16 && !accurate ? 2 : 1));
        p.rec3 = c->opt_rec3 ? (c->opt_rec3 == 2) : (!accurate && (p.qt == 16 || p.nb <= 2));
        p.npoly = accurate ? 1 : 0;
        if (p.rec3 && p.qt == 8 && p.nb > 2) return fail(c, NMS_E_ARG, "the three-term recurrence needs bases <= 2");
    } else if (p.variant != 8) {
        p.npoly = accurate ? p.qt : 0;
    }
    p.uni = c->g_n1 % AMP_THREADS == 0 && c->opt_uniform != 1;
    p.sh = rec && accurate && fabs(c->g_dq) * c->geo_rmax < 0.24 * 6.283185307179586 && c->opt_uniform != 1;
    // accurate variant, four channels, not split, default arrangement: generate every other point of a line and take the
    // points in between from the sums (k_amp_interp.cu) -- admissible while the step phase of every cell stays within 0.2
    // cycle (1 / (2 cos delta) <= 1.62) and the line has at least 3 points
    p.interp = rec && accurate && !split && p.nch == 4 && p.qt == 16 && c->opt_interp != 1 && c->opt_uniform != 1 &&
               c->g_n0 >= 3 && fabs(c->g_dq) * c->geo_rmax < 0.2 * 6.283185307179586;
    if (c->opt_interp == 2 && !p.interp)
        return fail(c, NMS_E_UNSUPPORTED, "the interpolating kernel needs the accurate four-channel line recurrence (not split, qt 0 / 16, "
                                          "default bases / recurrence) and a step phase below 0.2 cycle (d r_max = %.3g cycles)",
                    fabs(c->g_dq) * c->geo_rmax * INV_2PI);
    amp_kernel_t kern = pick_kernel(p);
    if (!kern) return fail(c, NMS_E_ARG, "no amplitude kernel for variant %d qt %d bases %d polynomial %d three-term %d",
                           p.variant, p.qt, p.nb, p.npoly, p.rec3);
    const size_t smem = p.variant == 8 ? 0 : p.interp ? AMP_SMEM_INTERP : amp_smem_bytes(p.qt, p.nch, split, p.npoly != 0 && !split);
    NMS_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int occ = 0;
    NMS_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, AMP_THREADS, smem));
    if (occ < 1) return fail(c, NMS_E_CUDA, "amplitude kernel does not fit on an SM");
    const int64_t slots = (int64_t)c->sm_count * occ;
    const int64_t n_qb = p.variant == 8 ? ceil_div(c->n_q, AMP_THREADS)
                         : p.interp     ? ceil_div(ceil_div(c->g_n0 / 2 + 1, 8) * c->g_n1, AMP_THREADS)   // 8 primaries per thread
                                        : ceil_div(ceil_div(c->g_n0, p.qt) * c->g_n1, AMP_THREADS);

    // (per-particle split: capping the chunks so that the (8 + n_kinds) planes per chunk stay within 0.3 GB -- 46 chunks
    // instead of 148 on C3 -- was tried: DRAM writes 1.96 -> 1.66 GB only (the reductions of the object flushes, not the
    // footprint, make them), 1 % slower: not kept)
    p.n_chunks = choose_chunks(c, n_qb, slots, units, 8.0 * (double)c->n_q * (split ? 8.0 + NMS_KIND_COUNT : p.interp ? 20.0 : 8.0), split ? 1 : 8, 2.0e9);
    p.n_qblocks = (int)n_qb; p.blocks_per_sm = occ;
    *plan = p;
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
    const size_t part_bytes = sizeof(double) * 8 * (size_t)c->n_q * n_chunks;
    const size_t form_bytes = sizeof(double) * (size_t)n_kinds * (size_t)c->n_q * n_chunks;
    if (nms_status st = ensure(c, c->part, part_bytes)) return st;
    if (plan.split) if (nms_status st = ensure(c, c->formpart, form_bytes)) return st;
    const int n_prim = c->g_n0 / 2 + 1;   // interpolating kernel: even lines, and one beyond the edge when n0 is even
    const size_t sb_bytes = sizeof(double) * 8 * (size_t)n_prim * (size_t)c->g_n1 * n_chunks;   // 8 planes
    if (plan.interp) {
        if (nms_status st = ensure(c, c->interp_sb, 2 * sb_bytes)) return st;    // A and B sets: 16 planes per chunk
        if (nms_status st = ensure(c, c->interp_spb, sb_bytes)) return st;
    }
    AmpArgs a;
    a.cells = (const Cell*)c->cells.p;
    a.tiles = (const TileMeta*)c->tile_meta.p;
    a.chunk_begin = plan.split ? (const int32_t*)c->chunk_begin.p : nullptr;
    a.n_tiles = (int)c->n_tiles;
    a.type = c->g_type; a.n0 = c->g_n0; a.n1 = c->g_n1; a.n_q = c->n_q;
    a.u0 = (const float*)c->u0.p; a.dq = c->g_dq; a.qc = (const double2*)c->qc.p; a.sc = (const double2*)c->sc.p;
    a.part = (double*)c->part.p; a.form = (double*)c->formpart.p;
    a.sb = (double*)c->interp_sb.p; a.spb = (double*)c->interp_spb.p; a.n_prim = n_prim;
    a.kinds = kinds_dev; a.n_kinds = n_kinds;
    a.rp.Px = c->P[0]; a.rp.Py = c->P[1]; a.rp.Pz = c->P[2]; a.rp.sN = c->sN; a.rp.sM = c->sM; a.rp.invV = c->invV;

    amp_kernel_t kern = pick_kernel(plan);
    const size_t smem = plan.variant == 8 ? 0 : plan.interp ? AMP_SMEM_INTERP : amp_smem_bytes(plan.qt, plan.nch, plan.split, plan.npoly != 0 && !plan.split);
    NMS_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    dim3 grid((unsigned)plan.n_qblocks, (unsigned)n_chunks);
    // the kernels accumulate into their chunk partials with reductions
    if (!plan.interp) NMS_CUDA(c, cudaMemsetAsync(c->part.p, 0, part_bytes, c->stream));   // (interp: written by the combine pass)
    if (plan.split) NMS_CUDA(c, cudaMemsetAsync(c->formpart.p, 0, form_bytes, c->stream));
    if (plan.interp) {
        NMS_CUDA(c, cudaMemsetAsync(c->interp_sb.p, 0, 2 * sb_bytes, c->stream));
        NMS_CUDA(c, cudaMemsetAsync(c->interp_spb.p, 0, sb_bytes, c->stream));
    }
    if (nms_status st = timer_begin(c, c->amp_timer)) return st;
    kern<<<grid, AMP_THREADS, smem, c->stream>>>(a);
    if (plan.interp) { launch_interp_combine(a, n_chunks, c->stream); c->launches += 1; }   // the odd lines, inside the timed region
    if (nms_status st = timer_end(c, c->amp_timer)) return st;
    c->launches += 1;
    NMS_CUDA(c, cudaGetLastError());
    c->variant_used = plan.variant; c->n_chunks_used = n_chunks; c->blocks_per_sm_used = plan.blocks_per_sm;
    c->qt_used = plan.qt; c->npoly_used = plan.npoly; c->nb_used = plan.nb; c->rec3_used = plan.rec3;
    c->interp_used = plan.interp ? 1 : 0;
    return NMS_OK;
}

}  // namespace nms
