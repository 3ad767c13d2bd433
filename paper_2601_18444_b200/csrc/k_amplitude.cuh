// k_amplitude.cuh -- a-2 (and a-6): the direct sums of Eq. 42-47 (L353-L368) on the FP32, FP64 and XU pipes.
// Kernel templates; instantiated in k_amp_direct.cu, k_amp_rec_polar.cu, k_amp_rec_cart.cu (three translation
// units so that the build runs in parallel) and dispatched from k_amplitude.cu.
//
//   A_c(q) = sum_j w_cj exp(-i Psi_j(q)),  Psi_j = q_y Y_j + q_z Z_j  (Eq. 41),  c in {N, x, y, z}.
//
// Work decomposition: grid = (detector blocks) x (cell chunks).  A block owns 128*QT detector points
// (thread = one position along the fast detector index i1 and QT consecutive positions along i0) and
// walks the tiles of its chunk.  Tiles (<= TILE = 256 Cell records of 32 B) are brought into shared memory by
// one elected thread with cp.async.bulk + mbarrier, double buffered; every lane of a warp reads the same
// record (2 LDS.128 broadcasts per cell, no bank conflicts).
//
// Arithmetic per (cell, detector point):
//   FP64 pipe : the phase in CYCLES by one DFMA with the addend MAGIC (nms_phasor.cuh): exact t - rint(t);
//   phasor    : phasor<false> (MUFU, XU pipe) or phasor<true> (polynomial, FMA + ALU pipes), nms_phasor.cuh;
//   FP32 pipe : 4 packed fma.rn.f32x2 per pair, one per weight channel: {w, w} * {cos, sin} + {Re, -Im},
//               the weight as a 32-bit broadcast operand.  A complex accumulator is ONE 64-bit register pair:
//               8 registers per detector point, 64 at QT = 8, 4 blocks of 128 threads per SM.
// Accumulators are fp32 over one tile only (<= 256 additions); at the end of a tile they are added to fp64
// chunk partials in global memory (RED.ADD.F64 into zeroed block-private slots: deterministic order per address).
//
// Phase variants (MODE): how t is formed for the thread's QT points
//   0  polar   : p = sin(th) Y + cos(th) Z per (cell, thread) [2 fp64 ops], t_k = q'_k p + magic [1 per pair]
//   1  cart.   : u = q'_y Y per (cell, thread) [1], t_k = (q'_z,k Z + u) + magic [2 per pair]
//   2  list    : t_k = (q'_z,k Z + q'_y,k Y) + magic [3 per pair]
//
// Direct kernels (NB = 0): every pair gets its own phasor: by MUFU (2 per pair: the XU pipe caps the kernel at
// 8 pairs/clk/SM), or, NPOLY = QT, by the polynomial phasor (the accurate variant, no MUFU at all).
//
// Line recurrence (NB > 0; north star (b): "advanced by a complex-rotation recurrence ... with periodic resync").
// Where the abscissa along the thread's line is equally spaced (|q| of a polar grid, q_z of a Cartesian one) the
// phases of a thread's QT points form an arithmetic progression with the step d' * p (polar) or d' * Z (Cartesian)
// per cell.  The QT points are cut into NB segments; one point per segment (its "base") is evaluated exactly --
// the resync, at EVERY cell -- and so is the step phasor (cd, sd).  The other points follow
//   REC3 = 0: by complex rotations from the base, forwards and backwards (2 FMUL + 2 FFMA per pair);
//   REC3 = 1: one rotation gives the base's neighbour, then the three-term recurrence
//             z_{k+1} = 2 cd z_k - z_{k-1} outwards on both sides (2 FFMA per pair).  An error e of cd enters a
//             point n steps from the exact pair as n (n + 1) e, so the runs are kept short (<= 3 steps).
// The abscissae of a float grid are NOT an exact progression (each is rounded to fp32): the kernel evaluates the
// line g_b + (k - k_b) d and corrects the tile sums at the flush, to first order, by the phase
// 2 pi (g_k - g_b - (k - k_b) d) p_0 with p_0 the projection of the tile's centre (TileMeta::Y0, Z0); what is left
// is that deviation times the extent of the tile (zero when the cells of a tile share (Y, Z)).
#pragma once
#include "nms_internal.h"
#include "nms_phasor.cuh"
#include "nms_response.cuh"

namespace nms {

constexpr int AMP_THREADS = 128;
constexpr int STAGE_CELLS = TILE;

struct AmpArgs {
    const Cell* cells;
    const TileMeta* tiles;
    const int32_t* chunk_begin;   // [n_chunks+1] or NULL (equal parts of n_tiles)
    int n_tiles;
    int type, n0, n1;
    int64_t n_q;
    const float* u0;
    double dq;           // recurrence kernels: spacing of u0 [rad/nm] (fp64, (u0[n0-1] - u0[0]) / (n0 - 1))
    const double2* qc;   // (q_y, q_z) [rad/nm] fp64
    const double2* sc;   // (sin th, cos th)
    double* part;        // [n_chunks][8][n_q]
    double* form;        // split: [n_chunks][n_kinds][n_q]
    double* sb;          // k_amp_interp: A and B sets of the primaries [n_chunks][8 + 8][n_prim * n1] ...
    double* spb;         // ... and the B sets weighted with the projection of the tile centres [n_chunks][8][n_prim * n1]
    int n_prim;          // k_amp_interp: primaries (even lines, one more beyond the edge when n0 is even) per line
    const int32_t* kinds;
    int n_kinds;
    RespParams rp;
};

typedef void (*amp_kernel_t)(const AmpArgs);

// shared memory of the fp32 kernels: two tile stages, two mbarriers, and in split mode the fp32 running
// amplitudes of the current object (QT * 2 * NCH floats per thread)
constexpr size_t AMP_SMEM_TILES = 2 * STAGE_CELLS * sizeof(Cell) + 2 * sizeof(uint64_t);
// ... and in the accurate non-split kernels the fp64 sub-accumulators of the nuclear channel (QT * 2 doubles per thread)
constexpr int NSUB_CELLS = 32;   // 16: 0.552 of the roofline on C5, worst signed-kind error 6.7e-4; 32: 0.566, 7.3e-4
constexpr size_t amp_smem_bytes(int qt, int nch, bool split, bool nsub)
{
    return AMP_SMEM_TILES + (split ? (size_t)qt * 2 * nch * AMP_THREADS * sizeof(float) : 0) +
           (nsub ? (size_t)qt * 2 * AMP_THREADS * sizeof(double) : 0);
}

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

__device__ __forceinline__ void issue_tile(const AmpArgs& a, int tile, Cell* dst, uint64_t* bar)
{
    const TileMeta tm = a.tiles[tile];
    const uint32_t bytes = (uint32_t)tm.n_slots * (uint32_t)sizeof(Cell);
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    mbar_expect_tx(bar, bytes);
    bulk_g2s(dst, a.cells + tm.first_slot, bytes, bar);
}

// ---- packed fp32x2 arithmetic (sm_100 PTX; SASS FFMA2) -------------------------------------------
__device__ __forceinline__ u64 ffma2(u64 a, u64 b, u64 c)
{
    u64 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}

// NCH packed accumulations of one (cell, detector point): acc[c] += {w_c, w_c} * {cos, sin}.  The pack of a
// register with itself compiles to the broadcast operand form (FFMA2 Rd, Rw.F32, Rph, Racc): no extra move.
// NCH = 4: nuclear + three magnetic channels; NCH = 1: nuclear only (sample without moments -- the activation
// switch of L242 -- and the pixel sums of the two-dimensional correlation function).
template <int NCH>
__device__ __forceinline__ void accumulate(u64 (&acc)[NCH], const float4& w, u64 ph)
{
    acc[0] = ffma2(pack2(w.x, w.x), ph, acc[0]);
    if (NCH > 1) {
        acc[1 % NCH] = ffma2(pack2(w.y, w.y), ph, acc[1 % NCH]);
        acc[2 % NCH] = ffma2(pack2(w.z, w.z), ph, acc[2 % NCH]);
        acc[3 % NCH] = ffma2(pack2(w.w, w.w), ph, acc[3 % NCH]);
    }
}

// Advance the phase of the phasor {c, s} by the step whose phasor is (cd, sd): {c cd - s sd, s cd + c sd}.
// The backward rotation passes (cd, -sd).  2 FMUL + 2 FFMA.
__device__ __forceinline__ u64 rotate(u64 ph, float cd, float sd)
{
    float c, s;
    unpack2(ph, c, s);
    return pack2(fmaf(c, cd, -(s * sd)), fmaf(c, sd, s * cd));
}
// Three-term step: z_next = 2 cd z - z_prev, per component (2 FFMA).
__device__ __forceinline__ u64 three_term(u64 z, u64 zprev, float two_cd)
{
    float c, s, cp, sp;
    unpack2(z, c, s);
    unpack2(zprev, cp, sp);
    return pack2(fmaf(two_cd, c, -cp), fmaf(two_cd, s, -sp));
}

__device__ __forceinline__ void chunk_range(const AmpArgs& a, int& tile_beg, int& tile_end)
{
    const int chunk = blockIdx.y;   // chunk boundaries: a table in split mode (object boundaries), else equal parts
    if (a.chunk_begin) { tile_beg = a.chunk_begin[chunk]; tile_end = a.chunk_begin[chunk + 1]; }
    else {
        tile_beg = (int)(((int64_t)a.n_tiles * chunk) / gridDim.y);
        tile_end = (int)(((int64_t)a.n_tiles * (chunk + 1)) / gridDim.y);
    }
}

// Add the complete amplitudes Ap[8] of one object at detector point f to the chunk's totals, and its responses
// B(A_p, A_p) to the chunk's form accumulators (a-6, Eq. 49-50).  Reductions into zeroed slots that
// belong to this thread alone: every address sees its additions in object order.
__device__ __forceinline__ void flush_object(const AmpArgs& a, int chunk, int64_t f, const double (&Ap)[8])
{
    const double2 d = a.sc[f];
    double val[NMS_KIND_COUNT];
    responses_at_point(Ap, d.x, d.y, a.rp, val);
    for (int i = 0; i < a.n_kinds; ++i)
        atomicAdd(a.form + ((int64_t)chunk * a.n_kinds + i) * a.n_q + f, val[a.kinds[i]]);
#pragma unroll
    for (int r = 0; r < 8; ++r) atomicAdd(a.part + ((int64_t)chunk * 8 + r) * a.n_q + f, Ap[r]);
}

// Segment b of the NB segments of a thread's QT points: [lo, hi], exactly evaluated at kb.
template <int QT, int NB> struct Seg {
    static __device__ __forceinline__ constexpr int lo(int b) { return (b * QT) / NB; }
    static __device__ __forceinline__ constexpr int hi(int b) { return ((b + 1) * QT) / NB - 1; }
    static __device__ __forceinline__ constexpr int kb(int b) { return lo(b) + (hi(b) - lo(b) + 1) / 2; }
    // exactly evaluated point: the middle (rotations both ways) or, for the three-term recurrence, the lower of the
    // two middle points (its upper neighbour follows by one rotation)
    static __device__ __forceinline__ constexpr int base(int b, bool rec3) { return rec3 ? lo(b) + (hi(b) - lo(b)) / 2 : kb(b); }
};

// NB = 0: direct evaluation of every pair (NPOLY of the QT phasors by polynomial, the others by MUFU);
// NB > 0: line recurrence with NB exactly evaluated points per QT (NPOLY != 0: bases and step by polynomial),
//         REC3 = 1: three-term recurrence instead of rotations.
// UNI: the launch guarantees n1 % 128 == 0, so a block lies inside ONE group of QT lines: the line abscissae are then
//      block-uniform values (derived from blockIdx only), which frees the 2 QT registers a thread needs for them.
// QT = 16 with four channels: 128 accumulator registers, built with MINB = 2 (255 registers, 8 warps per SM); measured on C5
//      against QT = 8 at 128 registers and 16 warps per SM: fast variant 0.805 -> 0.857 of the roofline, accurate 0.566 -> 0.634.
// SH:  polynomial recurrence kernels only: the step phase stays within a quarter cycle (checked on the host: d r_max <
//      pi / 2), so the step phasor needs no quadrant logic (sincos_poly_half).
template <int MODE, int QT, bool SPLIT, int MINB, int NB, int NCH, int NPOLY, int REC3, bool UNI = false, bool SH = false>
__global__ void __launch_bounds__(AMP_THREADS, MINB) k_amp(const AmpArgs a)
{
    static_assert(NB == 0 || (MODE != 2 && NB <= QT), "the recurrence needs a line of equally spaced abscissae");
    extern __shared__ __align__(128) unsigned char smem_raw[];
    Cell* sC = reinterpret_cast<Cell*>(smem_raw);                                          // [2][STAGE_CELLS]
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw + 2 * STAGE_CELLS * sizeof(Cell));
    float* obj = reinterpret_cast<float*>(smem_raw + AMP_SMEM_TILES);                       // split: [QT*2*NCH][128]
    // Accurate variant (polynomial phasors), nuclear channel: its weights are typically uniform (N_j = const inside the
    // sample), so a tile whose cells share one phase (an x-row of a lattice: q_x = 0) adds the SAME number 256 times and
    // the fp32 roundings drift instead of averaging out (measured: rms error of C5's nuclear amplitude 0.14 against 0.011
    // with fp64 accumulation -- all of the remaining north-star misses of NM).  Every NSUB_CELLS cells the nuclear
    // accumulators are therefore moved into fp64 sums in shared memory.
    constexpr bool NSUB = NPOLY != 0 && !SPLIT;
    double* nacc = reinterpret_cast<double*>(smem_raw + AMP_SMEM_TILES);                    // NSUB: [QT*2][128]

    const int tid = threadIdx.x;
    const int chunk = blockIdx.y;
    int tile_beg, tile_end;
    chunk_range(a, tile_beg, tile_end);

    // ---- this thread's detector points ---------------------------------------------------------
    const int n_groups = (a.n0 + QT - 1) / QT;
    const int64_t n_slots_q = (int64_t)n_groups * a.n1;
    int64_t slot = (int64_t)blockIdx.x * AMP_THREADS + tid;
    const bool valid = slot < n_slots_q;
    if (!valid) slot = 0;
    int grp, i1;
    if (UNI) {
        const int bpg = a.n1 / AMP_THREADS;            // blocks per group of QT lines
        grp = (int)blockIdx.x / bpg;
        i1 = ((int)blockIdx.x % bpg) * AMP_THREADS + tid;
    } else {
        grp = (int)(slot / a.n1);
        i1 = (int)(slot % a.n1);
    }
    const int i0 = grp * QT;
    const int kmax = valid ? min(QT, a.n0 - i0) : 0;
    const int kclamp = max(min(QT, a.n0 - i0), 1);
    const int64_t flat0 = (int64_t)i0 * a.n1 + i1;

    // per-thread constants in cycles/nm (q' = q / 2 pi)
    double c0 = 0.0, c1 = 0.0;     // MODE 0: sin th, cos th;  MODE 1: q'_y
    double g[QT], h[QT];           // MODE 0: q'_k;  MODE 1: q'_z,k;  MODE 2: q'_y,k and q'_z,k
#pragma unroll
    for (int k = 0; k < QT; ++k) {
        const int kk = min(k, kclamp - 1);
        if (MODE == 0 || (MODE == 1 && UNI)) {
            g[k] = (double)a.u0[i0 + kk] * INV_2PI;                          // |q|'_k, or q'_z,k of a Cartesian line
            h[k] = MODE == 1 ? a.qc[flat0].x * INV_2PI : 0.0;                // q'_y
        } else {
            const double2 q = a.qc[flat0 + (int64_t)kk * a.n1];
            g[k] = q.y * INV_2PI;      // q'_z
            h[k] = q.x * INV_2PI;      // q'_y
        }
    }
    // keep the abscissae as opaque fp64 values: where registers are short the compiler otherwise re-derives them from
    // the float grid inside the cell loop (F2F.F64.F32 + DMUL per point and iteration -- F2F runs on the XU pipe, the
    // very pipe the direct kernels are bound by: measured 4.7 % of its capacity in the per-particle kernel)
#pragma unroll
    for (int k = 0; k < QT; ++k) {
        asm volatile("" : "+d"(g[k]));
        if (MODE == 2) asm volatile("" : "+d"(h[k]));
    }
    if (MODE == 0) { const double2 d = a.sc[flat0]; c0 = d.x; c1 = d.y; }
    if (MODE == 1) c0 = h[0];
    (void)c1;
    const double dq = a.dq * INV_2PI;   // recurrence: spacing of the line in cycles/nm
    constexpr int NBX = NB > 0 ? NB : 1;
    typedef Seg<QT, NBX> S;
    double gb[NBX];                     // abscissae of the exactly evaluated points
#pragma unroll
    for (int b = 0; b < NBX; ++b) {     // a base beyond the detector edge continues the progression (never stored)
        const int kb = S::base(b, REC3 != 0);
        gb[b] = g[kb];
        if (NB > 0 && kb >= kclamp) gb[b] += (double)(kb - (kclamp - 1)) * dq;   // g[kb] was clamped to g[kclamp - 1]
    }

    if (tid == 0) {
        mbar_init(&bar[0], 1);
        mbar_init(&bar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (tid == 0) {
        if (tile_beg < tile_end) issue_tile(a, tile_beg, sC, &bar[0]);
        if (tile_beg + 1 < tile_end) issue_tile(a, tile_beg + 1, sC + STAGE_CELLS, &bar[1]);
    }

    u64 acc[QT][NCH];          // per point and channel: {sum w cos, sum w sin}

    for (int t = tile_beg; t < tile_end; ++t) {
        const int it = t - tile_beg;
        const int stage = it & 1;
        const TileMeta tm = a.tiles[t];
        const Cell* __restrict__ tC = sC + stage * STAGE_CELLS;
#pragma unroll
        for (int k = 0; k < QT; ++k)
#pragma unroll
            for (int r = 0; r < NCH; ++r) acc[k][r] = 0ull;
        mbar_wait(&bar[stage], (uint32_t)((it >> 1) & 1));

        const int nc = tm.n_slots;
        auto cell = [&](int j) {
            const double2 YZ = *reinterpret_cast<const double2*>(&tC[j].Y);
            const float4 w = *reinterpret_cast<const float4*>(&tC[j].wN);
            double p = 0.0;
            if (MODE == 0) p = fma(c1, YZ.y, c0 * YZ.x);   // Eq. 41 / q
            if (MODE == 1) p = c0 * YZ.x;
            u64 ph[QT];
            if (NB == 0) {
#pragma unroll
                for (int k = 0; k < QT; ++k) {
                    double m;
                    if (MODE == 0) m = fma(g[k], p, MAGIC);
                    else if (MODE == 1) m = fma(g[k], YZ.y, p) + MAGIC;
                    else m = fma(g[k], YZ.y, h[k] * YZ.x) + MAGIC;
                    ph[k] = (k < NPOLY) ? phasor<true>(m) : phasor<false>(m);
                }
            } else {
                // step phasor of this cell: phase step dq' p (polar) or dq' Z (Cartesian), exactly reduced
                float cd, sd;
                if (SH) sincos_poly_half(__double2loint(fma(dq, MODE == 0 ? p : YZ.y, MAGIC)), cd, sd);
                else unpack2(phasor<(NPOLY != 0)>(fma(dq, MODE == 0 ? p : YZ.y, MAGIC)), cd, sd);
                const float two_cd = cd + cd;
#pragma unroll
                for (int b = 0; b < NBX; ++b) {
                    const int kb = S::base(b, REC3 != 0);
                    ph[kb] = phasor<(NPOLY != 0)>(MODE == 0 ? fma(gb[b], p, MAGIC) : fma(gb[b], YZ.y, p) + MAGIC);
                    if (REC3) {
                        if (S::hi(b) > kb) ph[kb + 1] = rotate(ph[kb], cd, sd);
#pragma unroll
                        for (int k = kb + 2; k <= S::hi(b); ++k) ph[k] = three_term(ph[k - 1], ph[k - 2], two_cd);
#pragma unroll
                        for (int k = kb - 1; k >= S::lo(b); --k) ph[k] = three_term(ph[k + 1], ph[k + 2], two_cd);
                    } else if (QT / NBX >= 16) {
                        // long segments: two interleaved chains per direction, advanced by the squared step phasor
                        // (half the depth of the dependency chain and of the accumulated rotation roundings)
                        const float c2 = fmaf(-2.f * sd, sd, 1.f), s2 = 2.f * sd * cd;
                        if (S::hi(b) > kb) ph[kb + 1] = rotate(ph[kb], cd, sd);
                        if (S::lo(b) < kb) ph[kb - 1] = rotate(ph[kb], cd, -sd);
#pragma unroll
                        for (int k = kb + 2; k <= S::hi(b); ++k) ph[k] = rotate(ph[k - 2], c2, s2);
#pragma unroll
                        for (int k = kb - 2; k >= S::lo(b); --k) ph[k] = rotate(ph[k + 2], c2, -s2);
                    } else {
#pragma unroll
                        for (int k = kb + 1; k <= S::hi(b); ++k) ph[k] = rotate(ph[k - 1], cd, sd);
#pragma unroll
                        for (int k = kb - 1; k >= S::lo(b); --k) ph[k] = rotate(ph[k + 1], cd, -sd);
                    }
                }
            }
#pragma unroll
            for (int k = 0; k < QT; ++k) accumulate<NCH>(acc[k], w, ph[k]);
        };
        if (!NSUB) {
#pragma unroll 8
            for (int j = 0; j < nc; ++j) cell(j);
        } else {
#pragma unroll
            for (int r = 0; r < 2 * QT; ++r) nacc[r * AMP_THREADS + tid] = 0.0;
            for (int j0 = 0; j0 < nc; j0 += NSUB_CELLS) {
                const int j1 = min(nc, j0 + NSUB_CELLS);
#pragma unroll 8
                for (int j = j0; j < j1; ++j) cell(j);
#pragma unroll
                for (int k = 0; k < QT; ++k) {
                    float cs, sn;
                    unpack2(acc[k][0], cs, sn);
                    nacc[(2 * k) * AMP_THREADS + tid] += (double)cs;
                    nacc[(2 * k + 1) * AMP_THREADS + tid] += (double)sn;
                    acc[k][0] = 0ull;
                }
            }
        }

        __syncthreads();   // every thread is done with this stage: refill it while the flush runs
        if (tid == 0 && t + 2 < tile_end) issue_tile(a, t + 2, sC + stage * STAGE_CELLS, &bar[stage]);

        // ---- flush: add the fp32 tile sums to the fp64 chunk partials -----------------------------
        const bool p_first = SPLIT ? ((tm.flags & 2) != 0) : false;
        const bool p_last = SPLIT ? ((tm.flags & 1) != 0) : false;
        double p0 = 0.0;                                   // projection of the tile centre (recurrence correction)
        if (NB > 0) p0 = MODE == 0 ? fma(c1, tm.Z0, c0 * tm.Y0) : tm.Z0;
#pragma unroll
        for (int b = 0; b < NBX; ++b) {
#pragma unroll
            for (int k = S::lo(b); k <= S::hi(b); ++k) {
                if (k < kmax) {
                    const int64_t f = flat0 + (int64_t)k * a.n1;
                    float eps = 0.f;
                    if (NB > 0 && k != S::base(b, REC3 != 0)) {
                        // the float abscissa of point k against the evaluated progression, as a phase at the tile centre
                        const double gk = MODE == 0 ? (double)a.u0[i0 + k] * INV_2PI : a.qc[f].y * INV_2PI;
                        eps = (float)(6.283185307179586 * (gk - (gb[b] + (double)(k - S::base(b, REC3 != 0)) * dq)) * p0);
                    }
                    double Ap[8];
#pragma unroll
                    for (int w = 0; w < 4; ++w) {
                        float cs = 0.f, sn = 0.f;
                        if (NSUB && w == 0) {              // the nuclear tile sums are the fp64 sub-accumulators
                            const double dc = nacc[(2 * k) * AMP_THREADS + tid], ds = nacc[(2 * k + 1) * AMP_THREADS + tid];
                            Ap[0] = fma(-(double)eps, ds, dc);
                            Ap[1] = -fma((double)eps, dc, ds);
                            continue;
                        }
                        if (w < NCH) {
                            unpack2(acc[k][w % NCH], cs, sn);
                            if (NB > 0) {                  // cos(psi + eps), sin(psi + eps) to first order
                                const float c2 = fmaf(-eps, sn, cs);
                                sn = fmaf(eps, cs, sn);
                                cs = c2;
                            }
                            if (SPLIT) {                   // fp32 running amplitudes of the current object, on chip
                                float* oc = obj + ((k * NCH + w) * 2) * AMP_THREADS + tid;
                                if (!p_first) { cs += oc[0]; sn += oc[AMP_THREADS]; }
                                if (!p_last) { oc[0] = cs; oc[AMP_THREADS] = sn; }
                            }
                        }
                        Ap[2 * w] = (double)cs;          // Re: + sum w cos(Psi)   (Eq. 44, 46)
                        Ap[2 * w + 1] = -(double)sn;     // Im: - sum w sin(Psi)   (Eq. 45, 47)
                    }
                    if (!SPLIT) {
                        // fire-and-forget reductions (RED.ADD.F64); the slots are block-private and zeroed before the
                        // launch, so every address sees its additions in tile order: deterministic
#pragma unroll
                        for (int r = 0; r < 2 * NCH; ++r) atomicAdd(a.part + ((int64_t)chunk * 8 + r) * a.n_q + f, Ap[r]);
                    } else if (p_last) {
                        flush_object(a, chunk, f, Ap);
                    }
                }
            }
        }
    }
}

// k_amp_interp: the sub-accumulators of both sets (as amp_smem_bytes(16, 4, false, true)) and the fp32 p_0-weighted B sums
constexpr size_t AMP_SMEM_INTERP = amp_smem_bytes(16, 4, false, true) + (size_t)64 * AMP_THREADS * sizeof(float);

// lookup functions of the three instantiation units (NULL if the combination is not built)
amp_kernel_t amp_kernel_direct(int mode, int qt, bool split, int nch, int npoly, bool uni);
amp_kernel_t amp_kernel_rec_polar(int qt, int nb, bool split, int nch, bool poly, bool rec3, bool uni, bool sh);
amp_kernel_t amp_kernel_rec_cart(int qt, int nb, bool split, int nch, bool poly, bool rec3, bool uni, bool sh);
// k_amp_interp.cu: the accurate variant that generates every other point of a line (mode 0 polar, 1 Cartesian), and the
// pass that forms the points in between from the B sets
amp_kernel_t amp_kernel_interp(int mode);
void launch_interp_combine(const AmpArgs& a, int n_chunks, cudaStream_t stream);

}  // namespace nms
