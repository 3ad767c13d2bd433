// k_amplitude.cu -- a-2 (and a-6): the direct sums of Eq. 42-47 (L353-L368) on the FP32, FP64 and XU pipes.
//
//   A_c(q) = sum_j w_cj exp(-i Psi_j(q)),  Psi_j = q_y Y_j + q_z Z_j  (Eq. 41),  c in {N, x, y, z}.
//
// Work decomposition: grid = (detector blocks) x (cell chunks).  A block owns 128*QT detector points
// (thread = one position along the fast detector index i1 and QT consecutive positions along i0) and
// walks the tiles of its chunk.  Tiles (<= TILE = 256 Cell records of 32 B) are brought into shared memory by
// one elected thread with cp.async.bulk + mbarrier, double buffered; every lane of a warp reads the same
// record (2 LDS.128 broadcasts per cell, no bank conflicts).
//
// Arithmetic per (cell, detector point) -- B200 has three independent pipes that all get work:
//   FP64 pipe : the phase in CYCLES, t = (q/2pi).r, by DFMA with the addend 1.5*2^20: the sum is rounded
//               to a multiple of 2^-32, so the low mantissa word of the result is frac(t) * 2^32 as a
//               two's-complement integer in [-1/2, 1/2) cycle, whatever the magnitude of t -- the
//               "t - rint(t)" reduction of the north star, done by the rounding of the adder, with no fp32
//               phase rounding and no tile origins;
//   conversion: one I2FP turns that word into a float (|error| <= 2^-25 cycle = 1.9e-7 rad);
//   XU pipe   : sin.approx / cos.approx of x = 2 pi frac in [-pi, pi) (absolute error 2^-21.4, CUDA C
//               Programming Guide), written into an aligned register pair {cos, sin};
//   FP32 pipe : 4 packed fma.rn.f32x2 per pair, one per weight channel: {w, w} * {cos, sin} + {Re, -Im},
//               the weight as a 32-bit broadcast operand (an FFMA2 with three 64-bit register operands
//               was measured at 3 cycles instead of 2: register-file bandwidth).
//               A complex accumulator is ONE 64-bit register pair, so a detector point costs 8 registers
//               and a thread with QT = 8 points needs 64 accumulator registers: 4 blocks of 128 threads
//               per SM (16 warps) instead of 2, which is what hides the MUFU / FP64 / LDS latencies.
// Accumulators are fp32 over one tile only (<= 256 additions); at the end of a tile they are added to
// fp64 chunk partials in global memory (block-private slots, plain read-modify-write, deterministic).
// The epilogue kernel sums the chunks and forms the responses.
//
// Phase variants (MODE): how t is formed for the thread's QT points
//   0  polar   : p = sin(th) Y + cos(th) Z per (cell, thread) [2 fp64 ops], t_k = q'_k p + magic [1 per pair]
//   1  cart.   : u = q'_y Y per (cell, thread) [1], t_k = (q'_z,k Z + u) + magic [2 per pair]
//   2  list    : t_k = (q'_z,k Z + q'_y,k Y) + magic [3 per pair]
//
// Line recurrence (NB > 0; north star (b): "advanced by a complex-rotation recurrence ... with periodic
// resync").  The direct path is bound by the XU pipe (2 MUFU per pair at 16 lanes/clk/SM = 8 pairs/clk/SM).
// Where the abscissa along the thread's line is equally spaced (u0[k] = u0[0] + k d: |q| of a polar grid,
// q_z of a Cartesian one) the phases of a thread's QT points form an arithmetic progression with the step
// d' * p (polar) or d' * Z (Cartesian) per cell.  The QT points are cut into NB segments; the phasor of one
// point per segment (its "base") is evaluated exactly as above -- the resync, at EVERY cell -- and the
// others are reached from it by at most ceil((QT/NB - 1)/2) complex rotations with the step phasor
// (cos, sin of the exactly reduced step phase, one evaluation per cell and thread), forwards or backwards
// (conjugate step).  A rotation is 2 FMUL + 2 FFMA, so a pair costs 12 FP32 lane-operations and the MUFU
// load drops from 2 to (NB + 1) * 2 / QT per pair.  Error: a point s steps from its base carries (s + 1)
// MUFU errors (2^-21.4 each) and s fp32 roundings, and the deviation of the fp32 abscissae from the exact
// progression (<= 1 ulp of q, checked on the host) enters as a phase error <= ulp(q) * |r|; both are
// measured against the oracle in tests/test_gpu_parity.py.
#include "nms_internal.h"
#include "nms_response.cuh"

namespace nms {

constexpr int AMP_THREADS = 128;
constexpr int STAGE_CELLS = TILE;

typedef unsigned long long u64;

constexpr double MAGIC = 1572864.0;                 // 1.5 * 2^20: ulp = 2^-32 (needs |t| < 2^19 cycles)
constexpr double INV_2PI = 0.15915494309189533577;

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

__device__ __forceinline__ void issue_tile(const AmpArgs& a, int tile, Cell* dst, uint64_t* bar)
{
    const TileMeta tm = a.tiles[tile];
    const uint32_t bytes = (uint32_t)tm.n_slots * (uint32_t)sizeof(Cell);
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    mbar_expect_tx(bar, bytes);
    bulk_g2s(dst, a.cells + tm.first_slot, bytes, bar);
}

// ---- packed fp32x2 arithmetic (sm_100 PTX; SASS FFMA2) -------------------------------------------
__device__ __forceinline__ u64 pack2(float lo, float hi)
{
    u64 d;
    asm("mov.b64 %0, {%1, %2};" : "=l"(d) : "f"(lo), "f"(hi));
    return d;
}
__device__ __forceinline__ void unpack2(u64 v, float& lo, float& hi)
{
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ u64 ffma2(u64 a, u64 b, u64 c)
{
    u64 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ u64 fmul2(u64 a, u64 b)
{
    u64 d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}

// The low word of m holds frac(t) * 2^32 as a signed integer (t = phase in cycles, see MAGIC).  One I2FP
// (24 significant bits: |error| <= 2^-25 cycle) and one multiply give x = 2 pi frac in [-pi, pi); the
// phasor {cos x, sin x} comes back as one packed register pair.  (sin.approx / cos.approx multiply x by
// fl(1 / 2 pi) again -- FMUL.RZ, then MUFU on cycles; PTX offers no entry point that skips it.  A relative
// error of the phase SCALE acts like q -> q (1 + eps), a coherent error of 2 eps q L in the cross sections;
// measured against the oracle the net scale of this chain is 1 - 1e-8, small enough.)
__device__ __forceinline__ u64 phasor(double m)
{
    const float TWO_PI_2M32 = 0x1.921fb6p-30f;   // fl(2 pi) * 2^-32
    const float x = __int2float_rn(__double2loint(m)) * TWO_PI_2M32;
    return pack2(__cosf(x), __sinf(x));
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

// Add the sums Ap[8] of one tile at detector point f to the fp64 chunk partials (block-private slots, plain
// read-modify-write).  SPLIT (a-6, Eq. 49-50): ppart carries the running amplitudes of the
// current object across its tiles; when the object is complete its responses B(A_p, A_p) go to the form
// accumulators and A_p to the total amplitudes.
template <bool SPLIT>
__device__ __forceinline__ void flush_point(const AmpArgs& a, int chunk, int64_t f, double (&Ap)[8], bool first,
                                            bool p_first, bool p_last, bool first_total)
{
    if (!SPLIT) {
        // fire-and-forget reductions (RED.ADD.F64, no round trip to the thread); the slots are block-private
        // and zeroed before the launch, so every address sees its additions in tile order: deterministic
        (void)first;
#pragma unroll
        for (int r = 0; r < 8; ++r) atomicAdd(a.part + ((int64_t)chunk * 8 + r) * a.n_q + f, Ap[r]);
    } else {
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            double* pp = a.ppart + ((int64_t)chunk * 8 + r) * a.n_q + f;
            if (!p_first) Ap[r] += *pp;
            if (!p_last) *pp = Ap[r];
        }
        if (p_last) {
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

__device__ __forceinline__ void chunk_range(const AmpArgs& a, int& tile_beg, int& tile_end)
{
    const int chunk = blockIdx.y;   // chunk boundaries: a table in split mode (object boundaries), else equal parts
    if (a.chunk_begin) { tile_beg = a.chunk_begin[chunk]; tile_end = a.chunk_begin[chunk + 1]; }
    else {
        tile_beg = (int)(((int64_t)a.n_tiles * chunk) / gridDim.y);
        tile_end = (int)(((int64_t)a.n_tiles * (chunk + 1)) / gridDim.y);
    }
}

// ---- exact variant: everything in fp64 -----------------------------------------------------------
// One thread per detector point, cells read straight from global memory (every lane of a block reads the
// same record: L1 broadcast).  Phase t = (q/2pi).r in fp64, reduced exactly to [-1/2, 1/2] cycle, sincospi
// and the 8 accumulations in fp64.  ~50 fp64 operations per pair: 7x slower than the fp32 kernels, chosen
// automatically only for small problems (launch-bound anyway), where it makes the result exact to the
// fp32 rounding of the rotated weights.  See DESIGN.md section 7 (precision policy).
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
    bool first_total = true;
    for (int t = tile_beg; t < tile_end; ++t) {
        const TileMeta tm = a.tiles[t];
        const Cell* __restrict__ tC = a.cells + tm.first_slot;
        double Ap[8];
#pragma unroll
        for (int r = 0; r < 8; ++r) Ap[r] = 0.0;
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
        const bool p_first = SPLIT ? ((tm.flags & 2) != 0) : false;
        const bool p_last = SPLIT ? ((tm.flags & 1) != 0) : false;
        flush_point<SPLIT>(a, chunk, f, Ap, t == tile_beg, p_first, p_last, first_total);
        if (SPLIT && p_last) first_total = false;
    }
}

// Segment b of the NB segments of a thread's QT points: [lo, hi], exactly evaluated at kb.
template <int QT, int NB> struct Seg {
    static __device__ __forceinline__ constexpr int lo(int b) { return (b * QT) / NB; }
    static __device__ __forceinline__ constexpr int hi(int b) { return ((b + 1) * QT) / NB - 1; }
    static __device__ __forceinline__ constexpr int kb(int b) { return lo(b) + (hi(b) - lo(b) + 1) / 2; }
};

// NB = 0: direct evaluation of every pair; NB > 0: line recurrence with NB exactly evaluated points per QT
template <int MODE, int QT, bool SPLIT, int MINB, int NB, int NCH>
__global__ void __launch_bounds__(AMP_THREADS, MINB) k_amp(const AmpArgs a)
{
    static_assert(NB == 0 || (MODE != 2 && NB <= QT), "the recurrence needs a line of equally spaced abscissae");
    extern __shared__ __align__(128) unsigned char smem_raw[];
    Cell* sC = reinterpret_cast<Cell*>(smem_raw);                                          // [2][STAGE_CELLS]
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw + 2 * STAGE_CELLS * sizeof(Cell));

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
    const int grp = (int)(slot / a.n1), i1 = (int)(slot % a.n1);
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
        if (MODE == 0) {
            g[k] = (double)a.u0[i0 + kk] * INV_2PI;
            h[k] = 0.0;
        } else {
            const double2 q = a.qc[flat0 + (int64_t)kk * a.n1];
            g[k] = q.y * INV_2PI;      // q'_z
            h[k] = q.x * INV_2PI;      // q'_y
        }
    }
    if (MODE == 0) { const double2 d = a.sc[flat0]; c0 = d.x; c1 = d.y; }
    if (MODE == 1) c0 = h[0];
    (void)c1;
    const double dq = a.dq * INV_2PI;   // recurrence: spacing of the line in cycles/nm
    constexpr int NBX = NB > 0 ? NB : 1;
    typedef Seg<QT, NBX> S;
    double gb[NBX];                     // abscissae of the exactly evaluated points
    if (NB > 0) {                       // points beyond the detector edge continue the progression (never stored)
#pragma unroll
        for (int k = 1; k < QT; ++k)
            if (k >= kclamp) g[k] += (double)(k - (kclamp - 1)) * dq;   // g[k] was clamped to g[kclamp - 1]
    }
#pragma unroll
    for (int b = 0; b < NBX; ++b) gb[b] = g[S::kb(b)];

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
    bool first_total = true;   // SPLIT: no object of this chunk has been completed yet

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
#pragma unroll 8
        for (int j = 0; j < nc; ++j) {
            const double2 YZ = *reinterpret_cast<const double2*>(&tC[j].Y);
            const float4 w = *reinterpret_cast<const float4*>(&tC[j].wN);
            double p = 0.0;
            if (MODE == 0) p = fma(c1, YZ.y, c0 * YZ.x);   // Eq. 41 / q
            if (MODE == 1) p = c0 * YZ.x;
            if (NB == 0) {
                u64 ph[QT];
#pragma unroll
                for (int k = 0; k < QT; ++k) {
                    double m;
                    if (MODE == 0) m = fma(g[k], p, MAGIC);
                    else if (MODE == 1) m = fma(g[k], YZ.y, p) + MAGIC;
                    else m = fma(g[k], YZ.y, h[k] * YZ.x) + MAGIC;
                    ph[k] = phasor(m);
                }
#pragma unroll
                for (int k = 0; k < QT; ++k) accumulate<NCH>(acc[k], w, ph[k]);
            } else {
                // step phasor of this cell: phase step dq' p (polar) or dq' Z (Cartesian), exactly reduced
                float cd, sd;
                unpack2(phasor(fma(dq, MODE == 0 ? p : YZ.y, MAGIC)), cd, sd);
                u64 pb[NBX];
#pragma unroll
                for (int b = 0; b < NBX; ++b)
                    pb[b] = phasor(MODE == 0 ? fma(gb[b], p, MAGIC) : fma(gb[b], YZ.y, p) + MAGIC);
#pragma unroll
                for (int b = 0; b < NBX; ++b) {
                    accumulate<NCH>(acc[S::kb(b)], w, pb[b]);
                    u64 ph = pb[b];
#pragma unroll
                    for (int k = S::kb(b) + 1; k <= S::hi(b); ++k) {
                        ph = rotate(ph, cd, sd);
                        accumulate<NCH>(acc[k], w, ph);
                    }
                    ph = pb[b];
#pragma unroll
                    for (int k = S::kb(b) - 1; k >= S::lo(b); --k) {
                        ph = rotate(ph, cd, -sd);
                        accumulate<NCH>(acc[k], w, ph);
                    }
                }
            }
        }

        __syncthreads();   // every thread is done with this stage: refill it while the flush runs
        if (tid == 0 && t + 2 < tile_end) issue_tile(a, t + 2, sC + stage * STAGE_CELLS, &bar[stage]);

        // ---- flush: add the fp32 tile sums to the fp64 chunk partials -----------------------------
        const bool first = (t == tile_beg);
        const bool p_first = SPLIT ? ((tm.flags & 2) != 0) : false;
        const bool p_last = SPLIT ? ((tm.flags & 1) != 0) : false;
#pragma unroll
        for (int k = 0; k < QT; ++k) {
            if (k < kmax) {
                const int64_t f = flat0 + (int64_t)k * a.n1;
                double Ap[8];
#pragma unroll
                for (int w = 0; w < 4; ++w) {
                    float cs = 0.f, sn = 0.f;
                    if (w < NCH) unpack2(acc[k][w % NCH], cs, sn);
                    Ap[2 * w] = (double)cs;          // Re: + sum w cos(Psi)   (Eq. 44, 46)
                    Ap[2 * w + 1] = -(double)sn;     // Im: - sum w sin(Psi)   (Eq. 45, 47)
                }
                flush_point<SPLIT>(a, chunk, f, Ap, first, p_first, p_last, first_total);
            }
        }
        if (SPLIT && p_last) first_total = false;
    }
}

// ---- host side: planning and dispatch ------------------------------------------------------------
constexpr size_t AMP_SMEM = 2 * STAGE_CELLS * sizeof(Cell) + 2 * sizeof(uint64_t);

typedef void (*amp_kernel_t)(const AmpArgs);

template <int MODE, int QT, int MINB, int NB>
static amp_kernel_t pick_split(bool split, bool nuclear_only)
{
    if (nuclear_only)
        return split ? (amp_kernel_t)k_amp<MODE, QT, true, MINB, NB, 1> : (amp_kernel_t)k_amp<MODE, QT, false, MINB, NB, 1>;
    return split ? (amp_kernel_t)k_amp<MODE, QT, true, MINB, NB, 4> : (amp_kernel_t)k_amp<MODE, QT, false, MINB, NB, 4>;
}

template <int MODE>
static amp_kernel_t pick_rec(int qt, int nb, bool split, bool nuc)
{
    // one channel leaves room for 16 points per thread: the phasor set-up per pair halves (bases stay <= 2 steps away)
    if (qt == 16) return split ? (amp_kernel_t)k_amp<MODE, 16, true, 4, 4, 1> : (amp_kernel_t)k_amp<MODE, 16, false, 4, 4, 1>;
    switch (nb) {
    case 1: return pick_split<MODE, 8, 4, 1>(split, nuc);
    case 3: return pick_split<MODE, 8, 4, 3>(split, nuc);
    case 4: return pick_split<MODE, 8, 4, 4>(split, nuc);
    default: return pick_split<MODE, 8, 4, 2>(split, nuc);
    }
}

// variant: 1 list direct, 2 polar direct, 4 cartesian direct, 3 polar recurrence, 5 cartesian recurrence
// (all with fp32 accumulation over a tile), 8 exact (fp64); nuc: the sample has no magnetic channel
static amp_kernel_t pick_kernel(int variant, int qt, int nb, bool split, bool nuc)
{
    switch (variant) {
    case 1: return pick_split<2, 4, 4, 0>(split, nuc);
    case 2:
        if (qt == 4) return pick_split<0, 4, 4, 0>(split, nuc);
        return pick_split<0, 8, 4, 0>(split, nuc);
    case 4:
        if (qt == 4) return pick_split<1, 4, 4, 0>(split, nuc);
        return pick_split<1, 8, 4, 0>(split, nuc);
    case 3: return pick_rec<0>(qt, nb, split, nuc);
    case 5: return pick_rec<1>(qt, nb, split, nuc);
    default: return split ? (amp_kernel_t)k_amp_f64<true> : (amp_kernel_t)k_amp_f64<false>;
    }
}

static int64_t ceil_div(int64_t a, int64_t b) { return (a + b - 1) / b; }

nms_status plan_amplitude(nms_ctx* c, bool split, AmpPlan* plan)
{
    // precision policy: small problems run the exact fp64 kernel; otherwise the line
    // recurrence where the thread lines are equally spaced, else the direct kernel
    int variant;
    const bool small = (double)c->W * (double)c->n_q <= 1073741824.0;
    const bool line_ok = c->g_type != 2 && c->g_uniform && c->g_n0 >= 2;
    if (c->opt_variant == 2 && !line_ok)
        return fail(c, NMS_E_UNSUPPORTED, "the line-recurrence variant needs a polar or Cartesian detector with equally spaced u0");
    if (c->opt_variant == 3 || (c->opt_variant == 0 && small)) variant = 8;
    else if (c->g_type == 2) variant = 1;
    else if (c->opt_variant == 2 || (c->opt_variant == 0 && line_ok)) variant = (c->g_type == 0) ? 3 : 5;
    else variant = (c->g_type == 0) ? 2 : 4;

    // units of work along the cell dimension: tiles, or whole objects in split mode
    const int64_t units = split ? c->K : c->n_tiles;
    int dev_slots_guess = c->sm_count * 3;
    // q points per thread: the largest that still yields enough blocks to fill the device
    int qt_opts[3]; int n_opts = 0;
    if (variant == 8) { qt_opts[n_opts++] = 1; }
    else if (variant == 1) { qt_opts[n_opts++] = 4; }
    else if (variant == 3 || variant == 5) { if (!c->has_M && c->opt_bases == 0) qt_opts[n_opts++] = 16; qt_opts[n_opts++] = 8; }
    else { qt_opts[n_opts++] = 8; qt_opts[n_opts++] = 4; }
    int qt = qt_opts[n_opts - 1];
    if (c->opt_qt && variant != 8) {
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
    const size_t smem = variant == 8 ? 0 : AMP_SMEM;
    amp_kernel_t kern = pick_kernel(variant, qt, c->opt_bases, split, !c->has_M);
    NMS_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)AMP_SMEM));
    int occ = 0;
    NMS_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, AMP_THREADS, smem));
    if (occ < 1) return fail(c, NMS_E_CUDA, "amplitude kernel does not fit on an SM");
    const int64_t slots = (int64_t)c->sm_count * occ;
    const int64_t n_qb = variant == 8 ? ceil_div(c->n_q, AMP_THREADS)
                                      : ceil_div(ceil_div(c->g_n0, qt) * c->g_n1, AMP_THREADS);

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
    a.cells = (const Cell*)c->cells.p;
    a.tiles = (const TileMeta*)c->tile_meta.p;
    a.chunk_begin = plan.split ? (const int32_t*)c->chunk_begin.p : nullptr;
    a.n_tiles = (int)c->n_tiles;
    a.type = c->g_type; a.n0 = c->g_n0; a.n1 = c->g_n1; a.n_q = c->n_q;
    a.u0 = (const float*)c->u0.p; a.dq = c->g_dq; a.qc = (const double2*)c->qc.p; a.sc = (const double2*)c->sc.p;
    a.part = (double*)c->part.p; a.ppart = (double*)c->ppart.p; a.form = (double*)c->formpart.p;
    a.kinds = kinds_dev; a.n_kinds = n_kinds;
    a.rp.Px = c->P[0]; a.rp.Py = c->P[1]; a.rp.Pz = c->P[2]; a.rp.sN = c->sN; a.rp.sM = c->sM; a.rp.invV = c->invV;

    amp_kernel_t kern = pick_kernel(plan.variant, plan.qt, c->opt_bases, plan.split, !c->has_M);
    NMS_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)AMP_SMEM));
    dim3 grid((unsigned)plan.n_qblocks, (unsigned)n_chunks);
    if (!plan.split)   // the kernel accumulates into its chunk partials with reductions
        NMS_CUDA(c, cudaMemsetAsync(c->part.p, 0, sizeof(double) * 8 * (size_t)c->n_q * n_chunks, c->stream));
    timer_begin(c, NMS_T_AMPLITUDE);
    kern<<<grid, AMP_THREADS, plan.variant == 8 ? 0 : AMP_SMEM, c->stream>>>(a);
    timer_end(c, NMS_T_AMPLITUDE);
    c->launches += 1;
    NMS_CUDA(c, cudaGetLastError());
    c->variant_used = plan.variant; c->n_chunks_used = n_chunks; c->blocks_per_sm_used = plan.blocks_per_sm;
    c->qt_used = plan.qt;
    return NMS_OK;
}

}  // namespace nms
