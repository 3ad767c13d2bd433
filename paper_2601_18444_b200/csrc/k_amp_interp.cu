// k_amp_interp.cu -- a-2, accurate variant on equally spaced lines: every OTHER detector point of a line is generated,
// the points in between follow from the sums themselves.
//
// On a line of equally spaced abscissae (|q| of a polar grid, q_z of a Cartesian one; step d) the phasors of one cell at
// three consecutive points obey  z_{k-1} + z_{k+1} = 2 cos(delta) z_k,  delta = d p  (p: the cell's coordinate along the
// line's direction) -- the identity behind the three-term recurrence of the fast variant.  Chained forwards it amplifies
// the rounding of cos(delta) by n (n + 1), which is why the accurate variant generates its points
// by rotations: 4 FMA-pipe operations per point.  Read the other way, z_k = h (z_{k-1} + z_{k+1}) with h = 1 / (2 cos delta),
// it is an INTERPOLATION with no amplification as long as the step phase stays away from a quarter cycle (|delta| < 0.2
// cycle is checked on the host: h <= 1.62), and because the Fourier sums of Eq. 42-47 (L353-L368) are linear in the phasor
// it can be applied to the sums instead of the terms:
//
//   A_c(q_k) = sum_j w_cj z_k^j = B_c(q_{k-1}) + B_c(q_{k+1}),   B_c(q_m) = sum_j (h_j w_cj) z_m^j.
//
// So a thread generates only the EVEN points of its line (its "primaries": one exactly evaluated polynomial phasor, 4
// rotations by the doubled step alternating with 3 single three-term steps) and accumulates each primary twice -- with the weights w (set A: the amplitude at the
// primary itself) and with the weights h w (set B) -- and the odd points are the sums of their two neighbours' B sets.
// Per 16 detector points: 64 packed accumulations as before, but 4 rotations + 3 three-term steps instead of 15 rotations
// and 8 live phasors instead of 16 (13.4 -> 11.5 FMA-pipe cycles per pair).  The neighbour of a thread's last odd point belongs to another block, so
// both sets are flushed to compact chunk partials indexed by primary and k_interp_combine writes the detector-shaped
// partials afterwards (even lines: the A sets; odd lines: the sums of the neighbours' B sets; per chunk, the layout the other
// kernels fill: the epilogue is unchanged).  With an even number of lines the last line is odd
// and its upper neighbour is one more primary beyond the detector edge (the progression continues; only its B set is kept).
//
// Float-grid correction.  The kernel evaluates each thread's primaries on the exact progression a_k = g_b + 2 (k - k_b) d
// through the float abscissa g_b of its base; the float abscissae of the grid deviate from it by up to an ulp.  As in the
// other recurrence kernels (k_amplitude.cuh) the A sets are corrected at the flush, to first order, by that deviation times
// the projection p_0 of the tile's centre.  A B set serves two odd points, each with its own deviation, so it is flushed
// twice: as it is (SB, fp64 chunk partials like the A sets) and multiplied by p_0 (SPB: summed over the chunk's tiles in
// fp32 on chip, one flush per block -- it only carries a correction of ~1e-5 of the amplitude); the combine pass applies
// (target abscissa -/+ d - a_m) to SPB.
#include <type_traits>
#include "k_amplitude.cuh"

namespace nms {

constexpr int QP = 8;      // primaries per thread (16 detector points)
constexpr int QP_B = 4;    // the exactly evaluated one

// abscissa [cycles/nm] of line l of the grid; beyond the edge the progression continues
__device__ __forceinline__ double line_abscissa(const float* __restrict__ u0, int n0, double dq, int l)
{
    return l < n0 ? (double)u0[l] * INV_2PI : (double)u0[n0 - 1] * INV_2PI + (double)(l - (n0 - 1)) * dq;
}
// abscissa at which primary pr is evaluated: the progression through the base of its group
__device__ __forceinline__ double primary_abscissa(const float* __restrict__ u0, int n0, double dq, int pr)
{
    const int grp = pr / QP, k = pr % QP;
    return line_abscissa(u0, n0, dq, 2 * (grp * QP + QP_B)) + (double)(2 * (k - QP_B)) * dq;
}

__device__ __forceinline__ float rcp_refined(float x)   // 1 / x: MUFU.RCP and one Newton step (x in [0.6, 2])
{
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return fmaf(r, fmaf(-x, r, 1.0f), r);
}

template <int MODE>
__global__ void __launch_bounds__(AMP_THREADS, 2) k_amp_interp(const AmpArgs a)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    Cell* sC = reinterpret_cast<Cell*>(smem_raw);                                          // [2][STAGE_CELLS]
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw + 2 * STAGE_CELLS * sizeof(Cell));
    // fp64 sub-accumulators of the nuclear channel (k_amplitude.cuh, NSUB): [set A: 2 QP | set B: 2 QP][128]
    double* nacc = reinterpret_cast<double*>(smem_raw + AMP_SMEM_TILES);
    // sum over the chunk's tiles of p_0 x (set B of the tile), fp32: it only enters multiplied by the deviation of a float
    // abscissa from the progression (<= an ulp of q: a correction of ~1e-5 of the amplitude)   [QP * 8][128]
    float* spb_acc = reinterpret_cast<float*>(smem_raw + AMP_SMEM_TILES + 4 * QP * AMP_THREADS * sizeof(double));
#pragma unroll
    for (int r = 0; r < 8 * QP; ++r) spb_acc[r * AMP_THREADS + threadIdx.x] = 0.f;

    const int tid = threadIdx.x;
    const int chunk = blockIdx.y;
    int tile_beg, tile_end;
    chunk_range(a, tile_beg, tile_end);

    const int n_groups = (a.n_prim + QP - 1) / QP;
    int64_t slot = (int64_t)blockIdx.x * AMP_THREADS + tid;
    const bool valid = slot < (int64_t)n_groups * a.n1;
    if (!valid) slot = 0;
    const int grp = (int)(slot / a.n1), i1 = (int)(slot % a.n1);
    const int pr0 = grp * QP;

    // per-thread constants in cycles/nm (q' = q / 2 pi)
    double c0, c1 = 0.0;
    if (MODE == 0) { const double2 d = a.sc[i1]; c0 = d.x; c1 = d.y; }   // sin th, cos th (the same on every ring)
    else c0 = a.qc[i1].x * INV_2PI;                                       // q'_y (the same on every row)
    const double dq = a.dq * INV_2PI;
    const double gb = line_abscissa(a.u0, a.n0, dq, 2 * (pr0 + QP_B));
    const double g0 = gb + (double)(2 * (0 - QP_B)) * dq;   // abscissa of the thread's first primary
    (void)c1;
    const bool slim = __syncthreads_or(valid && a.n_prim - pr0 > 1) == 0;

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

    u64 accA[QP][4], accB[QP][4];   // per primary and channel: {sum w cos, sum w sin}, {sum h w cos, sum h w sin}

    for (int t = tile_beg; t < tile_end; ++t) {
        const int it = t - tile_beg;
        const int stage = it & 1;
        const TileMeta tm = a.tiles[t];
        const Cell* __restrict__ tC = sC + stage * STAGE_CELLS;
#pragma unroll
        for (int k = 0; k < QP; ++k)
#pragma unroll
            for (int r = 0; r < 4; ++r) { accA[k][r] = 0ull; accB[k][r] = 0ull; }
#pragma unroll
        for (int r = 0; r < 4 * QP; ++r) nacc[r * AMP_THREADS + tid] = 0.0;
        mbar_wait(&bar[stage], (uint32_t)((it >> 1) & 1));

        const int nc = tm.n_slots;
        // SLIM: no thread of the block has more than one primary to produce (the group that only holds the primary beyond
        // the detector edge): that primary is evaluated directly, no rotations, one A and one B set
        auto run = [&](auto slim_tag) {
            constexpr bool SLIM = decltype(slim_tag)::value;
            for (int j0 = 0; j0 < nc; j0 += NSUB_CELLS) {
                const int j1 = min(nc, j0 + NSUB_CELLS);
#pragma unroll 8
                for (int j = j0; j < j1; ++j) {
                    const double2 YZ = *reinterpret_cast<const double2*>(&tC[j].Y);
                    const float4 w = *reinterpret_cast<const float4*>(&tC[j].wN);
                    const double p = MODE == 0 ? fma(c1, YZ.y, c0 * YZ.x) : c0 * YZ.x;   // Eq. 41 / q; Cartesian: q'_y Y
                    const double pl = MODE == 0 ? p : YZ.y;                               // coordinate along the line
                    float cd, sd;                                                          // the step phasor of this cell
                    sincos_poly_half(__double2loint(fma(dq, pl, MAGIC)), cd, sd);
                    const float h = rcp_refined(cd + cd);
                    const float4 wh = make_float4(w.x * h, w.y * h, w.z * h, w.w * h);
                    if (SLIM) {
                        const u64 ph0 = phasor<true>(MODE == 0 ? fma(g0, p, MAGIC) : fma(g0, YZ.y, p) + MAGIC);
                        accumulate<4>(accA[0], w, ph0);
                        accumulate<4>(accB[0], wh, ph0);
                    } else {
                        const float c2 = fmaf(-2.f * sd, sd, 1.f), s2 = 2.f * sd * cd;     // ... and of the doubled step
                        u64 ph[QP];
                        ph[QP_B] = phasor<true>(MODE == 0 ? fma(gb, p, MAGIC) : fma(gb, YZ.y, p) + MAGIC);
                        // rotations alternate with SINGLE three-term steps z_{k+1} = 2 cos(2 delta) z_k - z_{k-1} (2 FFMA instead of 2 FMUL +
                    // 2 FFMA): a step whose two inputs come from the base and a rotation adds the rounding of 2 cos once and is
                    // not chained (two consecutive steps were measured: NM worst 9.8e-4 on the full C5 map against 6.5e-4 here)
                        const float t2 = c2 + c2;
                        ph[QP_B + 1] = rotate(ph[QP_B], c2, s2);
                        ph[QP_B - 1] = rotate(ph[QP_B], c2, -s2);
                        ph[QP_B + 2] = three_term(ph[QP_B + 1], ph[QP_B], t2);
                        ph[QP_B - 2] = three_term(ph[QP_B - 1], ph[QP_B], t2);
                        ph[QP_B + 3] = rotate(ph[QP_B + 2], c2, s2);
                        ph[QP_B - 3] = rotate(ph[QP_B - 2], c2, -s2);
                        ph[QP_B - 4] = three_term(ph[QP_B - 3], ph[QP_B - 2], t2);
#pragma unroll
                        for (int k = 0; k < QP; ++k) {
                            accumulate<4>(accA[k], w, ph[k]);
                            accumulate<4>(accB[k], wh, ph[k]);
                        }
                    }
                }
#pragma unroll
                for (int k = 0; k < (SLIM ? 1 : QP); ++k) {   // nuclear channel: fp32 sums of <= NSUB_CELLS cells into the fp64 sums
                    float cs, sn;
                    unpack2(accA[k][0], cs, sn);
                    nacc[(2 * k) * AMP_THREADS + tid] += (double)cs;
                    nacc[(2 * k + 1) * AMP_THREADS + tid] += (double)sn;
                    accA[k][0] = 0ull;
                    unpack2(accB[k][0], cs, sn);
                    nacc[(2 * QP + 2 * k) * AMP_THREADS + tid] += (double)cs;
                    nacc[(2 * QP + 2 * k + 1) * AMP_THREADS + tid] += (double)sn;
                    accB[k][0] = 0ull;
                }
            }
        };
        if (slim) run(std::true_type{}); else run(std::false_type{});

        __syncthreads();   // every thread is done with this stage: refill it while the flush runs
        if (tid == 0 && t + 2 < tile_end) issue_tile(a, t + 2, sC + stage * STAGE_CELLS, &bar[stage]);

        // ---- flush: fp32 tile sums -> fp64 chunk partials (RED.ADD.F64 into zeroed block-private slots) ----------
        const double p0 = MODE == 0 ? fma(c1, tm.Z0, c0 * tm.Y0) : tm.Z0;
        const float p0f = (float)p0;
        const int64_t n_pq = (int64_t)a.n_prim * a.n1;
        // both sets go to COMPACT partials indexed by primary ([chunk][A: 8 planes | B: 8 planes][n_prim n1]): writing the A
        // sets straight into every other line of the detector-shaped partials made the L2 evict the lines under
        // reduction nine times over (11 GB of DRAM writes per C5 launch against 0.6 GB with either set alone)
        double* const pS = a.sb + (int64_t)chunk * 16 * n_pq + i1;     // + primary n1 + plane n_pq
#pragma unroll
        for (int k = 0; k < QP; ++k) {
            const int pr = pr0 + k, line = 2 * pr;
            if (!valid || pr >= a.n_prim) continue;
            double A[8], B[8];
            A[0] = nacc[(2 * k) * AMP_THREADS + tid];
            A[1] = nacc[(2 * k + 1) * AMP_THREADS + tid];
            B[0] = nacc[(2 * QP + 2 * k) * AMP_THREADS + tid];
            B[1] = nacc[(2 * QP + 2 * k + 1) * AMP_THREADS + tid];
#pragma unroll
            for (int w = 1; w < 4; ++w) {
                float cs, sn;
                unpack2(accA[k][w], cs, sn); A[2 * w] = (double)cs; A[2 * w + 1] = (double)sn;
                unpack2(accB[k][w], cs, sn); B[2 * w] = (double)cs; B[2 * w + 1] = (double)sn;
            }
            if (line < a.n0) {   // set A: the amplitude at the primary, corrected to its float abscissa
                double* q = pS + (int64_t)pr * a.n1;
                double eps = 0.0;
                if (k != QP_B) eps = 6.283185307179586 * ((double)a.u0[line] * INV_2PI - (gb + (double)(2 * (k - QP_B)) * dq)) * p0;
#pragma unroll
                for (int w = 0; w < 4; ++w) {
                    const double cs = fma(-eps, A[2 * w + 1], A[2 * w]);          // cos(psi + eps), sin(psi + eps)
                    const double sn = fma(eps, A[2 * w], A[2 * w + 1]);
                    atomicAdd(q, cs); q += n_pq;         // Re: + sum w cos (Eq. 44, 46)
                    atomicAdd(q, -sn); q += n_pq;        // Im: - sum w sin (Eq. 45, 47)
                }
            }
            double* q = pS + 8 * n_pq + (int64_t)pr * a.n1;
#pragma unroll
            for (int w = 0; w < 4; ++w) {   // set B as (Re, Im) = (sum cos, - sum sin); times p_0: fp32 sums on chip
                atomicAdd(q, B[2 * w]); q += n_pq;
                atomicAdd(q, -B[2 * w + 1]); q += n_pq;
                float* sp = spb_acc + ((k * 4 + w) * 2) * AMP_THREADS + tid;
                sp[0] = fmaf(p0f, (float)B[2 * w], sp[0]);
                sp[AMP_THREADS] = fmaf(p0f, (float)B[2 * w + 1], sp[AMP_THREADS]);
            }
        }
    }
    // the p_0-weighted B sets of the whole chunk, once per block
#pragma unroll
    for (int k = 0; k < QP; ++k) {
        const int pr = pr0 + k;
        if (!valid || pr >= a.n_prim) continue;
        const int64_t n_pq = (int64_t)a.n_prim * a.n1, fp = (int64_t)pr * a.n1 + i1;
#pragma unroll
        for (int w = 0; w < 4; ++w) {
            const float* sp = spb_acc + ((k * 4 + w) * 2) * AMP_THREADS + tid;
            atomicAdd(a.spb + ((int64_t)chunk * 8 + 2 * w) * n_pq + fp, (double)sp[0]);
            atomicAdd(a.spb + ((int64_t)chunk * 8 + 2 * w + 1) * n_pq + fp, -(double)sp[AMP_THREADS]);
        }
    }
}

// The detector-shaped chunk partials from the compact ones, per chunk: an even line is the A set of its primary; an odd
// line is the sum of the B sets of its two neighbouring primaries.  A neighbour m was evaluated at the abscissa a_m; the
// identity needs it at (float abscissa of the odd line) -/+ d: the difference enters to first order through the
// p_0-weighted sums, (Re, Im) -> (Re + e Im, Im - e Re) summed over tiles with e = 2 pi (difference) p_0 (the rule of the
// flush in k_amplitude.cuh, written for (Re, Im) = (sum cos, - sum sin)).
__global__ void k_interp_combine(double* __restrict__ part, const double* __restrict__ sb, const double* __restrict__ spb,
                                 const float* __restrict__ u0, double dq_rad, int n0, int n1, int n_prim, int64_t n_q)
{
    const int64_t f = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (f >= n_q) return;
    const int chunk = blockIdx.y;
    const int line = (int)(f / n1), i1 = (int)(f % n1);
    const int64_t n_pq = (int64_t)n_prim * n1;
    const int m = line >> 1;
    const int64_t f_lo = (int64_t)m * n1 + i1, f_hi = f_lo + n1;
    if (!(line & 1)) {
        const double* sa = sb + (int64_t)chunk * 16 * n_pq + f_lo;
#pragma unroll
        for (int r = 0; r < 8; ++r) part[((int64_t)chunk * 8 + r) * n_q + f] = sa[r * n_pq];
        return;
    }
    const double dq = dq_rad * INV_2PI;
    const double gk = (double)u0[line] * INV_2PI;
    const double e_lo = 6.283185307179586 * ((gk - dq) - primary_abscissa(u0, n0, dq, m));
    const double e_hi = 6.283185307179586 * ((gk + dq) - primary_abscissa(u0, n0, dq, m + 1));
#pragma unroll
    for (int w = 0; w < 4; ++w) {
        const double* sre = sb + ((int64_t)chunk * 16 + 8 + 2 * w) * n_pq;
        const double* sim = sre + n_pq;
        const double* pre = spb + ((int64_t)chunk * 8 + 2 * w) * n_pq;
        const double* pim = pre + n_pq;
        const double re = fma(e_lo, pim[f_lo], sre[f_lo]) + fma(e_hi, pim[f_hi], sre[f_hi]);
        const double im = fma(-e_lo, pre[f_lo], sim[f_lo]) + fma(-e_hi, pre[f_hi], sim[f_hi]);
        part[((int64_t)chunk * 8 + 2 * w) * n_q + f] = re;
        part[((int64_t)chunk * 8 + 2 * w + 1) * n_q + f] = im;
    }
}

amp_kernel_t amp_kernel_interp(int mode)
{
    return mode == 0 ? (amp_kernel_t)k_amp_interp<0> : (amp_kernel_t)k_amp_interp<1>;
}

void launch_interp_combine(const AmpArgs& a, int n_chunks, cudaStream_t stream)
{
    const int64_t n = a.n_q;
    dim3 grid((unsigned)((n + 255) / 256), (unsigned)n_chunks);
    k_interp_combine<<<grid, 256, 0, stream>>>(a.part, a.sb, a.spb, a.u0, a.dq, a.n0, a.n1, a.n_prim, a.n_q);
}

}  // namespace nms
