/*
 * nms.h -- C ABI of the B200-native direct-summation SANS core
 * (data-parallel hot path of arxiv/paper_2601_18444, "NuMagSANS").
 *
 * Citations "Lnnn"/"Eq. n" refer to /root/reference/PAPER.md; "reading n" to
 * DESIGN.md section 3.  Everything behind this header is hand-written CUDA for
 * sm_100a in paper_2601_18444_b200/csrc/; there is no CPU fallback: without a
 * CUDA device nms_create() fails with NMS_E_CUDA.
 *
 * General conventions
 *  - Pointers are tagged [dev] (device memory, caller-owned, e.g. a torch tensor's
 *    data_ptr()) or [host].  The library never frees or keeps a caller pointer:
 *    nms_set_sample() copies what it needs into context-owned device storage.
 *  - Every call only ENQUEUES work on the context's CUDA stream (given to
 *    nms_create; 0 = legacy default stream).  Results are valid after
 *    nms_synchronize() or a stream synchronisation by the caller.  The *_host
 *    entry point is the exception: it synchronises before returning.
 *  - Errors: return code + nms_last_error(); no exceptions, no abort, no stdout.
 *    Argument errors are detected before any launch and leave the context usable.
 *  - Units: positions nm, q nm^-1 (L393), r nm (L404); only q.r must be dimensionless.
 *  - Geometry (Fig. 1 L33, Eq. 6): beam along x, detector in the y-z plane,
 *    q = (0, q_y, q_z) = q (0, sin th, cos th), th measured from +z towards +y.
 *  - Amplitude planes, in this order: Re N~, Im N~, Re M~x, Im M~x, Re M~y, Im M~y,
 *    Re M~z, Im M~z; they are the RAW sums of Eq. 42-47 (L353-L368) without the
 *    (2 pi)^-3/2 or (W N)^-1/2 prefactors (reading 4); the imaginary parts carry the
 *    minus sign of e^{-i q.r} (Eq. 45, 47).
 */
#ifndef NMS_H_
#define NMS_H_

#include <stdint.h>

#if defined(__GNUC__)
#define NMS_API __attribute__((visibility("default")))
#else
#define NMS_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef struct nms_ctx nms_ctx;

typedef enum {
    NMS_OK = 0,
    NMS_E_ARG = 1,          /* bad argument (NULL, non-positive size, unknown kind, non-orthonormal R, ...) */
    NMS_E_STATE = 2,        /* call order violated (e.g. nms_response before nms_amplitudes) */
    NMS_E_CUDA = 3,         /* CUDA runtime error or no usable device; text in nms_last_error() */
    NMS_E_NOMEM = 4,        /* host or device allocation failed */
    NMS_E_UNSUPPORTED = 5
} nms_status;

/* The 13 base response functions of Section II (L35-L174), all real, per detector point.
 * With N = sN N~, M = sM M~, q^ = (0, sin th, cos th), Q = q^ x (q^ x M) (Eq. 5, Eq. 7),
 * Pi = P.Q, every kind is multiplied by invV (see nms_set_scales):                              */
typedef enum {
    NMS_NUC = 0,        /* |N|^2                         Eq. 3  L48  */
    NMS_MAG = 1,        /* |Q|^2                         Eq. 4  L50  */
    NMS_UNPOL = 2,      /* NUC + MAG = (PP+MM+PM+MP)/2   Eq. 27-28 */
    NMS_PROJ = 3,       /* |Pi|^2                        Eq. 8  L66  */
    NMS_NM = 4,         /* P.(N Q* + N* Q) = 2 Re(N Pi*) Eq. 18 */
    NMS_SF = 5,         /* MAG - PROJ                    Eq. 13  */
    NMS_CHI = 6,        /* -i P.(Q x Q*)                 Eq. 14  */
    NMS_PM = 7,         /* (+-) = SF + CHI               Eq. 11  */
    NMS_MP = 8,         /* (-+) = SF - CHI               Eq. 12  */
    NMS_PP = 9,         /* (++) = NUC + NM + PROJ        Eq. 16 */
    NMS_MM = 10,        /* (--) = NUC - NM + PROJ        Eq. 17 */
    NMS_POL_PLUS = 11,  /* (+) = PP + PM                 Eq. 23 */
    NMS_POL_MINUS = 12, /* (-) = MM + MP                 Eq. 24 */
    NMS_KIND_COUNT = 13
} nms_kind;

/* Detector grid.  The abscissa arrays are HOST arrays (they are tiny and the library analyses
 * them on the host to pick the kernel variant); they are copied during the call.
 *  type 0 polar     : u0 = |q| [n0], u1 = theta [n1] (radians); q_y = q sin th, q_z = q cos th (L343),
 *                     evaluated in fp64 from the float values.
 *  type 1 cartesian : u0 = q_z [n0], u1 = q_y [n1]; theta = atan2(q_y, q_z), theta(0,0) = 0 (reading 5).
 *  type 2 list      : u0 = q_y [n0], u1 = q_z [n0], n1 must be 1; theta as for cartesian.
 * Flat detector index = i0 * n1 + i1 (i1 fastest); n_q = n0 * n1.                                 */
typedef struct {
    int type;
    int n0, n1;
    const float* u0;   /* [host] */
    const float* u1;   /* [host] */
} nms_qgrid;

/* Kernels whose device time nms_kernel_time_ms() can report (CUDA events on the context stream). */
typedef enum {
    NMS_T_PREP = 0,         /* a-1 rotate + pack                                    */
    NMS_T_AMPLITUDE = 1,    /* a-2 direct sums (also the a-6 per-particle variant)  */
    NMS_T_EPILOGUE = 2,     /* a-3 reduce + responses                               */
    NMS_T_AZIMUTHAL = 3,    /* a-4                                                  */
    NMS_T_CORRELATION = 4,  /* a-5                                                  */
    NMS_T_MODAL = 5,        /* f-2 angular modal decomposition                      */
    NMS_T_CORR2D = 6,       /* f-1 two-dimensional correlation function (its amplitude kernel) */
    NMS_T_BATCH = 7,        /* f-3 amplitude kernel of the batched magnetisation fields */
    NMS_T_COUNT = 8
} nms_timer;

/* ---- context ---------------------------------------------------------------------------------- */

/* Create a context on CUDA device `device` that enqueues on `cuda_stream` (a cudaStream_t cast to
 * void*; NULL = default stream).  Fails with NMS_E_CUDA if no device is usable or the device is not
 * compute capability 10.x.  *out is NULL on failure.                                              */
NMS_API nms_status nms_create(nms_ctx** out, int device, void* cuda_stream);
/* Synchronise the stream and free everything the context owns.  NULL is allowed. */
NMS_API void nms_destroy(nms_ctx* ctx);
/* Text of the last error on this context ("" if none).  Valid until the next call on the context. */
NMS_API const char* nms_last_error(const nms_ctx* ctx);
/* Block until all work enqueued by this context has finished. */
NMS_API nms_status nms_synchronize(nms_ctx* ctx);

/* ---- sample (a-1, Eq. 37-41) --------------------------------------------------------- */

/* Define the real-space sample: W cells with positions pos [dev][W][3] (x,y,z), nuclear weights
 * N [dev][W] or NULL (nuclear channel absent, N~ = 0) and moments m [dev][W][3] or NULL (magnetic
 * channel absent) -- the activation switches of L242.  R [host][9] is the row-major sample rotation
 * (Eq. 37), NULL = identity; it must be orthonormal within 1e-6 (else NMS_E_ARG).  Positions AND
 * moments are rotated (reading 2): r' = R (x + r^k), m' = R m, in fp64, rounded once.  The arrays are
 * copied; they may be released once the stream has passed this call.  Resets particles to "none". */
NMS_API nms_status nms_set_sample(nms_ctx* ctx, const float* pos, const float* N, const float* m, int64_t W,
                          const double* R);
/* Optional object structure (L310-L317): offsets [host][K+1], offsets[0] = 0, non-decreasing,
 * offsets[K] = W; cells of object k are [offsets[k], offsets[k+1]).  centres [dev][K][3] are the
 * StructData positions r^k added to the local coordinates before rotation (Eq. 38-40), or NULL
 * (r^k = 0, L341).  K = 0 removes the structure.  Needed by nms_form_factor_split.              */
NMS_API nms_status nms_set_particles(nms_ctx* ctx, const int64_t* offsets, int64_t K, const float* centres);
/* Change the rotation only (rocking scans): re-runs the prep pass on the stored sample. */
NMS_API nms_status nms_set_rotation(nms_ctx* ctx, const double* R);
/* Polarisation direction P [host][3] (L64, L272); normalised on input; default (0,0,1). */
NMS_API nms_status nms_set_polarization(nms_ctx* ctx, const double* P);
/* Scale factors (reading 4): N = sN N~, M = sM M~, every response is multiplied by invV.  Defaults 1.
 * Absolute units of the paper: sN = N_s V_cell, sM = b_H M_s V_cell, invV = 1/V (Eq. 48).   */
NMS_API nms_status nms_set_scales(nms_ctx* ctx, double sN, double sM, double invV);

/* ---- amplitudes and responses (a-2, a-3) -------------------------------------------------------- */

/* Direct sums A_c(q) = sum_j w_cj exp(-i q.r'_j) for every detector point (Eq. 42-47).  The result
 * is kept in the context (fp64) for nms_response; if out_amp [dev][8][n_q] (float) is not NULL the
 * eight planes are also written there.  The grid becomes the context's current grid.             */
NMS_API nms_status nms_amplitudes(nms_ctx* ctx, const nms_qgrid* grid, float* out_amp);
/* Response maps out [dev][n_kinds][n_q] (float) from the amplitudes of the last nms_amplitudes call
 * (NMS_E_STATE if there was none since the last sample change).                                  */
NMS_API nms_status nms_response(nms_ctx* ctx, const nms_kind* kinds, int n_kinds, float* out);
/* Fourier cross-correlation components of the magnetisation (f-4, Eq. 51-52) from the amplitudes of the
 * last nms_amplitudes call (NMS_E_STATE if there was none since the last sample change):
 *   G_ab = invV sM^2 M~_a M~_b^*,  a, b in (x, y, z),  out_GR = Re G, out_GI = Im G, each [dev][9][n_q] (float) with
 * row 3 a + b; either may be NULL (not both).  G^R is symmetric, G^I antisymmetric.                      */
NMS_API nms_status nms_cross_spectra(nms_ctx* ctx, float* out_GR, float* out_GI);
/* Fused a-2 + a-3: amplitudes and all requested responses without materialising the amplitudes.
 * This is the call bench.py times.  out [dev][n_kinds][n_q] (float).                             */
NMS_API nms_status nms_compute(nms_ctx* ctx, const nms_qgrid* grid, const nms_kind* kinds, int n_kinds, float* out);

/* ---- batched magnetisation fields on a fixed geometry (f-3; the paper's loop mode L254, L323, L391, L686) -------- */

/* n_fields magnetisation fields m_batch [dev][n_fields][W][3] on the geometry of the current sample (positions, N, object
 * centres and rotation as set by nms_set_sample / nms_set_particles / nms_set_rotation; the sample's own m is not used).
 * The phasors and the nuclear sum are evaluated once per group of 3 fields and shared; field b gets the same results as
 * nms_set_sample(pos, N, m_batch[b]) + nms_compute would give.  out_maps [dev][n_fields][n_kinds][n_q] (float) or NULL;
 * out_amp [dev][n_fields][8][n_q] (float, plane order as nms_amplitudes; planes 0-1 are the shared nuclear amplitude) or
 * NULL (not both NULL).  fp32 kernels at every problem size, fast or accurate variant by the "precision" rule below;
 * the accurate variant runs a line recurrence over 8 points per thread where u0 is equally spaced and the cell order
 * spatially coherent; otherwise (fast variant, list detectors, "variant" 1) the direct kernel with 4 points per thread;
 * "variant" 2 forces the recurrence (NMS_E_UNSUPPORTED without equally spaced lines).                                 */
NMS_API nms_status nms_compute_batch(nms_ctx* ctx, const nms_qgrid* grid, const float* m_batch, int n_fields,
                             const nms_kind* kinds, int n_kinds, float* out_maps, float* out_amp);

/* ---- azimuthal average (a-4, Eq. 30) ------------------------------------------------------ */

/* Average maps [dev][n_maps][n_q] (float) over the azimuth on the context's current grid.
 *  - polar grid and q_hi <= q_lo: n_bins must equal n0; bin i is ring i, value = arithmetic mean
 *    over theta (periodic trapezoid, reading 7), abscissa q_i, count n1.
 *  - otherwise: n_bins uniform bins on [q_lo, q_hi): bin = floor((|q|-q_lo)/(q_hi-q_lo)*n_bins) in
 *    fp64 exactly in this order with |q| = sqrt(q_y^2+q_z^2); points outside are dropped; value =
 *    mean of the members; empty bins give 0 with count 0; abscissa = bin centre (reading 8).
 * out_I [dev][n_maps][n_bins] (float); out_q [dev][n_bins] (float) or NULL; out_count
 * [dev][n_bins] (int32) or NULL.                                                                 */
NMS_API nms_status nms_azimuthal_average(nms_ctx* ctx, const float* maps, int n_maps, int n_bins, double q_lo,
                                 double q_hi, float* out_I, float* out_q, int32_t* out_count);
/* The |q|-histogram mode of nms_azimuthal_average (q_hi > q_lo, any grid type; Eq. 30, reading 8) for callers that
 * cannot allocate device memory (CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc): same
 * arguments, same results (counts identical, averages equal up to the order of the fp64 additions), but the call
 * allocates and frees nothing.  Its scratch -- per-bin counts and per-(map, bin) fp64 sums -- is one static device array
 * of 576 KB inside libnms.so, held by every GPU that loads the library until the process exits.  Limits: n_bins <= 16384
 * and n_maps * n_bins <= 65536 (NMS_E_UNSUPPORTED beyond them); q_hi <= q_lo (the ring mode, which uses no scratch) is
 * NMS_E_ARG.  The first call on a device resolves the array's address (cudaGetSymbolAddress): make it outside any graph
 * capture.  Every call on a device shares the array, and it keeps the last call's contents: each call clears what it uses
 * on the context's stream first; calls that overlap on the GPU (two streams, two contexts) RACE -- serialise them.
 * Asynchronous on the context's stream like the other calls.                                                          */
NMS_API nms_status nms_azimuthal_average_noalloc(nms_ctx* ctx, const float* maps, int n_maps, int n_bins, double q_lo,
                                         double q_hi, float* out_I, float* out_q, int32_t* out_count);

/* ---- angular modal decomposition (f-2, Eq. 31-33) -------------------------------------- */

/* Sine and cosine harmonics of maps [dev][n_maps][n_q] (float) on the context's current grid, which must be
 * polar with theta_j = 2 pi j / n1 (reading 7; NMS_E_UNSUPPORTED otherwise): for k = 0..k_max (k_max <= 63)
 *   I_k^{s,c}(q_i) = (2 - delta_k0) / n1 * sum_j f(q_i, theta_j) {sin, cos}(k theta_j)      (Eq. 31, trapezoid L183)
 *   a_k^{s,c} = sum_i I_k^{s,c}(q_i)                                                        (Eq. 32)
 *   A_k^{s,c} = a_k^{s,c} / sum_{j=0..k_max} sqrt(a_j^s^2 + a_j^c^2)   (0 if that sum is 0) (Eq. 33)
 * in fp64, outputs rounded once to float.  out_Is, out_Ic [dev][n_maps][k_max+1][n0]; out_a, out_A
 * [dev][n_maps][2][k_max+1] with index 0 = sine, 1 = cosine.  Any output may be NULL (not all).        */
NMS_API nms_status nms_modal_decomposition(nms_ctx* ctx, const float* maps, int n_maps, int k_max, float* out_Is,
                                   float* out_Ic, float* out_a, float* out_A);

/* ---- correlation function (a-5, Eq. 34-35) -------------------------------------------- */

/* c(r_k) = (1/2pi^2) trapz_q[ I(q) j0(q r_k) q^2 ], p(r_k) = r_k^2 c(r_k), for each of n_maps curves
 * I [dev][n_maps][n_bins] (float) on abscissae q_of_bin [dev][n_bins] (float, ascending).  Bins whose
 * count [dev][n_bins] (int32) is 0 are skipped (count NULL = none skipped); the trapezoid runs over the
 * remaining abscissae only, no extrapolation (reading 9); j0(x) = 1 - x^2/6 for |x| < 1e-4.  Arithmetic
 * in fp64.  r [dev][n_r] (float); out_c, out_p [dev][n_maps][n_r] (float).                       */
NMS_API nms_status nms_correlation(nms_ctx* ctx, const float* I, const float* q_of_bin, const int32_t* count,
                           int n_maps, int n_bins, const float* r, int n_r, float* out_c, float* out_p);

/* ---- two-dimensional correlation function (f-1, Eq. 36) -------------------------------------- */

/* C(rho, alpha) = int int f(q, theta) exp(i q rho cos(theta - alpha)) q dq dtheta of ONE map [dev][n_q] (float) given
 * on the context's current grid, which must be polar (NMS_E_UNSUPPORTED otherwise), evaluated on the polar grid
 * rgrid (type 0: u0 = rho [n0], u1 = alpha [n1] radians, host arrays).  Trapezoidal rule (L183): periodic in theta
 * (weight 2 pi / n1, reading 7), non-uniform in q over the given abscissae without extrapolation (as reading 9):
 * wq_0 = (q_1 - q_0)/2, wq_i = (q_{i+1} - q_{i-1})/2, wq_last = (q_last - q_{last-1})/2 (a single ring: wq = 1).
 * It is the direct Fourier sum of a-2 with the roles exchanged -- the n_q detector pixels are the "cells"
 * (position (q sin theta, q cos theta) in fp64, weight f q wq dtheta rounded once to fp32) and the (rho, alpha) points
 * are the "detector" -- and runs the same amplitude kernels.  out_re, out_im [dev][n0*n1] (float; either may be
 * NULL).  The context's sample, detector grid and stored amplitudes are left untouched.                       */
NMS_API nms_status nms_correlation_2d(nms_ctx* ctx, const float* map, const nms_qgrid* rgrid, float* out_re, float* out_im);

/* ---- form factor / interference split (a-6, Eq. 49-50) -------------------------------- */

/* For every requested kind B: out_total = B(sum_p A_p, sum_p A_p), out_form = sum_p B(A_p, A_p), where
 * A_p are the amplitudes of object p alone (with its centre); interference = total - form (reading 13).
 * Needs nms_set_particles (NMS_E_STATE otherwise).  Each output [dev][n_kinds][n_q] (float); either
 * may be NULL.                                                                                   */
NMS_API nms_status nms_form_factor_split(nms_ctx* ctx, const nms_qgrid* grid, const nms_kind* kinds, int n_kinds,
                                 float* out_total, float* out_form);

/* ---- end-to-end host entry point ---------------------------------------------------------------- */

/* One whole step from HOST buffers: copy pos/N/m [host] to the device, prep, amplitudes + responses,
 * optional azimuthal average and correlation, copy the results back to HOST buffers and synchronise.
 * out_maps [host][n_kinds][n_q] (float) or NULL.  If n_bins > 0: out_I [host][n_kinds][n_bins], and if
 * additionally n_r > 0 (r [host][n_r]): out_c, out_p [host][n_kinds][n_r].  Pinned host memory makes
 * the copies asynchronous; pageable memory also works.                                           */
NMS_API nms_status nms_run_host(nms_ctx* ctx, const float* pos, const float* N, const float* m, int64_t W,
                        const double* R, const nms_qgrid* grid, const nms_kind* kinds, int n_kinds,
                        float* out_maps, int n_bins, double q_lo, double q_hi, float* out_I,
                        const float* r, int n_r, float* out_c, float* out_p);

/* The same for a sample with object structure (a-6): copies pos/N/m [host][W], centres [host][K][3] (or NULL), runs
 * nms_set_sample + nms_set_particles(offsets [host][K+1], K, centres) + nms_form_factor_split, copies out_total and
 * out_form [host][n_kinds][n_q] (either may be NULL) back and synchronises.                                       */
NMS_API nms_status nms_run_host_split(nms_ctx* ctx, const float* pos, const float* N, const float* m, int64_t W,
                              const int64_t* offsets, int64_t K, const float* centres, const double* R,
                              const nms_qgrid* grid, const nms_kind* kinds, int n_kinds, float* out_total,
                              float* out_form);
/* Rocking scan from HOST buffers (L7 "full rotational control"; config C4): the sample is copied once, then for each of
 * the n_rot rotations R [host][n_rot][9] the prep pass and nms_compute run and the maps are copied to
 * out_maps [host][n_rot][n_kinds][n_q]; synchronises before returning.                                             */
NMS_API nms_status nms_run_host_scan(nms_ctx* ctx, const float* pos, const float* N, const float* m, int64_t W,
                             const double* R, int n_rot, const nms_qgrid* grid, const nms_kind* kinds, int n_kinds,
                             float* out_maps);

/* ---- introspection / tuning --------------------------------------------------------------------- */

/* sum_j |w_cj| of the rotated weights, c = N, m'x, m'y, m'z, into out [host][4] (the denominators of
 * the amplitude tolerance 1e-5 sum|w|); synchronises.                                            */
NMS_API nms_status nms_get_weight_sums(nms_ctx* ctx, double* out);

/* Integer options.  "variant": 0 auto (exact fp64 kernel for W * n_q <= 2^30, else the line-recurrence
 * kernel where u0 is equally spaced and the cell order is spatially coherent, else the direct kernel), 1 force the
 * direct (one phasor per pair) kernel, 2 force the line-recurrence kernel (NMS_E_UNSUPPORTED at compute time if the
 * detector is a point list or u0 is not an arithmetic progression within one fp32 ulp), 3 force the exact fp64
 * kernel.  "precision": which variant of the fp32 kernels runs.  1 fast: MUFU phasors (sin.approx /
 * cos.approx on the exactly reduced phase), three-term recurrence; amplitudes and the positive kinds meet the north-star
 * tolerances, the signed difference kinds NM and CHI miss them at a fraction of a percent of their points.  2 accurate:
 * polynomial phasors to fp32 rounding, rotations, fp64 sub-accumulation of the nuclear channel; 20-30 % slower; meets the
 * tolerances for all 13 kinds on every config.  0 (default) automatic: accurate where NM / CHI may be formed from the sums
 * (nms_amplitudes, whose result nms_response and nms_cross_spectra use later; nms_compute, nms_form_factor_split and
 * nms_compute_batch when NMS_NM or NMS_CHI is among the kinds or amplitudes are returned), fast otherwise.
 * "bases": exactly evaluated points per 8 in the recurrence kernel (0 auto = 1, else
 * 1..4).  "recurrence": 0 auto (three-term in the fast variant, rotations in the accurate one), 1 complex rotations, 2 three-term
 * recurrence (bases <= 2).  "timing": 1 records a
 * CUDA event pair around every kernel launch (and resets the record).  "chunks": 0 auto, else the number of cell
 * chunks.  "qt": 0 auto, else detector points per thread (4 or 8; 16 for the recurrence kernel on a sample without
 * moments).  "friedel" (f-4): 1 = on a polar grid with an even number of angles closed under theta -> theta + pi
 * (within one ulp of 2 pi; NMS_E_UNSUPPORTED otherwise, and for nms_form_factor_split) the amplitude sums are evaluated
 * for the first half of every ring only and the second half is taken as the conjugate, A(-q) = A(q)^* for real weights
 * (Eq. 42-43): half the pair evaluations; the second half then belongs to the float angle rotated by
 * its deviation from theta + pi (<= 2.4e-7 rad).  Off by default; bench.py reports it as an EFFECTIVE rate only.
 * "uniform": 1 = do not use the block-uniform instantiation of the polar recurrence kernel (testing).
 * "interp": the accurate variant of the line-recurrence kernels (four channels, not split, 16 points per thread) generates
 * only every other point of a line and takes the points in between from the sums -- the three-term identity
 * z_{k-1} + z_{k+1} = 2 cos(delta) z_k read as an interpolation and applied, by the linearity of Eq. 42-47 (L353-L368), to
 * h-weighted sums of the two neighbours (csrc/k_amp_interp.cu; the generated points follow from one exactly evaluated
 * point by rotations alternating with single, unchained three-term steps) -- wherever the step phase of every cell along the line
 * stays below 0.2 cycle (d r_max < 0.4 pi).  0 automatic (used where admissible), 1 never, 2 required (NMS_E_UNSUPPORTED at
 * compute time if it is not admissible).
 * Unknown keys: NMS_E_ARG.  The fp32 kernels need q_max r_max / 2 pi < 2^19 cycles (NMS_E_UNSUPPORTED
 * otherwise; the exact kernel has no such limit).                                                        */
NMS_API nms_status nms_set_option(nms_ctx* ctx, const char* key, int64_t value);
/* Read back integers: "launches" (kernels launched by this context so far), "variant_used" (1 list direct,
 * 2 polar direct, 4 cartesian direct, 3 polar recurrence, 5 cartesian recurrence, 8 exact fp64, 16 / 17 batched-field
 * kernel direct / line recurrence),
 * "n_chunks", "n_tiles", "n_slots", "sm_count", "blocks_per_sm", "qt", "poly_phasors" (non-zero: polynomial phasors),
 * "bases", "three_term", "interp" (1: the interpolating kernel ran), "corr2d_variant" (variant_used of the last
 * nms_correlation_2d).                                                                              */
NMS_API nms_status nms_get_info(nms_ctx* ctx, const char* key, int64_t* value);
/* Device time in ms of the most recent launch of the given kernel class ("timing" must be 1);
 * synchronises on that kernel's end event.  NMS_E_STATE if it has not run.                       */
NMS_API nms_status nms_kernel_time_ms(nms_ctx* ctx, nms_timer which, float* ms);
/* Sum of the device times [ms] and the number of launches of the given kernel class recorded since
 * "timing" was last set (setting the option resets the record); synchronises on the recorded events.
 * This is what bench.py divides the algorithmic work by for the roofline figure.                  */
NMS_API nms_status nms_kernel_time_total(nms_ctx* ctx, nms_timer which, double* total_ms, int64_t* count);

/* ---- measured properties of the machine and of the phasor routines (diagnostics) ------------------------------------ */

/* Instruction classes timed by nms_pipe_rates, in this order. */
typedef enum {
    NMS_PIPE_FFMA = 0,        /* fma.rn.f32                                   lane-FMAs per clock and SM              */
    NMS_PIPE_FFMA2_REG = 1,   /* fma.rn.f32x2, three 64-bit register operands (2 lane-FMAs per instruction and lane)  */
    NMS_PIPE_FFMA2_BCAST = 2, /* fma.rn.f32x2 with a broadcast 32-bit operand -- the form the amplitude kernels use   */
    NMS_PIPE_FMUL = 3,
    NMS_PIPE_MUFU_SIN = 4,    /* sin.approx (FMUL.RZ + MUFU.SIN)              MUFU per clock and SM                   */
    NMS_PIPE_MUFU_EX2 = 5,    /* ex2.approx (MUFU.EX2 alone)                                                          */
    NMS_PIPE_DFMA = 6,
    NMS_PIPE_I2FP = 7,
    NMS_PIPE_IALU = 8,        /* SHF + IADD3                                   integer operations per clock and SM    */
    NMS_PIPE_LOP3 = 9,
    NMS_PIPE_F2F = 10,        /* double -> float -> double round trip + DMUL   round trips per clock and SM           */
    NMS_PIPE_PHASOR_MUFU = 11,/* whole MUFU phasor (nms_phasor.cuh)            phasors per clock and SM               */
    NMS_PIPE_PHASOR_POLY = 12,/* whole polynomial phasor                                                              */
    NMS_PIPE_COUNT = 13
} nms_pipe;
/* Micro-benchmark behind the roofline figures of DESIGN.md section 6: for each class above, 16 warps per SM each run
 * 8 independent chains of the instruction for 4096 rounds between two clock64() reads; out [host][NMS_PIPE_COUNT]
 * receives operations per clock and SM (slowest block).  Synchronises.                                                  */
NMS_API nms_status nms_pipe_rates(nms_ctx* ctx, double* out);
/* Error statistics of the phasor routine of the amplitude kernels (polynomial = 0: MUFU, 1: polynomial) over 2^log2_n
 * stratified phases (10 <= log2_n <= 30) against fp64: out [host][23] = largest |error| of cos, of sin, rms error of cos,
 * of sin, then |e_n| for n = -8 ... 8, the Fourier coefficients of the complex error function e(phi) = z_computed -
 * exp(-i phi) (e_n multiplies A(n q) in the error of A(q); e_1 is a harmless relative error), then Re e_0, Im e_0 (the
 * mean errors of cos and of -sin).  Synchronises.                                                                      */
NMS_API nms_status nms_phasor_selftest(nms_ctx* ctx, int polynomial, int log2_n, double* out);

#ifdef __cplusplus
}
#endif
#endif /* NMS_H_ */
