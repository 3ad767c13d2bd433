// nms_internal.h -- shared declarations of the CUDA implementation behind include/nms.h.
// Nothing here is part of the ABI.  Citations "Lnnn"/"Eq. n" refer to PAPER.md (see include/nms.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <vector>
#include "../../include/nms.h"

namespace nms {

// ---- packed real-space layout (a-1) ----------------------------------------------------------
// Cells are grouped into tiles of at most TILE consecutive cells (never straddling an object when
// an object structure is set).  A tile is an array of 32-byte Cell records.  Coordinates are the
// rotated detector-plane coordinates Y, Z (Eq. 39-40) in fp64 -- the phase is formed in fp64 (one DFMA
// per evaluated phasor on the FP64 pipe), see k_amplitude.cu; X is never needed: q_x = 0 (Eq. 41).
// Weights are rounded once to fp32.  The amplitude kernel keeps each complex accumulator as one packed
// register pair {sum w cos, sum w sin} and updates it with a single fma.rn.f32x2 {w, w} * {cos, sin} + acc
// whose first operand is the 32-bit weight register broadcast to both halves (SASS: FFMA2 Rd, Rw.F32, ...),
// so an accumulation reads one 32-bit and two 64-bit registers.
constexpr int TILE = 256;
constexpr int SLOT_PAD = 1;

struct Cell {              // 32 B, the unit of the bulk copies (16-byte aligned)
    double Y, Z;           // [nm]
    float wN, wx, wy, wz;  // nuclear weight, m'_x, m'_y, m'_z
};

struct TileMeta {          // consumed by the amplitude kernel (32 B)
    double Y0, Z0;         // centre of the tile's bounding box in the detector plane [nm]: the recurrence kernels
                           // correct the deviation of a float abscissa from the evaluated progression there
    int64_t first_slot;    // index into the cell array
    int32_t n_slots;       // cell count of the tile
    int32_t flags;         // bit 0: last tile of its object, bit 1: first tile (form-factor split)
};
struct TileSrc {           // consumed by the prep kernel
    int64_t src_first;     // first source cell
    int32_t n_src;         // number of source cells (<= TILE)
    int32_t particle;      // object index (for centres), -1 if none
};

struct Timer {                         // "timing" option: one CUDA event pair per launch, kept until the next reset
    std::vector<cudaEvent_t> beg, end;
    size_t used = 0;                   // pairs recorded since the last reset
};

struct DevBuf {
    void* p = nullptr;
    size_t cap = 0;
};

}  // namespace nms

struct nms_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    int sm_count = 0;
    char err[512] = {0};

    // options
    int opt_variant = 0;   // 0 auto, 1 direct, 2 recurrence, 3 exact fp64
    int opt_timing = 0;
    int opt_chunks = 0;
    int opt_qt = 0;        // 0 auto, else 4/8/16
    int opt_bases = 0;     // recurrence kernels: exactly evaluated points per 8 (0 auto = 2, else 1..4)
    int opt_precision = 0; // 0 auto (accurate where NM / CHI may be formed from the sums, else fast), 1 fast, 2 accurate
    int opt_friedel = 0;   // f-4: 1 = evaluate half of every ring and take the other half as the conjugate (polar grids)
    bool friedel_active = false;   // the partials of the last amplitude launch cover the first half of every ring only
    nms::DevBuf qc_half, sc_half;  // detector constants of the half rings
    int opt_uniform = 0;   // 1: never use the block-uniform instantiations (testing)
    int opt_rec3 = 0;      // recurrence kernels: 0 auto, 1 rotations, 2 three-term recurrence
    int opt_interp = 0;    // accurate recurrence kernels: 0 auto (interpolating kernel where admissible), 1 never, 2 required
    int amp_timer = NMS_T_AMPLITUDE;   // timer class of the amplitude launch (-1: none, the caller times it)
    int64_t launches = 0;
    int variant_used = 0, n_chunks_used = 0, blocks_per_sm_used = 0, qt_used = 0;
    int npoly_used = 0, nb_used = 0, rec3_used = 0, corr2d_variant = 0, interp_used = 0;

    // sample (raw copy kept for nms_set_rotation)
    int64_t W = 0;
    bool has_N = false, has_M = false;
    nms::DevBuf raw_pos, raw_N, raw_m, centres;
    std::vector<int64_t> offsets;      // host, K+1 entries (empty = no object structure)
    int64_t K = 0;
    bool has_centres = false;
    double R[9] = {1, 0, 0, 0, 1, 0, 0, 0, 1};
    double P[3] = {0, 0, 1};
    double sN = 1.0, sM = 1.0, invV = 1.0;

    // packed sample
    bool packed_valid = false;
    int64_t n_tiles = 0, n_slots = 0;
    std::vector<nms::TileSrc> h_tile_src;
    std::vector<int32_t> h_tile_flags;
    std::vector<int64_t> h_tile_first_slot;
    nms::DevBuf tile_wsum;             // double [n_tiles][7]: per-tile sum |w|, largest r^2, squared half diagonal, half Z extent
    nms::DevBuf tile_src, tile_meta, cells, wsum;   // cells: Cell[n_slots]; wsum: double[7] (4 sums, r_max, tile half diagonal, tile half Z extent)
    double* h_geo = nullptr;           // pinned [3]: r_max, largest tile half diagonal and half Z extent of the packed sample
    cudaEvent_t geo_event = nullptr;   // recorded after the copy into h_geo
    bool geo_pending = false;
    double geo_rmax = 0.0, geo_ext = 0.0, geo_extz = 0.0;   // host copies (valid once geo_pending is false)

    // current detector grid
    bool grid_valid = false;
    int g_type = 0, g_n0 = 0, g_n1 = 0;
    int64_t n_q = 0;
    bool g_uniform = false;            // abscissa along the thread line (u0) is equally spaced (within 1 ulp)
    double g_dq = 0.0;                 // its spacing (u0[n0-1] - u0[0]) / (n0 - 1)
    double g_dev = 0.0;                // largest deviation of u0 from that progression [rad/nm]
    double g_qmax = 0.0;               // largest |q| on the grid [rad/nm]
    std::vector<float> h_u0, h_u1;
    nms::DevBuf u0, u1, qc, sc;        // qc: double2[n_q] (q_y,q_z) rad/nm; sc: double2[n_q] (sin th, cos th)

    // amplitudes / scratch
    bool amp_valid = false;
    nms::DevBuf amp64;                 // double [8][n_q]
    nms::DevBuf part, formpart;        // chunk partials
    nms::DevBuf interp_sb, interp_spb; // k_amp_interp: chunk partials of the B sets (plain, and weighted with the tile centres)
    nms::DevBuf chunk_begin;           // int32 [n_chunks+1] (split mode only)
    std::vector<int32_t> h_chunk_begin;
    nms::DevBuf kinds_dev;             // int32 [<=13]
    nms::DevBuf bin_idx, bin_sum, bin_cnt;
    nms::DevBuf pix_cells, pix_meta, pix_u0, pix_u1, pix_qc, pix_sc;   // 2-D correlation: detector pixels as a sample, r-grid
    nms::DevBuf modal_tab, modal_ring; // (sin, cos)(k theta_j) table; fp64 ring values of the modal decomposition
    nms::DevBuf batch_cells, batch_ampN;   // f-3: packed records of one pass of fields; the shared nuclear amplitude (fp64)
    nms::DevBuf diag;                  // scratch of the diagnostics (k_diag.cu)
    nms::DevBuf host_stage[8];         // device staging for nms_run_host

    nms::Timer timers[NMS_T_COUNT];
};

namespace nms {

nms_status fail(nms_ctx* c, nms_status st, const char* fmt, ...);
nms_status cuda_fail(nms_ctx* c, cudaError_t e, const char* where);
nms_status ensure(nms_ctx* c, DevBuf& b, size_t bytes);
nms_status timer_begin(nms_ctx* c, int which);   // no-ops unless the "timing" option is set (which < 0: never)
nms_status timer_end(nms_ctx* c, int which);

#define NMS_CUDA(c, call)                                          \
    do {                                                           \
        cudaError_t e__ = (call);                                  \
        if (e__ != cudaSuccess) return nms::cuda_fail((c), e__, #call); \
    } while (0)

// ---- kernel launchers (each only enqueues on c->stream) ----------------------------------------
// k_prep.cu
nms_status launch_prep(nms_ctx* c);                       // a-1: raw sample -> packed tiles, wsum
nms_status launch_qsetup(nms_ctx* c);                     // detector abscissae -> qc, sc
// nms_api.cu
nms_status set_grid(nms_ctx* c, const nms_qgrid* g);      // install a detector grid as the current one
// k_amplitude.cu
struct AmpPlan {
    int variant;       // 1 list direct, 2 polar direct, 4 cartesian direct, 3 polar / 5 cartesian recurrence, 8 exact
    int qt;            // q points per thread
    int n_chunks;
    int n_qblocks;
    int blocks_per_sm;
    bool split;
    int nch;           // weight channels the kernel accumulates: 4, or 1 for a sample without moments
    int npoly;         // direct: phasors per thread evaluated by polynomial (qt = all: accurate); recurrence: 0 / 1
    int nb;            // recurrence: exactly evaluated points per thread
    int rec3;          // recurrence: three-term recurrence instead of rotations
    bool sh;           // accurate recurrence: the step phase stays within a quarter cycle (no quadrant logic)
    bool uni;          // n1 % 128 == 0: a block lies inside one group of lines (block-uniform abscissae)
    bool interp;       // accurate recurrence: every other point of a line generated, the others interpolated (k_amp_interp.cu)
};
nms_status plan_amplitude(nms_ctx* c, bool split, bool want_accurate, AmpPlan* plan);
int choose_chunks(nms_ctx* c, int64_t n_qb, int64_t slots, int64_t units, double chunk_bytes, int64_t min_units, double mem_bytes);
nms_status wait_geometry(nms_ctx* c);                     // r_max / tile extents of the packed sample (k_prep) on the host
nms_status launch_amplitude(nms_ctx* c, const AmpPlan& plan, const int32_t* kinds_dev, int n_kinds);
// k_epilogue.cu
nms_status launch_epilogue(nms_ctx* c, int n_chunks, const int32_t* kinds_dev, int n_kinds, float* out_maps,
                           float* out_amp, bool keep_amp64);
nms_status launch_cross_spectra(nms_ctx* c, float* out_GR, float* out_GI);
nms_status launch_response_from_amp(nms_ctx* c, const int32_t* kinds_dev, int n_kinds, float* out_maps);
nms_status launch_split_epilogue(nms_ctx* c, int n_chunks, const int32_t* kinds_dev, int n_kinds, float* out_total,
                                 float* out_form);
// k_batch.cu
nms_status launch_batch(nms_ctx* c, const float* m_batch, int B, const int32_t* kinds_dev, int n_kinds, float* out_maps,
                        float* out_amp, bool accurate);
// k_post.cu
nms_status launch_azimuthal(nms_ctx* c, const float* maps, int n_maps, int n_bins, double q_lo, double q_hi,
                            float* out_I, float* out_q, int32_t* out_count);
nms_status launch_modal(nms_ctx* c, const float* maps, int n_maps, int k_max, float* out_Is, float* out_Ic, float* out_a,
                        float* out_A);
nms_status launch_correlation_2d(nms_ctx* c, const float* map, const nms_qgrid* rgrid, float* out_re, float* out_im);
nms_status launch_correlation(nms_ctx* c, const float* I, const float* q_of_bin, const int32_t* count, int n_maps,
                              int n_bins, const float* r, int n_r, float* out_c, float* out_p);

}  // namespace nms
