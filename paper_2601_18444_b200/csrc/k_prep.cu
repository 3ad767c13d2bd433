// k_prep.cu -- a-1: rotate + pack the real-space sample into tiles, and detector set-up.
//
//  prep kernel   (Eq. 37-41):  r' = R (x + r^k), m' = R m in fp64; only Y, Z (rows 2, 3 of R)
//                are kept because q_x = 0 on the detector (Eq. 41).  One block per tile, TILE/256 cells per
//                thread: it writes the Cell records (fp64 Y, Z; weights rounded once to fp32), the tile's sum_j |w_cj|
//                and the centre of its bounding box in the detector plane; k_wsum_reduce adds the tiles in a fixed
//                order (the tolerance denominators, deterministic) and takes the largest radius and tile extent
//                (host checks: |t| < 2^19 cycles for the exact phase reduction; residual of the recurrence correction).
//  qsetup kernel (Eq. 6): per detector point (q_y, q_z) in fp64 [rad/nm] and
//                (sin th, cos th) for the response epilogue.
#include "nms_internal.h"

namespace nms {

constexpr int PREP_THREADS = 256;
constexpr int PREP_PER_THREAD = TILE / PREP_THREADS;

struct PrepArgs {
    const float* pos;
    const float* N;
    const float* m;
    const float* centres;
    const TileSrc* src;
    const int64_t* first_slot;
    const int32_t* flags;
    TileMeta* meta;
    Cell* cells;
    double* tile_wsum;   // [n_tiles][7]: per-tile sum_j |w_cj|, largest Y^2 + Z^2, squared half diagonal and half Z extent of the bounding box
    double R[9];
};

__device__ __forceinline__ double warp_sum(double v)
{
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Bounding box and radius need no more than float accuracy (tile centres for a first-order correction, a range check):
// order-preserving integer images of the floats go through the warp-wide REDUX instruction (1 instead of 10 shuffles).
__device__ __forceinline__ int float_order(float f)
{
    const int i = __float_as_int(f);
    return i >= 0 ? i : i ^ 0x7fffffff;
}
__device__ __forceinline__ float order_float(int i) { return __int_as_float(i >= 0 ? i : i ^ 0x7fffffff); }
__device__ __forceinline__ float warp_minf(float v) { return order_float(__reduce_min_sync(0xffffffffu, float_order(v))); }
__device__ __forceinline__ float warp_maxf(float v) { return order_float(__reduce_max_sync(0xffffffffu, float_order(v))); }
__device__ __forceinline__ double warp_min(double v)
{
    for (int o = 16; o > 0; o >>= 1) v = fmin(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
__device__ __forceinline__ double warp_max(double v)
{
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

__global__ void __launch_bounds__(PREP_THREADS) k_prep(const PrepArgs a)
{
    __shared__ double red[9][PREP_THREADS / 32];
    const int tile = blockIdx.x;
    const TileSrc ts = a.src[tile];
    const int64_t first_slot = a.first_slot[tile];
    const int n_slots = (ts.n_src + SLOT_PAD - 1) / SLOT_PAD * SLOT_PAD;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    double cx = 0.0, cy = 0.0, cz = 0.0;
    if (a.centres && ts.particle >= 0) {
        cx = (double)a.centres[3 * (int64_t)ts.particle + 0];
        cy = (double)a.centres[3 * (int64_t)ts.particle + 1];
        cz = (double)a.centres[3 * (int64_t)ts.particle + 2];
    }
    double Y[PREP_PER_THREAD], Z[PREP_PER_THREAD];
    float wN[PREP_PER_THREAD], wx[PREP_PER_THREAD], wy[PREP_PER_THREAD], wz[PREP_PER_THREAD];
    double sN = 0.0, sx = 0.0, sy = 0.0, sz = 0.0;
    double ylo = 1e300, yhi = -1e300, zlo = 1e300, zhi = -1e300, r2 = 0.0;
#pragma unroll
    for (int u = 0; u < PREP_PER_THREAD; ++u) {
        const int i = PREP_PER_THREAD * tid + u;
        Y[u] = Z[u] = 0.0;
        wN[u] = wx[u] = wy[u] = wz[u] = 0.f;
        if (i < ts.n_src) {
            const int64_t j = ts.src_first + i;
            const double x = (double)a.pos[3 * j + 0] + cx;
            const double y = (double)a.pos[3 * j + 1] + cy;
            const double z = (double)a.pos[3 * j + 2] + cz;
            Y[u] = a.R[3] * x + a.R[4] * y + a.R[5] * z;   // Eq. 39
            Z[u] = a.R[6] * x + a.R[7] * y + a.R[8] * z;   // Eq. 40
            ylo = fmin(ylo, Y[u]); yhi = fmax(yhi, Y[u]); zlo = fmin(zlo, Z[u]); zhi = fmax(zhi, Z[u]);
            r2 = fmax(r2, Y[u] * Y[u] + Z[u] * Z[u]);
            if (a.N) { wN[u] = a.N[j]; sN += fabs((double)wN[u]); }
            if (a.m) {
                const double mx = (double)a.m[3 * j + 0], my = (double)a.m[3 * j + 1], mz = (double)a.m[3 * j + 2];
                const double rx = a.R[0] * mx + a.R[1] * my + a.R[2] * mz;   // m' = R m (reading 2)
                const double ry = a.R[3] * mx + a.R[4] * my + a.R[5] * mz;
                const double rz = a.R[6] * mx + a.R[7] * my + a.R[8] * mz;
                sx += fabs(rx); sy += fabs(ry); sz += fabs(rz);
                wx[u] = (float)rx; wy[u] = (float)ry; wz[u] = (float)rz;
            }
        }
    }
    sN = warp_sum(sN); sx = warp_sum(sx); sy = warp_sum(sy); sz = warp_sum(sz);
    // rounded outwards by one float ulp at most: harmless for a centre, conservative for the radius
    ylo = (double)warp_minf((float)ylo); yhi = (double)warp_maxf((float)yhi);
    zlo = (double)warp_minf((float)zlo); zhi = (double)warp_maxf((float)zhi); r2 = (double)warp_maxf((float)r2 * 1.0000002f);
    if (lane == 0) {
        red[0][warp] = sN; red[1][warp] = sx; red[2][warp] = sy; red[3][warp] = sz;
        red[4][warp] = ylo; red[5][warp] = yhi; red[6][warp] = zlo; red[7][warp] = zhi; red[8][warp] = r2;
    }
    __syncthreads();
    if (tid == 0) {
        double v[9];
        for (int r = 0; r < 9; ++r) v[r] = red[r][0];
        for (int w = 1; w < PREP_THREADS / 32; ++w) {
            for (int r = 0; r < 4; ++r) v[r] += red[r][w];
            v[4] = fmin(v[4], red[4][w]); v[5] = fmax(v[5], red[5][w]);
            v[6] = fmin(v[6], red[6][w]); v[7] = fmax(v[7], red[7][w]); v[8] = fmax(v[8], red[8][w]);
        }
        const bool any = ts.n_src > 0;
        TileMeta tm;
        tm.Y0 = any ? 0.5 * (v[4] + v[5]) : 0.0; tm.Z0 = any ? 0.5 * (v[6] + v[7]) : 0.0;
        tm.first_slot = first_slot; tm.n_slots = n_slots; tm.flags = a.flags[tile];
        a.meta[tile] = tm;
        for (int r = 0; r < 4; ++r) a.tile_wsum[7 * (int64_t)tile + r] = v[r];
        a.tile_wsum[7 * (int64_t)tile + 4] = v[8];
        a.tile_wsum[7 * (int64_t)tile + 5] = any ? 0.25 * ((v[5] - v[4]) * (v[5] - v[4]) + (v[7] - v[6]) * (v[7] - v[6])) : 0.0;
        a.tile_wsum[7 * (int64_t)tile + 6] = any ? 0.5 * (v[7] - v[6]) : 0.0;
    }
#pragma unroll
    for (int u = 0; u < PREP_PER_THREAD; ++u) {
        const int i = PREP_PER_THREAD * tid + u;
        if (i < n_slots) {
            Cell ce;
            ce.Y = Y[u]; ce.Z = Z[u];
            ce.wN = wN[u]; ce.wx = wx[u]; ce.wy = wy[u]; ce.wz = wz[u];
            a.cells[first_slot + i] = ce;
        }
    }
}

// sum_j |w_cj| over all tiles: one block, fixed order (deterministic, unlike atomics on four addresses)
__global__ void __launch_bounds__(1024) k_wsum_reduce(const double* __restrict__ tile_wsum, int64_t n_tiles,
                                                      double* __restrict__ wsum)
{
    __shared__ double red[7][32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double s[7] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    for (int64_t t = threadIdx.x; t < n_tiles; t += blockDim.x) {
#pragma unroll
        for (int r = 0; r < 4; ++r) s[r] += tile_wsum[7 * t + r];
        s[4] = fmax(s[4], tile_wsum[7 * t + 4]); s[5] = fmax(s[5], tile_wsum[7 * t + 5]); s[6] = fmax(s[6], tile_wsum[7 * t + 6]);
    }
#pragma unroll
    for (int r = 0; r < 7; ++r) {
        s[r] = r < 4 ? warp_sum(s[r]) : warp_max(s[r]);
        if (lane == 0) red[r][warp] = s[r];
    }
    __syncthreads();
    if (threadIdx.x < 7) {
        double v = 0.0;
        for (int w = 0; w < 32; ++w) v = threadIdx.x < 4 ? v + red[threadIdx.x][w] : fmax(v, red[threadIdx.x][w]);
        wsum[threadIdx.x] = (threadIdx.x < 4 || threadIdx.x == 6) ? v : sqrt(v);   // [4]: largest radius in the detector plane, [5]: largest tile half diagonal, [6]: largest tile half extent in Z
    }
}

nms_status launch_prep(nms_ctx* c)
{
    PrepArgs a;
    a.pos = (const float*)c->raw_pos.p;
    a.N = c->has_N ? (const float*)c->raw_N.p : nullptr;
    a.m = c->has_M ? (const float*)c->raw_m.p : nullptr;
    a.centres = c->has_centres ? (const float*)c->centres.p : nullptr;
    a.src = (const TileSrc*)c->tile_src.p;
    // first_slot and flags live behind the TileSrc array in the same buffer (see build_tiles in nms_api.cu)
    const char* base = (const char*)c->tile_src.p + sizeof(TileSrc) * (size_t)c->n_tiles;
    a.first_slot = (const int64_t*)base;
    a.flags = (const int32_t*)(base + sizeof(int64_t) * (size_t)c->n_tiles);
    a.meta = (TileMeta*)c->tile_meta.p;
    a.cells = (Cell*)c->cells.p;
    if (nms_status st = ensure(c, c->tile_wsum, sizeof(double) * 7 * (size_t)c->n_tiles)) return st;
    a.tile_wsum = (double*)c->tile_wsum.p;
    for (int i = 0; i < 9; ++i) a.R[i] = c->R[i];
    if (nms_status ts_ = timer_begin(c, NMS_T_PREP)) return ts_;
    k_prep<<<(unsigned)c->n_tiles, PREP_THREADS, 0, c->stream>>>(a);
    k_wsum_reduce<<<1, 1024, 0, c->stream>>>((const double*)c->tile_wsum.p, c->n_tiles, (double*)c->wsum.p);
    if (nms_status ts_ = timer_end(c, NMS_T_PREP)) return ts_;
    c->launches += 2;
    NMS_CUDA(c, cudaGetLastError());
    // the two geometry figures go to pinned host memory; the planner waits for this event only
    NMS_CUDA(c, cudaMemcpyAsync(c->h_geo, (const double*)c->wsum.p + 4, 3 * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    NMS_CUDA(c, cudaEventRecord(c->geo_event, c->stream));
    c->geo_pending = true;
    return NMS_OK;
}

// ---- detector set-up ---------------------------------------------------------------------------
__global__ void k_qsetup(int type, int n0, int n1, const float* __restrict__ u0, const float* __restrict__ u1,
                         double2* __restrict__ qc, double2* __restrict__ sc)
{
    const int64_t f = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t nq = (int64_t)n0 * n1;
    if (f >= nq) return;
    const int i0 = (int)(f / n1), i1 = (int)(f % n1);
    double qy, qz, s, c;
    if (type == 0) {                       // polar: q_y = q sin th, q_z = q cos th (L343)
        const double q = (double)u0[i0], th = (double)u1[i1];
        sincos(th, &s, &c);
        qy = q * s; qz = q * c;
    } else {
        if (type == 1) { qz = (double)u0[i0]; qy = (double)u1[i1]; }
        else           { qy = (double)u0[i0]; qz = (double)u1[i0]; }
        const double n = sqrt(qy * qy + qz * qz);
        if (n > 0.0) { s = qy / n; c = qz / n; }     // th = atan2(q_y, q_z)
        else         { s = 0.0; c = 1.0; }           // th(0,0) = 0 (reading 5)
    }
    qc[f] = make_double2(qy, qz);
    sc[f] = make_double2(s, c);
}

nms_status launch_qsetup(nms_ctx* c)
{
    const int threads = 256;
    const unsigned blocks = (unsigned)((c->n_q + threads - 1) / threads);
    k_qsetup<<<blocks, threads, 0, c->stream>>>(c->g_type, c->g_n0, c->g_n1, (const float*)c->u0.p,
                                                (const float*)c->u1.p, (double2*)c->qc.p, (double2*)c->sc.p);
    c->launches += 1;
    NMS_CUDA(c, cudaGetLastError());
    return NMS_OK;
}

}  // namespace nms
