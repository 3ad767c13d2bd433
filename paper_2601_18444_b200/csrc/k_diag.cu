// k_diag.cu -- measured properties of the machine and of the phasor routines that DESIGN.md and bench.py quote:
//   nms_pipe_rates      issue rates (lane-operations per clock and SM) of the instructions the amplitude kernels are made
//                       of: FFMA, packed FFMA2, FMUL, MUFU (sin/cos/ex2), DFMA, I2FP, integer ALU, F2F, and whole phasors
//                       (MUFU and polynomial) -- the numbers behind the "148 SMs x 128 FP32 lanes" roofline and the
//                       "16 MUFU lanes/clk/SM" ceiling of the direct kernels;
//   nms_phasor_selftest error statistics of phasor<false> / phasor<true> (nms_phasor.cuh) over 2^24 phases against
//                       fp64 sincospi: largest and rms error per component and the Fourier coefficients e_n of the
//                       complex error function (e_n leaks A(n q) into A(q): e_0 the forward amplitude sum w).
#include "nms_internal.h"
#include "nms_phasor.cuh"

namespace nms {

constexpr int RATE_THREADS = 256;
constexpr int RATE_ITERS = 4096;
constexpr int RATE_CHAINS = 8;

// One timed loop per instruction class: RATE_CHAINS independent dependency chains per thread, RATE_ITERS rounds.
// cycles[block] = clock64 span of the block; sink keeps the results alive.
template <int OP>
__global__ void __launch_bounds__(RATE_THREADS) k_rate(long long* __restrict__ cycles, float* __restrict__ sink, float seed,
                                                       unsigned* __restrict__ arrived)
{
    float x[RATE_CHAINS];
    u64 y[RATE_CHAINS];
    double d[RATE_CHAINS];
    int n[RATE_CHAINS];
#pragma unroll
    for (int c = 0; c < RATE_CHAINS; ++c) {
        x[c] = seed + 0.001f * (float)(threadIdx.x + c);
        y[c] = pack2(x[c], x[c] + 0.5f);
        d[c] = (double)x[c];
        n[c] = (int)threadIdx.x * 2654435 + c * 40503;
    }
    const float a = 0.999f + seed * 1e-6f, b = 1e-3f;
    const u64 a2 = pack2(a, a), b2 = pack2(b, b);
    const double ad = 0.999 + (double)seed * 1e-9, bd = 1e-3;
    // all blocks start the timed loop together (the grid is one resident wave: 2 blocks per SM), so that the two blocks
    // of an SM share it for the whole of both spans
    if (threadIdx.x == 0) {
        atomicAdd(arrived, 1u);
        while (*(volatile unsigned*)arrived < gridDim.x) { }
    }
    __syncthreads();
    const long long t0 = clock64();
    for (int it = 0; it < RATE_ITERS; ++it) {
#pragma unroll
        for (int c = 0; c < RATE_CHAINS; ++c) {
            if (OP == 0) x[c] = fmaf(x[c], a, b);                                            // FFMA
            if (OP == 1) asm volatile("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(y[c]) : "l"(y[c]), "l"(a2), "l"(b2));   // FFMA2, three 64-bit operands
            if (OP == 2) asm volatile("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(y[c]) : "l"(pack2(a, a)), "l"(y[c]), "l"(b2));  // FFMA2, broadcast 32-bit operand
            if (OP == 3) x[c] = x[c] * a;                                                    // FMUL
            if (OP == 4) x[c] = __sinf(x[c]);                                                // FMUL.RZ + MUFU.SIN
            if (OP == 5) asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(x[c]));            // MUFU.EX2 alone
            if (OP == 6) d[c] = fma(d[c], ad, bd);                                           // DFMA
            if (OP == 7) x[c] = __int2float_rn(__float_as_int(x[c]));                        // I2FP
            if (OP == 8) n[c] = n[c] + (n[c] >> 3);                                          // SHF + IADD3 (2 integer ALU operations)
            if (OP == 9) n[c] = (n[c] ^ 0x5bd1e995) & (n[c] | 0x1b873593);                   // LOP3 (one instruction)
            if (OP == 10) d[c] = (double)__double2float_rn(d[c]) * ad;                        // F2F.F32.F64 + F2F.F64.F32 + DMUL
            if (OP == 11) { float cs, sn; sincos_mufu(n[c], cs, sn); n[c] += __float_as_int(cs) ^ __float_as_int(sn); }   // MUFU phasor
            if (OP == 12) { float cs, sn; sincos_poly(n[c], cs, sn); n[c] += __float_as_int(cs) ^ __float_as_int(sn); }   // polynomial phasor
        }
    }
    const long long t1 = clock64();
    float s = 0.f;
#pragma unroll
    for (int c = 0; c < RATE_CHAINS; ++c) {
        float lo, hi;
        unpack2(y[c], lo, hi);
        s += x[c] + lo + hi + (float)d[c] + (float)n[c];
    }
    if (s == 12345.678f) sink[0] = s;
    if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
}

typedef void (*rate_kernel_t)(long long*, float*, float, unsigned*);
static const rate_kernel_t RATE_KERNELS[NMS_PIPE_COUNT] = {
    k_rate<0>, k_rate<1>, k_rate<2>, k_rate<3>, k_rate<4>, k_rate<5>, k_rate<6>, k_rate<7>, k_rate<8>, k_rate<9>, k_rate<10>,
    k_rate<11>, k_rate<12>};
// operations counted per loop round and chain (the figure reported is per OPERATION, not per instruction: an FFMA2 counts
// as 2 lane-FMAs, the integer pair as 2, the conversion round trip as 1 round trip, a phasor as 1 phasor)
static const double RATE_OPS[NMS_PIPE_COUNT] = {1, 2, 2, 1, 1, 1, 1, 1, 2, 1, 1, 1, 1};

// ---- phasor error statistics ---------------------------------------------------------------------
constexpr int SELF_HARM = 8;                 // Fourier coefficients e_n for n = -8 ... 8
struct SelfOut {
    double max_c, max_s, sum_c2, sum_s2;
    double re[2 * SELF_HARM + 1], im[2 * SELF_HARM + 1];
};

template <bool POLY>
__global__ void __launch_bounds__(256) k_phasor_selftest(int log2_n, SelfOut* __restrict__ out)
{
    const int64_t n = (int64_t)1 << log2_n;
    double mc = 0.0, ms = 0.0, c2 = 0.0, s2 = 0.0;
    double re[2 * SELF_HARM + 1], im[2 * SELF_HARM + 1];
    for (int h = 0; h <= 2 * SELF_HARM; ++h) re[h] = im[h] = 0.0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        // a stratified sample of the 2^32 phases: one per stratum of 2^(32 - log2_n), at a hashed offset inside it
        const unsigned stride = 1u << (32 - log2_n);
        unsigned hsh = (unsigned)i * 2654435761u;
        hsh ^= hsh >> 15;
        const int k = (int)((unsigned)i * stride + (hsh & (stride - 1u)) - 0x80000000u);
        float c, s;
        if (POLY) sincos_poly(k, c, s); else sincos_mufu(k, c, s);
        double sr, cr;
        sincospi((double)k * (1.0 / 2147483648.0), &sr, &cr);
        const double ec = (double)c - cr, es = (double)s - sr;
        mc = fmax(mc, fabs(ec)); ms = fmax(ms, fabs(es));
        c2 += ec * ec; s2 += es * es;
        // error of z = c - i s; coefficient e_n = mean(e exp(+i n phi))
        for (int h = -SELF_HARM; h <= SELF_HARM; ++h) {
            double sh, ch;
            sincospi((double)h * (double)k * (1.0 / 2147483648.0), &sh, &ch);
            re[h + SELF_HARM] += ec * ch + es * sh;      // (ec - i es)(ch + i sh)
            im[h + SELF_HARM] += ec * sh - es * ch;
        }
    }
    // block reduction through shared memory, then fp64 atomics (max through a compare-and-swap loop on the bits)
    __shared__ double sh[256];
    auto block_sum = [&](double v) {
        sh[threadIdx.x] = v;
        __syncthreads();
        for (int o = 128; o > 0; o >>= 1) { if (threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o]; __syncthreads(); }
        const double r = sh[0];
        __syncthreads();
        return r;
    };
    auto block_max = [&](double v) {
        sh[threadIdx.x] = v;
        __syncthreads();
        for (int o = 128; o > 0; o >>= 1) { if (threadIdx.x < o) sh[threadIdx.x] = fmax(sh[threadIdx.x], sh[threadIdx.x + o]); __syncthreads(); }
        const double r = sh[0];
        __syncthreads();
        return r;
    };
    const double bmc = block_max(mc), bms = block_max(ms), bc2 = block_sum(c2), bs2 = block_sum(s2);
    if (threadIdx.x == 0) {
        atomicMax((unsigned long long*)&out->max_c, (unsigned long long)__double_as_longlong(bmc));   // non-negative doubles order like their bits
        atomicMax((unsigned long long*)&out->max_s, (unsigned long long)__double_as_longlong(bms));
        atomicAdd(&out->sum_c2, bc2); atomicAdd(&out->sum_s2, bs2);
    }
    for (int h = 0; h <= 2 * SELF_HARM; ++h) {
        const double r = block_sum(re[h]), m = block_sum(im[h]);
        if (threadIdx.x == 0) { atomicAdd(&out->re[h], r); atomicAdd(&out->im[h], m); }
    }
}

}  // namespace nms

using namespace nms;

extern "C" {

nms_status nms_pipe_rates(nms_ctx* c, double* out)
{
    if (!c) return NMS_E_ARG;
    c->err[0] = 0;
    cudaSetDevice(c->device);
    if (!out) return fail(c, NMS_E_ARG, "out is NULL");
    const int blocks = c->sm_count * 2;                       // 2 x 256 threads = 16 warps per SM, one wave
    if (nms_status st = ensure(c, c->diag, sizeof(long long) * (size_t)blocks + 64)) return st;
    long long* d_cyc = (long long*)c->diag.p;
    float* d_sink = (float*)((char*)c->diag.p + sizeof(long long) * (size_t)blocks);
    unsigned* d_arrived = (unsigned*)(d_sink + 4);
    int occ = 0;
    NMS_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, RATE_KERNELS[NMS_PIPE_PHASOR_POLY], RATE_THREADS, 0));
    if (occ < 2) return fail(c, NMS_E_CUDA, "the rate kernels need two resident blocks per SM");
    std::vector<long long> h(blocks);
    for (int op = 0; op < NMS_PIPE_COUNT; ++op) {
        for (int rep = 0; rep < 2; ++rep) {                   // the first launch warms the instruction cache
            NMS_CUDA(c, cudaMemsetAsync(d_arrived, 0, sizeof(unsigned), c->stream));
            RATE_KERNELS[op]<<<blocks, RATE_THREADS, 0, c->stream>>>(d_cyc, d_sink, 0.25f, d_arrived);
            c->launches += 1;
        }
        NMS_CUDA(c, cudaGetLastError());
        NMS_CUDA(c, cudaMemcpyAsync(h.data(), d_cyc, sizeof(long long) * (size_t)blocks, cudaMemcpyDeviceToHost, c->stream));
        NMS_CUDA(c, cudaStreamSynchronize(c->stream));
        long long worst = 1;
        for (long long v : h) worst = v > worst ? v : worst;
        // operations per clock and SM: two co-resident blocks share the SM for the whole span
        out[op] = RATE_OPS[op] * 2.0 * RATE_THREADS * (double)RATE_CHAINS * (double)RATE_ITERS / (double)worst;
    }
    return NMS_OK;
}

nms_status nms_phasor_selftest(nms_ctx* c, int polynomial, int log2_n, double* out)
{
    if (!c) return NMS_E_ARG;
    c->err[0] = 0;
    cudaSetDevice(c->device);
    if (!out || log2_n < 10 || log2_n > 30) return fail(c, NMS_E_ARG, "out NULL or log2_n outside 10..30");
    if (nms_status st = ensure(c, c->diag, sizeof(SelfOut))) return st;
    NMS_CUDA(c, cudaMemsetAsync(c->diag.p, 0, sizeof(SelfOut), c->stream));
    if (polynomial) k_phasor_selftest<true><<<c->sm_count * 8, 256, 0, c->stream>>>(log2_n, (SelfOut*)c->diag.p);
    else k_phasor_selftest<false><<<c->sm_count * 8, 256, 0, c->stream>>>(log2_n, (SelfOut*)c->diag.p);
    c->launches += 1;
    NMS_CUDA(c, cudaGetLastError());
    SelfOut h;
    NMS_CUDA(c, cudaMemcpyAsync(&h, c->diag.p, sizeof(SelfOut), cudaMemcpyDeviceToHost, c->stream));
    NMS_CUDA(c, cudaStreamSynchronize(c->stream));
    const double n = (double)((int64_t)1 << log2_n);
    out[0] = h.max_c; out[1] = h.max_s; out[2] = sqrt(h.sum_c2 / n); out[3] = sqrt(h.sum_s2 / n);
    for (int k = 0; k <= 2 * SELF_HARM; ++k) out[4 + k] = sqrt(h.re[k] * h.re[k] + h.im[k] * h.im[k]) / n;
    out[21] = h.re[SELF_HARM] / n; out[22] = h.im[SELF_HARM] / n;          // e_0 itself: the mean error of cos, of -sin
    return NMS_OK;
}

}  // extern "C"
