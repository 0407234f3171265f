// landscape.cu -- landscape ingest (a1) and contagion-threshold precompute (a2).
//
// a1  fire_landscape_create : rasters -> FP64 covariates of Eq. 1 per TARGET cell + burnable bitmap
//     (I_f, psi, omega, sigma; the raster layers).
// a2  fire_params_upload    : T[p][cell][d] = min(rint(2^32 * logistic(x)), 2^32 - 1), Eq. 1,
//     x = (((b0 + b1 I_f) + b2 psi) + b3 omega_d) + b4 sigma_d, every operation one IEEE double
//     operation in this order (explicit __dmul_rn/__dadd_rn: no FMA contraction).
//
// Both kernels are HBM streams: a1 reads 13 B and writes 90 B per cell once per landscape; a2 writes
// 32 B per (p, cell) -- one DRAM sector holding the 8 directions of a target cell -- and re-reads the
// covariates of a cell once per CTA, i.e. once per `vectors_per_cta` parameter vectors (all of them on large lattices).
#include "fire_internal.cuh"

#include <new>

namespace {

constexpr double kPi = 3.14159265358979323846;

// ------------------------------------------------------------------------------------------ a1
// One thread per cell; a warp covers 32 consecutive x of one row and assembles the row's bitmap
// word with a ballot (lane = bit = x & 31, LSB = lowest x).
__global__ void __launch_bounds__(256)
fire_covariates_kernel(const uint8_t* __restrict__ veg, const float* __restrict__ slope,
                       const float* __restrict__ aspect, const float* __restrict__ wind,
                       int W, int H, int Ww,
                       uint8_t* __restrict__ flags, uint8_t* __restrict__ uphill, double* __restrict__ psi,
                       double* __restrict__ tan_slope, double* __restrict__ omega, uint32_t* __restrict__ burnable)
{
    const int lane = threadIdx.x & 31;
    const long long warp = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;   // one warp per bitmap word
    const long long nwords = (long long)H * Ww;
    if (warp >= nwords) return;
    const int y = (int)(warp / Ww), wx = (int)(warp % Ww);
    const int x = wx * 32 + lane;
    const bool inside = x < W;
    const size_t cells = (size_t)W * H;
    bool can_burn = false;
    if (inside) {
        const size_t c = (size_t)y * W + x;
        const uint8_t v = veg[c];
        const double s = (double)slope[c], a = (double)aspect[c], w = (double)wind[c];
        can_burn = (v != 0);                                              // PAPER.md:113; R-9
        flags[c] = (uint8_t)((v != 0 ? 1 : 0) | (v == 1 ? 2 : 0));       // bit1: forest indicator I_f
        // psi = cos(aspect - 315 deg) where slope > 5 deg, else 0 (R-4, R-10)
        const double five_deg = 5.0 * kPi / 180.0;
        psi[c] = (s > five_deg) ? cos(a - 7.0 * (kPi / 4.0)) : 0.0;
        tan_slope[c] = tan(s);                                            // slope/100 with slope in percent (R-8)
        uint32_t up = 0;
#pragma unroll
        for (int d = 0; d < 8; ++d) {
            const double phi = (double)d * (kPi / 4.0);                   // compass bearing of travel direction d
            omega[(size_t)d * cells + c] = cos(w - phi);                  // +1 when the target is downwind (R-6)
            // target higher than the burning cell <=> travelling against the downslope bearing (R-7, R-14)
            if (s > 0.0 && cos(phi - a) < 0.0) up |= 1u << d;
        }
        uphill[c] = (uint8_t)up;
    }
    const uint32_t word = __ballot_sync(0xFFFFFFFFu, can_burn);
    if (lane == 0) burnable[warp] = word;                                 // tail bits of a row stay zero
}

// ------------------------------------------------------------------------------------------ a2
// The table is SOURCE-indexed: thr[p][b][d] = T of the trial "burning cell b spreads in direction d",
// i.e. Eq. 1 evaluated with the covariates of the TARGET b + offset(d) ("covariates of the
// target cell"); 0 where the target is non-burnable.  The 8 outgoing trials of one burning cell are one
// 32 B DRAM sector, and a cell burns for exactly one step, so the propagation kernel
// reads every sector it needs exactly once.  Slots whose target lies outside the lattice are never
// written and never read.
//
// One thread per TARGET cell of a 32 x 8 tile, covariates in registers, loop over a group of parameter
// vectors.  The 8 thresholds of a target go through shared memory to the slots of their 8 sources, so
// that sources whose targets all lie in the tile (30 x 6 of 32 x 8) are written as whole sectors; the
// others are completed, 4 B at a time, by the neighbouring tiles (merged in L2).
#define FIRE_THR_PGROUP 64      // parameter vectors staged in shared memory at a time
constexpr int kThrTX = 32, kThrTY = 8;

// T = min(rint(2^32 / (1 + exp(-x))), 2^32 - 1) in double precision, written for the FP64 pipe: the kernel is bound by it (about 30
// double-precision operations per logistic with the library's exp and a correctly rounded reciprocal, 2.1e9 logistics per
// generation), so every step is the cheapest one that keeps the result within a few ulp of p, i.e. within ONE count and only
// when p 2^32 lies within 1e-6 of a rounding boundary (tests count these on the whole table of config 3; north_star allows <= 1):
//   exp(y), |y| <= 40 (beyond |x| = 40 the threshold is saturated either way: p 2^32 rounds to 2^32 from x = 22.9 on and to 0
//            below -22.9): y = (64 k + j) ln 2 / 64 + r with a Cody-Waite split of ln 2 / 64, 2^(j/64) from a 64-entry table in
//            shared memory, exp(r) by a Taylor polynomial of degree 5 on |r| <= ln 2 / 128 (truncation 3e-17), 2^k added to the
//            exponent field: 10 operations instead of 16;
//   1 / d:   the hardware's 20-bit estimate and two Newton steps (full double precision, not correctly rounded);
//   rint:    p 2^32 + 2^52 in ONE fused operation: the product is exact and the addition rounds it to an integer, ties to even
//            (R-11), exactly as llrint(ldexp(p, 32)) does.
__constant__ double kExp2Table[64] = {      // 2^(j/64), j = 0..63, correctly rounded
    1.0, 1.0108892860517005, 1.0218971486541166, 1.0330248790212284,
    1.0442737824274138, 1.0556451783605572, 1.0671404006768237, 1.0787607977571199,
    1.0905077326652577, 1.102382583307841, 1.1143867425958924, 1.1265216186082418,
    1.1387886347566916, 1.1511892299529827, 1.1637248587775775, 1.1763969916502812,
    1.189207115002721, 1.202156731452703, 1.215247359980469, 1.22848053610687,
    1.241857812073484, 1.255380757024691, 1.2690509571917332, 1.2828700160787783,
    1.2968395546510096, 1.3109612115247644, 1.3252366431597413, 1.339667524053303,
    1.3542555469368927, 1.3690024229745905, 1.383909881963832, 1.3989796725383112,
    1.4142135623730951, 1.42961333839197, 1.4451808069770467, 1.460917794180647,
    1.4768261459394993, 1.4929077282912648, 1.5091644275934228, 1.5255981507445384,
    1.5422108254079407, 1.559004400237837, 1.5759808451078865, 1.593142151342267,
    1.6104903319492543, 1.6280274218573478, 1.645755478153965, 1.6636765803267364,
    1.681792830507429, 1.7001063537185235, 1.718619298122478, 1.7373338352737062,
    1.7562521603732995, 1.7753764925265212, 1.7947090750031072, 1.8142521755003989,
    1.8340080864093424, 1.8539791250833855, 1.8741676341103, 1.8945759815869656,
    1.9152065613971474, 1.9360617934922943, 1.9571441241754002, 1.978456026387951
};

// N independent arguments, written step by step across them so that the N dependent chains interleave in the instruction stream
// (one chain alone waits for the latency of every operation).  kSafe = false leaves out the clamp and the saturation: the caller
// guarantees |x| < 21 (no clamp needed, and rint(p 2^32) < 2^32 because p 2^32 reaches 2^32 - 0.5 at x = 22.9 only); both
// variants run the same operations on the same values there, so they return the same bits.
template <int N, bool kSafe>
__device__ __forceinline__ void fire_thresholds_from_x(const double (&x)[N], const double* __restrict__ tbl, uint32_t (&T)[N])
{
    double y[N], t[N], r[N], q[N], d[N], rc[N];
    int n[N];
#pragma unroll
    for (int i = 0; i < N; ++i) {
        y[i] = -x[i];
        if (kSafe) {      // clamp to [-40, 40] with integer operations on the high word (the FP64 pipe is the bottleneck)
            const uint32_t yh = (uint32_t)__double2hiint(y[i]);
            if ((yh & 0x7FFFFFFFu) >= 0x40440000u) y[i] = __hiloint2double((int)((yh & 0x80000000u) | 0x40440000u), 0);
        }
    }
#pragma unroll
    for (int i = 0; i < N; ++i) t[i] = __fma_rn(y[i], 92.33248261689366, 6755399441055744.0);      // 2^52 + 2^51: low word = n = rint(64 y log2 e)
#pragma unroll
    for (int i = 0; i < N; ++i) {
        const double nf = t[i] - 6755399441055744.0;
        r[i] = __fma_rn(nf, -0.010830424667801708, y[i]);                  // ln 2 / 64, high part (24 trailing zero bits)
        r[i] = __fma_rn(nf, -2.8447437476627285e-11, r[i]);                // low part
        n[i] = __double2loint(t[i]);
    }
#pragma unroll
    for (int i = 0; i < N; ++i) q[i] = __fma_rn(8.33333333333333333333e-03, r[i], 4.16666666666666666667e-02);
#pragma unroll
    for (int i = 0; i < N; ++i) q[i] = __fma_rn(q[i], r[i], 1.66666666666666666667e-01);
#pragma unroll
    for (int i = 0; i < N; ++i) q[i] = __fma_rn(q[i], r[i], 0.5);
#pragma unroll
    for (int i = 0; i < N; ++i) q[i] = __fma_rn(q[i], r[i], 1.0);
#pragma unroll
    for (int i = 0; i < N; ++i) q[i] = __fma_rn(q[i], r[i], 1.0);
#pragma unroll
    for (int i = 0; i < N; ++i) q[i] = q[i] * tbl[n[i] & 63];
#pragma unroll
    for (int i = 0; i < N; ++i) {
        const double e = __hiloint2double(__double2hiint(q[i]) + ((n[i] >> 6) << 20), __double2loint(q[i]));   // q 2^k, |k| <= 58
        d[i] = 1.0 + e;
        asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(rc[i]) : "d"(d[i]));
    }
    // one cubic step from the 20-bit estimate: err = 1 - d rc, rc (1 + err + err^2) leaves err^3 = 2^-60
#pragma unroll
    for (int i = 0; i < N; ++i) d[i] = __fma_rn(-d[i], rc[i], 1.0);
#pragma unroll
    for (int i = 0; i < N; ++i) d[i] = __fma_rn(d[i], d[i], d[i]);
#pragma unroll
    for (int i = 0; i < N; ++i) rc[i] = __fma_rn(rc[i], d[i], rc[i]);
#pragma unroll
    for (int i = 0; i < N; ++i) {
        const double v = __fma_rn(rc[i], 4294967296.0, 4503599627370496.0);          // 2^52 + rint(p 2^32), 0 <= rint <= 2^32
        const uint32_t lo = (uint32_t)__double2loint(v), hi = (uint32_t)__double2hiint(v);
        T[i] = (kSafe && (hi & 1u)) ? 0xFFFFFFFFu : lo;                              // min(., 2^32 - 1)
    }
}

__device__ __forceinline__ uint32_t fire_threshold_from_x(double x, const double* __restrict__ tbl)
{
    const double x1[1] = { x };
    uint32_t T1[1];
    fire_thresholds_from_x<1, true>(x1, tbl, T1);
    return T1[0];
}

// x of Eq. 1 for one (target, direction): every operation one IEEE double operation, in the order of C-3
__device__ __forceinline__ uint32_t fire_threshold(double b0, double b1, double b2, double b3, double b4,
                                                   double If, double ps, double om, double sg, const double* __restrict__ tbl)
{
    const double base = __dadd_rn(__dadd_rn(b0, __dmul_rn(b1, If)), __dmul_rn(b2, ps));
    const double x = __dadd_rn(__dadd_rn(base, __dmul_rn(b3, om)), __dmul_rn(b4, sg));
    return fire_threshold_from_x(x, tbl);
}

constexpr int kThrChains = 4;      // directions evaluated side by side (4 x 2 passes; 8 at once needs 108 registers and is slower)

// The 8 thresholds of one target cell into the transposition buffer; returns the sum of the 8 probabilities (scheduling hint).
template <bool kSafe>
__device__ __forceinline__ float fire_thresholds_of_cell(double base, double b3, double b4ts, const double (&om)[8], uint32_t up, bool live,
                                                         const double* __restrict__ tbl, uint32_t (*sT)[kThrTY + 2][kThrTX + 2], int lx, int ly)
{
    float fsum = 0.0f;
#pragma unroll
    for (int h = 0; h < 8 / kThrChains; ++h) {
        double x4[kThrChains];
        uint32_t T4[kThrChains];
#pragma unroll
        for (int i = 0; i < kThrChains; ++i) {
            const int d = kThrChains * h + i;
            x4[i] = __dadd_rn(__dadd_rn(base, __dmul_rn(b3, om[d])), ((up >> d) & 1u) ? b4ts : 0.0);
        }
        fire_thresholds_from_x<kThrChains, kSafe>(x4, tbl, T4);
#pragma unroll
        for (int i = 0; i < kThrChains; ++i) {
            const int d = kThrChains * h + i;
            const uint32_t T = live ? T4[i] : 0u;
            sT[d][ly - fire_dy(d) + 1][lx - fire_dx(d) + 1] = T;      // slot d of the source = target - offset(d)
            fsum += (float)T * 2.3283064365386963e-10f;
        }
    }
    return fsum;
}
__global__ void __launch_bounds__(kThrTX * kThrTY, 4)
fire_thresholds_kernel(const float* __restrict__ beta, int P, int vectors_per_cta, int W, int H, int tiles_x,
                       const uint8_t* __restrict__ flags, const uint8_t* __restrict__ uphill,
                       const double* __restrict__ psi, const double* __restrict__ tan_slope,
                       const double* __restrict__ omega, const double* __restrict__ if_cell, uint32_t* __restrict__ thr,
                       float* __restrict__ param_mean)
{
    __shared__ double sb[FIRE_THR_PGROUP][5];
    __shared__ float sab[FIRE_THR_PGROUP][5];                             // |beta|
    __shared__ double s_exp2[64];
    __shared__ float s_mean[FIRE_THR_PGROUP];
    __shared__ uint32_t sT2[2][8][kThrTY + 2][kThrTX + 2];                // [buffer][d][source row + 1][source column + 1]
    const int tid = threadIdx.x, lx = tid & 31, ly = tid >> 5;
    // this CTA's parameter vectors: [p_begin, p_end), staged through shared memory FIRE_THR_PGROUP at a time.  The covariates of the
    // tile are loaded once per CTA (a cold DRAM round trip with nothing to overlap it), so the more vectors a CTA takes the better,
    // as long as the grid still has a few waves (the host picks vectors_per_cta)
    const int p_begin = blockIdx.y * vectors_per_cta;
    const int p_end = min(P, p_begin + vectors_per_cta);
    if (tid < 64) s_exp2[tid] = kExp2Table[tid];
    const int x0 = (int)(blockIdx.x % tiles_x) * kThrTX, y0 = (int)(blockIdx.x / tiles_x) * kThrTY;
    const int x = x0 + lx, y = y0 + ly;
    const size_t cells = (size_t)W * H;
    const bool inside = x < W && y < H;
    const size_t c = inside ? (size_t)y * W + x : 0;
    const uint32_t f = inside ? flags[c] : 0u;
    const bool live = (f & 1u) != 0;                                      // impossible to burn: T = 0
    double If = 0.0, ps = 0.0, ts = 0.0, om[8];
    uint32_t up = 0;
#pragma unroll
    for (int d = 0; d < 8; ++d) om[d] = 0.0;
    if (live) {
        If = if_cell ? if_cell[c] : ((f & 2u) ? 1.0 : 0.0);           // per-class table (fire_landscape_set_class_indicator) or forest bit
        ps = psi[c]; ts = tan_slope[c]; up = uphill[c];
#pragma unroll
        for (int d = 0; d < 8; ++d) om[d] = omega[(size_t)d * cells + c];
    }
    // largest |covariate| over the warp, in single precision (non-negative floats order like their bit patterns; a NaN wins)
    uint32_t om_bits = 0u;
#pragma unroll
    for (int d = 0; d < 8; ++d) om_bits = max(om_bits, __float_as_uint(fabsf((float)om[d])));
    const float m_om = __uint_as_float(__reduce_max_sync(0xFFFFFFFFu, om_bits));
    const float m_if = __uint_as_float(__reduce_max_sync(0xFFFFFFFFu, __float_as_uint(fabsf((float)If))));
    const float m_ps = __uint_as_float(__reduce_max_sync(0xFFFFFFFFu, __float_as_uint(fabsf((float)ps))));
    const float m_ts = __uint_as_float(__reduce_max_sync(0xFFFFFFFFu, __float_as_uint(fabsf((float)ts))));
    // the sources this thread writes out: its own cell, and (threads 0..83) one cell of the ring around the tile.  Which of
    // their 8 slots this tile holds does not depend on the parameter vector: one bit mask each, worked out once.
    int hx = -2, hy = -2;                                                 // ring cell in tile coordinates, if any
    if (tid < 2 * kThrTX) { hx = tid & 31; hy = (tid < kThrTX) ? -1 : kThrTY; }
    else if (tid < 2 * kThrTX + 2 * kThrTY) { const int k = tid - 2 * kThrTX; hx = (k < kThrTY) ? -1 : kThrTX; hy = k % kThrTY; }
    else if (tid < 2 * kThrTX + 2 * kThrTY + 4) { const int k = tid - 2 * kThrTX - 2 * kThrTY; hx = (k & 1) ? kThrTX : -1; hy = (k & 2) ? kThrTY : -1; }
    uint32_t own_mask = 0u, ring_mask = 0u;
    uint32_t ring_c = 0;                                                  // the host checks W * H < 2^31
    if (inside) {
#pragma unroll
        for (int d = 0; d < 8; ++d) {
            const int tx = lx + fire_dx(d), ty = ly + fire_dy(d);
            if (tx >= 0 && tx < kThrTX && ty >= 0 && ty < kThrTY) own_mask |= 1u << d;
        }
    }
    if (hx != -2) {
        const int gx = x0 + hx, gy = y0 + hy;
        if (gx >= 0 && gx < W && gy >= 0 && gy < H) {
            ring_c = (uint32_t)gy * (uint32_t)W + (uint32_t)gx;
#pragma unroll
            for (int d = 0; d < 8; ++d) {
                const int tx = hx + fire_dx(d), ty = hy + fire_dy(d);
                if (tx >= 0 && tx < kThrTX && ty >= 0 && ty < kThrTY) ring_mask |= 1u << d;
            }
        }
    }
    const int hx1 = hx + 1, hy1 = hy + 1;
    for (int p0 = p_begin; p0 < p_end; p0 += FIRE_THR_PGROUP) {
    const int np = min(FIRE_THR_PGROUP, p_end - p0);
    __syncthreads();                                                      // the previous chunk's last reads of sb, s_mean and sT2
    for (int i = tid; i < np * 5; i += kThrTX * kThrTY) { const float bv = beta[(size_t)p0 * 5 + i]; sb[i / 5][i % 5] = (double)bv; sab[i / 5][i % 5] = fabsf(bv); }
    if (tid < FIRE_THR_PGROUP) s_mean[tid] = 0.0f;
    __syncthreads();
    for (int q = 0; q < np; ++q) {
        const double b0 = sb[q][0], b1 = sb[q][1], b2 = sb[q][2], b3 = sb[q][3], b4 = sb[q][4];
        uint32_t (*sT)[kThrTY + 2][kThrTX + 2] = sT2[q & 1];         // double-buffered: one barrier per parameter vector
        float fsum = 0.0f;
        // Eq. 1 for the 8 directions of this target: x in the order of C-3, one IEEE operation each; non-burnable targets run
        // the same arithmetic on zeros and are masked at the end (no branch: the chains of 4 directions interleave).
        // b4 sigma_d is b4 tan(slope) or b4 0 = +-0; adding +-0 changes nothing (x = +-0 gives the same threshold).
        const double base = __dadd_rn(__dadd_rn(b0, __dmul_rn(b1, If)), __dmul_rn(b2, ps));
        const double b4ts = __dmul_rn(b4, ts);
        // |x| <= |b0| + |b1| max|If| + |b2| max|psi| + |b3| max|omega| + |b4| max|tan| over the warp (single precision is enough
        // for a bound): below 20, neither the clamp (|x| >= 40) nor the saturation (x >= 22.9) can act.  NaN compares false.
        const float bound = fmaf(sab[q][4], m_ts, fmaf(sab[q][3], m_om, fmaf(sab[q][2], m_ps, fmaf(sab[q][1], m_if, sab[q][0]))));
        const bool fast = __all_sync(0xFFFFFFFFu, bound < 20.0f);
        if (fast) fsum = fire_thresholds_of_cell<false>(base, b3, b4ts, om, up, live, s_exp2, sT, lx, ly);
        else fsum = fire_thresholds_of_cell<true>(base, b3, b4ts, om, up, live, s_exp2, sT, lx, ly);
        // scheduling hint only (never enters a result): sum of the contagion probabilities of this parameter vector
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) fsum += __shfl_xor_sync(0xFFFFFFFFu, fsum, o);
        if (lx == 0) atomicAdd(&s_mean[q], fsum);
        __syncthreads();
        uint32_t* const tp = thr + (size_t)(p0 + q) * cells * 8;
        if (own_mask == 0xFFu) {                                          // own cell as a source: a whole sector
            uint32_t* const out = tp + c * 8;
            reinterpret_cast<uint4*>(out)[0] = make_uint4(sT[0][ly + 1][lx + 1], sT[1][ly + 1][lx + 1], sT[2][ly + 1][lx + 1], sT[3][ly + 1][lx + 1]);
            reinterpret_cast<uint4*>(out)[1] = make_uint4(sT[4][ly + 1][lx + 1], sT[5][ly + 1][lx + 1], sT[6][ly + 1][lx + 1], sT[7][ly + 1][lx + 1]);
        } else if (own_mask) {                                            // on the tile's edge: the slots whose targets are in the tile
            uint32_t* const out = tp + c * 8;
#pragma unroll
            for (int d = 0; d < 8; ++d)
                if ((own_mask >> d) & 1u) out[d] = sT[d][ly + 1][lx + 1];
        }
        if (ring_mask) {                                                  // one cell of the ring around the tile
            uint32_t* const out = tp + (size_t)ring_c * 8;
#pragma unroll
            for (int d = 0; d < 8; ++d)
                if ((ring_mask >> d) & 1u) out[d] = sT[d][hy1][hx1];
        }
    }
    __syncthreads();
    if (tid < np) atomicAdd(param_mean + p0 + tid, s_mean[tid]);
    }
}

// Test hook: the table of one parameter vector in TARGET-indexed form out[c][d] = T(target c, direction d).
// Entries whose source c - offset(d) lies outside the lattice are in no sector; they are evaluated here by the
// same device function.
__global__ void __launch_bounds__(256)
fire_thresholds_gather_kernel(const float* __restrict__ beta5, int W, int H,
                              const uint8_t* __restrict__ flags, const uint8_t* __restrict__ uphill,
                              const double* __restrict__ psi, const double* __restrict__ tan_slope,
                              const double* __restrict__ omega, const double* __restrict__ if_cell, const uint32_t* __restrict__ thr_p,
                              uint32_t* __restrict__ out)
{
    const size_t cells = (size_t)W * H;
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;      // one thread per (cell, d)
    if (i >= cells * 8) return;
    const size_t c = i >> 3;
    const int d = (int)(i & 7), x = (int)(c % W), y = (int)(c / W);
    const int sx = x - fire_dx(d), sy = y - fire_dy(d);
    uint32_t T;
    if (sx >= 0 && sx < W && sy >= 0 && sy < H) {
        T = thr_p[((size_t)sy * W + sx) * 8 + d];
    } else {
        const uint32_t f = flags[c];
        T = 0u;
        if (f & 1u)
            T = fire_threshold((double)beta5[0], (double)beta5[1], (double)beta5[2], (double)beta5[3], (double)beta5[4],
                               if_cell ? if_cell[c] : ((f & 2u) ? 1.0 : 0.0), psi[c], omega[(size_t)d * cells + c], ((uphill[c] >> d) & 1u) ? tan_slope[c] : 0.0, kExp2Table);
    }
    out[i] = T;
}

// f4 variant (PAPER.md:87 read literally): uphill in direction d <=> slope > 0 and elevation[target] > elevation[source],
// source = target - offset(d) inside the lattice; replaces the aspect-based mask written by fire_covariates_kernel.
__global__ void __launch_bounds__(256)
fire_uphill_from_dem_kernel(const float* __restrict__ elevation, const double* __restrict__ tan_slope, int W, int H,
                            uint8_t* __restrict__ uphill)
{
    const size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= (size_t)W * H) return;
    const int x = (int)(c % W), y = (int)(c / W);
    uint32_t up = 0u;
    if (tan_slope[c] > 0.0) {                                              // tan(s) > 0 <=> s > 0 on [0, pi/2)
        const float z = elevation[c];
#pragma unroll
        for (int d = 0; d < 8; ++d) {
            const int sx = x - fire_dx(d), sy = y - fire_dy(d);
            if (sx >= 0 && sx < W && sy >= 0 && sy < H && z > elevation[(size_t)sy * W + sx]) up |= 1u << d;
        }
    }
    uphill[c] = (uint8_t)up;
}

struct class_table { float w[256]; };
__global__ void __launch_bounds__(256)
fire_class_indicator_kernel(const uint8_t* __restrict__ veg, const class_table tab, size_t cells, double* __restrict__ if_cell)
{
    const size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c < cells) if_cell[c] = (double)tab.w[veg[c]];
}

}  // namespace

extern "C" int fire_landscape_set_class_indicator(fire_landscape* L, const float* class_if_host, int32_t n_classes, void* stream)
{
    if (L == nullptr || n_classes < 0 || n_classes > 256 || (n_classes > 0 && class_if_host == nullptr)) return FIRE_EINVAL;
    if (L->sticky) return L->sticky;
    fire_device_guard g(L->device);
    if (!g.ok) return FIRE_ECUDA;
    cudaStream_t st = (cudaStream_t)stream;
    L->P = 0;                                                              // any table built before is stale
    if (n_classes == 0) {                                                  // back to the paper's indicator: forest (class 1) only
        FIRE_CUDA_TRY(L, cudaStreamSynchronize(st));
        if (L->if_cell) { cudaFree(L->if_cell); L->if_cell = nullptr; }
        return FIRE_OK;
    }
    class_table tab;
    for (int v = 0; v < 256; ++v) tab.w[v] = v < n_classes ? class_if_host[v] : 0.0f;
    if (L->if_cell == nullptr) {
        size_t cap = 0;
        int rc = fire_reserve(L, (void**)&L->if_cell, &cap, L->cells * sizeof(double));
        if (rc != FIRE_OK) return rc;
    }
    fire_class_indicator_kernel<<<(unsigned)((L->cells + 255) / 256), 256, 0, st>>>(L->veg_class, tab, L->cells, L->if_cell);
    FIRE_CUDA_TRY(L, cudaGetLastError());
    L->launches += 1;
    return FIRE_OK;
}

extern "C" int fire_landscape_set_elevation(fire_landscape* L, const float* elevation, void* stream)
{
    if (L == nullptr || elevation == nullptr) return FIRE_EINVAL;
    if (L->sticky) return L->sticky;
    fire_device_guard g(L->device);
    if (!g.ok) return FIRE_ECUDA;
    fire_uphill_from_dem_kernel<<<(unsigned)((L->cells + 255) / 256), 256, 0, (cudaStream_t)stream>>>(elevation, L->tan_slope, L->W, L->H, L->uphill);
    FIRE_CUDA_TRY(L, cudaGetLastError());
    L->launches += 1;
    L->P = 0;                                                              // any table built before is stale
    return FIRE_OK;
}

// ----------------------------------------------------------------------------------------------
extern "C" int fire_landscape_destroy(fire_landscape* L)
{
    if (L == nullptr) return FIRE_EINVAL;
    fire_device_guard g(L->device);
    if (g.ok) {
        cudaDeviceSynchronize();
        void* ptrs[] = { L->flags, L->uphill, L->psi, L->tan_slope, L->omega, L->burnable, L->thr, L->beta_dev,
                         L->work_counter, L->status, L->spill, L->rescue_planes, L->ref_area, L->counts_scratch,
                         L->burnable_tiles, L->tiles, L->order, L->param_mean, L->veg_class, L->ktime, L->gt_planes, L->if_cell,
                         L->gen_buf };
        for (void* p : ptrs) if (p) cudaFree(p);
        if (L->prof_ev[0]) for (int i = 0; i < 2 * 64; ++i) if (L->prof_ev[i]) cudaEventDestroy(L->prof_ev[i]);
        (void)cudaGetLastError();
    }
    delete L;
    return g.ok ? FIRE_OK : FIRE_ECUDA;
}

extern "C" int fire_landscape_create(fire_landscape** out, const uint8_t* veg, const float* slope,
                                     const float* aspect, const float* wind, int32_t W, int32_t H, void* stream)
{
    if (out == nullptr) return FIRE_EINVAL;
    *out = nullptr;
    if (!veg || !slope || !aspect || !wind || W < 1 || H < 1 || W > 8192 || H > 8192) return FIRE_EINVAL;
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) { (void)cudaGetLastError(); return FIRE_ECUDA; }   // no CUDA device: no fallback
    fire_landscape* L = new (std::nothrow) fire_landscape();
    if (L == nullptr) return FIRE_ENOMEM;
    L->device = dev;
    L->W = W; L->H = H; L->Ww = (W + 31) / 32; L->cells = (size_t)W * H;
    L->Tw = (W + 7) / 8; L->Th = (H + 7) / 8;
    int sms = 0;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1) {
        (void)cudaGetLastError(); delete L; return FIRE_ECUDA;
    }
    L->num_sms = sms;
    const size_t n = L->cells, nw = (size_t)H * L->Ww;
    bool ok = cudaMalloc(&L->flags, n) == cudaSuccess && cudaMalloc(&L->uphill, n) == cudaSuccess &&
              cudaMalloc(&L->psi, n * 8) == cudaSuccess && cudaMalloc(&L->tan_slope, n * 8) == cudaSuccess &&
              cudaMalloc(&L->omega, n * 64) == cudaSuccess && cudaMalloc(&L->burnable, nw * 4) == cudaSuccess &&
              cudaMalloc(&L->veg_class, n) == cudaSuccess &&
              cudaMalloc(&L->work_counter, 4 * sizeof(unsigned int)) == cudaSuccess &&
              cudaMalloc(&L->ref_area, 4 * sizeof(uint32_t)) == cudaSuccess;
    if (!ok) { (void)cudaGetLastError(); fire_landscape_destroy(L); return FIRE_ENOMEM; }
    cudaStream_t st = (cudaStream_t)stream;
    const long long threads = (long long)nw * 32;
    const int block = 256;
    const unsigned grid = (unsigned)((threads + block - 1) / block);
    if (cudaMemcpyAsync(L->veg_class, veg, n, cudaMemcpyDeviceToDevice, st) != cudaSuccess) { (void)cudaGetLastError(); fire_landscape_destroy(L); return FIRE_ECUDA; }
    fire_covariates_kernel<<<grid, block, 0, st>>>(veg, slope, aspect, wind, W, H, L->Ww, L->flags, L->uphill, L->psi,
                                                   L->tan_slope, L->omega, L->burnable);
    L->launches += 1;
    if (cudaGetLastError() != cudaSuccess) { fire_landscape_destroy(L); return FIRE_ECUDA; }
    *out = L;
    return FIRE_OK;
}

extern "C" int fire_params_upload(fire_landscape* L, const float* beta, int32_t P, void* stream)
{
    if (L == nullptr || beta == nullptr || P < 1) return FIRE_EINVAL;
    if (L->sticky) return L->sticky;
    fire_device_guard g(L->device);
    if (!g.ok) return FIRE_ECUDA;
    if ((size_t)P * L->cells >= ((size_t)1 << 32)) return FIRE_EINVAL;   // sectors are addressed by 32-bit indices (2^32 sectors = 137 GB)
    const size_t bytes = (size_t)P * L->cells * 32;
    if (L->thr_capacity < bytes) {
        // growing the table must not race with work still using the old one
        FIRE_CUDA_TRY(L, cudaStreamSynchronize((cudaStream_t)stream));
        L->P = 0;
        int rc = fire_reserve(L, (void**)&L->thr, &L->thr_capacity, bytes);
        if (rc != FIRE_OK) return rc;
    }
    if (L->beta_capacity < (size_t)P * 5 * sizeof(float)) {
        FIRE_CUDA_TRY(L, cudaStreamSynchronize((cudaStream_t)stream));
        int rc = fire_reserve(L, (void**)&L->beta_dev, &L->beta_capacity, (size_t)P * 5 * sizeof(float));
        if (rc != FIRE_OK) return rc;
    }
    // the handle keeps its own copy of beta (fire_thresholds_download evaluates the lattice-edge entries from it)
    FIRE_CUDA_TRY(L, cudaMemcpyAsync(L->beta_dev, beta, (size_t)P * 5 * sizeof(float), cudaMemcpyDeviceToDevice, (cudaStream_t)stream));
    if (L->param_mean_capacity < (size_t)P * sizeof(float)) {
        FIRE_CUDA_TRY(L, cudaStreamSynchronize((cudaStream_t)stream));
        int rc = fire_reserve(L, (void**)&L->param_mean, &L->param_mean_capacity, (size_t)P * sizeof(float));
        if (rc != FIRE_OK) return rc;
    }
    FIRE_CUDA_TRY(L, cudaMemsetAsync(L->param_mean, 0, (size_t)P * sizeof(float), (cudaStream_t)stream));
    const int tiles_x = (L->W + kThrTX - 1) / kThrTX, tiles_y = (L->H + kThrTY - 1) / kThrTY;
    // vectors per CTA: as many as leave about eight waves of CTAs (4 resident per SM), at least 8 (one group of the old scheme)
    const long long tiles = (long long)tiles_x * tiles_y;
    long long gy = (8ll * 4 * L->num_sms + tiles - 1) / tiles;
    if (gy < 1) gy = 1;
    if (gy > (P + 7) / 8) gy = (P + 7) / 8;
    const int vectors_per_cta = (int)((P + gy - 1) / gy);
    dim3 grid((unsigned)tiles, (unsigned)((P + vectors_per_cta - 1) / vectors_per_cta));
    fire_thresholds_kernel<<<grid, kThrTX * kThrTY, 0, (cudaStream_t)stream>>>(L->beta_dev, P, vectors_per_cta, L->W, L->H, tiles_x, L->flags,
                                                                                L->uphill, L->psi, L->tan_slope, L->omega, L->if_cell, L->thr, L->param_mean);
    L->launches += 1;
    FIRE_CUDA_TRY(L, cudaGetLastError());
    L->P = P;
    return FIRE_OK;
}

extern "C" int fire_thresholds_download(fire_landscape* L, int32_t p, uint32_t* out, void* stream)
{
    if (L == nullptr || out == nullptr) return FIRE_EINVAL;
    if (L->sticky) return L->sticky;
    if (L->P == 0 || p < 0 || p >= L->P) return FIRE_ESTATE;
    fire_device_guard g(L->device);
    if (!g.ok) return FIRE_ECUDA;
    const size_t n = L->cells * 8;
    fire_thresholds_gather_kernel<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(
        L->beta_dev + (size_t)p * 5, L->W, L->H, L->flags, L->uphill, L->psi, L->tan_slope, L->omega, L->if_cell,
        L->thr + (size_t)p * L->cells * 8, out);
    L->launches += 1;
    FIRE_CUDA_TRY(L, cudaGetLastError());
    return FIRE_OK;
}
