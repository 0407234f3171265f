// fire_internal.cuh -- private declarations of libfire (sm_100a).  Not installed; the public
// surface is include/fire.h.  Nothing under oracle/ is included, linked or called from here.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "fire.h"

// ---------------------------------------------------------------------------------------------
// Handle.  All pointers are device memory owned by the handle.
// ---------------------------------------------------------------------------------------------
struct fire_landscape {
    int device;
    int W, H, Ww;            // lattice width/height in cells, words per bitmap row = ceil(W/32)
    int num_sms;
    size_t cells;            // W*H

    // a1: covariates of Eq. 1 per TARGET cell, structure of arrays, FP64
    uint8_t*  flags;         // [cells]  bit0 burnable, bit1 forest (I_f)
    uint8_t*  uphill;        // [cells]  bit d set iff travelling in direction d into this cell goes uphill
    double*   psi;           // [cells]
    double*   tan_slope;     // [cells]
    double*   omega;         // [8][cells]  cos(wind - phi_d)
    uint32_t* burnable;      // [H][Ww] bitmap
    double*   if_cell;       // [cells] I_f of the cell's class (fire_landscape_set_class_indicator), or null = forest bit of `flags`

    // a2: thresholds, [P][cells][8] u32, SOURCE-indexed: thr[p][b][d] = T(target b + offset(d), direction d);
    // one 32 B DRAM sector holds the 8 outgoing trials of a burning cell b
    uint32_t* thr;
    size_t    thr_capacity;  // bytes allocated
    int       P;             // 0 until fire_params_upload
    float*    beta_dev;      // [P][5] staging (device copy made by the caller's pointer -> ours)
    size_t    beta_capacity;

    // a3-a6: propagation scratch
    int Tw, Th;                   // 8 x 8-cell tiles per row / column of the lattice: ceil(W/8), ceil(H/8)
    uint64_t* burnable_tiles;     // [Th][Tw] burnable bitmap in tile layout: bit (y&7)*8 + (x&7) of tile (y>>3, x>>3)
    uint64_t* tiles;              // [S][Th][Tw] susceptible plane (burnable & ~burned) of every simulation of a batch
    size_t    tiles_capacity;     // bytes
    uint32_t* order;              // [S] launch order of the simulations (largest expected first)
    size_t    order_capacity;     // bytes
    float*    param_mean;         // [P] mean contagion probability per parameter vector (written by fire_params_upload)
    size_t    param_mean_capacity;
    unsigned int* work_counter;   // [4] simulations taken by the fast kernel, simulations handed to the rescue kernel, 2 spare
    uint32_t* status;             // [S] 0 = finished by the fast kernel, 1 = needs the rescue kernel
    size_t    status_capacity;    // entries
    uint32_t* spill;              // per resident CTA: frontier + success lists beyond shared memory
    size_t    spill_capacity;     // bytes
    uint32_t* rescue_planes;      // rescue kernel: 2 burning planes per rescue CTA, kept all-zero between sims
    size_t    rescue_capacity;    // bytes

    // f3: fuel-dependent burn-out times (fire_set_burn_time)
    uint8_t*  veg_class;          // [cells] the caller's vegetation classes (kept: burn times are per class)
    uint8_t*  ktime;              // [cells] burn time - 1 of the cell's class
    uint32_t* gt_planes;          // [7][H][Ww] bit set iff burn time > j + 1
    size_t    gt_capacity;
    int       burn_kmax;          // largest burn time set; <= 1 = the base model (every cell burns one step)
    int32_t*  out_time;           // fire_set_time_output: the caller's [S][H][W] ignition-time array, or null
    const uint32_t* fit_ref;      // fire_set_fused_counts: the caller's reference bitmap and [S][2] counts, or null
    uint32_t* fit_counts;

    // a7: fitness scratch
    uint32_t* ref_area;           // [1]
    uint32_t* counts_scratch;     // [S][2] when the caller passes out_counts = NULL
    size_t    counts_capacity;    // entries of 2 x u32

    // end-to-end path (fire_generation_host): device staging owned by the handle
    void*     gen_buf;
    size_t    gen_capacity;

    // launch geometry knobs (fire_set_launch_geometry) and test knobs
    int threads_per_cta;          // 0 = default
    int ctas_per_sm;              // 0 = default
    int list_capacity;            // total frontier-list capacity per CTA (0 = default); tests shrink it to force the rescue path
    int kernel_family;            // fire_set_kernel: 0 = automatic, 1 = two-phase kernel, 2 = asynchronous-warp kernel
    int schedule;                 // 0 = largest expected fires first, 1 = batch order
    int list_shared;              // shared-memory part of it (0 = default); tests shrink it to force the global spill

    // optional device timing of the propagation kernel alone (fire_set_profiling / fire_profile_read)
    int          prof_enabled;
    int          prof_count;               // event pairs recorded since the last read
    cudaEvent_t  prof_ev[2 * 64];

    int64_t launches;             // kernels enqueued so far
    int     sticky;               // first CUDA error seen (as FIRE_E*), 0 if none
};

// ---------------------------------------------------------------------------------------------
// Error plumbing: never throw, never abort, never print.
// ---------------------------------------------------------------------------------------------
#define FIRE_CUDA_TRY(L, expr)                                            \
    do {                                                                  \
        cudaError_t e__ = (expr);                                         \
        if (e__ != cudaSuccess) {                                         \
            int c__ = (e__ == cudaErrorMemoryAllocation) ? FIRE_ENOMEM : FIRE_ECUDA; \
            if ((L) != nullptr && (L)->sticky == 0 && c__ == FIRE_ECUDA) (L)->sticky = c__; \
            (void)cudaGetLastError();                                     \
            return c__;                                                   \
        }                                                                 \
    } while (0)

// grow-only device buffer
static inline int fire_reserve(fire_landscape* L, void** p, size_t* cap, size_t bytes)
{
    if (*cap >= bytes && *p != nullptr) return FIRE_OK;
    if (*p) { cudaFree(*p); *p = nullptr; *cap = 0; }
    cudaError_t e = cudaMalloc(p, bytes ? bytes : 1);
    if (e != cudaSuccess) { (void)cudaGetLastError(); *p = nullptr; return FIRE_ENOMEM; }
    *cap = bytes;
    (void)L;
    return FIRE_OK;
}

struct fire_device_guard {
    int prev; bool ok;
    explicit fire_device_guard(int dev) : prev(-1), ok(false) {
        if (cudaGetDevice(&prev) != cudaSuccess) { (void)cudaGetLastError(); return; }
        if (prev != dev && cudaSetDevice(dev) != cudaSuccess) { (void)cudaGetLastError(); return; }
        ok = true;
    }
    ~fire_device_guard() { if (ok && prev >= 0) cudaSetDevice(prev); }
};

// ---------------------------------------------------------------------------------------------
// Geometry (C-2).  d = 0..7 = N, NE, E, SE, S, SW, W, NW = direction of travel from the
// burning cell to the target; row 0 is north, x grows east: target = source + (dx, dy).
// ---------------------------------------------------------------------------------------------
__host__ __device__ __forceinline__ int fire_dx(int d) { return (d == 1 || d == 2 || d == 3) ? 1 : ((d == 5 || d == 6 || d == 7) ? -1 : 0); }
__host__ __device__ __forceinline__ int fire_dy(int d) { return (d == 3 || d == 4 || d == 5) ? 1 : ((d == 7 || d == 0 || d == 1) ? -1 : 0); }

// ---------------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon et al., SC'11; the Random123 generator of PAPER.md:139-141).  Written from
// the round description: two 32x32->64 products per round, xor with the other counter words and the
// round key, key bumped by the Weyl constants before every round but the first.
// ---------------------------------------------------------------------------------------------
struct philox_out { uint32_t r0, r1, r2, r3; };

__device__ __forceinline__ philox_out philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                                    uint32_t k0, uint32_t k1)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint64_t a = (uint64_t)c0 * 0xD2511F53ull;   // IMAD.WIDE.U32
        const uint64_t b = (uint64_t)c2 * 0xCD9E8D57ull;
        const uint32_t n0 = (uint32_t)(b >> 32) ^ c1 ^ k0; // LOP3
        const uint32_t n2 = (uint32_t)(a >> 32) ^ c3 ^ k1;
        c1 = (uint32_t)b;
        c3 = (uint32_t)a;
        c0 = n0;
        c2 = n2;
        k0 += 0x9E3779B9u;                                 // the bump after round 9 is dead code
        k1 += 0xBB67AE85u;
    }
    philox_out o; o.r0 = c0; o.r1 = c1; o.r2 = c2; o.r3 = c3;
    return o;
}

// Random word of trial (seed, sim, step, target cell, d): word d&3 of
// Philox4x32-10(counter = (cell, step, sim, d>>2), key = (seed lo, seed hi))   (C-1)
__device__ __forceinline__ uint32_t fire_rnd(uint32_t key_lo, uint32_t key_hi, uint32_t sim, uint32_t step,
                                             uint32_t cell, int d)
{
    const philox_out o = philox4x32_10(cell, step, sim, (uint32_t)(d >> 2), key_lo, key_hi);
    const int w = d & 3;
    const uint32_t lo = (w & 1) ? o.r1 : o.r0;
    const uint32_t hi = (w & 1) ? o.r3 : o.r2;
    return (w & 2) ? hi : lo;
}

// A trial succeeds iff rnd < T, and T = 2^32 - 1 means certain (R-11).
__device__ __forceinline__ bool fire_trial(uint32_t rnd, uint32_t T) { return rnd < T || T == 0xFFFFFFFFu; }

