// fitness.cu -- fitness reduction (a7) and per-candidate statistics (a8).
//
// Eq. 2: delta = (#(A u A*) - #(A n A*)) / #A with A the reference burnt map,
// A* the simulated one and # the number of burnt cells.  With I = #(A n A*), N = #A, N* = #A*:
// #(A u A*) - #(A n A*) = N + N* - 2I.  The integers come from popcounts of the bit-packed maps;
// the score is ONE IEEE float divide of those integers (C-5).
//
// The counting kernel is a pure HBM stream: it reads S*H*ceil(W/32)*4 bytes once with 16 B loads;
// the reference map (one plane) stays in L2.
#include "fire_internal.cuh"

#include <atomic>

// Scratch of fire_fitness_static, the entry point that allocates nothing (fire.h): counts (I, N*) of up to
// FIRE_FITNESS_STATIC_MAX_SIMS simulations, then #A of the reference map in the first word of a 256 B tail.  Every GPU that
// loads the library holds these 128.25 KiB until the process exits.  In host code this name is a host-side stand-in, not a
// device address: the address a kernel can use comes from cudaGetSymbolAddress (fire_static_scratch below).
static __device__ __align__(256) uint32_t g_fitness_static_scratch[2 * FIRE_FITNESS_STATIC_MAX_SIMS + 64];

namespace {

__device__ __forceinline__ uint32_t warp_sum(uint32_t v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, o);
    return v;
}

// grid = (chunks, S); each CTA counts a contiguous chunk of one simulation's plane and adds its
// partial sums into counts[s] = (I, N*).  Integer atomics: the result does not depend on order.
__global__ void __launch_bounds__(256)
fire_fitness_counts_kernel(const uint32_t* __restrict__ reference, const uint32_t* __restrict__ burned,
                           size_t nw, uint32_t words_per_cta, uint32_t* __restrict__ counts)
{
    const size_t s = blockIdx.y;
    const size_t lo = (size_t)blockIdx.x * words_per_cta;
    const size_t hi = (lo + words_per_cta < nw) ? lo + words_per_cta : nw;
    const uint32_t* b = burned + s * nw;
    uint32_t inter = 0, area = 0;
    // 16 B vector body when the plane offset is 16 B aligned (nw % 4 == 0 keeps every sim aligned)
    if ((nw & 3) == 0 && (words_per_cta & 3) == 0 &&
        ((reinterpret_cast<uintptr_t>(burned) | reinterpret_cast<uintptr_t>(reference)) & 15) == 0) {
        const uint4* b4 = reinterpret_cast<const uint4*>(b + lo);
        const uint4* r4 = reinterpret_cast<const uint4*>(reference + lo);
        const size_t n4 = (hi - lo) >> 2;
        for (size_t i = threadIdx.x; i < n4; i += blockDim.x) {
            const uint4 v = __ldcs(b4 + i);            // streamed once
            const uint4 r = __ldg(r4 + i);
            area += __popc(v.x) + __popc(v.y) + __popc(v.z) + __popc(v.w);
            inter += __popc(v.x & r.x) + __popc(v.y & r.y) + __popc(v.z & r.z) + __popc(v.w & r.w);
        }
    } else {
        for (size_t i = lo + threadIdx.x; i < hi; i += blockDim.x) {
            const uint32_t v = b[i], r = __ldg(reference + i);
            area += __popc(v);
            inter += __popc(v & r);
        }
    }
    inter = warp_sum(inter); area = warp_sum(area);
    __shared__ uint32_t sh[2][8];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0) { sh[0][warp] = inter; sh[1][warp] = area; }
    __syncthreads();
    if (warp == 0) {
        const int nwarps = blockDim.x >> 5;
        uint32_t a = lane < nwarps ? sh[0][lane] : 0u, c = lane < nwarps ? sh[1][lane] : 0u;
        a = warp_sum(a); c = warp_sum(c);
        if (lane == 0) {
            if (a) atomicAdd(counts + 2 * s, a);
            if (c) atomicAdd(counts + 2 * s + 1, c);
        }
    }
}

// #A of the reference map: grid-stride popcount, one integer atomic per CTA (*out zeroed before the launch).
__global__ void __launch_bounds__(256)
fire_reference_area_kernel(const uint32_t* __restrict__ reference, size_t nw, uint32_t* __restrict__ out)
{
    uint32_t n = 0;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nw; i += (size_t)gridDim.x * blockDim.x)
        n += __popc(__ldg(reference + i));
    n = warp_sum(n);
    __shared__ uint32_t sh[8];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0) sh[warp] = n;
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t t = 0;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) t += sh[w];
        if (t) atomicAdd(out, t);
    }
}

__global__ void __launch_bounds__(256)
fire_fitness_score_kernel(const uint32_t* __restrict__ counts, const uint32_t* __restrict__ ref_area, int S,
                          int metric, float* __restrict__ score, uint32_t* __restrict__ out_ref_area)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    const uint32_t N = *ref_area;
    if (s == 0 && out_ref_area) *out_ref_area = N;
    if (s >= S) return;
    const uint32_t I = counts[2 * s], Ns = counts[2 * s + 1];
    const uint32_t uni = N + Ns - I;
    score[s] = (metric == FIRE_METRIC_DELTA) ? __fdiv_rn((float)(uni - I), (float)N)      // Eq. 2
                                             : __fdiv_rn((float)I, (float)uni);           // Jaccard
}

// a8: one warp per candidate; x = N + N* - 2I per replicate, sums in u64 (exact), then
// mean = sum x / (R N), var = (R sum x^2 - (sum x)^2) / (R (R-1)) / N^2, one IEEE op per step (R-16).
__global__ void __launch_bounds__(256)
fire_group_stats_kernel(const uint32_t* __restrict__ counts, uint32_t N, int G, int R,
                        unsigned long long* __restrict__ sums, double* __restrict__ mean_var)
{
    const int g = (int)((blockIdx.x * (size_t)blockDim.x + threadIdx.x) >> 5);
    const int lane = threadIdx.x & 31;
    if (g >= G) return;
    unsigned long long sx = 0, sxx = 0;
    for (int r = lane; r < R; r += 32) {
        const size_t k = (size_t)g * R + r;
        const unsigned long long I = counts[2 * k], Ns = counts[2 * k + 1];
        const unsigned long long x = (unsigned long long)N + Ns - 2ull * I;
        sx += x; sxx += x * x;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        sx += __shfl_xor_sync(0xFFFFFFFFu, sx, o);
        sxx += __shfl_xor_sync(0xFFFFFFFFu, sxx, o);
    }
    if (lane == 0) {
        sums[2 * g] = sx; sums[2 * g + 1] = sxx;
        const double mean = __ddiv_rn((double)sx, __dmul_rn((double)R, (double)N));
        // numerator R sum x^2 - (sum x)^2 >= 0 as a 128-bit integer (x reaches 2 W H: the 64-bit expression wraps from
        // R = 33 on an 8192 x 8192 lattice); one conversion to double when it fits 64 bits (always, at BASELINE's sizes)
        const unsigned long long a_lo = (unsigned long long)R * sxx, a_hi = __umul64hi((unsigned long long)R, sxx);
        const unsigned long long b_lo = sx * sx, b_hi = __umul64hi(sx, sx);
        const unsigned long long n_lo = a_lo - b_lo, n_hi = a_hi - b_hi - (a_lo < b_lo ? 1ull : 0ull);
        const double num = n_hi == 0ull ? (double)n_lo : __fma_rn((double)n_hi, 18446744073709551616.0, (double)n_lo);
        double var = __ddiv_rn(num, (double)((unsigned long long)R * (unsigned long long)(R - 1)));
        var = __ddiv_rn(var, __dmul_rn((double)N, (double)N));
        mean_var[2 * g] = mean; mean_var[2 * g + 1] = var;
    }
}

// Hazard map (f4): per-cell number of maps in which the cell is burnt.  One thread per bitmap word and slab of maps:
// the 32 counts of the word live in registers while the slab streams by (one coalesced 4 B load per map), then go to the output
// with one integer atomic each.
__global__ void __launch_bounds__(256)
fire_burn_count_kernel(const uint32_t* __restrict__ burned, size_t nw, int W, int Ww, int S, int slab, uint32_t* __restrict__ out)
{
    const size_t wi = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (wi >= nw) return;
    const int s0 = blockIdx.y * slab, s1 = min(S, s0 + slab);
    uint32_t cnt[32];
#pragma unroll
    for (int b = 0; b < 32; ++b) cnt[b] = 0u;
    for (int s = s0; s < s1; ++s) {
        const uint32_t w = __ldcs(burned + (size_t)s * nw + wi);
#pragma unroll
        for (int b = 0; b < 32; ++b) cnt[b] += (w >> b) & 1u;
    }
    const int y = (int)(wi / Ww), x0 = (int)(wi % Ww) * 32;
#pragma unroll
    for (int b = 0; b < 32; ++b)
        if (x0 + b < W && cnt[b]) atomicAdd(out + (size_t)y * W + x0 + b, cnt[b]);
}

}  // namespace

extern "C" int fire_burn_count(fire_landscape* L, const uint32_t* burned, int32_t S, uint32_t* out_count, void* stream)
{
    if (L == nullptr || burned == nullptr || out_count == nullptr || S < 1) return FIRE_EINVAL;
    if (L->sticky) return L->sticky;
    fire_device_guard g(L->device);
    if (!g.ok) return FIRE_ECUDA;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t nw = (size_t)L->H * L->Ww;
    FIRE_CUDA_TRY(L, cudaMemsetAsync(out_count, 0, L->cells * sizeof(uint32_t), st));
    const int slab = 64;
    const unsigned gy = (unsigned)((S + slab - 1) / slab);
    for (unsigned y0 = 0; y0 < gy; y0 += 65535) {                           // gridDim.y <= 65535
        const unsigned ny = gy - y0 < 65535 ? gy - y0 : 65535;
        fire_burn_count_kernel<<<dim3((unsigned)((nw + 255) / 256), ny), 256, 0, st>>>(burned + (size_t)y0 * slab * nw, nw, L->W, L->Ww,
                                                                                       S - (int)(y0 * slab), slab, out_count);
        FIRE_CUDA_TRY(L, cudaGetLastError());
        L->launches += 1;
    }
    return FIRE_OK;
}

extern "C" int fire_fitness(fire_landscape* L, const uint32_t* reference, const uint32_t* burned, int32_t S,
                            int32_t metric, float* out_score, uint32_t* out_counts, uint32_t* out_ref_area, void* stream)
{
    if (L == nullptr || !reference || !burned || !out_score || S < 1) return FIRE_EINVAL;
    if (metric != FIRE_METRIC_DELTA && metric != FIRE_METRIC_JACCARD) return FIRE_EINVAL;
    if (L->sticky) return L->sticky;
    fire_device_guard g(L->device);
    if (!g.ok) return FIRE_ECUDA;
    cudaStream_t st = (cudaStream_t)stream;
    uint32_t* counts = out_counts;
    if (counts == nullptr) {
        if (L->counts_capacity < (size_t)S) {
            FIRE_CUDA_TRY(L, cudaStreamSynchronize(st));
            size_t cap_bytes = L->counts_capacity * 8;
            int rc = fire_reserve(L, (void**)&L->counts_scratch, &cap_bytes, (size_t)S * 8);
            if (rc != FIRE_OK) return rc;
            L->counts_capacity = cap_bytes / 8;
        }
        counts = L->counts_scratch;
    }
    const size_t nw = (size_t)L->H * L->Ww;
    // chunks of <= 16 Ki words (64 KiB) so that small batches of big lattices still fill the SMs
    uint32_t words_per_cta = 16384;
    if ((size_t)words_per_cta > nw) words_per_cta = (uint32_t)((nw + 3) & ~(size_t)3);
    const unsigned chunks = (unsigned)((nw + words_per_cta - 1) / words_per_cta);
    FIRE_CUDA_TRY(L, cudaMemsetAsync(counts, 0, (size_t)S * 8, st));
    FIRE_CUDA_TRY(L, cudaMemsetAsync(L->ref_area, 0, sizeof(uint32_t), st));
    {
        unsigned ctas = (unsigned)((nw + 256 * 4 - 1) / (256 * 4));
        if (ctas > 256) ctas = 256;
        fire_reference_area_kernel<<<ctas, 256, 0, st>>>(reference, nw, L->ref_area);
    }
    for (int s0 = 0; s0 < S; s0 += 65535) {                    // gridDim.y limit
        const int ns = (S - s0 < 65535) ? S - s0 : 65535;
        fire_fitness_counts_kernel<<<dim3(chunks, (unsigned)ns), 256, 0, st>>>(reference, burned + (size_t)s0 * nw, nw,
                                                                              words_per_cta, counts + 2 * (size_t)s0);
        L->launches += 1;
    }
    fire_fitness_score_kernel<<<(S + 255) / 256, 256, 0, st>>>(counts, L->ref_area, S, metric, out_score, out_ref_area);
    L->launches += 2;
    FIRE_CUDA_TRY(L, cudaGetLastError());
    return FIRE_OK;
}

extern "C" int fire_fitness_group_stats(const uint32_t* counts, uint32_t ref_area, int32_t G, int32_t R,
                                        uint64_t* out_sums, double* out_mean_var, void* stream)
{
    if (!counts || !out_sums || !out_mean_var || G < 1 || R < 2) return FIRE_EINVAL;
    const size_t threads = (size_t)G * 32;
    fire_group_stats_kernel<<<(unsigned)((threads + 255) / 256), 256, 0, (cudaStream_t)stream>>>(
        counts, ref_area, G, R, (unsigned long long*)out_sums, out_mean_var);
    if (cudaGetLastError() != cudaSuccess) return FIRE_ECUDA;
    return FIRE_OK;
}

// Device address of g_fitness_static_scratch on the CURRENT device, looked up once per device (with that device current) and
// kept; cudaGetSymbolAddress allocates nothing (the array is part of the loaded module) and is idempotent, so two threads
// that race here store the same value.
static int fire_static_scratch(uint32_t** out)
{
    constexpr int kMaxDevices = 64;
    static std::atomic<uint32_t*> table[kMaxDevices];
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return FIRE_ECUDA;
    uint32_t* p = table[dev].load(std::memory_order_acquire);
    if (p == nullptr) {
        void* sym = nullptr;
        if (cudaGetSymbolAddress(&sym, g_fitness_static_scratch) != cudaSuccess || sym == nullptr) {
            (void)cudaGetLastError();
            return FIRE_ECUDA;
        }
        p = static_cast<uint32_t*>(sym);
        table[dev].store(p, std::memory_order_release);
    }
    *out = p;
    return FIRE_OK;
}

// Eq. 2 without a handle and without any allocation (fire.h): the kernels of fire_fitness on the static scratch array.
extern "C" int fire_fitness_static(const uint32_t* reference, const uint32_t* burned, int32_t W, int32_t H, int32_t S,
                                   int32_t metric, float* out_score, uint32_t* out_ref_area, void* stream)
{
    if (!reference || !burned || !out_score || S < 1 || W < 1 || H < 1 || W > 8192 || H > 8192) return FIRE_EINVAL;
    if (metric != FIRE_METRIC_DELTA && metric != FIRE_METRIC_JACCARD) return FIRE_EINVAL;
    if (S > FIRE_FITNESS_STATIC_MAX_SIMS) return FIRE_ELIMIT;
    uint32_t* scratch = nullptr;
    const int rc = fire_static_scratch(&scratch);
    if (rc != FIRE_OK) return rc;
    uint32_t* const counts = scratch;
    uint32_t* const ref_area = scratch + 2 * FIRE_FITNESS_STATIC_MAX_SIMS;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t nw = (size_t)H * (size_t)((W + 31) / 32);
    uint32_t words_per_cta = 16384;
    if ((size_t)words_per_cta > nw) words_per_cta = (uint32_t)((nw + 3) & ~(size_t)3);
    const unsigned chunks = (unsigned)((nw + words_per_cta - 1) / words_per_cta);
    // the array keeps the last call's contents: the sums of this call start at zero
    if (cudaMemsetAsync(counts, 0, (size_t)S * 8, st) != cudaSuccess) return FIRE_ECUDA;
    if (cudaMemsetAsync(ref_area, 0, sizeof(uint32_t), st) != cudaSuccess) return FIRE_ECUDA;
    {
        unsigned ctas = (unsigned)((nw + 256 * 4 - 1) / (256 * 4));
        if (ctas > 256) ctas = 256;
        fire_reference_area_kernel<<<ctas, 256, 0, st>>>(reference, nw, ref_area);
    }
    fire_fitness_counts_kernel<<<dim3(chunks, (unsigned)S), 256, 0, st>>>(reference, burned, nw, words_per_cta, counts);   // S <= 16,384 < 65,535
    fire_fitness_score_kernel<<<(S + 255) / 256, 256, 0, st>>>(counts, ref_area, S, metric, out_score, out_ref_area);
    if (cudaGetLastError() != cudaSuccess) return FIRE_ECUDA;
    return FIRE_OK;
}
