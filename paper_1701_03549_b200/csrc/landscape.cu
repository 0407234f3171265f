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
// covariates of a cell once per group of FIRE_THR_PGROUP parameter vectors.
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
// One thread per cell, looping over a group of parameter vectors with the cell's covariates held in
// registers.  For a fixed p a warp writes 32 x 32 B = 1 KiB contiguous (two 16 B stores per thread).
#define FIRE_THR_PGROUP 8

__device__ __forceinline__ uint32_t fire_threshold_from_x(double x)
{
    const double e = exp(-x);
    const double p = __ddiv_rn(1.0, __dadd_rn(1.0, e));                   // Eq. 1
    const long long t = __double2ll_rn(p * 4294967296.0);                 // exact scaling, ties-to-even (R-11)
    return (uint32_t)(t > 0xFFFFFFFFll ? 0xFFFFFFFFll : (t < 0 ? 0 : t));
}

__global__ void __launch_bounds__(128)
fire_thresholds_kernel(const float* __restrict__ beta, int P, size_t cells,
                       const uint8_t* __restrict__ flags, const uint8_t* __restrict__ uphill,
                       const double* __restrict__ psi, const double* __restrict__ tan_slope,
                       const double* __restrict__ omega, uint32_t* __restrict__ thr)
{
    __shared__ double sb[FIRE_THR_PGROUP][5];
    const int p0 = blockIdx.y * FIRE_THR_PGROUP;
    const int np = min(FIRE_THR_PGROUP, P - p0);
    if (threadIdx.x < np * 5) sb[threadIdx.x / 5][threadIdx.x % 5] = (double)beta[(size_t)p0 * 5 + threadIdx.x];
    __syncthreads();
    const size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= cells) return;
    const uint32_t f = flags[c];
    uint4* out = reinterpret_cast<uint4*>(thr) + ((size_t)p0 * cells + c) * 2;
    if ((f & 1u) == 0) {                                                  // impossible to burn: T = 0
        for (int q = 0; q < np; ++q) {
            out[0] = make_uint4(0, 0, 0, 0); out[1] = make_uint4(0, 0, 0, 0);
            out += cells * 2;
        }
        return;
    }
    const double If = (f & 2u) ? 1.0 : 0.0;
    const double ps = psi[c], ts = tan_slope[c];
    const uint32_t up = uphill[c];
    double om[8];
#pragma unroll
    for (int d = 0; d < 8; ++d) om[d] = omega[(size_t)d * cells + c];
    for (int q = 0; q < np; ++q) {
        const double b0 = sb[q][0], b1 = sb[q][1], b2 = sb[q][2], b3 = sb[q][3], b4 = sb[q][4];
        const double base = __dadd_rn(__dadd_rn(b0, __dmul_rn(b1, If)), __dmul_rn(b2, ps));
        uint32_t T[8];
#pragma unroll
        for (int d = 0; d < 8; ++d) {
            const double sg = ((up >> d) & 1u) ? ts : 0.0;
            const double x = __dadd_rn(__dadd_rn(base, __dmul_rn(b3, om[d])), __dmul_rn(b4, sg));
            T[d] = fire_threshold_from_x(x);
        }
        out[0] = make_uint4(T[0], T[1], T[2], T[3]);
        out[1] = make_uint4(T[4], T[5], T[6], T[7]);
        out += cells * 2;
    }
}

}  // namespace

// ----------------------------------------------------------------------------------------------
extern "C" int fire_landscape_destroy(fire_landscape* L)
{
    if (L == nullptr) return FIRE_EINVAL;
    fire_device_guard g(L->device);
    if (g.ok) {
        cudaDeviceSynchronize();
        void* ptrs[] = { L->flags, L->uphill, L->psi, L->tan_slope, L->omega, L->burnable, L->thr, L->beta_dev,
                         L->work_counter, L->status, L->spill, L->rescue_planes, L->ref_area, L->counts_scratch,
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
    int sms = 0;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1) {
        (void)cudaGetLastError(); delete L; return FIRE_ECUDA;
    }
    L->num_sms = sms;
    const size_t n = L->cells, nw = (size_t)H * L->Ww;
    bool ok = cudaMalloc(&L->flags, n) == cudaSuccess && cudaMalloc(&L->uphill, n) == cudaSuccess &&
              cudaMalloc(&L->psi, n * 8) == cudaSuccess && cudaMalloc(&L->tan_slope, n * 8) == cudaSuccess &&
              cudaMalloc(&L->omega, n * 64) == cudaSuccess && cudaMalloc(&L->burnable, nw * 4) == cudaSuccess &&
              cudaMalloc(&L->work_counter, 2 * sizeof(unsigned int)) == cudaSuccess &&
              cudaMalloc(&L->ref_area, 4 * sizeof(uint32_t)) == cudaSuccess;
    if (!ok) { (void)cudaGetLastError(); fire_landscape_destroy(L); return FIRE_ENOMEM; }
    cudaStream_t st = (cudaStream_t)stream;
    const long long threads = (long long)nw * 32;
    const int block = 256;
    const unsigned grid = (unsigned)((threads + block - 1) / block);
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
    const size_t bytes = (size_t)P * L->cells * 32;
    if (L->thr_capacity < bytes) {
        // growing the table must not race with work still using the old one
        FIRE_CUDA_TRY(L, cudaStreamSynchronize((cudaStream_t)stream));
        L->P = 0;
        int rc = fire_reserve(L, (void**)&L->thr, &L->thr_capacity, bytes);
        if (rc != FIRE_OK) return rc;
    }
    const int block = 128;
    dim3 grid((unsigned)((L->cells + block - 1) / block), (unsigned)((P + FIRE_THR_PGROUP - 1) / FIRE_THR_PGROUP));
    fire_thresholds_kernel<<<grid, block, 0, (cudaStream_t)stream>>>(beta, P, L->cells, L->flags, L->uphill, L->psi,
                                                                      L->tan_slope, L->omega, L->thr);
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
    FIRE_CUDA_TRY(L, cudaMemcpyAsync(out, L->thr + (size_t)p * L->cells * 8, L->cells * 32, cudaMemcpyDeviceToDevice,
                                     (cudaStream_t)stream));
    return FIRE_OK;
}
