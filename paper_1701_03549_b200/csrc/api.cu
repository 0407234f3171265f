// api.cu -- the end-to-end call with HOST buffers and the small utility entry points of fire.h.
#include "fire_internal.cuh"

namespace {
inline size_t align256(size_t n) { return (n + 255) & ~(size_t)255; }
}

// One GA generation: H2D of the generation's inputs, a2 + a3-a6 + a7 on the device, D2H of the
// scores.  The burnt maps stay on the device (the GA only needs the fitness; App. B).
extern "C" int fire_generation_host(fire_landscape* L, const float* beta_host, int32_t P,
                                    const int32_t* ignitions_host, const int32_t* sim_param_host,
                                    const uint64_t* seeds_host, const int32_t* sim_ids_host, int32_t S,
                                    uint32_t max_steps, const uint32_t* reference_host, int32_t metric,
                                    float* out_score_host, uint32_t* out_counts_host, uint32_t* out_steps_host,
                                    uint32_t** out_burned_dev, void* stream)
{
    if (L == nullptr || !beta_host || !ignitions_host || !sim_param_host || !seeds_host || !reference_host ||
        !out_score_host || P < 1 || S < 1)
        return FIRE_EINVAL;
    if (L->sticky) return L->sticky;
    fire_device_guard g(L->device);
    if (!g.ok) return FIRE_ECUDA;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t nw = (size_t)L->H * L->Ww;

    // carve the staging buffer
    size_t off = 0;
    const size_t o_beta = off;   off += align256((size_t)P * 5 * sizeof(float));
    const size_t o_ign = off;    off += align256((size_t)S * 2 * sizeof(int32_t));
    const size_t o_par = off;    off += align256((size_t)S * sizeof(int32_t));
    const size_t o_seed = off;   off += align256((size_t)S * sizeof(uint64_t));
    const size_t o_ids = off;    off += align256((size_t)S * sizeof(int32_t));
    const size_t o_ref = off;    off += align256(nw * sizeof(uint32_t));
    const size_t o_score = off;  off += align256((size_t)S * sizeof(float));
    const size_t o_counts = off; off += align256((size_t)S * 2 * sizeof(uint32_t));
    const size_t o_steps = off;  off += align256((size_t)S * sizeof(uint32_t));
    const size_t o_burned = off; off += align256((size_t)S * nw * sizeof(uint32_t));
    if (L->gen_capacity < off) {
        FIRE_CUDA_TRY(L, cudaStreamSynchronize(st));
        int rc = fire_reserve(L, &L->gen_buf, &L->gen_capacity, off);
        if (rc != FIRE_OK) return rc;
    }
    char* base = (char*)L->gen_buf;
    float* d_beta = (float*)(base + o_beta);
    int32_t* d_ign = (int32_t*)(base + o_ign);
    int32_t* d_par = (int32_t*)(base + o_par);
    uint64_t* d_seed = (uint64_t*)(base + o_seed);
    int32_t* d_ids = sim_ids_host ? (int32_t*)(base + o_ids) : nullptr;
    uint32_t* d_ref = (uint32_t*)(base + o_ref);
    float* d_score = (float*)(base + o_score);
    uint32_t* d_counts = (uint32_t*)(base + o_counts);
    uint32_t* d_steps = (uint32_t*)(base + o_steps);
    uint32_t* d_burned = (uint32_t*)(base + o_burned);

    FIRE_CUDA_TRY(L, cudaMemcpyAsync(d_beta, beta_host, (size_t)P * 5 * sizeof(float), cudaMemcpyHostToDevice, st));
    FIRE_CUDA_TRY(L, cudaMemcpyAsync(d_ign, ignitions_host, (size_t)S * 2 * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    FIRE_CUDA_TRY(L, cudaMemcpyAsync(d_par, sim_param_host, (size_t)S * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    FIRE_CUDA_TRY(L, cudaMemcpyAsync(d_seed, seeds_host, (size_t)S * sizeof(uint64_t), cudaMemcpyHostToDevice, st));
    if (d_ids) FIRE_CUDA_TRY(L, cudaMemcpyAsync(d_ids, sim_ids_host, (size_t)S * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    FIRE_CUDA_TRY(L, cudaMemcpyAsync(d_ref, reference_host, nw * sizeof(uint32_t), cudaMemcpyHostToDevice, st));

    int rc = fire_params_upload(L, d_beta, P, stream);
    if (rc != FIRE_OK) return rc;
    rc = fire_simulate_batch(L, d_ign, d_par, d_seed, d_ids, S, max_steps, d_burned, d_steps, nullptr, stream);
    if (rc != FIRE_OK) return rc;
    rc = fire_fitness(L, d_ref, d_burned, S, metric, d_score, d_counts, nullptr, stream);
    if (rc != FIRE_OK) return rc;

    FIRE_CUDA_TRY(L, cudaMemcpyAsync(out_score_host, d_score, (size_t)S * sizeof(float), cudaMemcpyDeviceToHost, st));
    if (out_counts_host)
        FIRE_CUDA_TRY(L, cudaMemcpyAsync(out_counts_host, d_counts, (size_t)S * 2 * sizeof(uint32_t), cudaMemcpyDeviceToHost, st));
    if (out_steps_host)
        FIRE_CUDA_TRY(L, cudaMemcpyAsync(out_steps_host, d_steps, (size_t)S * sizeof(uint32_t), cudaMemcpyDeviceToHost, st));
    FIRE_CUDA_TRY(L, cudaStreamSynchronize(st));
    if (out_burned_dev) *out_burned_dev = d_burned;
    return FIRE_OK;
}

extern "C" int fire_set_profiling(fire_landscape* L, int32_t enabled)
{
    if (L == nullptr) return FIRE_EINVAL;
    fire_device_guard g(L->device);
    if (!g.ok) return FIRE_ECUDA;
    if (enabled && L->prof_ev[0] == nullptr)
        for (int i = 0; i < 2 * 64; ++i) FIRE_CUDA_TRY(L, cudaEventCreate(&L->prof_ev[i]));
    L->prof_enabled = enabled ? 1 : 0;
    L->prof_count = 0;
    return FIRE_OK;
}

extern "C" int fire_profile_read(fire_landscape* L, float* ms_host, int32_t max_entries, int32_t* n_out)
{
    if (L == nullptr || ms_host == nullptr || n_out == nullptr || max_entries < 0) return FIRE_EINVAL;
    fire_device_guard g(L->device);
    if (!g.ok) return FIRE_ECUDA;
    int n = 0;
    for (; n < L->prof_count && n < max_entries; ++n) {
        FIRE_CUDA_TRY(L, cudaEventSynchronize(L->prof_ev[2 * n + 1]));
        FIRE_CUDA_TRY(L, cudaEventElapsedTime(ms_host + n, L->prof_ev[2 * n], L->prof_ev[2 * n + 1]));
    }
    *n_out = n;
    L->prof_count = 0;
    return FIRE_OK;
}

extern "C" int64_t fire_launch_count(const fire_landscape* L) { return L ? L->launches : 0; }

extern "C" const char* fire_error_string(int code)
{
    switch (code) {
        case FIRE_OK:     return "ok";
        case FIRE_EINVAL: return "invalid argument";
        case FIRE_ENOMEM: return "device allocation failed";
        case FIRE_ESTATE: return "call out of order (no thresholds uploaded, or parameter index out of range)";
        case FIRE_ECUDA:  return "CUDA error or no CUDA device";
        case FIRE_ELIMIT: return "size beyond the limit of the static scratch array (FIRE_FITNESS_STATIC_MAX_SIMS)";
        default:          return "unknown error code";
    }
}
