/* drive_cfg.c -- a plain C program (no Python, no ctypes) that drives one workload through the C ABI of include/fire.h:
 * reads rasters, parameter vectors and the batch from a binary file written by tests/test_gpu_parity.py, runs
 * fire_landscape_create -> fire_params_upload -> fire_simulate_batch (reference + batch) -> fire_fitness, and writes burnt maps,
 * steps, trials, counts and scores to another binary file.  The test compares that file with the oracle's stored values.
 *   usage: drive_cfg <in.bin> <out.bin>
 *   in : i32 W, H, P, S, metric; veg u8[H*W]; slope, aspect, wind f32[H*W]; beta f32[(P+1)*5] (last = reference vector);
 *        ign i32[S*2]; par i32[S]; seeds u64[S]; ref_ign i32[2]; ref_seed u64
 *   out: burned u32[S*H*Ww]; steps u32[S]; trials u64[S]; counts u32[S*2]; score f32[S]; ref_area u32 */
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <cuda_runtime_api.h>
#include "fire.h"

#define CHECK(x) do { int rc__ = (x); if (rc__ != 0) { fprintf(stderr, "%s failed: %d (%s)\n", #x, rc__, fire_error_string(rc__)); return 2; } } while (0)
#define CU(x) do { cudaError_t e__ = (x); if (e__ != cudaSuccess) { fprintf(stderr, "%s: %s\n", #x, cudaGetErrorString(e__)); return 3; } } while (0)

static void* rd(FILE* f, size_t n) { void* p = malloc(n ? n : 1); if (fread(p, 1, n, f) != n) { fprintf(stderr, "short read\n"); exit(4); } return p; }
static void* up(const void* h, size_t n) { void* d = NULL; if (cudaMalloc(&d, n ? n : 1) != cudaSuccess || cudaMemcpy(d, h, n, cudaMemcpyHostToDevice) != cudaSuccess) { fprintf(stderr, "upload failed\n"); exit(5); } return d; }

int main(int argc, char** argv)
{
    if (argc != 3) { fprintf(stderr, "usage: %s in.bin out.bin\n", argv[0]); return 1; }
    FILE* f = fopen(argv[1], "rb");
    if (!f) { perror(argv[1]); return 1; }
    int32_t hdr[5];
    if (fread(hdr, 4, 5, f) != 5) return 4;
    const int32_t W = hdr[0], H = hdr[1], P = hdr[2], S = hdr[3], metric = hdr[4];
    const size_t n = (size_t)W * H, Ww = (size_t)(W + 31) / 32, nw = (size_t)H * Ww;
    uint8_t* veg = rd(f, n); float* slope = rd(f, 4 * n); float* aspect = rd(f, 4 * n); float* wind = rd(f, 4 * n);
    float* beta = rd(f, (size_t)(P + 1) * 20);
    int32_t* ign = rd(f, (size_t)S * 8); int32_t* par = rd(f, (size_t)S * 4); uint64_t* seeds = rd(f, (size_t)S * 8);
    int32_t* ref_ign = rd(f, 8); uint64_t* ref_seed = rd(f, 8);
    fclose(f);

    fire_landscape* L = NULL;
    void *d_veg = up(veg, n), *d_slope = up(slope, 4 * n), *d_aspect = up(aspect, 4 * n), *d_wind = up(wind, 4 * n);
    CHECK(fire_landscape_create(&L, d_veg, d_slope, d_aspect, d_wind, W, H, NULL));
    void* d_beta = up(beta, (size_t)(P + 1) * 20);
    CHECK(fire_params_upload(L, d_beta, P + 1, NULL));
    /* the reference burnt map: the stored vector (index P), ignition and seed, sim id 0 */
    int32_t ref_par = P, ref_id = 0;
    void *d_rign = up(ref_ign, 8), *d_rpar = up(&ref_par, 4), *d_rseed = up(ref_seed, 8), *d_rid = up(&ref_id, 4);
    uint32_t* d_ref = NULL; CU(cudaMalloc((void**)&d_ref, nw * 4));
    CHECK(fire_simulate_batch(L, d_rign, d_rpar, d_rseed, d_rid, 1, 0, d_ref, NULL, NULL, NULL));
    void *d_ign = up(ign, (size_t)S * 8), *d_par = up(par, (size_t)S * 4), *d_seeds = up(seeds, (size_t)S * 8);
    uint32_t *d_burned = NULL, *d_steps = NULL, *d_counts = NULL, *d_area = NULL; uint64_t* d_trials = NULL; float* d_score = NULL;
    CU(cudaMalloc((void**)&d_burned, (size_t)S * nw * 4)); CU(cudaMalloc((void**)&d_steps, (size_t)S * 4));
    CU(cudaMalloc((void**)&d_trials, (size_t)S * 8)); CU(cudaMalloc((void**)&d_counts, (size_t)S * 8));
    CU(cudaMalloc((void**)&d_score, (size_t)S * 4)); CU(cudaMalloc((void**)&d_area, 4));
    CHECK(fire_simulate_batch(L, d_ign, d_par, d_seeds, NULL, S, 0, d_burned, d_steps, d_trials, NULL));
    CHECK(fire_fitness(L, d_ref, d_burned, S, metric, d_score, d_counts, d_area, NULL));
    CU(cudaDeviceSynchronize());

    FILE* o = fopen(argv[2], "wb");
    if (!o) { perror(argv[2]); return 1; }
    size_t sizes[6] = { (size_t)S * nw * 4, (size_t)S * 4, (size_t)S * 8, (size_t)S * 8, (size_t)S * 4, 4 };
    void* devs[6] = { d_burned, d_steps, d_trials, d_counts, d_score, d_area };
    for (int i = 0; i < 6; ++i) {
        void* h = malloc(sizes[i]);
        CU(cudaMemcpy(h, devs[i], sizes[i], cudaMemcpyDeviceToHost));
        if (fwrite(h, 1, sizes[i], o) != sizes[i]) return 6;
        free(h);
    }
    fclose(o);
    printf("launches %lld\n", (long long)fire_launch_count(L));
    CHECK(fire_landscape_destroy(L));
    return 0;
}
