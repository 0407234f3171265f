/* abi_c99.c -- compiled (never run) by tests/test_abi.py with `gcc -std=c99 -pedantic -Wall -Werror -c`: include/fire.h must
 * be a valid C99 header on its own, and every call it declares must have exactly the prototype written here. */
#include "fire.h"

typedef void (*any_fn)(void);

typedef int (*create_fn)(fire_landscape**, const uint8_t*, const float*, const float*, const float*, int32_t, int32_t, void*);
typedef int (*destroy_fn)(fire_landscape*);
typedef int (*upload_fn)(fire_landscape*, const float*, int32_t, void*);
typedef int (*simulate_fn)(fire_landscape*, const int32_t*, const int32_t*, const uint64_t*, const int32_t*, int32_t, uint32_t,
                           uint32_t*, uint32_t*, uint64_t*, void*);
typedef int (*fitness_fn)(fire_landscape*, const uint32_t*, const uint32_t*, int32_t, int32_t, float*, uint32_t*, uint32_t*, void*);
typedef int (*stats_fn)(const uint32_t*, uint32_t, int32_t, int32_t, uint64_t*, double*, void*);
typedef int (*download_fn)(fire_landscape*, int32_t, uint32_t*, void*);
typedef int (*generation_fn)(fire_landscape*, const float*, int32_t, const int32_t*, const int32_t*, const uint64_t*, const int32_t*,
                             int32_t, uint32_t, const uint32_t*, int32_t, float*, uint32_t*, uint32_t*, uint32_t**, void*);
typedef int64_t (*count_fn)(const fire_landscape*);
typedef int (*set1_fn)(fire_landscape*, int32_t);
typedef int (*set2_fn)(fire_landscape*, int32_t, int32_t);
typedef int (*profread_fn)(fire_landscape*, float*, int32_t, int32_t*);
typedef const char* (*errstr_fn)(int);

typedef int (*burn_fn)(fire_landscape*, const uint8_t*, int32_t, void*);
typedef int (*elev_fn)(fire_landscape*, const float*, void*);
typedef int (*hazard_fn)(fire_landscape*, const uint32_t*, int32_t, uint32_t*, void*);
typedef int (*timeout_fn)(fire_landscape*, int32_t*);
typedef int (*fused_fn)(fire_landscape*, const uint32_t*, uint32_t*);
typedef int (*static_fn)(const uint32_t*, const uint32_t*, int32_t, int32_t, int32_t, int32_t, float*, uint32_t*, void*);
typedef int (*classif_fn)(fire_landscape*, const float*, int32_t, void*);
any_fn fire_abi_table[23];

void fire_abi_fill(void)
{
    create_fn f0 = fire_landscape_create;       destroy_fn f1 = fire_landscape_destroy;
    upload_fn f2 = fire_params_upload;          simulate_fn f3 = fire_simulate_batch;
    fitness_fn f4 = fire_fitness;               stats_fn f5 = fire_fitness_group_stats;
    download_fn f6 = fire_thresholds_download;  generation_fn f7 = fire_generation_host;
    count_fn f8 = fire_launch_count;            set2_fn f9 = fire_set_launch_geometry;
    set2_fn f10 = fire_set_list_capacity;       set1_fn f11 = fire_set_schedule;
    set1_fn f12 = fire_set_kernel;              set1_fn f13 = fire_set_profiling;
    profread_fn f14 = fire_profile_read;        errstr_fn f15 = fire_error_string;
    burn_fn f16 = fire_set_burn_time;
    elev_fn f17 = fire_landscape_set_elevation;
    hazard_fn f18 = fire_burn_count;
    timeout_fn f19 = fire_set_time_output;
    classif_fn f20 = fire_landscape_set_class_indicator;
    fused_fn f21 = fire_set_fused_counts;
    static_fn f22 = fire_fitness_static;
    fire_abi_table[22] = (any_fn)f22;
    fire_abi_table[21] = (any_fn)f21;
    fire_abi_table[20] = (any_fn)f20;
    fire_abi_table[19] = (any_fn)f19;
    fire_abi_table[16] = (any_fn)f16; fire_abi_table[17] = (any_fn)f17; fire_abi_table[18] = (any_fn)f18;
    fire_abi_table[0] = (any_fn)f0;   fire_abi_table[1] = (any_fn)f1;
    fire_abi_table[2] = (any_fn)f2;   fire_abi_table[3] = (any_fn)f3;
    fire_abi_table[4] = (any_fn)f4;   fire_abi_table[5] = (any_fn)f5;
    fire_abi_table[6] = (any_fn)f6;   fire_abi_table[7] = (any_fn)f7;
    fire_abi_table[8] = (any_fn)f8;   fire_abi_table[9] = (any_fn)f9;
    fire_abi_table[10] = (any_fn)f10; fire_abi_table[11] = (any_fn)f11;
    fire_abi_table[12] = (any_fn)f12; fire_abi_table[13] = (any_fn)f13;
    fire_abi_table[14] = (any_fn)f14; fire_abi_table[15] = (any_fn)f15;
    { int codes[6] = { FIRE_OK, FIRE_EINVAL, FIRE_ENOMEM, FIRE_ESTATE, FIRE_ECUDA, FIRE_ELIMIT }; (void)codes; }
    { int limits[1] = { FIRE_FITNESS_STATIC_MAX_SIMS }; (void)limits; }
    { int metrics[2] = { FIRE_METRIC_DELTA, FIRE_METRIC_JACCARD }; (void)metrics; }
}
