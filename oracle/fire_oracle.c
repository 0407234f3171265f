/*
 * fire_oracle.c -- CPU ORACLE for the hot path of arXiv 1701.03549 (Denham & Laneri).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  It is a plain, slow, obviously
 * correct restatement of what the paper's method computes, written from PAPER.md
 * and the readings R-1..R-20 listed in DESIGN.md.  Only tests/, bench.py's
 * cpu_baseline / --impl reference legs and __graft_entry__.smoke() may load it.
 * It shares no code, header, table or constant generator with the CUDA library
 * in paper_1701_03549_b200/csrc (that library has its own Philox, its own trig,
 * its own bit tricks).  No blocking, fusion or reordering beyond what the paper's
 * algorithm states: one cell, one neighbour, one trial at a time.
 *
 * Build:  gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC -o libfire_oracle.so fire_oracle.c -lm
 *         (-ffp-contract=off: every double operation below is one IEEE operation,
 *          evaluated in the order written; no FMA.)
 *
 * Pins (tests/test_oracle_*.py, all `-m "not gpu"`):
 *   orc_philox4x32_10   : the three published Philox4x32-10 known-answer vectors.
 *   orc_probability /
 *   orc_threshold       : closed forms (beta0=0 -> 2^31; T(x)+T(-x)=2^32+-1; monotone;
 *                         saturation), scipy.special.expit, worked values of Eq. 1 with
 *                         the paper's Table 2 reference vector, compass-geometry cases.
 *   orc_simulate        : p==0 -> ignition only; p==1 -> 8-connected burnable component
 *                         and burn time = BFS depth (scipy.ndimage); invariants;
 *                         1-D strip closed form (chi^2); <=3x3 exact Markov enumeration
 *                         (chi^2); percolation identity vs an independent numpy sampler (KS).
 *   orc_fitness_*       : per-cell numpy set arithmetic, special cases of Eq. 2.
 *   orc_group_stats     : numpy mean / var(ddof=1) on the same integers.
 *   parity unpinned     : the paper's own outputs (delta ~ 0.05 floor PAPER.md:137,
 *                         delta = 0.15 PAPER.md:163, Tables 2-3) -- they need the
 *                         authors' Patagonia maps, which are not available.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif

/* ------------------------------------------------------------------------- *
 * Random numbers.  PAPER.md:139-141 (Sec. 3.3): "a counter based random number
 * generator: the Random123 library ... Philox generator was used".  Variant,
 * rounds and keying are not given; reading R-3 fixes Philox4x32-10 (Salmon,
 * Moraes, Dror, Shaw, SC'11) keyed by (seed, sim, step, cell, direction).
 * ------------------------------------------------------------------------- */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        if (round > 0) {             /* key schedule: bumped before every round but the first */
            k0 += 0x9E3779B9u;       /* golden ratio */
            k1 += 0xBB67AE85u;       /* sqrt(3) - 1  */
        }
        uint64_t prod0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        uint64_t prod1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        uint32_t hi0 = (uint32_t)(prod0 >> 32), lo0 = (uint32_t)prod0;
        uint32_t hi1 = (uint32_t)(prod1 >> 32), lo1 = (uint32_t)prod1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* C-1: the random word of trial (seed, sim, step, cell, d): word d&3 of
 * Philox4x32-10(counter = (cell, step, sim, d>>2), key = (seed lo, seed hi)).
 * cell = y*W + x of the TARGET cell, step = index t of the transition t -> t+1. */
uint32_t orc_rnd(uint64_t seed, uint32_t sim, uint32_t step, uint32_t cell, int d)
{
    uint32_t ctr[4] = { cell, step, sim, (uint32_t)(d >> 2) };
    uint32_t key[2] = { (uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32) };
    uint32_t out[4];
    orc_philox4x32_10(ctr, key, out);
    return out[d & 3];
}

/* ------------------------------------------------------------------------- *
 * Geometry.  Direction d = 0..7 = N, NE, E, SE, S, SW, W, NW is the direction of
 * travel from the burning (source) cell to the target cell; row 0 is north and
 * x grows east (R-5), so target = source + (DX[d], DY[d]).  phi_d = d * pi/4 is
 * the compass bearing of that travel direction (R-4).
 * ------------------------------------------------------------------------- */
static const int DX[8] = { 0, 1, 1, 1, 0, -1, -1, -1 };
static const int DY[8] = { -1, -1, 0, 1, 1, 1, 0, -1 };

void orc_direction_offset(int d, int* dx, int* dy) { *dx = DX[d]; *dy = DY[d]; }

static double phi(int d) { return (double)d * (M_PI / 4.0); }

typedef struct {
    int    burnable;   /* veg != 0 */
    double I_f;        /* 1 for forest (veg == 1), else 0  */
    double psi;        /* cos(aspect - 315 deg) if slope > 5 deg  */
    double omega[8];   /* cos(wind - phi_d)  */
    double sigma[8];   /* tan(slope) if travelling uphill, else 0  */
} orc_cov;

/* C-2: covariates of a TARGET cell ("... of the target cell"). */
void orc_covariates(uint8_t veg, float slope, float aspect, float wind, orc_cov* c)
{
    double s = (double)slope, a = (double)aspect, w = (double)wind;
    c->burnable = (veg != 0);
    c->I_f = (veg == 1) ? 1.0 : 0.0;                                  /* R-9  */
    if (s > 5.0 * M_PI / 180.0) c->psi = cos(a - phi(7));             /* 315 deg = NW; R-4 */
    else                        c->psi = 0.0;                         /* R-10 */
    for (int d = 0; d < 8; ++d) {
        c->omega[d] = cos(w - phi(d));                                /* R-6: wind blows TOWARD w */
        int uphill = (s > 0.0) && (cos(phi(d) - a) < 0.0);            /* R-7, R-14 */
        c->sigma[d] = uphill ? tan(s) : 0.0;                          /* R-8: slope/100 with slope in percent */
    }
}

/* Eq. 1 for one (target cell, direction). */
double orc_probability(const float beta[5], uint8_t veg, float slope, float aspect, float wind, int d)
{
    orc_cov c;
    orc_covariates(veg, slope, aspect, wind, &c);
    double b0 = (double)beta[0], b1 = (double)beta[1], b2 = (double)beta[2],
           b3 = (double)beta[3], b4 = (double)beta[4];
    double x = b0 + b1 * c.I_f;
    x = x + b2 * c.psi;
    x = x + b3 * c.omega[d];
    x = x + b4 * c.sigma[d];
    return 1.0 / (1.0 + exp(-x));
}

/* Mean of Eq. 1 over the 8 directions of n cells (used by oracle/make_workloads.py to
 * choose beta_0 for a target mean spread probability). */
double orc_mean_probability(const float beta[5], const uint8_t* veg, const float* slope,
                            const float* aspect, const float* wind, int n)
{
    double sum = 0.0;
    for (int i = 0; i < n; ++i)
        for (int d = 0; d < 8; ++d)
            sum += orc_probability(beta, veg[i], slope[i], aspect[i], wind[i], d);
    return sum / (8.0 * (double)n);
}

/* C-3: 32-bit contagion threshold. */
uint32_t orc_threshold(const float beta[5], uint8_t veg, float slope, float aspect, float wind, int d)
{
    if (veg == 0) return 0u;                          /* impossible to burn */
    double p = orc_probability(beta, veg, slope, aspect, wind, d);
    long long t = llrint(ldexp(p, 32));               /* ties-to-even (default rounding mode) */
    if (t > 0xFFFFFFFFLL) t = 0xFFFFFFFFLL;
    if (t < 0) t = 0;
    return (uint32_t)t;
}

/* R-11: a trial succeeds iff rnd < T, and T = 0xFFFFFFFF means certain. */
int orc_trial_succeeds(uint32_t rnd, uint32_t T) { return (rnd < T) || (T == 0xFFFFFFFFu); }

/* Whole table for one parameter vector: out[(y*W + x)*8 + d]. */
void orc_threshold_table(const float beta[5], const uint8_t* veg, const float* slope,
                         const float* aspect, const float* wind, int W, int H, uint32_t* out)
{
#ifdef _OPENMP
#pragma omp parallel for schedule(static)      /* rows are independent; arithmetic unchanged */
#endif
    for (int y = 0; y < H; ++y)
        for (int x = 0; x < W; ++x) {
            size_t c = (size_t)y * W + x;
            for (int d = 0; d < 8; ++d)
                out[c * 8 + d] = orc_threshold(beta, veg[c], slope[c], aspect[c], wind[c], d);
        }
}

/* Variant of C-2 / C-3 (PAPER.md:87 read literally): "Slope is calculated based on the digital elevation map (DEM)
 * and is ignored whenever the target landscape cell is at a lower elevation or when slope is zero. The normalized slope is used
 * when the target cell is higher in elevation than the burning cell."  With an elevation raster the uphill test of direction d
 * is  elevation[target] > elevation[source]  (strictly, R-14), source = target - offset(d), instead of R-7's local-plane test on
 * the aspect; everything else is orc_probability.  Entries whose source lies outside the lattice are never tried; they get
 * sigma = 0. */
void orc_threshold_table_dem(const float beta[5], const uint8_t* veg, const float* slope, const float* aspect,
                             const float* wind, const float* elevation, int W, int H, uint32_t* out)
{
    double b0 = (double)beta[0], b1 = (double)beta[1], b2 = (double)beta[2], b3 = (double)beta[3], b4 = (double)beta[4];
    for (int y = 0; y < H; ++y)
        for (int x = 0; x < W; ++x) {
            size_t c = (size_t)y * W + x;
            orc_cov cv;
            orc_covariates(veg[c], slope[c], aspect[c], wind[c], &cv);
            for (int d = 0; d < 8; ++d) {
                int sx = x - DX[d], sy = y - DY[d];
                int inside = sx >= 0 && sx < W && sy >= 0 && sy < H;
                int uphill = inside && ((double)slope[c] > 0.0) && (elevation[c] > elevation[(size_t)sy * W + sx]);
                double sigma = uphill ? tan((double)slope[c]) : 0.0;
                double xx = b0 + b1 * cv.I_f;
                xx = xx + b2 * cv.psi;
                xx = xx + b3 * cv.omega[d];
                xx = xx + b4 * sigma;
                double p = 1.0 / (1.0 + exp(-xx));
                long long t = llrint(ldexp(p, 32));
                out[c * 8 + d] = cv.burnable ? (uint32_t)(t > 0xFFFFFFFFll ? 0xFFFFFFFFll : t) : 0u;
            }
        }
}

/* Variant of C-2 / C-3 ("per-class I_f table"): Eq. 1 has ONE vegetation term, beta_1 I_f with I_f = 1 for forest
 * (PAPER.md:76, :81); with more fuel classes than the paper's two (BASELINE configs have 4 and 6) a table gives every class v its
 * own value I_f = class_if[v] (double of the f32 given).  class_if = {0, 1, 0, 0, ...} is orc_threshold_table. */
void orc_threshold_table_classes(const float beta[5], const uint8_t* veg, const float* slope, const float* aspect,
                                 const float* wind, const float class_if[256], int W, int H, uint32_t* out)
{
    double b0 = (double)beta[0], b1 = (double)beta[1], b2 = (double)beta[2], b3 = (double)beta[3], b4 = (double)beta[4];
    for (int y = 0; y < H; ++y)
        for (int x = 0; x < W; ++x) {
            size_t c = (size_t)y * W + x;
            orc_cov cv;
            orc_covariates(veg[c], slope[c], aspect[c], wind[c], &cv);
            for (int d = 0; d < 8; ++d) {
                double xx = b0 + b1 * (double)class_if[veg[c]];
                xx = xx + b2 * cv.psi;
                xx = xx + b3 * cv.omega[d];
                xx = xx + b4 * cv.sigma[d];
                double p = 1.0 / (1.0 + exp(-xx));
                long long t = llrint(ldexp(p, 32));
                out[c * 8 + d] = cv.burnable ? (uint32_t)(t > 0xFFFFFFFFll ? 0xFFFFFFFFll : t) : 0u;
            }
        }
}

/* ------------------------------------------------------------------------- *
 * C-4: one simulation (PAPER.md:91 states; :97 ignition; :99, :133 synchronous
 * update, independent trial per burning neighbour = 1 - prod(1 - p_i) in law,
 * R-1/R-2; :91, :145 a cell is active for exactly one step; :100, :135 the run
 * ends when the fire stops by itself).
 *
 * table: NULL  -> every threshold is computed on demand from the rasters;
 *        else  -> u32[H][W][8] used instead (lets a test feed a given table).
 * out_burned : canonical bitmap, cell (x,y) = bit (x&31) of word y*ceil(W/32)+(x>>5).
 * out_time   : optional i32[H][W], step at which the cell ignited (0 = ignition), -1 never.
 * counters   : optional u64[3] = { trials, candidate cell-steps, distinct target cells }.
 * ------------------------------------------------------------------------- */
int orc_simulate(const uint8_t* veg, const float* slope, const float* aspect, const float* wind,
                 int W, int H, const float beta[5], const uint32_t* table,
                 int ix, int iy, uint64_t seed, uint32_t sim, uint32_t max_steps,
                 uint32_t* out_burned, int32_t* out_time, uint32_t* out_steps, uint64_t* counters)
{
    size_t ncell = (size_t)W * H;
    int Ww = (W + 31) / 32;
    uint8_t*  burned   = (uint8_t*)calloc(ncell, 1);
    uint8_t*  is_new   = (uint8_t*)calloc(ncell, 1);    /* ignited during the current step */
    uint32_t* tried_at = (uint32_t*)calloc(ncell, 4);   /* t+1 of the last step the cell was a target */
    uint32_t* burning  = (uint32_t*)malloc(ncell * 4);  /* list of burning cells */
    uint32_t* fresh    = (uint32_t*)malloc(ncell * 4);  /* list of cells ignited this step */
    if (!burned || !is_new || !tried_at || !burning || !fresh) {
        free(burned); free(is_new); free(tried_at); free(burning); free(fresh);
        return -1;
    }
    size_t n_burning = 0;
    uint64_t trials = 0, cand_steps = 0, distinct = 0;
    uint32_t t = 0;
    if (out_time) for (size_t c = 0; c < ncell; ++c) out_time[c] = -1;

    /* step 1: ignition (R-12: outside the lattice or non-burnable -> nothing burns) */
    if (ix >= 0 && ix < W && iy >= 0 && iy < H && veg[(size_t)iy * W + ix] != 0) {
        size_t c = (size_t)iy * W + ix;
        burned[c] = 1;
        burning[n_burning++] = (uint32_t)c;
        if (out_time) out_time[c] = 0;
    }

    /* step 2 */
    while (n_burning > 0 && (max_steps == 0 || t < max_steps)) {
        size_t n_fresh = 0;
        for (size_t i = 0; i < n_burning; ++i) {
            int sx = (int)(burning[i] % (uint32_t)W), sy = (int)(burning[i] / (uint32_t)W);
            for (int d = 0; d < 8; ++d) {
                int tx = sx + DX[d], ty = sy + DY[d];
                if (tx < 0 || tx >= W || ty < 0 || ty >= H) continue;   /* R-13: no wrap-around */
                size_t c = (size_t)ty * W + tx;
                if (veg[c] == 0) continue;                              /* impossible to burn */
                if (burned[c]) continue;                                /* burnt (state at time t) */
                ++trials;
                if (tried_at[c] != t + 1) {
                    if (tried_at[c] == 0) ++distinct;
                    tried_at[c] = t + 1;
                    ++cand_steps;
                }
                uint32_t T = table ? table[c * 8 + d]
                                   : orc_threshold(beta, veg[c], slope[c], aspect[c], wind[c], d);
                uint32_t r = orc_rnd(seed, sim, t, (uint32_t)c, d);
                if (orc_trial_succeeds(r, T) && !is_new[c]) {
                    is_new[c] = 1;
                    fresh[n_fresh++] = (uint32_t)c;
                }
            }
        }
        /* synchronous update: burning -> burnt-inactive, fresh -> burning */
        for (size_t i = 0; i < n_fresh; ++i) {
            size_t c = fresh[i];
            burned[c] = 1;
            is_new[c] = 0;
            if (out_time) out_time[c] = (int32_t)(t + 1);
        }
        uint32_t* tmp = burning; burning = fresh; fresh = tmp;
        n_burning = n_fresh;
        ++t;
    }

    /* step 3: output */
    memset(out_burned, 0, (size_t)H * Ww * 4);
    for (int y = 0; y < H; ++y)
        for (int x = 0; x < W; ++x)
            if (burned[(size_t)y * W + x])
                out_burned[(size_t)y * Ww + (x >> 5)] |= (1u << (x & 31));
    if (out_steps) *out_steps = t;
    if (counters) { counters[0] = trials; counters[1] = cand_steps; counters[2] = distinct; }
    free(burned); free(is_new); free(tried_at); free(burning); free(fresh);
    return 0;
}

/* ---------------------------------------------------------------------------
 * C-4', fuel-dependent burn-out time (reading R-21).
 * PAPER.md:91 "A burnt cell gets inactive after a given time that depends on the vegetation type of the cell", :145
 * "cells have a turn off time that depends on vegetation fuel type", :68 / :273 (fuel consumption times are the extension the
 * authors announce).  burn_time[v] >= 1 is that time, in steps, for vegetation class v (0 is read as 1).  A cell ignited by
 * the transition t -> t+1 is ACTIVE during steps t+1 .. t+burn_time (the ignition cell during steps 0 .. burn_time-1); at
 * every step every active cell is a source for each of its susceptible neighbours: one trial rnd(seed, sim, t, target, d)
 * against T(target, d), exactly as in C-4 (the key contains the step, so a pair that is tried again draws a fresh word).
 * The run ends when no cell is active.  burn_time == 1 everywhere is orc_simulate, byte for byte.
 * out_time: optional, step at which the cell ignited (0 = ignition, -1 never).
 * counters: trials, candidate cell-steps, distinct targets, as in orc_simulate.
 * ------------------------------------------------------------------------- */
int orc_simulate_burn_time(const uint8_t* veg, const float* slope, const float* aspect, const float* wind,
                           int W, int H, const float beta[5], const uint32_t* table, const uint8_t burn_time[256],
                           int ix, int iy, uint64_t seed, uint32_t sim, uint32_t max_steps,
                           uint32_t* out_burned, int32_t* out_time, uint32_t* out_steps, uint64_t* counters)
{
    size_t ncell = (size_t)W * H;
    int Ww = (W + 31) / 32;
    uint8_t*  burned   = (uint8_t*)calloc(ncell, 1);
    uint8_t*  is_new   = (uint8_t*)calloc(ncell, 1);
    uint8_t*  left     = (uint8_t*)calloc(ncell, 1);    /* steps the cell stays active, 0 = inactive */
    uint32_t* tried_at = (uint32_t*)calloc(ncell, 4);
    uint32_t* active   = (uint32_t*)malloc(ncell * 4);  /* list of active cells */
    uint32_t* next     = (uint32_t*)malloc(ncell * 4);
    uint32_t* fresh    = (uint32_t*)malloc(ncell * 4);
    if (!burned || !is_new || !left || !tried_at || !active || !next || !fresh) {
        free(burned); free(is_new); free(left); free(tried_at); free(active); free(next); free(fresh);
        return -1;
    }
    size_t n_active = 0;
    uint64_t trials = 0, cand_steps = 0, distinct = 0;
    uint32_t t = 0;
    if (out_time) for (size_t c = 0; c < ncell; ++c) out_time[c] = -1;

    if (ix >= 0 && ix < W && iy >= 0 && iy < H && veg[(size_t)iy * W + ix] != 0) {
        size_t c = (size_t)iy * W + ix;
        burned[c] = 1;
        left[c] = burn_time[veg[c]] ? burn_time[veg[c]] : 1;
        active[n_active++] = (uint32_t)c;
        if (out_time) out_time[c] = 0;
    }

    while (n_active > 0 && (max_steps == 0 || t < max_steps)) {
        size_t n_fresh = 0, n_next = 0;
        for (size_t i = 0; i < n_active; ++i) {
            int sx = (int)(active[i] % (uint32_t)W), sy = (int)(active[i] / (uint32_t)W);
            for (int d = 0; d < 8; ++d) {
                int tx = sx + DX[d], ty = sy + DY[d];
                if (tx < 0 || tx >= W || ty < 0 || ty >= H) continue;
                size_t c = (size_t)ty * W + tx;
                if (veg[c] == 0) continue;
                if (burned[c]) continue;
                ++trials;
                if (tried_at[c] != t + 1) {
                    if (tried_at[c] == 0) ++distinct;
                    tried_at[c] = t + 1;
                    ++cand_steps;
                }
                uint32_t T = table ? table[c * 8 + d]
                                   : orc_threshold(beta, veg[c], slope[c], aspect[c], wind[c], d);
                uint32_t r = orc_rnd(seed, sim, t, (uint32_t)c, d);
                if (orc_trial_succeeds(r, T) && !is_new[c]) {
                    is_new[c] = 1;
                    fresh[n_fresh++] = (uint32_t)c;
                }
            }
        }
        /* synchronous update: one step of fuel is consumed in every active cell; the newly ignited become active */
        for (size_t i = 0; i < n_active; ++i) {
            size_t c = active[i];
            if (--left[c] > 0) next[n_next++] = (uint32_t)c;
        }
        for (size_t i = 0; i < n_fresh; ++i) {
            size_t c = fresh[i];
            burned[c] = 1;
            is_new[c] = 0;
            left[c] = burn_time[veg[c]] ? burn_time[veg[c]] : 1;
            next[n_next++] = (uint32_t)c;
            if (out_time) out_time[c] = (int32_t)(t + 1);
        }
        uint32_t* tmp = active; active = next; next = tmp;
        n_active = n_next;
        ++t;
    }

    memset(out_burned, 0, (size_t)H * Ww * 4);
    for (int y = 0; y < H; ++y)
        for (int x = 0; x < W; ++x)
            if (burned[(size_t)y * W + x])
                out_burned[(size_t)y * Ww + (x >> 5)] |= (1u << (x & 31));
    if (out_steps) *out_steps = t;
    if (counters) { counters[0] = trials; counters[1] = cand_steps; counters[2] = distinct; }
    free(burned); free(is_new); free(left); free(tried_at); free(active); free(next); free(fresh);
    return 0;
}

/* A batch of independent simulations (each individual /
 * replicate is its own CA run).  Parallel over simulations only; each one is
 * orc_simulate unchanged.  tables: NULL, or P pointers (each NULL or u32[H][W][8]).
 * Returns the number of threads used (>=1) or a negative error. */
int orc_simulate_batch(const uint8_t* veg, const float* slope, const float* aspect, const float* wind,
                       int W, int H, const float* betas /*[P][5]*/, int P,
                       const uint32_t* const* tables,
                       const int32_t* ignitions /*[S][2]*/, const int32_t* sim_param /*[S]*/,
                       const uint64_t* seeds /*[S]*/, const int32_t* sim_index /*[S] or NULL*/, int S,
                       uint32_t max_steps, uint32_t* out_burned /*[S][H][Ww]*/,
                       uint32_t* out_steps /*[S]*/, uint64_t* counters /*[S][3] or NULL*/, int nthreads)
{
    int Ww = (W + 31) / 32;
    int used = 1, err = 0;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
    used = (nthreads > 0) ? nthreads : omp_get_max_threads();
#pragma omp parallel for schedule(dynamic, 1)
#endif
    for (int s = 0; s < S; ++s) {
        uint32_t* ob = out_burned + (size_t)s * H * Ww;
        int p = sim_param[s];
        uint32_t sim = sim_index ? (uint32_t)sim_index[s] : (uint32_t)s;
        if (p < 0 || p >= P) {                         /* R-12: burns nothing */
            memset(ob, 0, (size_t)H * Ww * 4);
            if (out_steps) out_steps[s] = 0;
            if (counters) counters[3 * s] = counters[3 * s + 1] = counters[3 * s + 2] = 0;
            continue;
        }
        int rc = orc_simulate(veg, slope, aspect, wind, W, H, betas + 5 * p,
                              tables ? tables[p] : NULL, ignitions[2 * s], ignitions[2 * s + 1],
                              seeds[s], sim, max_steps, ob, NULL,
                              out_steps ? out_steps + s : NULL, counters ? counters + 3 * s : NULL);
        if (rc != 0) err = rc;
    }
    return err ? err : used;
}

/* ------------------------------------------------------------------------- *
 * C-5: fitness, Eq. 2.  A = reference map, A* = simulated
 * map; # = number of burnt cells.  Counted cell by cell.
 * counts = { I = #(A and A*), Nstar = #A*, N = #A }.
 * ------------------------------------------------------------------------- */
void orc_fitness_counts(const uint32_t* reference, const uint32_t* burned, int W, int H, uint32_t counts[3])
{
    int Ww = (W + 31) / 32;
    uint32_t I = 0, Nstar = 0, N = 0;
    for (int y = 0; y < H; ++y)
        for (int x = 0; x < W; ++x) {
            int in_ref = (reference[(size_t)y * Ww + (x >> 5)] >> (x & 31)) & 1u;
            int in_sim = (burned[(size_t)y * Ww + (x >> 5)] >> (x & 31)) & 1u;
            N += in_ref; Nstar += in_sim; I += (in_ref && in_sim);
        }
    counts[0] = I; counts[1] = Nstar; counts[2] = N;
}

/* metric 0: delta = (#(A u A*) - #(A n A*)) / #A      (Eq. 2)
 * metric 1: Jaccard  #(A n A*) / #(A u A*)             (BASELINE config 2)
 * one IEEE float divide of (rounded-to-float) exact integers; N = 0 -> inf/NaN. */
float orc_fitness_score(uint32_t I, uint32_t Nstar, uint32_t N, int metric)
{
    uint32_t uni = N + Nstar - I;
    if (metric == 0) return (float)(uni - I) / (float)N;
    return (float)I / (float)uni;
}

/* Group statistics over R replicates of each of G candidates (BASELINE config 4;
 * PAPER.md:177, :404 "error = standard deviation of the ensemble"; R-16 sample variance).
 * counts [G*R][2] = (I, Nstar); x = N + Nstar - 2I; sums [G][2] = (sum x, sum x^2);
 * mean_var [G][2] = mean and sample variance of delta = x / N. */
void orc_group_stats(const uint32_t* counts, uint32_t N, int G, int R, uint64_t* sums, double* mean_var)
{
    for (int g = 0; g < G; ++g) {
        uint64_t sx = 0, sxx = 0;
        for (int r = 0; r < R; ++r) {
            uint64_t I = counts[2 * ((size_t)g * R + r)], Nstar = counts[2 * ((size_t)g * R + r) + 1];
            uint64_t x = (uint64_t)N + Nstar - 2 * I;
            sx += x; sxx += x * x;
        }
        sums[2 * g] = sx; sums[2 * g + 1] = sxx;
        double mean = (double)sx / ((double)R * (double)N);
        uint64_t num = (uint64_t)R * sxx - sx * sx;      /* exact integer, >= 0 */
        double var = (double)num / (double)((uint64_t)R * (uint64_t)(R - 1));
        var = var / ((double)N * (double)N);
        mean_var[2 * g] = mean; mean_var[2 * g + 1] = var;
    }
}

int orc_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
