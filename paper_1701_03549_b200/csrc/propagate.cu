// propagate.cu -- batched CA fire propagation (a3-a6): fire_simulate_batch.
//
// What is computed (PAPER.md:91 states, :97 ignition, :99/:133 synchronous update with one
// independent trial per burning neighbour = 1 - prod(1 - p_i) in law, :91/:145 a cell burns for one
// step, :100/:135 the run ends when the fire stops by itself; C-4):
//   t = 0: burning = burned = {ignition} if it is inside the lattice and burnable.
//   step t: for every burning cell b and direction d, target c = b + offset(d); if c is inside the
//   lattice, burnable and not burned at time t: one trial rnd(seed, sim, t, c, d) against T[p][c][d].
//   new = targets with >= 1 success; burned |= new; burning = new.
//
// Design: one persistent CTA per simulation, simulations handed out by a device
// counter, all CA steps inside ONE launch, no host round trip and no grid-wide barrier.  State per
// simulation = ONE bit plane, the SUSCEPTIBLE plane  sus = burnable & ~burned  (it lives in the caller's
// output buffer: fire_init_planes_kernel fills it with `burnable`, fire_finish_planes_kernel turns it
// into the burnt map  burnable & ~sus  at the end), plus a CELL-LEVEL FRONTIER LIST of the burning
// cells, so work is proportional to the number of trials and idle lattice is never touched.  A step:
//   phase 1  one lane per burning cell: three words of `sus` give the 3 x 3 susceptibility window; the
//            (target, direction) pairs of the warp are compacted into the trial queue (warp prefix sum,
//            unrolled predicated stores, one shared atomic per warp);
//   -- barrier: every read of `sus` for step t happens before any update of step t (synchronous update)
//   phase 2  one lane per trial, four trials per lane in flight: one 4 B threshold load (the 32 B sector
//            of a target cell holds its 8 directions), one Philox4x32-10 call with the round keys of the
//            simulation held in registers, one compare; a success clears the target's bit with
//            atomicAnd, and the lane whose atomic saw the bit still set owns the new burning cell and
//            appends it to the next frontier (ballot / popc compaction, one shared atomic per warp).
//   -- barrier
// Lists live in shared memory and continue in a per-CTA global spill area (coalesced); if the frontier
// outgrows even that, the simulation is handed to the rescue kernel below: a plain full-sweep,
// three-plane, pull-style restatement of the same rules with no lists at all.
#include "fire_internal.cuh"

namespace {

struct prop_params {
    const uint32_t* burnable;     // [H][Ww]
    const uint32_t* thr;          // [P][cells][8]
    const int32_t*  ignitions;    // [S][2]
    const int32_t*  sim_param;    // [S]
    const uint64_t* seeds;        // [S]
    const int32_t*  sim_ids;      // [S] or null
    uint32_t* out_burned;         // [S][H][Ww]: the susceptible plane while the fast kernel runs
    uint32_t* out_steps;          // [S] or null
    unsigned long long* out_trials;  // [S] or null
    unsigned int* work_counter;   // [0] next sim of the fast kernel, [1] number of sims handed to the rescue kernel
    uint32_t* rescue_list;        // [S]
    uint32_t* spill;              // [grid][2 * (capA - capA_s) + (capQ - capQ_s)]
    int S, P, W, H, Ww;
    uint32_t max_steps;
    uint32_t capA_s, capQ_s;      // shared-memory entries: each frontier list, the trial queue
    uint32_t capA, capQ;          // total entries (shared + spill); capQ >= 8 * capA
};

__device__ __forceinline__ uint32_t list_get(const uint32_t* s, const uint32_t* g, uint32_t cap_s, uint32_t i)
{
    return i < cap_s ? s[i] : __ldcg(g + (i - cap_s));
}
__device__ __forceinline__ void list_put(uint32_t* s, uint32_t* g, uint32_t cap_s, uint32_t i, uint32_t v)
{
    if (i < cap_s) s[i] = v; else __stcg(g + (i - cap_s), v);
}

__device__ __forceinline__ uint32_t lanemask_lt()
{
    uint32_t m; asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m)); return m;
}

// Frontier entry: (y << 16) | x.  Trial item: (ty << 16) | (tx << 3) | d  (x, y < 8192).
// Item of the trial "burning cell e spreads in direction d": item(e) + kItemDelta(d).
__device__ __forceinline__ uint32_t item_delta(int d)
{
    return (uint32_t)(fire_dy(d) * 65536 + fire_dx(d) * 8 + d);
}

// Window of three susceptibility bits (x-1, x, x+1) -> bits 0..2, from the word holding x and, at the
// word's ends, bit 31 of the word to the left / bit 0 of the word to the right.
__device__ __forceinline__ uint32_t win3(uint32_t mid, uint32_t lft, uint32_t rgt, int bx)
{
    return (bx ? __funnelshift_r(mid, rgt, bx - 1) : ((mid << 1) | (lft >> 31))) & 7u;
}

// Threshold load: read-only path, and ask L2 to fetch the whole 256 B around a miss (the thresholds of the 8
// x-adjacent cells): HBM serves a random 32 B sector and a random 256 B chunk at nearly the same rate, and the
// neighbours are the next cells the front reaches.
__device__ __forceinline__ uint32_t ldg_thr(const uint32_t* p)
{
    uint32_t v;
#ifndef FIRE_NO_L2_PREFETCH
    asm volatile("ld.global.nc.L2::256B.u32 %0, [%1];" : "=r"(v) : "l"(p));
#else
    v = __ldg(p);
#endif
    return v;
}

constexpr int kTrialsInFlight = 4;   // trials per lane issued together in phase 2
constexpr int kCellsInFlight = 2;    // burning cells per lane issued together in phase 1

// ------------------------------------------------------------------------------------------------
// Fast kernel: one persistent CTA per simulation.
// ------------------------------------------------------------------------------------------------
#ifndef FIRE_LB_THREADS      // tuning builds: -DFIRE_LB_THREADS=256 -DFIRE_LB_CTAS=6 caps the registers for that geometry
#define FIRE_LB_THREADS 1024
#define FIRE_LB_CTAS 1
#endif
__global__ void __launch_bounds__(FIRE_LB_THREADS, FIRE_LB_CTAS)
fire_propagate_kernel(const prop_params prm)
{
    extern __shared__ uint32_t smem[];
    const uint32_t capA_s = prm.capA_s, capQ_s = prm.capQ_s;
    uint32_t* const As0 = smem;
    uint32_t* const As1 = As0 + capA_s;
    uint32_t* const Qs = As1 + capA_s;
    const size_t spill_per_cta = (size_t)2 * (prm.capA - capA_s) + (prm.capQ - capQ_s);
    uint32_t* const Ag0 = prm.spill + (size_t)blockIdx.x * spill_per_cta;
    uint32_t* const Ag1 = Ag0 + (prm.capA - capA_s);
    uint32_t* const Qg = Ag1 + (prm.capA - capA_s);

    __shared__ unsigned int s_sim, s_cntA[2], s_cntQ[2], s_over;
    __shared__ unsigned long long s_trials;

    const int tid = threadIdx.x, lane = tid & 31, nthr = blockDim.x;
    const int W = prm.W, H = prm.H, Ww = prm.Ww;
    const uint32_t lt = lanemask_lt();

    for (;;) {
        __syncthreads();                       // the previous simulation's last reads of s_* are done
        if (tid == 0) s_sim = atomicAdd(prm.work_counter, 1u);
        __syncthreads();
        const uint32_t s = s_sim;
        if (s >= (uint32_t)prm.S) break;
#ifdef FIRE_TRACE
        unsigned long long trace_t0; asm volatile("mov.u64 %0, %globaltimer;" : "=l"(trace_t0));
#endif

        const int p = prm.sim_param[s];
        const int ix = prm.ignitions[2 * s], iy = prm.ignitions[2 * s + 1];
        const uint64_t seed = prm.seeds[s];
        const uint32_t sim = prm.sim_ids ? (uint32_t)prm.sim_ids[s] : s;
        uint32_t* const sus = prm.out_burned + (size_t)s * H * Ww;
        bool valid = p >= 0 && p < prm.P && ix >= 0 && ix < W && iy >= 0 && iy < H;     // R-12
        if (valid) valid = (__ldg(prm.burnable + (size_t)iy * Ww + (ix >> 5)) >> (ix & 31)) & 1u;
        const uint32_t* const thr = prm.thr + (valid ? (size_t)p * W * H * 8 : 0);

        // round keys of Philox4x32-10 for this simulation's seed (bumped before every round but the first)
        uint32_t rk0[10], rk1[10];
#pragma unroll
        for (int r = 0; r < 10; ++r) {
            rk0[r] = (uint32_t)seed + (uint32_t)r * 0x9E3779B9u;
            rk1[r] = (uint32_t)(seed >> 32) + (uint32_t)r * 0xBB67AE85u;
        }

        if (tid == 0) {
            s_cntA[0] = valid ? 1u : 0u; s_cntA[1] = 0u; s_cntQ[0] = 0u; s_cntQ[1] = 0u;
            s_over = 0u; s_trials = 0ull;
            if (valid) {
                list_put(As0, Ag0, capA_s, 0u, ((uint32_t)iy << 16) | (uint32_t)ix);
                atomicAnd(sus + (size_t)iy * Ww + (ix >> 5), ~(1u << (ix & 31)));
            }
        }
        __syncthreads();

        uint32_t t = 0, my_trials = 0;
        uint32_t nA = valid ? 1u : 0u;
        bool over = false;
        while (nA > 0 && (prm.max_steps == 0 || t < prm.max_steps)) {
            const int par = t & 1;
            uint32_t* const Ac_s = par ? As1 : As0;  uint32_t* const Ac_g = par ? Ag1 : Ag0;
            uint32_t* const An_s = par ? As0 : As1;  uint32_t* const An_g = par ? Ag0 : Ag1;

            // ---- phase 1: susceptible neighbours of the burning cells -> trial queue
            // kCellsInFlight burning cells per lane; all their `sus` loads are issued before any is used.
            for (uint32_t i0 = (uint32_t)(tid & ~31) * kCellsInFlight; i0 < nA; i0 += (uint32_t)nthr * kCellsInFlight) {
                uint32_t e[kCellsInFlight], mid[kCellsInFlight], upw[kCellsInFlight], dnw[kCellsInFlight], m[kCellsInFlight];
#pragma unroll
                for (int k = 0; k < kCellsInFlight; ++k) {
                    const uint32_t i = i0 + 32u * k + lane;
                    e[k] = 0xFFFFFFFFu; mid[k] = 0u; upw[k] = 0u; dnw[k] = 0u;
                    if (i < nA) {
                        e[k] = list_get(Ac_s, Ac_g, capA_s, i);
                        const uint32_t x = e[k] & 0xFFFFu, y = e[k] >> 16;
                        const uint32_t* const r1 = sus + (y * (uint32_t)Ww + (x >> 5));
                        mid[k] = __ldcg(r1);
                        if (y > 0) upw[k] = __ldcg(r1 - Ww);
                        if (y + 1 < (uint32_t)H) dnw[k] = __ldcg(r1 + Ww);
                    }
                }
                uint32_t cnt = 0;
#pragma unroll
                for (int k = 0; k < kCellsInFlight; ++k) {
                    m[k] = 0u;
                    if (e[k] != 0xFFFFFFFFu) {
                        const uint32_t x = e[k] & 0xFFFFu, y = e[k] >> 16;
                        const int wx = (int)(x >> 5), bx = (int)(x & 31u);
                        uint32_t l0 = 0, l1 = 0, l2 = 0, g0 = 0, g1 = 0, g2 = 0;
                        if (bx == 0 || bx == 31) {                         // the window crosses into a neighbouring word (1 cell in 16)
                            const uint32_t* const r1 = sus + (y * (uint32_t)Ww + (uint32_t)wx);
                            const bool has_up = y > 0, has_dn = y + 1 < (uint32_t)H;
                            if (bx == 0 && wx > 0) {
                                l1 = __ldcg(r1 - 1);
                                if (has_up) l0 = __ldcg(r1 - Ww - 1);
                                if (has_dn) l2 = __ldcg(r1 + Ww - 1);
                            } else if (bx == 31 && wx + 1 < Ww) {
                                g1 = __ldcg(r1 + 1);
                                if (has_up) g0 = __ldcg(r1 - Ww + 1);
                                if (has_dn) g2 = __ldcg(r1 + Ww + 1);
                            }
                        }
                        const uint32_t up = win3(upw[k], l0, g0, bx), md = win3(mid[k], l1, g1, bx), dn = win3(dnw[k], l2, g2, bx);
                        // bit d of m: the neighbour reached by travelling in direction d can still burn
                        m[k] = ((up >> 1) & 3u) | (md & 4u) | ((dn & 4u) << 1) | ((dn & 2u) << 3) | ((dn & 1u) << 5) |
                               ((md & 1u) << 6) | ((up & 1u) << 7);
                    }
                    cnt += __popc(m[k]);
                }
                uint32_t incl = cnt;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const uint32_t v = __shfl_up_sync(0xFFFFFFFFu, incl, o);
                    if (lane >= o) incl += v;
                }
                const uint32_t total = __shfl_sync(0xFFFFFFFFu, incl, 31);
                if (total == 0) continue;
                uint32_t qbase = 0;
                if (lane == 31) qbase = atomicAdd(&s_cntQ[par], total);
                qbase = __shfl_sync(0xFFFFFFFFu, qbase, 31);
                uint32_t pos = qbase + incl - cnt;
                my_trials += cnt;
                const bool in_shared = qbase + total <= capQ_s;           // warp-uniform: the whole batch fits in shared memory
#pragma unroll
                for (int k = 0; k < kCellsInFlight; ++k) {
                    const uint32_t base = ((e[k] & 0xFFFFu) << 3) | (e[k] & 0xFFFF0000u);
                    if (in_shared) {
#pragma unroll
                        for (int d = 0; d < 8; ++d)
                            if (m[k] & (1u << d)) Qs[pos + __popc(m[k] & ((1u << d) - 1u))] = base + item_delta(d);
                    } else {
#pragma unroll
                        for (int d = 0; d < 8; ++d)
                            if (m[k] & (1u << d)) list_put(Qs, Qg, capQ_s, pos + __popc(m[k] & ((1u << d) - 1u)), base + item_delta(d));
                    }
                    pos += __popc(m[k]);
                }
            }
            __syncthreads();
            const uint32_t nQ = s_cntQ[par];
            if (tid == 0) { s_cntA[par] = 0u; s_cntQ[par ^ 1] = 0u; }     // next step's counters; nobody reads them now

            // ---- phase 2: one Bernoulli trial per lane-slot, kTrialsInFlight per lane, in stages so that each
            // long latency (threshold load, atomic) is waited for once per batch: loads -> Philox -> atomics -> compaction
            for (uint32_t j0 = (uint32_t)(tid & ~31) * kTrialsInFlight; j0 < nQ; j0 += (uint32_t)nthr * kTrialsInFlight) {
                uint32_t item[kTrialsInFlight], T[kTrialsInFlight], old[kTrialsInFlight];
#pragma unroll
                for (int u = 0; u < kTrialsInFlight; ++u) {
                    const uint32_t j = j0 + 32u * u + lane;
                    item[u] = 0xFFFFFFFFu;
                    T[u] = 0u;
                    if (j < nQ) {
                        item[u] = list_get(Qs, Qg, capQ_s, j);
                        const uint32_t c = (item[u] >> 16) * (uint32_t)W + ((item[u] >> 3) & 0x1FFFu);
                        T[u] = ldg_thr(thr + (c * 8u + (item[u] & 7u)));
                    }
                }
                bool succ[kTrialsInFlight];
#pragma unroll
                for (int u = 0; u < kTrialsInFlight; ++u) {
                    succ[u] = false;
                    if (j0 + 32u * u < nQ) {                               // warp-uniform
                        const uint32_t ty = item[u] >> 16, tx = (item[u] >> 3) & 0x1FFFu, d = item[u] & 7u;
                        // Philox4x32-10(counter = (c, t, sim, d >> 2), key = seed), word d & 3   (C-1)
                        uint32_t c0 = ty * (uint32_t)W + tx, c1 = t, c2 = sim, c3 = d >> 2;
#pragma unroll
                        for (int r = 0; r < 10; ++r) {
                            const uint64_t a = (uint64_t)c0 * 0xD2511F53ull;
                            const uint64_t b = (uint64_t)c2 * 0xCD9E8D57ull;
                            const uint32_t n0 = (uint32_t)(b >> 32) ^ c1 ^ rk0[r];
                            const uint32_t n2 = (uint32_t)(a >> 32) ^ c3 ^ rk1[r];
                            c1 = (uint32_t)b; c3 = (uint32_t)a; c0 = n0; c2 = n2;
                        }
                        const uint32_t lo = (d & 1u) ? c1 : c0, hi = (d & 1u) ? c3 : c2;
                        const uint32_t rnd = (d & 2u) ? hi : lo;
                        succ[u] = item[u] != 0xFFFFFFFFu && fire_trial(rnd, T[u]);
                    }
                }
#pragma unroll
                for (int u = 0; u < kTrialsInFlight; ++u) {
                    old[u] = 0u;
                    if (succ[u]) {
                        const uint32_t ty = item[u] >> 16, tx = (item[u] >> 3) & 0x1FFFu;
                        old[u] = atomicAnd(sus + (ty * (uint32_t)Ww + (tx >> 5)), ~(1u << (tx & 31u)));
                    }
                }
                uint32_t fresh_mask[kTrialsInFlight];
                uint32_t n_fresh = 0;
#pragma unroll
                for (int u = 0; u < kTrialsInFlight; ++u) {
                    const bool fresh = succ[u] && ((old[u] >> ((item[u] >> 3) & 31u)) & 1u);
                    fresh_mask[u] = __ballot_sync(0xFFFFFFFFu, fresh);
                    n_fresh += __popc(fresh_mask[u]);
                }
                if (n_fresh == 0) continue;                                // warp-uniform
                uint32_t abase = 0;
                if (lane == 0) abase = atomicAdd(&s_cntA[par ^ 1], n_fresh);
                abase = __shfl_sync(0xFFFFFFFFu, abase, 0);
#pragma unroll
                for (int u = 0; u < kTrialsInFlight; ++u) {
                    if (fresh_mask[u] & (1u << lane)) {
                        const uint32_t pos = abase + __popc(fresh_mask[u] & lt);
                        if (pos < prm.capA) list_put(An_s, An_g, capA_s, pos, (item[u] & 0xFFFF0000u) | ((item[u] >> 3) & 0x1FFFu));
                        else s_over = 1u;
                    }
                    abase += __popc(fresh_mask[u]);
                }
            }
            __syncthreads();
            ++t;
            if (s_over) { over = true; break; }       // written in phase 2 only, read after its closing barrier
            nA = s_cntA[par ^ 1];
        }

        // ---- end of the simulation
        if (my_trials) atomicAdd(&s_trials, (unsigned long long)my_trials);
        __syncthreads();
        if (tid == 0) {
            if (over) {
                prm.rescue_list[atomicAdd(prm.work_counter + 1, 1u)] = s;
            } else {
                if (prm.out_steps) prm.out_steps[s] = t;
                if (prm.out_trials) prm.out_trials[s] = s_trials;
#ifdef FIRE_TRACE   // diagnostic build only: out_trials = (start us << 32) | duration us of this simulation, for schedule plots
                unsigned long long trace_t1; asm volatile("mov.u64 %0, %globaltimer;" : "=l"(trace_t1));
                if (prm.out_trials) prm.out_trials[s] = (((trace_t0 / 1000ull) & 0xFFFFFFFFull) << 32) | (((trace_t1 - trace_t0) / 1000ull) & 0xFFFFFFFFull);
#endif
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// Plane set-up and tear-down around the fast kernel: sus = burnable before, burnt = burnable & ~sus after.
// Pure streams over S planes; grid = (chunks of the plane, S).
// ------------------------------------------------------------------------------------------------
template <bool kFinish>
__global__ void __launch_bounds__(256)
fire_planes_kernel(const uint32_t* __restrict__ burnable, uint32_t* __restrict__ planes, size_t nw, int vec4)
{
    uint32_t* const plane = planes + (size_t)blockIdx.y * nw;
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    if (vec4) {
        const uint4* const b4 = reinterpret_cast<const uint4*>(burnable);
        uint4* const p4 = reinterpret_cast<uint4*>(plane);
        for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nw / 4; i += stride) {
            uint4 b = __ldg(b4 + i);
            if (kFinish) {
                const uint4 s = __ldcs(p4 + i);
                b.x &= ~s.x; b.y &= ~s.y; b.z &= ~s.z; b.w &= ~s.w;
            }
            p4[i] = b;
        }
    } else {
        for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nw; i += stride) {
            uint32_t b = __ldg(burnable + i);
            if (kFinish) b &= ~__ldcs(plane + i);
            plane[i] = b;
        }
    }
}

// ------------------------------------------------------------------------------------------------
// Rescue kernel: plain restatement with three bit planes and a full sweep of the rows the fire has
// reached; every word of the next burning plane has exactly one writer, so there are no atomics and
// no lists.  planes: [gridDim.x][2][H*Ww], all-zero on entry and on exit.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t plane_word(const uint32_t* plane, int y, int wx, int H, int Ww)
{
    return ((unsigned)y < (unsigned)H && (unsigned)wx < (unsigned)Ww) ? __ldcg(plane + (size_t)y * Ww + wx) : 0u;
}

__global__ void __launch_bounds__(256)
fire_propagate_rescue_kernel(const prop_params prm, uint32_t* planes)
{
    __shared__ int s_y0, s_y1;
    __shared__ unsigned long long s_trials;
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int W = prm.W, H = prm.H, Ww = prm.Ww;
    const size_t nw = (size_t)H * Ww;
    const unsigned int n_rescue = *((volatile unsigned int*)(prm.work_counter + 1));

    for (unsigned int k = blockIdx.x; k < n_rescue; k += gridDim.x) {
        const uint32_t s = prm.rescue_list[k];
        const int p = prm.sim_param[s];
        const int ix = prm.ignitions[2 * s], iy = prm.ignitions[2 * s + 1];
        const uint64_t seed = prm.seeds[s];
        const uint32_t key_lo = (uint32_t)seed, key_hi = (uint32_t)(seed >> 32);
        const uint32_t sim = prm.sim_ids ? (uint32_t)prm.sim_ids[s] : s;
        const uint32_t* const thr = prm.thr + (size_t)p * W * H * 8;
        uint32_t* const burned = prm.out_burned + (size_t)s * nw;
        uint32_t* cur = planes + (size_t)blockIdx.x * 2 * nw;
        uint32_t* nxt = cur + nw;

        for (size_t w = tid; w < nw; w += nthr) burned[w] = 0u;      // the fast kernel left it half-done
        if (tid == 0) { s_y0 = iy; s_y1 = iy; s_trials = 0ull; }
        __syncthreads();
        if (tid == 0) {
            burned[(size_t)iy * Ww + (ix >> 5)] = 1u << (ix & 31);
            cur[(size_t)iy * Ww + (ix >> 5)] = 1u << (ix & 31);
        }
        __syncthreads();

        uint32_t t = 0;
        unsigned long long my_trials = 0;
        int burning = 1;
        while (burning && (prm.max_steps == 0 || t < prm.max_steps)) {
            const int ylo = max(s_y0 - 1, 0), yhi = min(s_y1 + 1, H - 1);
            const int nwords = (yhi - ylo + 1) * Ww;
            int any_new = 0, ny0 = H, ny1 = -1;
            for (int idx = tid; idx < nwords; idx += nthr) {
                const int y = ylo + idx / Ww, wx = idx % Ww;
                const uint32_t uL = plane_word(cur, y - 1, wx - 1, H, Ww), uC = plane_word(cur, y - 1, wx, H, Ww),
                               uR = plane_word(cur, y - 1, wx + 1, H, Ww);
                const uint32_t mL = plane_word(cur, y, wx - 1, H, Ww), mC = plane_word(cur, y, wx, H, Ww),
                               mR = plane_word(cur, y, wx + 1, H, Ww);
                const uint32_t dL = plane_word(cur, y + 1, wx - 1, H, Ww), dC = plane_word(cur, y + 1, wx, H, Ww),
                               dR = plane_word(cur, y + 1, wx + 1, H, Ww);
                // src[d]: bit x set iff the cell the fire would come FROM, (x, y) - offset(d), is burning
                uint32_t src[8];
                src[0] = dC;                          // travelling N: source is the row below
                src[1] = (dC << 1) | (dL >> 31);      // NE: source (x-1, y+1)
                src[2] = (mC << 1) | (mL >> 31);      // E : source (x-1, y)
                src[3] = (uC << 1) | (uL >> 31);      // SE: source (x-1, y-1)
                src[4] = uC;                          // S : source (x, y-1)
                src[5] = (uC >> 1) | (uR << 31);      // SW: source (x+1, y-1)
                src[6] = (mC >> 1) | (mR << 31);      // W : source (x+1, y)
                src[7] = (dC >> 1) | (dR << 31);      // NW: source (x+1, y+1)
                const size_t wi = (size_t)y * Ww + wx;
                const uint32_t sus = __ldg(prm.burnable + wi) & ~__ldcg(burned + wi);
                uint32_t cand = (src[0] | src[1] | src[2] | src[3] | src[4] | src[5] | src[6] | src[7]) & sus;
                uint32_t fresh = 0;
                while (cand) {
                    const int bx = __ffs(cand) - 1;
                    cand &= cand - 1;
                    const uint32_t c = (uint32_t)(y * W + wx * 32 + bx);
                    bool hit = false;
#pragma unroll 1
                    for (int d = 0; d < 8; ++d) {
                        if (((src[d] >> bx) & 1u) == 0u) continue;
                        ++my_trials;
                        const uint32_t T = __ldg(thr + (size_t)c * 8 + d);
                        hit |= fire_trial(fire_rnd(key_lo, key_hi, sim, t, c, d), T);
                    }
                    if (hit) fresh |= 1u << bx;
                }
                nxt[wi] = fresh;                      // always written: the region only grows, so stale words are overwritten
                if (fresh) { any_new = 1; ny0 = min(ny0, y); ny1 = max(ny1, y); }
            }
            __syncthreads();
            for (int idx = tid; idx < nwords; idx += nthr) {
                const size_t wi = (size_t)ylo * Ww + idx;
                const uint32_t f = __ldcg(nxt + wi);
                if (f) burned[wi] |= f;
            }
            if (any_new) { atomicMin(&s_y0, ny0); atomicMax(&s_y1, ny1); }
            burning = __syncthreads_or(any_new);
            uint32_t* tmp = cur; cur = nxt; nxt = tmp;
            ++t;
        }
        // leave both planes all-zero for the next simulation
        {
            const int ylo = max(s_y0 - 1, 0), yhi = min(s_y1 + 1, H - 1);
            const size_t lo = (size_t)ylo * Ww, n = (size_t)(yhi - ylo + 1) * Ww;
            for (size_t w = tid; w < n; w += nthr) { cur[lo + w] = 0u; nxt[lo + w] = 0u; }
        }
        if (my_trials) atomicAdd(&s_trials, my_trials);
        __syncthreads();
        if (tid == 0) {
            if (prm.out_steps) prm.out_steps[s] = t;
            if (prm.out_trials) prm.out_trials[s] = s_trials;
        }
        __syncthreads();
    }
}

constexpr int kRescueCtas = 16;

}  // namespace

// ----------------------------------------------------------------------------------------------
extern "C" int fire_set_launch_geometry(fire_landscape* L, int32_t threads_per_cta, int32_t ctas_per_sm)
{
    if (L == nullptr) return FIRE_EINVAL;
    if (threads_per_cta != 0 && (threads_per_cta < 32 || threads_per_cta > 1024 || threads_per_cta % 32 != 0)) return FIRE_EINVAL;
    if (ctas_per_sm < 0 || ctas_per_sm > 32) return FIRE_EINVAL;
    L->threads_per_cta = threads_per_cta;
    L->ctas_per_sm = ctas_per_sm;
    return FIRE_OK;
}

extern "C" int fire_set_list_capacity(fire_landscape* L, int32_t shared_entries, int32_t total_entries)
{
    if (L == nullptr || shared_entries < 0 || total_entries < 0) return FIRE_EINVAL;
    L->list_shared = shared_entries;
    L->list_capacity = total_entries;
    return FIRE_OK;
}

extern "C" int fire_simulate_batch(fire_landscape* L, const int32_t* ignitions, const int32_t* sim_param,
                                   const uint64_t* seeds, const int32_t* sim_ids, int32_t S, uint32_t max_steps,
                                   uint32_t* out_burned, uint32_t* out_steps, uint64_t* out_trials, void* stream)
{
    if (L == nullptr || !ignitions || !sim_param || !seeds || !out_burned || S < 1) return FIRE_EINVAL;
    if (L->sticky) return L->sticky;
    if (L->P == 0) return FIRE_ESTATE;
    fire_device_guard g(L->device);
    if (!g.ok) return FIRE_ECUDA;
    cudaStream_t st = (cudaStream_t)stream;

    // ---- geometry and list capacities
    const int threads = L->threads_per_cta ? L->threads_per_cta : 256;
    const int per_sm = L->ctas_per_sm ? L->ctas_per_sm : 4;
    const int grid = (int)((long long)S < (long long)L->num_sms * per_sm ? S : L->num_sms * per_sm);
    prop_params prm;
    uint32_t capA_s = L->list_shared ? (uint32_t)L->list_shared : 1536u;
    uint32_t capA = L->list_capacity ? (uint32_t)L->list_capacity : 0u;
    if (capA == 0) {
        // generous: a BFS level set of an open W x H lattice has at most 2(W+H) cells
        size_t want = (size_t)16 * (size_t)(L->W + L->H);
        if (want < 8192) want = 8192;
        if (want > L->cells) want = L->cells;
        capA = (uint32_t)want;
    }
    if (capA < 1) capA = 1;
    if (capA_s > capA) capA_s = capA;
    prm.capA_s = capA_s; prm.capA = capA;
    prm.capQ = 8u * capA;
    prm.capQ_s = 2u * capA_s < prm.capQ ? 2u * capA_s : prm.capQ;
    const size_t smem = ((size_t)2 * prm.capA_s + prm.capQ_s) * sizeof(uint32_t);
    if (smem > 200 * 1024) return FIRE_EINVAL;

    // ---- scratch owned by the handle (grow-only; growing waits for the stream first)
    const size_t spill_per_cta = (size_t)2 * (prm.capA - prm.capA_s) + (prm.capQ - prm.capQ_s);
    const size_t spill_bytes = spill_per_cta * (size_t)grid * 4 + 16;
    const size_t nw = (size_t)L->H * L->Ww;
    const size_t plane_bytes = nw * 4;
    const size_t rescue_bytes = plane_bytes * 2 * kRescueCtas;
    if (L->status_capacity < (size_t)S || L->spill_capacity < spill_bytes || L->rescue_capacity < rescue_bytes) {
        FIRE_CUDA_TRY(L, cudaStreamSynchronize(st));
        size_t cap_bytes = L->status_capacity * 4;
        int rc = fire_reserve(L, (void**)&L->status, &cap_bytes, (size_t)S * 4);
        if (rc != FIRE_OK) return rc;
        L->status_capacity = cap_bytes / 4;
        rc = fire_reserve(L, (void**)&L->spill, &L->spill_capacity, spill_bytes);
        if (rc != FIRE_OK) return rc;
        if (L->rescue_capacity < rescue_bytes) {
            rc = fire_reserve(L, (void**)&L->rescue_planes, &L->rescue_capacity, rescue_bytes);
            if (rc != FIRE_OK) return rc;
            FIRE_CUDA_TRY(L, cudaMemsetAsync(L->rescue_planes, 0, rescue_bytes, st));
        }
    }

    prm.burnable = L->burnable; prm.thr = L->thr;
    prm.ignitions = ignitions; prm.sim_param = sim_param; prm.seeds = seeds; prm.sim_ids = sim_ids;
    prm.out_burned = out_burned; prm.out_steps = out_steps; prm.out_trials = (unsigned long long*)out_trials;
    prm.work_counter = L->work_counter; prm.rescue_list = L->status; prm.spill = L->spill;
    prm.S = S; prm.P = L->P; prm.W = L->W; prm.H = L->H; prm.Ww = L->Ww; prm.max_steps = max_steps;

    // ---- planes: sus = burnable, then the simulations, then burnt = burnable & ~sus
    const int vec4 = (nw % 4 == 0 && ((uintptr_t)out_burned & 15u) == 0) ? 1 : 0;
    const size_t units = vec4 ? nw / 4 : nw;
    unsigned chunks = (unsigned)((units + 256 * 4 - 1) / (256 * 4));
    if (chunks < 1) chunks = 1;
    if (chunks > 64) chunks = 64;
    const dim3 plane_grid(chunks, (unsigned)S);
    fire_planes_kernel<false><<<plane_grid, 256, 0, st>>>(L->burnable, out_burned, nw, vec4);
    FIRE_CUDA_TRY(L, cudaGetLastError());
    FIRE_CUDA_TRY(L, cudaMemsetAsync(L->work_counter, 0, 2 * sizeof(unsigned int), st));
    if (smem > 48 * 1024)
        FIRE_CUDA_TRY(L, cudaFuncSetAttribute(fire_propagate_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const bool prof = L->prof_enabled && L->prof_count < 64;
    if (prof) FIRE_CUDA_TRY(L, cudaEventRecord(L->prof_ev[2 * L->prof_count], st));
    fire_propagate_kernel<<<grid, threads, smem, st>>>(prm);
    FIRE_CUDA_TRY(L, cudaGetLastError());
    if (prof) { FIRE_CUDA_TRY(L, cudaEventRecord(L->prof_ev[2 * L->prof_count + 1], st)); L->prof_count += 1; }
    fire_planes_kernel<true><<<plane_grid, 256, 0, st>>>(L->burnable, out_burned, nw, vec4);
    FIRE_CUDA_TRY(L, cudaGetLastError());
    fire_propagate_rescue_kernel<<<kRescueCtas, 256, 0, st>>>(prm, L->rescue_planes);
    FIRE_CUDA_TRY(L, cudaGetLastError());
    L->launches += 4;
    return FIRE_OK;
}
