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
// Design: one persistent CTA per simulation, all CA steps inside
// ONE launch, no host round trip and no grid-wide barrier.  The state is the bit-packed burned plane
// in the caller's output buffer plus a CELL-LEVEL FRONTIER LIST of the burning cells, so work is
// proportional to the number of trials and idle lattice is never touched.  Each step:
//   phase 1  one lane per burning cell: 3x3 susceptibility bits from the burnable and burned planes,
//            then the (target, direction) pairs are compacted into a shared-memory trial queue with a
//            warp prefix sum (shfl) -- so that
//   phase 2  every lane holds exactly one trial: one 4 B threshold load (the 32 B sector of a target
//            cell holds its 8 directions), one Philox4x32-10 call, one compare; successes are
//            compacted with __ballot_sync/__popc into the raw success list.
//   phase 3  the burned plane is only updated AFTER all trials of the step (synchronous update):
//            atomicOr per success; the lanes that flipped the bit own the new burning cell and append
//            it to the next frontier.
// Lists live in shared memory and continue in a per-CTA global spill area; if even that overflows,
// the simulation is handed to the rescue kernel below: a plain full-sweep, three-plane, pull-style
// restatement of the same rules with no lists at all (bounded memory, always terminates).
#include "fire_internal.cuh"

namespace {

struct prop_params {
    const uint32_t* burnable;     // [H][Ww]
    const uint32_t* thr;          // [P][cells][8]
    const int32_t*  ignitions;    // [S][2]
    const int32_t*  sim_param;    // [S]
    const uint64_t* seeds;        // [S]
    const int32_t*  sim_ids;      // [S] or null
    uint32_t* out_burned;         // [S][H][Ww], zeroed before the launch
    uint32_t* out_steps;          // [S] or null
    unsigned long long* out_trials;  // [S] or null
    unsigned int* work_counter;   // [0] next sim of the fast kernel, [1] number of sims handed to the rescue kernel
    uint32_t* rescue_list;        // [S]
    uint32_t* spill;              // [grid][capA_g + capB_g]
    int S, P, W, H, Ww;
    uint32_t max_steps;
    uint32_t capA_s, capB_s, capQ;   // shared-memory entries: frontier, raw successes, trial queue
    uint32_t capA, capB;             // total entries (shared + spill)
};

__device__ __forceinline__ uint32_t list_get(const uint32_t* s, const uint32_t* g, uint32_t cap_s, uint32_t i)
{
    return i < cap_s ? s[i] : __ldcg(g + (i - cap_s));
}
__device__ __forceinline__ void list_put(uint32_t* s, uint32_t* g, uint32_t cap_s, uint32_t i, uint32_t v)
{
    if (i < cap_s) s[i] = v; else __stcg(g + (i - cap_s), v);
}

// Susceptibility (burnable and not burned) of cells (x-1, y), (x, y), (x+1, y) as bits 0..2; cells
// outside the lattice do not exist (R-13).  The burned plane is read through L2 (it is updated
// with atomics by other lanes of this CTA in phase 3 of the previous step).
__device__ __forceinline__ uint32_t sus3(const uint32_t* __restrict__ burnable, const uint32_t* burned,
                                         int x, int y, int H, int Ww)
{
    if ((unsigned)y >= (unsigned)H) return 0u;
    const int wx = x >> 5, bx = x & 31;
    const size_t row = (size_t)y * Ww;
    const uint32_t mid = __ldg(burnable + row + wx) & ~__ldcg(burned + row + wx);
    uint32_t lo, hi; int sh;
    if (bx == 0) {
        lo = (wx > 0) ? (__ldg(burnable + row + wx - 1) & ~__ldcg(burned + row + wx - 1)) : 0u;
        hi = mid; sh = 31;
    } else {
        lo = mid;
        hi = (bx == 31 && wx + 1 < Ww) ? (__ldg(burnable + row + wx + 1) & ~__ldcg(burned + row + wx + 1)) : 0u;
        sh = bx - 1;
    }
    return __funnelshift_r(lo, hi, sh) & 7u;
}

__device__ __forceinline__ uint32_t lanemask_lt()
{
    uint32_t m; asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m)); return m;
}

// ------------------------------------------------------------------------------------------------
// Fast kernel: one persistent CTA per simulation.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(1024)
fire_propagate_kernel(const prop_params prm)
{
    extern __shared__ uint32_t smem[];
    uint32_t* const As = smem;
    uint32_t* const Bs = As + prm.capA_s;
    uint32_t* const Qs = Bs + prm.capB_s;
    uint32_t* const Ag = prm.spill + (size_t)blockIdx.x * ((prm.capA - prm.capA_s) + (prm.capB - prm.capB_s));
    uint32_t* const Bg = Ag + (prm.capA - prm.capA_s);

    __shared__ unsigned int s_sim, s_cntA[2], s_cntB[2], s_cntQ, s_overA, s_overB;
    __shared__ unsigned long long s_trials;

    const int tid = threadIdx.x, lane = tid & 31, nthr = blockDim.x;
    const int W = prm.W, H = prm.H, Ww = prm.Ww;
    const uint32_t chunk = prm.capQ >> 3;            // burning cells per chunk: at most 8 trials each
    const uint32_t lt = lanemask_lt();

    for (;;) {
        if (tid == 0) s_sim = atomicAdd(prm.work_counter, 1u);
        __syncthreads();
        const uint32_t s = s_sim;
        if (s >= (uint32_t)prm.S) break;

        const int p = prm.sim_param[s];
        const int ix = prm.ignitions[2 * s], iy = prm.ignitions[2 * s + 1];
        const uint64_t seed = prm.seeds[s];
        const uint32_t key_lo = (uint32_t)seed, key_hi = (uint32_t)(seed >> 32);
        const uint32_t sim = prm.sim_ids ? (uint32_t)prm.sim_ids[s] : s;
        uint32_t* const burned = prm.out_burned + (size_t)s * H * Ww;
        bool valid = p >= 0 && p < prm.P && ix >= 0 && ix < W && iy >= 0 && iy < H;     // R-12
        if (valid) valid = (__ldg(prm.burnable + (size_t)iy * Ww + (ix >> 5)) >> (ix & 31)) & 1u;
        const uint32_t* const thr = prm.thr + (valid ? (size_t)p * W * H * 8 : 0);

        if (tid == 0) {
            s_cntA[0] = valid ? 1u : 0u; s_cntA[1] = 0u; s_cntB[0] = 0u; s_cntB[1] = 0u; s_cntQ = 0u;
            s_overA = 0u; s_overB = 0u; s_trials = 0ull;
            if (valid) {
                list_put(As, Ag, prm.capA_s, 0u, (uint32_t)(iy * W + ix));
                burned[(size_t)iy * Ww + (ix >> 5)] = 1u << (ix & 31);
            }
        }
        __syncthreads();

        uint32_t t = 0, my_trials = 0;
        uint32_t nA = valid ? 1u : 0u;
        bool over = false;
        while (nA > 0 && (prm.max_steps == 0 || t < prm.max_steps)) {
            const int par = t & 1;
            for (uint32_t base = 0; base < nA; base += chunk) {
                const uint32_t end = min(base + chunk, nA);
                if (base > 0) {                       // multi-chunk step: recycle the trial queue
                    if (tid == 0) s_cntQ = 0u;
                    __syncthreads();
                }
                // ---- phase 1: susceptible neighbours of the burning cells -> trial queue
                for (uint32_t i0 = base + (uint32_t)(tid & ~31); i0 < end; i0 += nthr) {
                    const uint32_t i = i0 + lane;
                    uint32_t b = 0, m = 0;
                    if (i < end) {
                        b = list_get(As, Ag, prm.capA_s, i);
                        const int y = (int)(b / (uint32_t)W), x = (int)(b - (uint32_t)y * W);
                        const uint32_t up = sus3(prm.burnable, burned, x, y - 1, H, Ww);
                        const uint32_t md = sus3(prm.burnable, burned, x, y, H, Ww);
                        const uint32_t dn = sus3(prm.burnable, burned, x, y + 1, H, Ww);
                        // bit d of m: the neighbour reached by travelling in direction d can still burn
                        m = ((up >> 1) & 1u) | (((up >> 2) & 1u) << 1) | (((md >> 2) & 1u) << 2) | (((dn >> 2) & 1u) << 3) |
                            (((dn >> 1) & 1u) << 4) | ((dn & 1u) << 5) | ((md & 1u) << 6) | ((up & 1u) << 7);
                    }
                    const uint32_t cnt = __popc(m);
                    uint32_t incl = cnt;
#pragma unroll
                    for (int o = 1; o < 32; o <<= 1) {
                        const uint32_t v = __shfl_up_sync(0xFFFFFFFFu, incl, o);
                        if (lane >= o) incl += v;
                    }
                    const uint32_t total = __shfl_sync(0xFFFFFFFFu, incl, 31);
                    if (total == 0) continue;
                    uint32_t qbase = 0;
                    if (lane == 31) qbase = atomicAdd(&s_cntQ, total);
                    qbase = __shfl_sync(0xFFFFFFFFu, qbase, 31);
                    uint32_t pos = qbase + incl - cnt;
                    my_trials += cnt;
                    while (m) {
                        const int d = __ffs(m) - 1;
                        m &= m - 1;
                        const uint32_t c = (uint32_t)((int)b + fire_dx(d) + fire_dy(d) * W);
                        Qs[pos++] = (c << 3) | (uint32_t)d;
                    }
                }
                __syncthreads();
                const uint32_t nQ = s_cntQ;
                if (tid == 0 && base == 0) { s_cntA[par ^ 1] = 0u; s_cntB[par ^ 1] = 0u; }
                // ---- phase 2: one Bernoulli trial per lane
                for (uint32_t j0 = (uint32_t)(tid & ~31); j0 < nQ; j0 += nthr) {
                    const uint32_t j = j0 + lane;
                    bool succ = false;
                    uint32_t c = 0;
                    if (j < nQ) {
                        const uint32_t item = Qs[j];
                        c = item >> 3;
                        const int d = (int)(item & 7u);
                        const uint32_t T = __ldg(thr + (size_t)item);          // item == c*8 + d
                        const uint32_t r = fire_rnd(key_lo, key_hi, sim, t, c, d);
                        succ = fire_trial(r, T);
                    }
                    const uint32_t mask = __ballot_sync(0xFFFFFFFFu, succ);
                    if (mask == 0) continue;
                    uint32_t bbase = 0;
                    if (lane == 0) bbase = atomicAdd(&s_cntB[par], (unsigned)__popc(mask));
                    bbase = __shfl_sync(0xFFFFFFFFu, bbase, 0);
                    if (succ) {
                        const uint32_t pos = bbase + __popc(mask & lt);
                        if (pos < prm.capB) list_put(Bs, Bg, prm.capB_s, pos, c);
                        else s_overB = 1u;
                    }
                }
                __syncthreads();
            }
            // ---- phase 3: synchronous update of the burned plane; the lane that flips a bit owns the cell
            if (s_overB) { over = true; break; }     // written in phase 2 only, read after its closing barrier
            const uint32_t nB = s_cntB[par];
            for (uint32_t j0 = (uint32_t)(tid & ~31); j0 < nB; j0 += nthr) {
                const uint32_t j = j0 + lane;
                bool fresh = false;
                uint32_t c = 0;
                if (j < nB) {
                    c = list_get(Bs, Bg, prm.capB_s, j);
                    const uint32_t y = c / (uint32_t)W, x = c - y * (uint32_t)W;
                    const uint32_t bit = 1u << (x & 31);
                    const uint32_t old = atomicOr(burned + (size_t)y * Ww + (x >> 5), bit);
                    fresh = (old & bit) == 0u;
                }
                const uint32_t mask = __ballot_sync(0xFFFFFFFFu, fresh);
                if (mask == 0) continue;
                uint32_t abase = 0;
                if (lane == 0) abase = atomicAdd(&s_cntA[par ^ 1], (unsigned)__popc(mask));
                abase = __shfl_sync(0xFFFFFFFFu, abase, 0);
                if (fresh) {
                    const uint32_t pos = abase + __popc(mask & lt);
                    if (pos < prm.capA) list_put(As, Ag, prm.capA_s, pos, c);
                    else s_overA = 1u;
                }
            }
            if (tid == 0) s_cntQ = 0u;
            __syncthreads();
            ++t;
            if (s_overA) { over = true; break; }     // written in phase 3 only
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
            }
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
    uint32_t capA_s = L->list_shared ? (uint32_t)L->list_shared : 2048u;
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
    prm.capB_s = capA_s + capA_s / 2; prm.capB = 2 * capA;
    if (prm.capB_s > prm.capB) prm.capB_s = prm.capB;
    prm.capQ = 8u * (capA_s < 512u ? (capA_s < 4u ? 4u : capA_s) : 512u);
    const size_t smem = ((size_t)prm.capA_s + prm.capB_s + prm.capQ) * sizeof(uint32_t);
    if (smem > 200 * 1024) return FIRE_EINVAL;

    // ---- scratch owned by the handle (grow-only; growing waits for the stream first)
    const size_t spill_per_cta = (size_t)(prm.capA - prm.capA_s) + (prm.capB - prm.capB_s);
    const size_t spill_bytes = spill_per_cta * (size_t)grid * 4 + 16;
    const size_t plane_bytes = (size_t)L->H * L->Ww * 4;
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

    FIRE_CUDA_TRY(L, cudaMemsetAsync(out_burned, 0, (size_t)S * plane_bytes, st));
    FIRE_CUDA_TRY(L, cudaMemsetAsync(L->work_counter, 0, 2 * sizeof(unsigned int), st));
    if (smem > 48 * 1024)
        FIRE_CUDA_TRY(L, cudaFuncSetAttribute(fire_propagate_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const bool prof = L->prof_enabled && L->prof_count < 64;
    if (prof) FIRE_CUDA_TRY(L, cudaEventRecord(L->prof_ev[2 * L->prof_count], st));
    fire_propagate_kernel<<<grid, threads, smem, st>>>(prm);
    FIRE_CUDA_TRY(L, cudaGetLastError());
    if (prof) { FIRE_CUDA_TRY(L, cudaEventRecord(L->prof_ev[2 * L->prof_count + 1], st)); L->prof_count += 1; }
    fire_propagate_rescue_kernel<<<kRescueCtas, 256, 0, st>>>(prm, L->rescue_planes);
    FIRE_CUDA_TRY(L, cudaGetLastError());
    L->launches += 2;
    return FIRE_OK;
}
